// pdv_optics.hpp -- host-side (double precision) optics of one ejecta cloud: Mie efficiencies and phase
// tables (Eq. 12-14), class probabilities and extinction (Eq. 8-10), depth table (Eq. 20).
// Product code: shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/pdv.h"

namespace pdv {

struct HostCloud {
    int n_classes = 0, K = 0, n_depth = 0;
    std::vector<double> diameter, weight;            // normalised number weights
    std::vector<double> k_ext, k_sca, g, p_class;    // per class
    std::vector<double> phase;                       // [n_classes][K+1]
    std::vector<double> T_edge;                      // [n_depth+1], T at v_max - j dv
    double tau_ext = 0, kappa = 0, sauter = 0, v_fs = 0, v_max = 0, R = 0;
    int surface_model = 0;
    int depth_model = 0;                             // 1: closed-form v(T) of the exponential profile (then beta > 0)
    double beta = 0;
    double m_re = 0, m_im = 0, wavelength = 0;       // kept for pdv_phase_sampling_check
    int phase_model = 0;
    // gas environment (pdv_cloud_params.gas_density > 0; R35-R38): what the per-snapshot tables are built from
    double gas_density = 0, drag_coefficient = 0, density = 0;
    int profile_kind = 0;
    std::vector<double> prof_v, prof_cum;            // profile_kind 1
    bool gas() const { return gas_density > 0.0; }
};

// Depth tables of one (cloud, snapshot) unit in a gas environment: bins uniform in the height zeta above the free surface.
struct GasUnit {
    std::vector<double> zeta_edge, T_edge;           // [n_depth+1]: zeta_top ... 0, 0 ... tau_ext
    std::vector<double> class_cum;                   // [n_depth][n_classes]
    std::vector<double> L;                           // [n_classes] drag lengths (infinity: no drag)
    double t = 0;
};
void build_gas_unit(const HostCloud &h, double t, GasUnit &out);

// Mie coefficients a_n, b_n (n = 1..n_max) of a homogeneous sphere, size parameter x, relative index m.
void mie_coefficients(double x, double m_re, double m_im, std::vector<double> &a_re, std::vector<double> &a_im,
                      std::vector<double> &b_re, std::vector<double> &b_im);

// Eq. 12: efficiencies and asymmetry parameter.
void mie_efficiencies(double x, double m_re, double m_im, double *k_ext, double *k_sca, double *g);

// Inverse-CDF table of the unpolarised phase function in mu = cos(theta): M[k] = F^-1(k/K), k = 0..K.
// The nodes of the angular integral are evaluated on up to min(8, max_threads) host threads.
void mie_phase_quantiles(double x, double m_re, double m_im, int K, double *M, int max_threads = 8);

// Validates params and fills `out`.  Returns PDV_OK or PDV_E_INVALID with a message in `err`.
pdv_status build_host_cloud(const pdv_cloud_params &p, HostCloud &out, std::string &err);

pdv_status lognormal_classes(double d_median, double sigma_ln, int n, double *diameter, double *weight, int *n_out);

}  // namespace pdv
