// pdv_device.h -- structures shared by the C-ABI layer (pdv_api.cu) and the kernels (pdv_kernels.cu).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/pdv.h"

// transport_kernel is compiled for PDV_LB_THREADS threads per block at most and PDV_LB_BLOCKS resident blocks per SM
// (its register budget = 65536 / (PDV_LB_THREADS * PDV_LB_BLOCKS)).  The polydisperse instantiations, whose tables leave room
// for one block per SM anyway, are compiled for PDV_LB_THREADS_POLY threads.  Round 1 (kernel v10, 80 registers): 1024 / 896 /
// 768 / 640 threads on config 3: 1.45 / 1.48 / 1.52 / 1.44e11 events/s.  Round 2 (76 registers after the per-history bookkeeping
// went; it now fits 64 registers without a spill): 768 / 896 / 960 / 1024 threads: config 5 280.7 / 276.4 / 275.0 / 273.1 ms,
// Figs. 13-15 sweep (one draw per pass) 75.6 / 74.2 / 74.3 / 73.4 ms, config 3 at 4e6 photons per snapshot 76.4 / 75.7 / 75.5 /
// 74.9 ms -- 1024 threads = 32 warps per SM, as for one class.
#ifndef PDV_LB_THREADS
#define PDV_LB_THREADS 1024
#endif
#ifndef PDV_LB_THREADS_POLY
#define PDV_LB_THREADS_POLY 1024
#endif
// The long-history instantiations of the one-class kernel (ALT, four draws per pass) are compiled for PDV_LB_THREADS_LONG resident
// threads (80 registers: no spill; at 64 registers they spilled 16 ... 40 bytes) and launched as blocks of half that size.  Config 4:
// 512 x 2 at 64 registers 118.3 ms; 384 x 2 at 80 registers 111.2; 256 x 3 111.4; 320 x 2 at 102 registers 109.9; 256 x 4 at 64: 120.2.
#ifndef PDV_LB_THREADS_LONG
#define PDV_LB_THREADS_LONG 768
#endif
#ifndef PDV_LB_BLOCKS
#define PDV_LB_BLOCKS 1
#endif

namespace pdv {

// Fixed point of every tally: Q31, one photon = 2^31.  A history carries its weight in fp32 (a product of albedos in
// event order: the same bits for any launch shape) and converts it once, when the history ends.
constexpr uint32_t kWOne = 0x80000000u;
constexpr float kWOneF = 2147483648.0f;
constexpr double kWScale = 1.0 / 2147483648.0;

// Per-unit statistics slots (u64 each) in the device workspace.
enum StatSlot {
    ST_DETECTED = 0, ST_UNDER, ST_OVER, ST_ESCAPED, ST_ABS_PART, ST_ABS_SURF, ST_KILLED, ST_GAINED, ST_TRUNC,
    ST_HISTORIES, ST_EVENTS, ST_REFLECT, ST_MAXEV, ST_COUNT = 16
};

// Device image of one cloud: one contiguous blob [DevCloudHeader | phase | depth rows | class thr | albedo f32 | albedo thr | guide],
// every section 16-byte aligned, copied verbatim into shared memory by each block.
//
// Phase table (one float2 per class c and phase bin k, k = 0..K-1): x = M_c[k], y = (M_c[k+1] - M_c[k]) * 2^-shiftK with
// shiftK = 32 - log2 K, so that for a 32-bit word b:  k = b >> shiftK,  cos(theta) = x + y * (b & frac_mask)  -- the canonical
// D_K sample M[k] + (M[k+1]-M[k]) frac with frac = the 12 bits of b below the index bits: one 64-bit load,
// one FFMA.
//
// UNITS: every optical depth of the image (rows.x, tau_ext, the guide's float bits, an_c3) is in units of ln 2, T / ln 2: the
// kernel's free flight is then  T' = T + mu lg2(xi)  with the SFU's base-2 logarithm and no multiplication by ln 2.
// Depth rows (one float4 per depth bin j, bins uniform in v, j = 0 at the cloud top):
//   x = T_{j+1}                      vertical optical depth of the LOWER edge of bin j
//   y = v(T_{j+1}) / 2               half the particle velocity at that edge (the Doppler update uses v/2)
//   z = d(v/2)/dT inside bin j       (0 for an empty bin)
//   w = d(v/2)/dT inside bin j+1     (0 past the last bin)
// so that for T_j <= T < T_{j+2}:  v(T)/2 = y + (T - x) * (T < x ? z : w)   -- T linear in v inside each bin
// (the canonical depth discretisation), one branch-free probe.
// Guide: cell = (float bits of T) >> guide_shift, minus guide_base; guide[cell] = largest j with T_j <= every T of the
// cell.  The host picks guide_shift so that no cell straddles two bin edges (then one probe is exact); if it cannot,
// depth_bisect = 1 and the kernel bisects the rows instead.
// Class guide (polydisperse clouds): the class of a class word cw is  c = #{j < n_classes-1 : thr[j] <= cw}  (cumulative
// pick probabilities of Eq. 8, R12).  cguide[cw >> cguide_shift] holds that count for the first word of the cell in
// its low 7 bits, and bit 7 is set if more than one threshold lies inside the cell; so  c = low7 + (thr[low7] <= cw)  settles
// every cell but the flagged ones, which walk on.  The host takes the coarsest guide of 2^8 ... 2^12 cells in which no cell
// holds two thresholds (config 3: 2^10); if even 2^12 cells leave flagged ones (config 5: the two smallest classes, hit with
// probability 1.7e-6 and 2.7e-5) it stays at 2^12 and one flight in 4096 walks.
// Class thresholds: two tables of PDV_MAX_CLASSES words.  thr[j] = 32-bit threshold of the cumulative pick probability (padded with
// 0xffffffff); thr24[j] = 256 ceil((thr[j] - 128) / 256): a class word W whose low byte counts as 0x80 (first and second flight
// of a three-flight group, D2) satisfies  thr[j] <= (W & ~0xff | 0x80)  exactly when  W >= thr24[j].
struct DevCloudHeader {
    uint32_t blob_bytes;       // multiple of 16
    uint32_t n_classes, K, log2K, n_depth, n_guide;
    uint32_t off_phase, off_rows, off_thr, off_albedo, off_albthr, off_guide;   // byte offsets from the blob start
    uint32_t guide_base;       // (float bits of T) >> guide_shift of guide cell 0
    uint32_t guide_shift;
    uint32_t depth_bisect;     // 0: one guide probe; 1: bisect the rows; 2: closed form  v/2 = an_c0 + an_c1 lg2(an_c2 + an_c3 T)
    float tau_ext, vh_fs;      // tau_ext in units of ln 2 (see above); vh_fs = v_fs / 2
    float R_f;                 // surface reflectivity
    uint32_t R_thr;            // analog mode: reflected iff xi_absorb word < R_thr
    uint32_t surface_model;
    uint32_t frac_mask;        // the 12 bits of a phase word below its log2K index bits
    uint32_t off_cguide;       // class guide: 2^(32 - cguide_shift) bytes, see above
    float an_c0, an_c1, an_c2, an_c3;   // closed-form depth model (pdv_cloud_params.depth_model 1)
    uint32_t cguide_shift;     // 24 ... 20
    // Gas environment (R35-R37; one image per (cloud, snapshot) unit): the depth rows hold the HEIGHT zeta above the
    // free surface instead of v/2 (y = zeta_{j+1}, z / w = dzeta/dT inside bins j / j+1), bins uniform in zeta;
    // gas thresholds u32 [n_depth][n_pad + 1] (an ODD row length: the lanes of a warp read the same column of different rows, which
    // with rows of 2^k words fell on two banks: 13 wavefronts per load): row j = cumulative class pick probabilities inside bin j as 32-bit thresholds
    // (c = #{k : thr[j][k] <= cw}, padded with 0xffffffff to n_pad = 2^gas_steps entries, found by gas_steps bisection steps);
    // gas class constants float2 [n_pad]: (L_c / (2 t), -1 / L_c), or (0, 0) for a class without drag, so that half the
    // class-c particle velocity at zeta is  v_fs/2 + x (1 - e^{y zeta}),  = v_fs/2 + gas_inv_2t zeta (1 + y zeta / 2 + ...) for small y zeta.
    uint32_t gas;              // 1: this image is a gas unit
    uint32_t off_gthr, off_gcls, gas_steps;
    float omr_q31;             // (1 - R_f) 2^31: weight that reached the surface -> Q31 weight left in it
    uint32_t cguide_flagged;   // number of class-guide cells that hold several thresholds (0: an entry is the class count itself)
    float gas_inv_2t;          // gas unit: 1 / (2 t) of its snapshot
    uint32_t pad[2];
};
static_assert(sizeof(DevCloudHeader) % 16 == 0, "header must keep 16-byte alignment");

struct UnitDesc {
    const unsigned char *cloud_blob;   // device pointer
    uint32_t stream;                   // Philox counter word 2 (unit index)
    uint32_t visit;                    // entry k of the table: the k-th unit of the visiting order (descending cost)
    // Guided self-scheduling of the unit's photon ids: a warp claims 32 * clamp(remaining * chunk_per_remaining, 1, chunk)
    // ids at a time; chunk_per_remaining = 1 / (2 * threads expected to work on the unit)
    uint32_t chunk;
    float chunk_per_remaining;
};

struct RunParams {
    const UnitDesc *units;
    unsigned long long *next_id;       // [n_units] photons handed out so far (relative to first_id)
    unsigned long long *hist;          // [n_units][n_bins] Q31 sum w
    unsigned long long *hist2;         // [n_units][n_bins] Q31 sum w^2
    unsigned long long *stats;         // [n_units][ST_COUNT]
    pdv_trace_record *trace;           // TRACE only: [n_photons]
    const uint32_t *block_start;       // [grid] entry of the visiting order at which block b starts.  The units are laid on a
                                       // line in descending cost, each as long as its estimated cost, and block b starts in the
                                       // unit that holds point (b + 1/2) / grid of the line: a unit is staged by about as many
                                       // blocks as its share of the work, each block stages few units, and a block that runs out
                                       // of work walks on along the order (wrapping) and helps wherever photons are left
    uint32_t n_units;
    uint32_t n_bins;
    uint32_t max_events;               // roulette once n_scatter >= max_events; 0xffffffff: never
    uint32_t roulette_thr;             // survive iff the roulette word < roulette_thr
    float roulette_p;                  // play only while w <= p (then w / p <= 1)
    float roulette_inv_p;
    float v_lo, inv_dv, mu_aperture;
    uint32_t launch_model;             // 1: diffuse illumination (general kernel only), see pdv_run_opts
    unsigned long long n_photons, first_id;
    uint32_t key0[10], key1[10];       // Philox round keys
};

struct LaunchShape { int grid, block, smem; };

// Host wrappers implemented in pdv_kernels.cu.
// alt: run the second production instantiation (transport_kernel's ALT).  One-class launches: the histories are long
// (cost-weighted mean of the estimated flights per history >= 22), a lane then flies several random draws between two
// end-of-history passes -- that pass runs at one or two lanes when histories are long, and running it less often costs fewer
// issue slots than the lanes that wait for it (measured: profiles/README.md).  Polydisperse launches: no class-guide cell of
// any cloud holds two thresholds (DevCloudHeader::cguide_flagged == 0 everywhere).
struct KernelVariant { bool poly, analog, sso, trace, roulette; int dm; bool alt; };   // dm: see transport_kernel
cudaError_t launch_transport(const RunParams &rp, KernelVariant v, LaunchShape shape, cudaStream_t st);
cudaError_t transport_max_blocks_per_sm(KernelVariant v, int block, int smem, int *out);
cudaError_t transport_static_smem(KernelVariant v, size_t *out);      // static shared memory of the instantiation (warp queues, keys, stats)
// Test-only (pin P13): raw Philox4x32-10 blocks of n counters through the three key paths of the kernels; key0/key1: HOST [10]
// round keys, ctr and the outputs: DEVICE [n].
cudaError_t launch_philox_check(const uint32_t *key0, const uint32_t *key1, const uint4 *ctr, int n, uint4 *out_static,
                                uint4 *out_shared, uint4 *out_param, cudaStream_t st);
cudaError_t launch_finalize(const unsigned long long *hist, const unsigned long long *hist2, const unsigned long long *stats,
                            uint32_t n_units, uint32_t n_bins, double *out_hist, double *out_hist2, pdv_run_stats *out_stats,
                            cudaStream_t st);
cudaError_t launch_spectrogram(const double *hist, int n_snap, int n_bins, double inv_n, double inv_dv, int scale,
                               float floor_db, float *out, cudaStream_t st);
cudaError_t launch_peaks(const double *hist, int n_units, int n_bins, double n_photons, double v_lo, double v_hi,
                         const double *v_fs, const pdv_peak_opts &o, pdv_peak *out, cudaStream_t st);
// Sampling check of one class (pdv_phase_sampling_check): phase = that class's float2 table in the device blob; coef = device
// float4 [n_terms] (fa_re, fa_im, fb_re, fb_im), f = (2n+1)/(n(n+1)); out_hist = u64 [2][n_bins] (table, exact);
// out_sum = double [2]; out_cnt = u64 [2] (trials, bound violations).  All outputs zeroed by the caller.
cudaError_t launch_phase_check(const float2 *phase, uint32_t K, uint32_t log2K, uint32_t frac_mask, const float4 *coef,
                               int n_terms, float i_max, unsigned long long n_samples, unsigned long long seed, int n_bins,
                               unsigned long long *out_hist, double *out_sum, unsigned long long *out_cnt, int n_sm,
                               cudaStream_t st);
cudaError_t launch_issue_peaks(double millis, double *ffma, double *mufu, double *mhz, int n_sm, cudaStream_t st);

}  // namespace pdv
