/* pdv.h -- C-ABI of the B200-native Monte-Carlo PDV spectrum library (libpdv_b200.so).
 *
 * The library computes what arXiv 2012.00963 (Shi et al., "Reconstruction and interpretation of photon
 * Doppler velocimetry spectrum for ejecta particles from shock-loaded sample in vacuum") section II.B
 * describes: Monte-Carlo multiple-scattering transport of the PDV probe photons through a cloud of
 * spherical ejecta particles above a moving free surface, with the Doppler shifts of the photons that
 * return to the probe histogrammed per time snapshot (steps (1)-(7) at PAPER.md:174-183).
 *
 * C99.  No C++ types and no exceptions cross this boundary.  Every pointer is a HOST pointer unless its
 * comment says "device".  All physical quantities are SI doubles.  Every function returns a pdv_status
 * (or void / const char*); on any status other than PDV_OK the caller's output buffers are untouched.
 * There is no CPU fallback: without a CUDA device pdv_cloud_create still builds the host-side optics
 * (so they can be inspected) but pdv_mc_run returns PDV_E_CUDA.
 *
 * Conventions (readings R1-R4): z points from the free surface to the probe; ejecta move in
 * +z with v = z/t; photons start at the cloud top with direction cosine mu = u_z = -1; the "Doppler
 * velocity" of a history is  v~ = 1/2 sum_k (mu_k_out - mu_k_in) v_k  = Eq. 4 times
 * c/(2 w_r); the frequency shift is 2 v~/lambda.  T is the vertical optical depth measured down from the
 * cloud top (T = 0 top, T = tau_ext at the free surface).
 */
#ifndef PDV_H_
#define PDV_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    PDV_OK = 0,
    PDV_E_INVALID = 1,      /* NULL where not allowed, out-of-range value, inconsistent sizes */
    PDV_E_NOMEM = 2,        /* host or device allocation failed */
    PDV_E_CUDA = 3,         /* no device, or a CUDA call failed; text in pdv_last_error() */
    PDV_E_UNSUPPORTED = 4   /* valid request the kernels do not implement (e.g. tables too large for shared memory) */
} pdv_status;

typedef struct pdv_cloud pdv_cloud;    /* opaque; owned by the library; immutable after creation */

/* ---- cloud definition: PAPER.md section II.C (187-203) ------------------------------------------------ */
typedef struct {
    size_t struct_size;          /* = sizeof(pdv_cloud_params); lets the struct grow */
    double area_mass;            /* m0, total area mass of the ejecta, kg/m^2 (1 mg/cm^2 = 1e-2); >= 0   (Eq. 9)  */
    double density;              /* rho0 of the particle material, kg/m^3; > 0                          (Eq. 9)  */
    double v_fs;                 /* free-surface velocity, m/s; > 0                                     (Eq. 20) */
    int32_t profile_kind;        /* 0: exponential law Eq. 20 truncated to [v_fs, vmax_ratio v_fs] and renormalised;
                                    1: tabulated cumulative mass prof_cum_mass(prof_v) */
    double beta;                 /* velocity distribution coefficient of Eq. 20; > 0 (kind 0) */
    double vmax_ratio;           /* cloud top velocity / v_fs; > 1 */
    int32_t n_prof;              /* kind 1: number of table points (>= 2) */
    const double *prof_v;        /* kind 1: [n_prof] strictly increasing velocities, prof_v[0] = v_fs, last = v_max */
    const double *prof_cum_mass; /* kind 1: [n_prof] non-decreasing cumulative mass below v (any units)  */
    int32_t n_classes;           /* size distribution as explicit classes (Eq. 21 discretised by the caller, or by
                                    pdv_lognormal_classes); 1..PDV_MAX_CLASSES */
    const double *diameter;      /* [n_classes] particle diameters d_c, m; > 0 */
    const double *number_weight; /* [n_classes] relative NUMBER of particles per class; > 0; normalised internally */
    double m_re, m_im;           /* complex refractive index of the particles, m = m_re + i m_im, m_im >= 0 absorbs */
    double wavelength;           /* probe wavelength lambda, m (1550e-9 in the paper) */
    double surface_reflectivity; /* R in [0,1]: weight kept by a photon reflected at the free surface (R = 1: paper) */
    int32_t surface_model;       /* 0: paper's "ideal diffuse reflection", polar angle uniform;
                                    1: Lambertian (mu = sqrt(xi)) */
    int32_t n_phase_bins;        /* K of the inverse-CDF phase table D_K; a power of two in [16, 4096]; 0 -> 1024 */
    int32_t n_depth_bins;        /* depth bins uniform in v (= in z at fixed t); [1, 4096]; 0 -> 1024 */
    int32_t phase_model;         /* 0: Mie, Eq. 12-14; 1: isotropic ("uniform") scattering, Fig. 6 case 2,
                                    with the Mie efficiencies kept for extinction and albedo */
    int32_t depth_model;         /* how the kernel gets the particle velocity at an optical depth T (counted from the top):
                                    0: the depth table (n_depth_bins bins uniform in v, T linear in v inside a bin);
                                    1: the closed form of the truncated Eq. 20,
                                       v = v_fs - (v_fs/beta) ln(E + (1 - E) T/tau_ext), E = exp(-beta (vmax_ratio - 1))
                                       (R26) -- profile_kind 0 only; no table error, one logarithm per event */
    /* ---- gas environment.  The paper treats the vacuum only and names this case as future work in one
     * sentence without an equation, so what follows is a reading that is NOT the paper's (R35-R38):
     * the gas ahead of the free surface moves with it (velocity v_fs, density gas_density); a particle of diameter d feels the
     * quasi-steady drag of a constant coefficient on its velocity u relative to the gas, du/dt = -u^2/L with
     * L = 4 density d / (3 drag_coefficient gas_density), hence u(t) = u0/(1 + u0 t/L) and the height above the free surface
     * zeta(t) = L ln(1 + u0 t/L).  Small particles stop first, the cloud sorts itself by size, and the spectrum depends on the
     * snapshot time: pdv_mc_run builds the depth tables of every (cloud, snapshot) unit at run time. */
    double gas_density;          /* rho_g, kg/m^3; 0: vacuum (the paper; every other field keeps its meaning and the run is bit-identical
                                    to one without these two fields) */
    double drag_coefficient;     /* C_d > 0 when gas_density > 0 (0.5 is typical of spheres at high Reynolds number).
                                    Limit: a gas unit keeps one row of class thresholds PER DEPTH BIN in shared memory
                                    (n_depth_bins x (2^ceil(log2 n_classes) + 1) words), so 16 classes with 1024-cell phase tables and
                                    512 velocity bins run with at most about 790 depth bins: the row-f4 workload uses n_depth_bins
                                    = 256, and 16 x 1024 is PDV_E_UNSUPPORTED.  256 bins are enough at the statistics this library is run at: two stored
                                    oracle runs of that workload's last snapshot at 1e8 histories, 256 against 1024 bins, agree
                                    bin by bin within their noise (tests/test_oracle_gas.py) */
} pdv_cloud_params;

#define PDV_MAX_CLASSES 32

/* Discretises the log-normal number distribution of Eq. 21 into n classes: n bins of equal
 * width in x = ln(d/d_median)/sigma_ln over [-3, 3 + 3 sigma_ln], representative diameter at the bin centre
 * in x, weight = standard-normal mass of the bin, renormalised to 1 (reading R11).
 * sigma_ln = 0 gives one class (n is ignored, diameter[0] = d_median, weight[0] = 1) and returns *n_out = 1.
 * diameter, weight: [n] outputs.  n_out may be NULL. */
pdv_status pdv_lognormal_classes(double d_median, double sigma_ln, int32_t n, double *diameter, double *weight,
                                 int32_t *n_out);

/* Builds the optics of one cloud on the host in double precision -- per class the Mie efficiencies K_ext,
 * K_sca, K_abs (Eq. 12) and the inverse-CDF table of the phase function |S1|^2+|S2|^2 (Eq. 13-14,
 * PAPER.md:128-135); the class hit probabilities P_c ~ w_c d_c^2 K_ext,c (Eq. 8); the mass-extinction
 * coefficient kappa = 3 sum w d^2 K_ext / (2 rho0 sum w d^3) and tau_ext = kappa m0 (Eq. 10);
 * the depth table T_j (Eq. 20) -- and, when a CUDA device is present, copies the fp32 tables to it.
 * *out receives the new cloud; release it with pdv_cloud_destroy.
 * Streams: the upload goes through a pinned staging buffer and a stream of the library's own and waits for that copy only; a
 * device buffer recycled from a destroyed cloud is reused once the runs that read the old cloud have finished (an event behind
 * its last launch), not after a device-wide synchronisation.  So creating or destroying clouds while a long pdv_mc_run with
 * device outputs is in flight on another stream neither waits for that run nor disturbs it. */
pdv_status pdv_cloud_create(const pdv_cloud_params *params, pdv_cloud **out);

/* NULL is a no-op.  The cloud must not be in use by a running pdv_mc_run. */
void pdv_cloud_destroy(pdv_cloud *cloud);

typedef struct {
    size_t struct_size;
    int32_t n_classes, n_phase_bins, n_depth_bins, on_device;
    double tau_ext;              /* vertical extinction optical thickness of the cloud */
    double kappa;                /* mass-extinction coefficient, m^2/kg */
    double sauter_diameter;      /* sum w d^3 / sum w d^2 of the class list */
    double v_fs, v_max;
    double mean_albedo;          /* sum_c P_c K_sca,c/K_ext,c */
    double mean_g;               /* scattering-weighted mean asymmetry parameter */
} pdv_cloud_info;

pdv_status pdv_cloud_get_info(const pdv_cloud *cloud, pdv_cloud_info *out);

/* The library's own estimate of the flights (particle events + surface reflections + the exit flight) of ONE history of this
 * cloud under the run options `opts` (a pdv_run_opts; only mode, max_events, roulette_survival and single_scatter_only are read;
 * NULL: defaults) -- the number pdv_mc_run lays its blocks out with (2.3 + 4.8 tau_ext, capped by the roulette, the analog
 * absorption and the single-scatter cut).  Only ratios matter.  A caller that splits a job over several GPUs cuts it into
 * stretches of equal estimated cost with it (paper_2012_00963_b200/_shard.py::plan_balanced).  No device needed. */
pdv_status pdv_estimated_flights(const pdv_cloud *cloud, const void *opts, double *out);

/* Copies the host (double) tables of the cloud into caller buffers; any pointer may be NULL to skip it.
 * k_ext,k_sca,g,p_class: [n_classes].  phase: [n_classes][n_phase_bins+1], M_c[k] = F_c^-1(k/K) in cos(theta).
 * T_edge: [n_depth_bins+1], T at velocity v_max - j (v_max - v_fs)/n_depth_bins. */
pdv_status pdv_cloud_get_tables(const pdv_cloud *cloud, double *k_ext, double *k_sca, double *g, double *p_class,
                                double *phase, double *T_edge);

/* Diagnostic: the DEVICE IMAGE of a cloud in vacuum -- the fp32 / integer tables each block stages in shared memory
 * (layout and meaning of every section: csrc/pdv_device.h) -- with the offsets and parameters needed to read it.  For
 * tests of the host logic that builds it (guides, thresholds, units); needs no GPU.  `image` may be NULL (layout only);
 * otherwise it receives min(capacity, image_bytes) bytes.  Optical depths in the image are in units of ln 2. */
typedef struct {
    size_t struct_size;
    uint32_t image_bytes, n_classes, n_phase_bins, log2_phase_bins, n_depth_bins;
    uint32_t off_phase;          /* float2 [max(n_classes, 2)][n_phase_bins]: (M[k], (M[k+1] - M[k]) 2^-(32 - log2 K)) */
    uint32_t off_rows;           /* float4 [n_depth_bins]; the 80 bytes in front of it are the block's round-key slot */
    uint32_t off_thr, off_thr24; /* uint32 [PDV_MAX_CLASSES] each */
    uint32_t off_albedo;         /* float [>= max(n_classes, 2)] */
    uint32_t off_guide, n_guide, guide_base, guide_shift, depth_bisect;   /* uint16 [n_guide] */
    uint32_t off_cguide, cguide_cells, cguide_shift, cguide_flagged;      /* uint8 [cguide_cells] */
    uint32_t frac_mask;
    float tau_ext_ln2, half_v_fs, surface_reflectivity;
} pdv_image_layout;
pdv_status pdv_cloud_get_image(const pdv_cloud *cloud, pdv_image_layout *layout, unsigned char *image, size_t capacity);

/* Host (double) depth tables of the (cloud, snapshot time t) unit of a cloud in a gas environment (gas_density > 0), as
 * pdv_mc_run builds them (R36, R37): n = n_depth_bins bins uniform in the height zeta above the free surface.
 *   zeta_edge [n+1]  heights of the bin edges, from the cloud top zeta_top(t) = max_c L_c ln(1 + u_max t / L_c) down to 0
 *   T_edge    [n+1]  vertical optical depth from the top at the edges, 0 ... tau_ext (T linear in zeta inside a bin)
 *   class_cum [n][n_classes]  cumulative probabilities that an interaction inside the bin hits class 0..c (last = 1)
 *   drag_length [n_classes]   L_c
 * Any pointer may be NULL to skip it.  PDV_E_INVALID for a vacuum cloud or t <= 0.  No device is needed. */
pdv_status pdv_cloud_gas_tables(const pdv_cloud *cloud, double t, double *zeta_edge, double *T_edge, double *class_cum,
                                double *drag_length);

/* ---- Monte-Carlo run: PAPER.md section II.B steps (1)-(7) (174-183) ---------------------------------- */
typedef struct {
    size_t struct_size;
    int32_t n_bins;              /* velocity bins, 1..PDV_MAX_BINS; bin k = [v_lo + k dv, v_lo + (k+1) dv) */
    double v_lo, v_hi;           /* m/s; v_hi > v_lo */
    double aperture_sr;          /* on-axis probe aperture, sr, in (0, 2 pi]: detected iff mu_exit >= 1 - aperture/(2 pi) */
    int32_t mode;                /* 0: implicit capture (weight *= K_sca/K_ext, Eq. 11 in expectation);
                                    1: analog (absorbed with probability K_abs/K_ext, the paper's step (4)) */
    int32_t max_events;          /* Russian roulette once a history has had >= max_events particle events; 0: never */
    double roulette_survival;    /* p in (0,1]; a photon survives with probability p and weight w/p.  The kernel plays
                                    only while w/p <= 1 (weights never exceed one photon; reading R20) */
    int32_t single_scatter_only; /* 1: a history is cut at its second particle event ("truncated" weight) */
    uint64_t first_photon_id;    /* histories are keyed by id in [first_photon_id, first_photon_id + n_photons) */
    int32_t output_on_device;    /* 0: hist/hist2/stats are host pointers, the call returns when they are filled;
                                    1: they are DEVICE pointers, the call only enqueues work on cuda_stream */
    int32_t blocks_per_sm;       /* launch shape override for tests; 0: library default */
    int32_t threads_per_block;   /* 0: library default; multiple of 32, <= 1024; lowered to what the kernel instantiation of the
                                    launch was compiled for (768 for long one-class histories).  Never changes a result */
    int32_t launch_model;        /* 0: the paper's collimated probe beam, u = (0,0,-1) at the cloud top (R1);
                                    1: diffuse (Lambertian) illumination of the cloud top, mu = -sqrt(xi) with xi from word 0 of
                                       the history's Philox block with counter word 3 = 0xffffffff.  Not in the paper: it makes
                                       the mean-path invariance of a non-absorbing medium (<events> = 4 tau_ext, pin P16)
                                       testable on the device without any reference implementation */
    const uint32_t *unit_streams; /* HOST [n_clouds][n_snap] or NULL.  Random sub-stream (Philox counter word 2) of each unit; NULL:
                                    the unit index u = i_cloud * n_snap + i_snap.  A process that runs a SUBSET of the units of a
                                    larger job (whole units per GPU) passes the units' indices in the whole job
                                    here, so that its spectra are bit-identical to the rows of the one-process run */
} pdv_run_opts;

#define PDV_MAX_BINS 8192

typedef struct {                 /* weights in units of photons; identity (exact in the kernel's fixed point):
                                    detected+underflow+overflow+escaped+absorbed_particles+absorbed_surface
                                    +roulette_killed-roulette_gained+truncated = histories */
    double detected;             /* inside the aperture and inside [v_lo, v_hi): = sum of hist */
    double underflow, overflow;  /* inside the aperture, v~ < v_lo / v~ >= v_hi */
    double escaped;              /* left through the top outside the aperture */
    double absorbed_particles;   /* Eq. 11, p_a */
    double absorbed_surface;     /* (1 - R) at the free surface */
    double roulette_killed, roulette_gained;
    double truncated;            /* single_scatter_only */
    uint64_t histories;
    uint64_t particle_events;    /* "scattering events": particle interactions (absorbing ones included) */
    uint64_t surface_reflections;
    uint64_t max_events_in_history;
} pdv_run_stats;

/* Runs n_photons histories for every (cloud, snapshot) unit, unit index u = i_cloud * n_snap + i_snap.
 *   clouds  [n_clouds] clouds created by pdv_cloud_create (n_clouds >= 1)
 *   t_snap  [n_snap] snapshot times in s, each > 0 (n_snap >= 1).  In vacuum z = v t makes the
 *           expected spectrum independent of t (reading R16): t selects the unit's random stream.
 *   hist    [n_clouds][n_snap][n_bins] sum of weights of detected photons per velocity bin (Eq. 19)
 *   hist2   same shape, sum of squared weights (variance estimate); may be NULL
 *   stats   [n_clouds][n_snap]; may be NULL
 *   cuda_stream  a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream), or NULL for the default stream
 * Reproducibility: the same (clouds, n_snap, n_photons, seed, first_photon_id, opts) give bit-identical
 * hist/hist2/stats for any launch shape -- tallies are integer fixed point (Q31) and every history draws
 * from its own Philox4x32-10 counter stream keyed by (seed, photon id, unit).  Runs over id ranges [a,b)
 * and [b,c) sum to the run over [a,c).  n_photons = 0 is valid and yields zeros.
 * Limits: n_photons < 2^33 per unit (a tally is a Q31 sum in 64 bits: the weight of 2^33 photons, 2^33 * 2^31 = 2^64, would wrap
 * it to 0 -- e.g. "escaped" of an empty cloud; larger runs are split by the caller into id ranges, whose results add), n_clouds * n_snap <= 2^20, photon ids below 2^63; otherwise
 * PDV_E_INVALID.
 * Streams: every call takes its device scratch (id cursors, Q31 tallies, unit table, output staging) from the device's
 * stream-ordered memory pool on cuda_stream and releases it there behind its last kernel, so calls enqueued on DIFFERENT
 * streams, from one host thread or several, are independent of each other, and calls on one stream run in order.  With
 * output_on_device = 1 the caller's device buffers must stay valid, and the clouds alive, until the work enqueued on
 * cuda_stream has finished. */
pdv_status pdv_mc_run(const pdv_cloud *const *clouds, int32_t n_clouds, const double *t_snap, int32_t n_snap,
                      uint64_t n_photons, uint64_t seed, const pdv_run_opts *opts,
                      double *hist, double *hist2, pdv_run_stats *stats, void *cuda_stream);

/* pdv_mc_run for callers that must not allocate device memory.
 *
 * Who that is: pdv_mc_run takes its workspace from the device's stream-ordered memory pool on every call.  That is the wrong
 * thing to do inside a host program that has already handed the whole HBM to an arena of its own (a hydrocode that calls this
 * library as an in-situ PDV diagnostic every few time steps, a framework with a caching allocator that was told to take all
 * free memory): there the pool has nothing left to give and the call fails with PDV_E_NOMEM at an unpredictable step, or it
 * succeeds by growing the pool and the host program's next allocation fails instead.  It is also wrong for a caller on a
 * real-time path (a shot-by-shot analysis loop next to a running experiment) who wants the footprint of the library fixed when
 * it is loaded, not decided per call by a pool whose first allocation costs milliseconds.
 *
 * What this call does instead: its workspace (photon-id cursors, Q31 tallies, per-unit statistics, unit table, block starts)
 * is a fixed array of PDV_STATIC_SCRATCH_BYTES that is part of the library's device image -- every GPU that loads the
 * library holds those 2 MiB from load to exit, whether this call is ever used or not.  The call itself runs no cudaMalloc,
 * cudaMallocAsync, cudaFree, cudaMallocHost or cudaEventCreate and uses no pinned staging buffer; the only memory it takes is a
 * few KB of host heap for the unit table it uploads.  The transport and finalize kernels are the ones pdv_mc_run launches, so
 * hist / hist2 / stats are bit-identical to pdv_mc_run's for the same arguments.
 *
 * Arguments as pdv_mc_run, except:
 *   - hist, hist2 (may be NULL), stats (may be NULL) are DEVICE pointers owned by the caller, and opts->output_on_device must
 *     be 1: the call only enqueues work on cuda_stream and returns;
 *   - every cloud must already be resident on the current device (pdv_cloud_create with that device current uploads it -- and
 *     allocates, so create the clouds during set-up); a host-only cloud or one on another device is PDV_E_INVALID;
 *   - clouds in a gas environment are PDV_E_UNSUPPORTED (their per-snapshot images are built and uploaded per call);
 *   - the workspace must fit:  n_units (8 + 16 n_bins + 8*16 + 24) + 4 * (blocks of the launch, <= 2 per SM) bytes, each
 *     section rounded up to 16, must not exceed PDV_STATIC_SCRATCH_BYTES (one unit of 8192 bins, 120 units of 1024 bins, or the
 *     paper's 200 x 512 spectrogram fit); a larger request is PDV_E_UNSUPPORTED and pdv_last_error() states both sizes.
 *     Split it over several calls (whole units, or id ranges whose results add) or use pdv_mc_run.
 * Set-up: the first call on each device looks the array's device address up (cudaGetSymbolAddress, with that device current)
 * and keeps it; make that first call during set-up, before any stream capture is begun on the thread.
 * Sharing: there is ONE array per device and every call uses it from offset 0.  It keeps whatever the previous call left; each
 * call clears the part that must start at zero (cursors and tallies) on cuda_stream before its kernel.  Calls on one stream
 * run in order and are safe.  Two calls whose work can overlap on the GPU -- different streams, or different host threads
 * without a common stream -- race on the array and give garbage: serialise them (one stream, or an event between them).
 * pdv_last_launch_info does not see these calls (it would need timing events). */
#define PDV_STATIC_SCRATCH_BYTES (2u << 20)
pdv_status pdv_mc_run_static(const pdv_cloud *const *clouds, int32_t n_clouds, const double *t_snap, int32_t n_snap,
                             uint64_t n_photons, uint64_t seed, const pdv_run_opts *opts,
                             double *hist, double *hist2, pdv_run_stats *stats, void *cuda_stream);

/* Per-history record of the diagnostic entry point below. */
typedef struct {
    float vt;                    /* Doppler velocity v~ at termination, m/s */
    float weight;                /* final weight */
    float mu_exit;               /* direction cosine when the history ended */
    int32_t fate;                /* 0 detected, 1 escaped, 2 absorbed (analog), 3 roulette-killed, 4 truncated,
                                    5 detected but under/overflow */
    int32_t n_scatter, n_reflect;
} pdv_trace_record;

/* Diagnostic: same transport as pdv_mc_run for ONE unit (cloud, unit index `unit`), and additionally one
 * record per history, records[id - first_photon_id] (HOST, [n_photons]).  Used by the tests to compare
 * single histories with the oracle run on the same Philox stream. */
pdv_status pdv_mc_trace(const pdv_cloud *cloud, uint32_t unit, uint64_t n_photons, uint64_t seed,
                        const pdv_run_opts *opts, double *hist, double *hist2, pdv_run_stats *stats,
                        pdv_trace_record *records, void *cuda_stream);

/* Stacks per-snapshot histograms into the spectrogram (Fig. 1 items 12-13; Eq. 19):
 *   scale 0: out = hist / n_photons            (probability per bin)
 *   scale 1: out = hist / (n_photons dv)       (spectral density per m/s), dv = (v_hi - v_lo)/n_bins
 *   scale 2: out = 10 log10(hist / n_photons), floor_db where hist = 0
 * hist [n_snap][n_bins] doubles, out [n_snap][n_bins] floats; both HOST when on_device = 0, both DEVICE when 1
 * (then the work is enqueued on cuda_stream). */
pdv_status pdv_spectrogram(const double *hist, int32_t n_snap, int32_t n_bins, uint64_t n_photons,
                           double v_lo, double v_hi, int32_t scale, float floor_db, float *out,
                           int32_t on_device, void *cuda_stream);

/* Characteristics of the main peak of each spectrum of a stack (section III.B: the three quantities of Eq. 35,
 * PAPER.md:356-365, which the paper reads off its MC spectra in Figs. 13-15).  For row i, with x = v/v_fs[i]:
 *   1. S[k] = hist[i][k] / (n_photons dx), dx = (v_hi - v_lo) / (n_bins v_fs[i]): density of detected weight per unit x;
 *      bin centre x_k = (v_lo + (k + 1/2) dv) / v_fs[i];
 *   2. k* = arg-max (first on ties) of S smoothed by `smooth_passes` passes of a centred moving average of half-width
 *      `smooth_half` bins (mean over the bins that exist at the array ends), over the bins with x_min <= x_k <= x_max
 *      (x_min > 1 keeps the free-surface peak of thin clouds, out of the search);
 *   3. unweighted least-squares parabola through the UNSMOOTHED S[k], |k - k*| <= fit_half (bins that exist):
 *      x_peak = vertex position, i_peak = vertex value, curvature = S''/S at the vertex (per unit x squared).
 * status: 0 ok; 1 no bin in the search range (k_peak = -1) or fewer than 3 bins in the fit window; 2 the parabola has no
 * maximum -- then x_peak = x_{k*}, i_peak = smoothed S[k*], curvature = 0.
 * All arithmetic is fp64.  Steps 1-2 use the same operation order as their definition (sequential sums, no fused
 * multiply-add), so k* is reproducible bit for bit. */
typedef struct {
    size_t struct_size;          /* sizeof(pdv_peak_opts) */
    int32_t smooth_half;         /* >= 0 */
    int32_t smooth_passes;       /* >= 0 */
    int32_t fit_half;            /* >= 1 */
    int32_t pad;
    double x_min, x_max;         /* search range in x = v / v_fs; x_max >= x_min */
} pdv_peak_opts;

typedef struct {
    double x_peak;               /* v~_peak / v_fs            (Eq. 31) */
    double i_peak;               /* spectrum value at the peak (Eq. 32), density per unit x */
    double curvature;            /* I''/I at the peak          (Eq. 34), per unit x squared */
    int32_t k_peak;              /* arg-max bin k*, -1 if none */
    int32_t status;
    double beta_eq35;            /* Eq. 35 read backwards: beta = sqrt(-curvature); 0 unless status = 0 */
    double tau0_eq35;            /* tau0 = exp(beta (x_peak - 1)); for this library's weight tally that is 2 g tau_ext (R31) */
} pdv_peak;

/* hist [n_units][n_bins] doubles, v_fs [n_units] doubles (m/s, > 0), out [n_units]: all three HOST when on_device = 0,
 * all three DEVICE when on_device = 1 (then the work is enqueued on cuda_stream and the call does not wait).
 * n_bins <= PDV_MAX_BINS; n_units = 0 is valid.  Errors: PDV_E_INVALID for NULLs / bad sizes / bad opts, PDV_E_CUDA. */
pdv_status pdv_spectrum_peaks(const double *hist, int32_t n_units, int32_t n_bins, uint64_t n_photons,
                              double v_lo, double v_hi, const double *v_fs, const pdv_peak_opts *opts,
                              pdv_peak *out, int32_t on_device, void *cuda_stream);

/* Scattering-angle sampling check (the paper's own sampler on the device, to report the error of the table): draws
 * cos(theta) n_samples times for ONE size class of a Mie cloud (phase_model 0) in two ways and histograms both over
 * n_bins equal bins of [-1, 1]:
 *   table  the transport kernel's sampler: cos(theta) = M[k] + (M[k+1] - M[k]) frac from one Philox word (Eq. 13-14
 *          through the inverse-CDF table D_K);
 *   exact  acceptance-rejection on the exact Mie function, the paper's step (4): mu uniform on [-1, 1],
 *          accepted if xi i_max <= I(mu), I = |S1|^2 + |S2|^2 summed from the Mie series (Eq. 13-14) in fp32 on the device,
 *          i_max = 1.02 x the maximum of I over 20001 angles, found on the host.
 * Sample i draws from Philox4x32-10 streams keyed by (seed, i): same (cloud, class, n_samples, seed) => same counts.
 * hist_table, hist_exact: HOST [n_bins] counts.  info: HOST, may be NULL.  1 <= n_bins <= 4096.
 * Errors: PDV_E_INVALID (NULLs, class_index, n_bins), PDV_E_UNSUPPORTED (isotropic cloud; more than 1024 Mie terms),
 * PDV_E_CUDA. */
typedef struct {
    double sum_cos_table;        /* sum of cos(theta) over the table samples (mean = sum / n_samples -> g) */
    double sum_cos_exact;        /* same over the rejection samples */
    double i_max;                /* the bound used */
    uint64_t n_trials;           /* rejection trials in total: n_samples / n_trials = int I dmu / (2 i_max) */
    uint64_t n_bound_violations; /* trials that found I(mu) > i_max; must be 0 */
} pdv_phase_check;

pdv_status pdv_phase_sampling_check(const pdv_cloud *cloud, int32_t class_index, uint64_t n_samples, uint64_t seed,
                                    int32_t n_bins, uint64_t *hist_table, uint64_t *hist_exact, pdv_phase_check *info,
                                    void *cuda_stream);

/* Diagnostic (pin P13 of the test suite): raw blocks of the kernels' own Philox4x32-10.  Block i = the generator applied to the
 * counter counters[4i .. 4i+3] with the key (low word of seed, high word of seed) -- the key pdv_mc_run derives from `seed` --
 * computed three times, once through each way the transport kernel reads its ten round keys: static shared memory, a shared
 * address held in a register, and the kernel parameters (constant bank).  All three must equal the published Random123 vectors.
 * counters: HOST [4 n] words; out_static / out_shared / out_param: HOST [4 n] words each; 0 <= n <= 2^20. */
pdv_status pdv_philox_blocks(const uint32_t *counters, int32_t n, uint64_t seed, uint32_t *out_static, uint32_t *out_shared,
                             uint32_t *out_param);

/* Measures the issue-rate denominators on the current device: a dependent-free FFMA stream and a MUFU
 * stream, each run for ~`millis` ms on every SM.  Outputs (any may be NULL): thread-instructions/s of each,
 * the SM clock in MHz observed meanwhile (clock64 over globaltimer), and the SM count. */
pdv_status pdv_issue_peaks(double millis, double *ffma_thread_inst_per_s, double *mufu_thread_inst_per_s,
                           double *sm_clock_mhz, int32_t *n_sm, void *cuda_stream);

/* Launch statistics of the last pdv_mc_run / pdv_mc_trace on this thread: kernels launched and the duration of
 * the transport kernel in ms measured with CUDA events on cuda_stream.  After an output_on_device = 1 run this
 * call waits (cudaEventSynchronize) for that run's transport kernel to finish.  Any pointer may be NULL.
 * variant: which instantiation of the transport kernel ran -- bit 0 several size classes, bit 1 analog absorption,
 * bit 2 single-scatter-only, bit 3 trace, bit 4 Russian roulette, bit 5 the second production instantiation (one
 * class: long histories, several draws per pass; several classes: clean class guides), bits 8.. the depth model
 * (0 depth table, 1 closed form, 2 general, 3 gas units).  The result of a run never depends on it. */
pdv_status pdv_last_launch_info(int32_t *n_kernels, float *transport_ms, int32_t *grid, int32_t *block,
                                int32_t *smem_bytes, int32_t *variant);

/* The same for the last run this thread enqueued on `cuda_stream` (the library remembers the 16 most recently used streams of
 * each host thread): after two asynchronous runs on two streams each one's kernel time can still be read.  Zeros if the thread
 * has not run anything on that stream. */
pdv_status pdv_launch_info_on_stream(void *cuda_stream, int32_t *n_kernels, float *transport_ms, int32_t *grid, int32_t *block,
                                     int32_t *smem_bytes, int32_t *variant);

/* Thread-local message of the last failing call on this thread; "" if none.  Valid until the next call. */
const char *pdv_last_error(void);

/* Library version string, e.g. "pdv_b200 0.1 (sm_100a)". */
const char *pdv_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PDV_H_ */
