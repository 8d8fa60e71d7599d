/* ORACLE (test infrastructure) -- plain double-precision CPU Monte-Carlo of the PDV photon
 * transport of arXiv 2012.00963, section II.B.
 *
 * This file is NOT part of the product.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header,
 * table generator or constant with the CUDA library and includes nothing from it.
 *
 * It follows SURVEY.md 8(c) "Algorithm, step by step" in the paper's order, one photon history at
 * a time, with the full direction 3-vector (paper-literal, Eq. 16/17):
 *
 *   step 1   photon starts at the top, u = (0,0,-1), weight 1, shift 0
 *   step 3  (Eq. 7/10) free flight: s = -ln xi in optical depth, T' = T - mu s
 *                             (exact free-path sampling = the step->0 limit of the paper's H/1000
 *                             marching; reading R15)
 *   step 4  (Eq. 11) scatter with probability K_sca/K_ext (analog) or weight *= omega0
 *                             (implicit capture: same expectation); theta from the discretised
 *                             phase function D_K (or, variant, acceptance-rejection on exact Mie,
 *                             the paper's own step 4); phi uniform (Eq. 15); rotate by Eq. 16/17
 *   Eq. 4     Doppler velocity  v~ += 1/2 (u_out - u_in) . v zhat   per event
 *   step 6 free surface: "ideal diffuse reflection", polar angle uniform,
 *                             azimuth uniform; counted as a Doppler event with velocity v_fs
 *   Eq. 19    photons leaving the top inside the aperture are histogrammed by v~
 *   step 7    until absorbed or out (+ Russian roulette, BASELINE.json config 5)
 *
 * Random numbers: rng_mode 0 = xoshiro256** seeded per photon by splitmix64 (53-bit uniforms),
 * unrelated to the GPU generator.  rng_mode 1 = the shared counter-based stream of DESIGN.md
 * ("each side implements the same counter-based generator"): Philox4x32-10, key = seed,
 * counter = (id_lo, id_hi, stream, 2*draw + sub), with the word->uniform maps of DESIGN.md D2.
 * Mode 1 exists so that single histories can be compared with the GPU; it is pinned by the
 * published known-answer vectors of Philox4x32-10 (tests/golden/philox4x32_10_kat.txt).
 *
 * Parity status: every closed-form consequence is pinned (tests/test_oracle_*.py, pins P1-P13 of
 * SURVEY.md 8(c)), and the multiple-scattering transport core (free paths, direction updates,
 * reflections, over many events) by the mean-path invariance of a non-absorbing medium under diffuse
 * illumination (P16: <events> = 4 tau_ext, <reflections> = 1, Lambertian exit; launch_model 1).  The
 * Doppler bookkeeping is pinned per event (P2, P3) and over whole multiple-scattering histories in
 * a rigid cloud, where it telescopes to the exit angle (P17); with a velocity PROFILE the spectrum of
 * the histories of exactly two particle events is pinned to a 4-D quadrature (P20).  The SHAPE of the
 * multiple-scattering spectrum of a cloud with a velocity profile at orders >= 3 has no closed form and
 * no figure data is available: "parity unpinned" for that output beyond those pins.
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    /* ---- cloud tables (built by oracle/cloud.py) ---- */
    int32_t n_classes, K, n_depth;
    const double *phase;      /* [n_classes][K+1] quantiles M_c[k] of cos(theta) */
    const double *p_cum;      /* [n_classes] cumulative class hit probabilities, last = 1 */
    const double *omega0;     /* [n_classes] K_sca/K_ext */
    const double *T_edge;     /* [n_depth+1], T_edge[j] at v = v_max - j (v_max-v_fs)/n_depth */
    double v_fs, v_max, tau_ext;
    int32_t analytic_profile; /* variant: v(T) from the closed form of the truncated Eq. 20 */
    double beta;
    double R;                 /* surface reflectivity */
    int32_t surface_model;    /* 0 paper (polar angle uniform), 1 Lambertian */
    /* ---- variant: exact Mie sampling by acceptance-rejection ---- */
    int32_t exact_mie;        /* 0 table D_K, 1 rejection */
    const int32_t *mie_nmax;  /* [n_classes] */
    const double *mie_ab;     /* [n_classes][4*mie_stride]: Re a, Im a, Re b, Im b for n=1..nmax */
    int32_t mie_stride;
    const double *mie_gmax;   /* [n_classes] upper bound of (|S1|^2+|S2|^2) sin(theta) */
    /* ---- run options ---- */
    int32_t n_bins;
    double v_lo, v_hi, mu_aperture;
    int32_t mode;             /* 0 implicit capture, 1 analog */
    int32_t max_events;       /* roulette once n_scatter >= max_events; <=0: never */
    double p_roulette;
    int32_t single_scatter_only;
    int32_t rng_mode;         /* 0 xoshiro (independent), 1 shared Philox stream */
    uint64_t seed;
    uint32_t stream;
    int32_t launch_model;     /* 0: the paper's collimated beam, u = (0,0,-1) (reading R1); 1: diffuse (Lambertian) illumination of
                               * the cloud top, pdf of the polar cosine proportional to it -- used only by the invariance pin
                               * (mean-chord-length theorem), rng_mode 0 only */
    /* ---- gas environment (readings R35-R38 of oracle/gas.py, NOT from the paper) ---- */
    int32_t gas;              /* 1: T_edge belongs to the depth bins uniform in the height zeta above the free surface */
    const double *zeta_edge;  /* [n_depth+1] heights of the bin edges, zeta_top ... 0 */
    const double *class_cum;  /* [n_depth][n_classes] cumulative class hit probabilities inside each bin, last = 1 */
    const double *gas_L;      /* [n_classes] drag length L_c = 4 rho0 d_c / (3 C_d rho_g); +inf: no drag */
    double t_snap;            /* snapshot time t */
} oracle_params;

typedef struct {
    double detected, underflow, overflow, escaped, absorbed_particles, absorbed_surface,
           roulette_killed, roulette_gained, truncated;
    uint64_t histories, particle_events, surface_reflections, max_events_in_history;
} oracle_stats;

/* per-history record for trace mode */
typedef struct {
    double vt;        /* Doppler velocity by Eq. 4 (per event) */
    double vt_leg;    /* same by the per-leg form (Eq. 18 sign-corrected, R2) */
    double w;         /* final weight */
    double mu_exit;
    int32_t fate;     /* 0 detected(in aperture) 1 escaped 2 absorbed(analog) 3 roulette-killed 4 truncated */
    int32_t n_scatter, n_reflect;
} oracle_trace;

/* ------------------------------------------------------------------ RNG ---------------------- */
static inline uint64_t splitmix64(uint64_t *s) {
    uint64_t z = (*s += 0x9e3779b97f4a7c15ULL);
    z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ULL;
    z = (z ^ (z >> 27)) * 0x94d049bb133111ebULL;
    return z ^ (z >> 31);
}
static inline uint64_t rotl64(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }

/* Philox4x32-10 written from its definition (Salmon et al., SC'11): 10 rounds of
 * (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)), key bumped by the
 * Weyl constants between rounds. */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

typedef struct {
    int mode;
    uint64_t s[4];                 /* xoshiro256** state */
    uint32_t key[2], id_lo, id_hi, stream;
} rng_t;

static void rng_init(rng_t *r, const oracle_params *p, uint64_t id) {
    r->mode = p->rng_mode;
    if (p->rng_mode == 0) {
        uint64_t s = p->seed ^ (0x632be59bd9b4e019ULL * (id + 1)) ^ ((uint64_t)p->stream << 40);
        for (int i = 0; i < 4; ++i) r->s[i] = splitmix64(&s);
    } else {
        r->key[0] = (uint32_t)p->seed; r->key[1] = (uint32_t)(p->seed >> 32);
        r->id_lo = (uint32_t)id; r->id_hi = (uint32_t)(id >> 32); r->stream = p->stream;
    }
}
static inline double rng_u53(rng_t *r) {           /* uniform in [0,1), 53 bits */
    uint64_t *s = r->s;
    uint64_t result = rotl64(s[1] * 5, 7) * 9, t = s[1] << 17;
    s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3]; s[2] ^= t; s[3] = rotl64(s[3], 45);
    return (double)(result >> 11) * (1.0 / 9007199254740992.0);
}

/* the uniforms one flight needs */
typedef struct { double xi_path, xi_class, xi_cos, xi_phi, xi_roulette, xi_absorb; } flight_draws;

static void draw_flight(rng_t *r, const oracle_params *p, uint32_t flight, flight_draws *d) {
    if (r->mode == 0) {
        d->xi_path = 1.0 - rng_u53(r);             /* (0,1] */
        d->xi_class = rng_u53(r); d->xi_cos = rng_u53(r); d->xi_phi = rng_u53(r);
        d->xi_roulette = rng_u53(r); d->xi_absorb = rng_u53(r);
    } else {                                       /* DESIGN.md D1/D2: the shared counter-based stream */
        /* D1/D2.  Counter word 3 of a block = 2 * (block index), + 1 for its companion block (absorption /
         * roulette words).  A flight reads a path word a, a phase word b and, with several size classes, a class word cw.
         * One class: block index = flight / 2; the block feeds two flights, (a, b) = (x0, x1) then (x2, x3); companion
         *   words: absorption y[half], roulette y[2 + half].
         * Several classes: flights come in groups of three, group g = flight / 3 reads blocks 2g and 2g + 1 as eight words
         *   W0..W7: (a, b, cw) = (W0, W1, W2'), (W3, W4, W5'), (W6, W7, cw2), where W' = the word with its low byte
         *   replaced by 0x80 and cw2 = (W2.byte0, W5.byte0, W6 bits 23..8) from the top; companions: absorption =
         *   word r of the companion of block 2g, roulette = word r of the companion of block 2g + 1 (r = flight % 3).
         * Azimuth word, both cases: bytes (a.byte0, b.byte0, a.byte1, a.byte2) from the top. */
        int mono = p->n_classes == 1;
        uint32_t a, b, pw, w_abs, w_roul;
        if (mono) {
            uint32_t draw = flight >> 1, half = flight & 1u;
            uint32_t c[4] = { r->id_lo, r->id_hi, r->stream, 2u * draw }, x[4], y[4];
            oracle_philox4x32_10(c, r->key, x);
            c[3] = 2u * draw + 1u;
            oracle_philox4x32_10(c, r->key, y);
            a = x[2 * half]; b = x[2 * half + 1];
            w_abs = y[half]; w_roul = y[2 + half];
            d->xi_class = 0.0;
        } else {
            uint32_t g = flight / 3u, rr = flight % 3u, W[8], ya[4], yr[4], cw;
            uint32_t c[4] = { r->id_lo, r->id_hi, r->stream, 2u * (2u * g) };
            oracle_philox4x32_10(c, r->key, W);
            c[3] = 2u * (2u * g) + 1u;
            oracle_philox4x32_10(c, r->key, ya);
            c[3] = 2u * (2u * g + 1u);
            oracle_philox4x32_10(c, r->key, W + 4);
            c[3] = 2u * (2u * g + 1u) + 1u;
            oracle_philox4x32_10(c, r->key, yr);
            if (rr == 0u)      { a = W[0]; b = W[1]; cw = (W[2] & 0xFFFFFF00u) | 0x80u; }
            else if (rr == 1u) { a = W[3]; b = W[4]; cw = (W[5] & 0xFFFFFF00u) | 0x80u; }
            else               { a = W[6]; b = W[7]; cw = ((W[2] & 0xFFu) << 24) | ((W[5] & 0xFFu) << 16) | ((W[6] >> 8) & 0xFFFFu); }
            w_abs = ya[rr]; w_roul = yr[rr];
            d->xi_class = ((double)cw + 0.5) * (1.0 / 4294967296.0);
        }
        pw = ((a & 0xFFu) << 24) | ((b & 0xFFu) << 16) | (((a >> 8) & 0xFFu) << 8) | ((a >> 16) & 0xFFu);
        /* D2: path = top 23 bits of a; phase = top (log2 K + 12) bits of b; azimuth = pw */
        int log2K = 0;
        while ((1 << log2K) < p->K) ++log2K;
        uint32_t keep = (uint32_t)(log2K + 12);
        d->xi_path = 1.0 - (double)(a >> 9) * (1.0 / 8388608.0);         /* (0,1], 23 bits */
        d->xi_cos = (double)(b >> (32u - keep)) / (double)(1ull << keep);
        d->xi_phi = (double)pw * (1.0 / 4294967296.0);
        d->xi_absorb = (double)w_abs * (1.0 / 4294967296.0);
        d->xi_roulette = (double)w_roul * (1.0 / 4294967296.0);
    }
}

/* ------------------------------------------------------------------ physics ------------------ */
/* velocity of the particles at vertical optical depth T (0 < T < tau_ext) */
static double velocity_at(const oracle_params *p, double T) {
    if (p->analytic_profile) {     /* closed form: invert T(v) = tau_ext (exp(-beta (v/v_fs - 1)) - E)/(1 - E), i.e.
                                    * T = tau_ext (1 - G(v)) with G the truncated, renormalised mass CDF of Eq. 20
                                    * (PAPER.md:189).  T is measured from the TOP (T = 0 at v_max), so the argument is
                                    * E + (1-E) T/tau_ext; SURVEY.md 8(c) step 4d prints (1 - T/tau_ext), which would
                                    * be depth measured from the free surface (reading R26). */
        double E = exp(-p->beta * (p->v_max / p->v_fs - 1.0));
        return p->v_fs - (p->v_fs / p->beta) * log(E + (1.0 - E) * (T / p->tau_ext));
    }
    /* canonical depth discretisation: T linear in v inside each of n_depth bins uniform in v */
    int lo = 0, hi = p->n_depth;                   /* T_edge[lo] <= T < T_edge[hi] */
    while (hi - lo > 1) {
        int mid = (lo + hi) / 2;
        if (p->T_edge[mid] <= T) lo = mid; else hi = mid;
    }
    double dv = (p->v_max - p->v_fs) / p->n_depth;
    double frac = (T - p->T_edge[lo]) / (p->T_edge[lo + 1] - p->T_edge[lo]);
    return p->v_max - (lo + frac) * dv;
}

/* Gas environment (R36, R37): the interaction at optical depth T lies in depth bin `lo` at height zeta (T linear in zeta inside
 * the bin); the class is picked with the bin's own probabilities; the class-c particle found there moves with
 * v_fs + (L_c/t)(1 - exp(-zeta/L_c)) -- the closed form of the drag law du/dt = -u^2/L_c (R35). */
static double gas_interaction(const oracle_params *p, double T, double xi_class, int *c_out) {
    int lo = 0, hi = p->n_depth;                   /* T_edge[lo] <= T < T_edge[hi] */
    while (hi - lo > 1) {
        int mid = (lo + hi) / 2;
        if (p->T_edge[mid] <= T) lo = mid; else hi = mid;
    }
    double frac = (T - p->T_edge[lo]) / (p->T_edge[lo + 1] - p->T_edge[lo]);
    double zeta = p->zeta_edge[lo] + frac * (p->zeta_edge[lo + 1] - p->zeta_edge[lo]);
    const double *cum = p->class_cum + (size_t)lo * p->n_classes;
    int c = 0;
    while (c < p->n_classes - 1 && xi_class >= cum[c]) ++c;
    *c_out = c;
    double L = p->gas_L[c];
    double u = isinf(L) ? zeta / p->t_snap : -(L / p->t_snap) * expm1(-zeta / L);
    return p->v_fs + u;
}

static int pick_class(const oracle_params *p, double xi) {
    int c = 0;
    while (c < p->n_classes - 1 && xi >= p->p_cum[c]) ++c;
    return c;
}

/* |S1|^2+|S2|^2 at mu for class c from stored a_n, b_n (Eq. 14) -- exact-Mie variant only */
static double mie_intensity(const oracle_params *p, int c, double mu) {
    int nmax = p->mie_nmax[c];
    const double *ab = p->mie_ab + (size_t)c * 4 * p->mie_stride;
    const double *ar = ab, *ai = ab + p->mie_stride, *br = ab + 2 * p->mie_stride, *bi = ab + 3 * p->mie_stride;
    double pim1 = 0.0, pi0 = 1.0;                  /* pi_0, pi_1 */
    double s1r = 0, s1i = 0, s2r = 0, s2i = 0;
    for (int n = 1; n <= nmax; ++n) {
        double tau = n * mu * pi0 - (n + 1) * pim1;
        double f = (2.0 * n + 1.0) / (n * (n + 1.0));
        s1r += f * (ar[n - 1] * pi0 + br[n - 1] * tau); s1i += f * (ai[n - 1] * pi0 + bi[n - 1] * tau);
        s2r += f * (ar[n - 1] * tau + br[n - 1] * pi0); s2i += f * (ai[n - 1] * tau + bi[n - 1] * pi0);
        double pin = ((2.0 * n + 1.0) / n) * mu * pi0 - ((n + 1.0) / n) * pim1;   /* pi_{n+1} */
        pim1 = pi0; pi0 = pin;
    }
    return s1r * s1r + s1i * s1i + s2r * s2r + s2i * s2i;
}

static double sample_cos_theta(const oracle_params *p, int c, double xi, rng_t *r) {
    if (!p->exact_mie) {           /* canonical D_K: SURVEY.md 8(c) step 2 */
        double t = xi * p->K;
        int k = (int)t;
        if (k >= p->K) k = p->K - 1;
        double frac = t - k;
        const double *M = p->phase + (size_t)c * (p->K + 1);
        return M[k] + (M[k + 1] - M[k]) * frac;
    }
    for (;;) {                     /* acceptance-rejection in theta, density I(theta) sin(theta) */
        double th = M_PI * rng_u53(r);
        double gval = mie_intensity(p, c, cos(th)) * sin(th);
        if (rng_u53(r) * p->mie_gmax[c] < gval) return cos(th);
    }
}

/* Eq. 16 (standard rotation, R7) and Eq. 17 near the pole */
static void rotate(double u[3], double ct, double phi) {
    double st = sqrt(fmax(0.0, (1.0 - ct) * (1.0 + ct)));
    double cp = cos(phi), sp = sin(phi);
    double ux = u[0], uy = u[1], uz = u[2];
    if (1.0 - fabs(uz) < 1e-12) {
        u[0] = st * cp; u[1] = st * sp; u[2] = ct * (uz >= 0 ? 1.0 : -1.0);
    } else {
        double q = sqrt(1.0 - uz * uz);
        u[0] = st * (ux * uz * cp - uy * sp) / q + ux * ct;
        u[1] = st * (uy * uz * cp + ux * sp) / q + uy * ct;
        u[2] = -st * cp * q + uz * ct;
    }
    double nrm = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);   /* keep |u| = 1 against drift */
    u[0] /= nrm; u[1] /= nrm; u[2] /= nrm;
}

typedef struct {
    double *hist, *hist2;          /* [n_bins] */
    oracle_stats st;
} tally_t;

static void run_history(const oracle_params *p, uint64_t id, tally_t *ty, oracle_trace *tr) {
    rng_t rng; rng_init(&rng, p, id);
    double T = 0.0, u[3] = { 0.0, 0.0, -1.0 }, w = 1.0, vt = 0.0;
    double vt_leg = 0.0, v_prev = 0.0;             /* per-leg bookkeeping: source at rest */
    int n_sc = 0, n_refl = 0, fate = -1;
    uint32_t flight = 0;
    flight_draws d;
    ty->st.histories += 1;
    if (p->launch_model == 1 && rng.mode == 0) {
        double m0 = sqrt(rng_u53(&rng)), ph = 6.283185307179586 * rng_u53(&rng), sn = sqrt(fmax(0.0, 1.0 - m0 * m0));
        u[0] = sn * cos(ph); u[1] = sn * sin(ph); u[2] = -m0;
    }
    for (;;) {
        draw_flight(&rng, p, flight++, &d);
        double s = -log(d.xi_path);
        double Tn = T - u[2] * s;
        if (Tn < 0.0) {                            /* leaves through the top (step 6) */
            vt_leg += -0.5 * u[2] * (0.0 - v_prev);/* last leg: detector at rest */
            if (u[2] >= p->mu_aperture) {
                fate = 0;
                double b = floor((vt - p->v_lo) / ((p->v_hi - p->v_lo) / p->n_bins));
                if (b < 0) ty->st.underflow += w;
                else if (b >= p->n_bins) ty->st.overflow += w;
                else { ty->st.detected += w; ty->hist[(int)b] += w; ty->hist2[(int)b] += w * w; }
            } else { fate = 1; ty->st.escaped += w; }
            break;
        }
        double mu_old = u[2], v_here;
        if (Tn >= p->tau_ext) {                    /* free surface */
            v_here = p->v_fs;
            if (p->mode == 1) {                    /* analog: absorbed with probability 1-R */
                if (d.xi_absorb >= p->R) { ty->st.absorbed_surface += w; fate = 2; w = 0.0; break; }
            } else { ty->st.absorbed_surface += w * (1.0 - p->R); w *= p->R; }
            /* two independent uniforms: xi_phi drives the polar angle here, xi_cos the azimuth (D2) */
            double mu_new = (p->surface_model == 1) ? sqrt(d.xi_phi) : cos(0.5 * M_PI * d.xi_phi);
            double sn = sqrt(fmax(0.0, 1.0 - mu_new * mu_new)), ph = 2.0 * M_PI * d.xi_cos;
            u[0] = sn * cos(ph); u[1] = sn * sin(ph); u[2] = mu_new;
            T = p->tau_ext;
            n_refl += 1; ty->st.surface_reflections += 1;
        } else {                                   /* particle interaction at depth Tn */
            if (p->single_scatter_only && n_sc >= 1) { ty->st.truncated += w; fate = 4; break; }
            int c;
            if (p->gas) v_here = gas_interaction(p, Tn, d.xi_class, &c);
            else { v_here = velocity_at(p, Tn); c = pick_class(p, d.xi_class); }
            if (p->mode == 1) {
                if (d.xi_absorb >= p->omega0[c]) { ty->st.absorbed_particles += w; fate = 2; w = 0.0;
                                                   ty->st.particle_events += 1; break; }
            } else { ty->st.absorbed_particles += w * (1.0 - p->omega0[c]); w *= p->omega0[c]; }
            double ct = sample_cos_theta(p, c, d.xi_cos, &rng);
            rotate(u, ct, 2.0 * M_PI * d.xi_phi);
            T = Tn;
            n_sc += 1; ty->st.particle_events += 1;
        }
        vt += 0.5 * (u[2] - mu_old) * v_here;      /* Eq. 4, z components only (v along z) */
        vt_leg += -0.5 * mu_old * (v_here - v_prev);
        v_prev = v_here;
        if (p->max_events > 0 && n_sc >= p->max_events) {      /* Russian roulette */
            if (d.xi_roulette < p->p_roulette) { ty->st.roulette_gained += w * (1.0 / p->p_roulette - 1.0); w /= p->p_roulette; }
            else { ty->st.roulette_killed += w; fate = 3; break; }
        }
    }
    if ((uint64_t)(n_sc + n_refl) > ty->st.max_events_in_history) ty->st.max_events_in_history = n_sc + n_refl;
    if (tr) { tr->vt = vt; tr->vt_leg = vt_leg; tr->w = w; tr->mu_exit = u[2]; tr->fate = fate;
              tr->n_scatter = n_sc; tr->n_reflect = n_refl; }
}

/* ------------------------------------------------------------------ driver ------------------- */
typedef struct { const oracle_params *p; uint64_t first, count; tally_t ty; oracle_trace *trace; } job_t;

static void *worker(void *arg) {
    job_t *j = (job_t *)arg;
    for (uint64_t i = 0; i < j->count; ++i)
        run_history(j->p, j->first + i, &j->ty, j->trace ? j->trace + i : NULL);
    return NULL;
}

/* Runs photon ids [first_id, first_id + n_photons) on n_threads threads.  hist/hist2: [n_bins]
 * (overwritten); stats overwritten; trace may be NULL or [n_photons].  Returns 0, or -1 on
 * allocation failure.  Results do not depend on n_threads except through summation order. */
int oracle_mc_run(const oracle_params *p, uint64_t first_id, uint64_t n_photons, int n_threads,
                  double *hist, double *hist2, oracle_stats *stats, oracle_trace *trace) {
    if (n_threads < 1) n_threads = 1;
    if ((uint64_t)n_threads > n_photons && n_photons > 0) n_threads = (int)n_photons;
    job_t *jobs = (job_t *)calloc(n_threads, sizeof(job_t));
    pthread_t *th = (pthread_t *)calloc(n_threads, sizeof(pthread_t));
    if (!jobs || !th) return -1;
    uint64_t per = n_photons / n_threads, rem = n_photons % n_threads, at = 0;
    for (int t = 0; t < n_threads; ++t) {
        jobs[t].p = p; jobs[t].first = first_id + at; jobs[t].count = per + ((uint64_t)t < rem ? 1 : 0);
        jobs[t].trace = trace ? trace + at : NULL;
        at += jobs[t].count;
        jobs[t].ty.hist = (double *)calloc(p->n_bins, sizeof(double));
        jobs[t].ty.hist2 = (double *)calloc(p->n_bins, sizeof(double));
        if (!jobs[t].ty.hist || !jobs[t].ty.hist2) return -1;
    }
    for (int t = 1; t < n_threads; ++t) pthread_create(&th[t], NULL, worker, &jobs[t]);
    worker(&jobs[0]);
    for (int t = 1; t < n_threads; ++t) pthread_join(th[t], NULL);
    memset(hist, 0, sizeof(double) * p->n_bins);
    memset(hist2, 0, sizeof(double) * p->n_bins);
    memset(stats, 0, sizeof(*stats));
    for (int t = 0; t < n_threads; ++t) {
        for (int k = 0; k < p->n_bins; ++k) { hist[k] += jobs[t].ty.hist[k]; hist2[k] += jobs[t].ty.hist2[k]; }
        const oracle_stats *s = &jobs[t].ty.st;
        stats->detected += s->detected; stats->underflow += s->underflow; stats->overflow += s->overflow;
        stats->escaped += s->escaped; stats->absorbed_particles += s->absorbed_particles;
        stats->absorbed_surface += s->absorbed_surface; stats->roulette_killed += s->roulette_killed;
        stats->roulette_gained += s->roulette_gained; stats->truncated += s->truncated;
        stats->histories += s->histories; stats->particle_events += s->particle_events;
        stats->surface_reflections += s->surface_reflections;
        if (s->max_events_in_history > stats->max_events_in_history) stats->max_events_in_history = s->max_events_in_history;
        free(jobs[t].ty.hist); free(jobs[t].ty.hist2);
    }
    free(jobs); free(th);
    return 0;
}

/* Exposed for the rotation pins (P6): rotates u in place. */
void oracle_rotate(double u[3], double cos_theta, double phi) { rotate(u, cos_theta, phi); }
