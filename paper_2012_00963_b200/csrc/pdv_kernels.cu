// pdv_kernels.cu -- CUDA kernels of the PDV Monte-Carlo transport for sm_100a (B200).
//
// transport_kernel: persistent-thread photon transport, section II.B steps (1)-(7) (174-183):
//   * one lane = one photon history at a time; dead lanes are re-filled ("photon regeneration") from a chunk of
//     photon ids the warp claims with one global atomic, so lanes stay busy whatever the history lengths are;
//   * every history draws from its own Philox4x32-10 counter stream, counter = (id_lo, id_hi, unit, 2*flight+sub),
//     key = seed: results do not depend on which lane, warp or block runs a history (D1/D2);
//   * the cloud tables (inverse-CDF phase tables, depth table + its guide, class thresholds) live in shared memory;
//   * free flight in vertical optical depth T (exact sampling of Eq. 7/10), interaction (Eq. 11), scattering angle
//     from the discretised phase function D_K (Eq. 13-14), azimuth (Eq. 15), direction update (z row of Eq. 16 /
//     Eq. 17 -- only mu = u_z matters in slab geometry, reading R7), Doppler update (Eq. 4);
//   * tallies are Q31 integers in a shared-memory histogram, warp-aggregated, flushed once per block and unit.
#include "pdv_device.h"

namespace pdv {

#define FULL_MASK 0xffffffffu

constexpr uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;

// Philox4x32-10 block function; round keys precomputed on the host (kernel parameter = constant bank).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              const uint32_t (&k0)[10], const uint32_t (&k1)[10],
                                              uint32_t &o0, uint32_t &o1, uint32_t &o2, uint32_t &o3) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)PHILOX_M0 * c0;
        const unsigned long long p1 = (unsigned long long)PHILOX_M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

__device__ __forceinline__ float fast_sqrt(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// w * q (q in Q31, 0..2^31) -> Q31, truncated.
__device__ __forceinline__ uint32_t mul_q31(uint32_t w, uint32_t q) {
    return (uint32_t)(((unsigned long long)w * q) >> 31);
}

struct CloudView {               // per-unit scalars and shared-memory table pointers
    const float *phase, *T_edge;
    const uint32_t *thr, *albedo;
    const uint16_t *guide;
    uint32_t n_classes, K1, shiftK, n_depth, n_guide, guide_base, cls_steps;
    float frac_scale, tau_ext, v_fs, v_max, dv_depth;
    uint32_t R_q31, R_thr, surface_model;
};

// particle velocity at vertical optical depth Tn, 0 <= Tn < tau_ext: piecewise-linear T(v) table, bins uniform in v.
__device__ __forceinline__ float depth_velocity(const CloudView &cv, float Tn) {
    int gi = (int)(__float_as_uint(Tn) >> 16) - (int)cv.guide_base;
    gi = max(gi, 0);
    gi = min(gi, (int)cv.n_guide - 1);
    uint32_t j = cv.guide[gi];
    float Tj1 = cv.T_edge[j + 1];
    int steps = 0;
    while (Tj1 <= Tn && j + 1 < cv.n_depth) {
        if (++steps > 4) {                               // pathological table: finish by bisection
            uint32_t lo = j, hi = cv.n_depth;            // T_edge[lo] <= Tn < T_edge[hi]
            while (hi - lo > 1) {
                const uint32_t mid = (lo + hi) >> 1;
                if (cv.T_edge[mid] <= Tn) lo = mid; else hi = mid;
            }
            j = lo;
            Tj1 = cv.T_edge[j + 1];
            break;
        }
        ++j;
        Tj1 = cv.T_edge[j + 1];
    }
    const float Tj = cv.T_edge[j];
    const float frac = __fdividef(Tn - Tj, Tj1 - Tj);
    return fmaf(-((float)j + frac), cv.dv_depth, cv.v_max);
}

template <bool POLY, bool ANALOG, bool TRACE>
__global__ void __launch_bounds__(512, 2) transport_kernel(const __grid_constant__ RunParams P) {
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ unsigned long long s_stats[ST_COUNT];
    __shared__ int s_go;

    const uint32_t tid = threadIdx.x, lane = tid & 31u;
    const uint32_t lanemask_lt = (1u << lane) - 1u;
    unsigned long long *s_hist = reinterpret_cast<unsigned long long *>(smem);
    unsigned long long *s_hist2 = s_hist + P.n_bins;
    unsigned char *s_blob = smem + 16u * (size_t)P.n_bins;

    for (uint32_t visit = 0; visit < P.n_units; ++visit) {
        const uint32_t u = (blockIdx.x + visit) % P.n_units;
        if (tid == 0) s_go = (*(volatile unsigned long long *)(P.next_id + u) < P.n_photons) ? 1 : 0;
        __syncthreads();
        const bool go = s_go != 0;
        __syncthreads();
        if (!go) continue;

        // ---- stage the unit's cloud tables, clear the private histogram --------------------------------------
        const UnitDesc ud = P.units[u];
        {
            const uint4 *src = reinterpret_cast<const uint4 *>(ud.cloud_blob);
            const uint32_t n16 = reinterpret_cast<const DevCloudHeader *>(ud.cloud_blob)->blob_bytes >> 4;
            uint4 *dst = reinterpret_cast<uint4 *>(s_blob);
            for (uint32_t i = tid; i < n16; i += blockDim.x) dst[i] = __ldg(src + i);
            for (uint32_t i = tid; i < 2u * P.n_bins; i += blockDim.x) s_hist[i] = 0ull;
            if (tid < ST_COUNT) s_stats[tid] = 0ull;
        }
        __syncthreads();
        CloudView cv;
        {
            const DevCloudHeader *h = reinterpret_cast<const DevCloudHeader *>(s_blob);
            cv.phase = reinterpret_cast<const float *>(s_blob + h->off_phase);
            cv.T_edge = reinterpret_cast<const float *>(s_blob + h->off_tedge);
            cv.thr = reinterpret_cast<const uint32_t *>(s_blob + h->off_thr);
            cv.albedo = reinterpret_cast<const uint32_t *>(s_blob + (ANALOG ? h->off_albthr : h->off_albedo));
            cv.guide = reinterpret_cast<const uint16_t *>(s_blob + h->off_guide);
            cv.n_classes = h->n_classes; cv.K1 = h->K + 1u; cv.shiftK = 32u - h->log2K;
            cv.n_depth = h->n_depth; cv.n_guide = h->n_guide; cv.guide_base = h->guide_base;
            cv.cls_steps = 0;
            while ((1u << cv.cls_steps) < cv.n_classes) ++cv.cls_steps;
            cv.frac_scale = __uint_as_float((127u - cv.shiftK) << 23);       // 2^-(32-log2K)
            cv.tau_ext = h->tau_ext; cv.v_fs = h->v_fs; cv.v_max = h->v_max; cv.dv_depth = h->dv_depth;
            cv.R_q31 = h->R_q31; cv.R_thr = h->R_thr; cv.surface_model = h->surface_model;
        }
        const uint32_t albedo0 = cv.albedo[0];            // monodisperse: the only class

        // ---- per-thread accumulators (flushed once per unit) ------------------------------------------------
        unsigned long long acc_esc = 0ull, acc_absp = 0ull, acc_abss = 0ull;
        uint32_t cnt_hist = 0u, cnt_ev = 0u, cnt_refl = 0u, max_ev = 0u;

        // ---- warp-uniform work-queue state ------------------------------------------------------------------
        unsigned long long chunk_base = 0ull;
        uint32_t chunk_pos = 0u, chunk_len = 0u;
        bool exhausted = false;

        // ---- lane state: one photon history (step (1)) -----------------------------------------
        bool alive = false;
        float T = 0.f, mu = -1.f, vt = 0.f;
        uint32_t w = 0u, n_sc = 0u, n_refl = 0u, flight = 0u, id_lo = 0u, id_hi = 0u;

        for (;;) {
            // ---------------- photon regeneration --------------------------------------------------------------
            const uint32_t need = __ballot_sync(FULL_MASK, !alive);
            if (need) {
                if (chunk_pos >= chunk_len && !exhausted) {
                    unsigned long long b = 0ull;
                    if (lane == 0) b = atomicAdd(P.next_id + u, (unsigned long long)P.chunk);
                    b = __shfl_sync(FULL_MASK, b, 0);
                    if (b >= P.n_photons) {
                        exhausted = true;
                    } else {
                        const unsigned long long left = P.n_photons - b;
                        chunk_base = b; chunk_pos = 0u;
                        chunk_len = left < (unsigned long long)P.chunk ? (uint32_t)left : P.chunk;
                    }
                }
                const uint32_t avail = chunk_len - chunk_pos;
                const uint32_t rank = __popc(need & lanemask_lt);
                if (!alive && rank < avail) {
                    const unsigned long long id = P.first_id + chunk_base + chunk_pos + rank;
                    id_lo = (uint32_t)id; id_hi = (uint32_t)(id >> 32);
                    alive = true; T = 0.f; mu = -1.f; vt = 0.f; w = kWOne; n_sc = 0u; n_refl = 0u; flight = 0u;
                    ++cnt_hist;
                }
                chunk_pos += min((uint32_t)__popc(need), avail);
                if (exhausted && !__any_sync(FULL_MASK, alive)) break;
            }

            int tally_bin = -1;                            // >= 0: this lane tallies w into that bin this iteration
            uint32_t tally_w = 0u;
            if (alive) {
                // ---------------- random numbers of this flight (step (3)) -------------------------------------
                uint32_t x0, x1, x2, x3;
                philox4x32_10(id_lo, id_hi, ud.stream, 2u * flight, P.key0, P.key1, x0, x1, x2, x3);
                uint32_t y0 = 0u, y1 = 0u;
                if (ANALOG) {
                    uint32_t y2, y3;
                    philox4x32_10(id_lo, id_hi, ud.stream, 2u * flight + 1u, P.key0, P.key1, y0, y1, y2, y3);
                }
                // ---------------- free flight: s = -ln(xi), xi in (0,1]; T' = T - mu s (Eq. 7/10) --------------
                const float xi = 2.0f - __uint_as_float(0x3F800000u | (x0 >> 9));
                const float s = __log2f(xi) * -0.69314718056f;
                const float Tn = fmaf(-mu, s, T);
                int fate = -1;
                if (Tn < 0.f) {
                    // ------------ leaves through the top (step (6)); Eq. 19 tally inside the aperture ----------
                    if (mu >= P.mu_aperture) {
                        const float fb = (vt - P.v_lo) * P.inv_dv;
                        fate = 5;
                        if (fb < 0.f) {
                            atomicAdd(&s_stats[ST_UNDER], (unsigned long long)w);
                        } else if (fb >= (float)P.n_bins) {
                            atomicAdd(&s_stats[ST_OVER], (unsigned long long)w);
                        } else {
                            tally_bin = (int)fb; tally_w = w; fate = 0;
                        }
                    } else {
                        acc_esc += w; fate = 1;
                    }
                } else {
                    float mu_new, v_here;
                    if (Tn >= cv.tau_ext) {
                        // -------- free surface: "ideal diffuse reflection", Doppler event at v_fs
                        v_here = cv.v_fs;
                        if (ANALOG) {
                            if (y1 >= cv.R_thr) { acc_abss += w; fate = 2; }
                        } else {
                            const uint32_t wn = mul_q31(w, cv.R_q31);
                            acc_abss += w - wn; w = wn;
                        }
                        const float xc = __uint2float_rn(x2) * 2.3283064365386963e-10f;
                        mu_new = cv.surface_model ? fast_sqrt(xc) : __cosf(1.57079632679f * xc);
                        T = cv.tau_ext;
                        if (fate < 0) { ++n_refl; ++cnt_refl; }
                    } else if (P.single_scatter_only && n_sc >= 1u) {
                        atomicAdd(&s_stats[ST_TRUNC], (unsigned long long)w);
                        fate = 4; mu_new = mu; v_here = 0.f;
                    } else {
                        // -------- particle interaction at depth Tn (steps (4)-(5)) ------------------------------
                        v_here = depth_velocity(cv, Tn);
                        uint32_t c = 0u, alb = albedo0;
                        if (POLY) {
                            for (uint32_t stp = 1u << cv.cls_steps; stp > 1u;) {     // thr padded with 0xffffffff
                                stp >>= 1;
                                if (cv.thr[c + stp - 1u] <= x1) c += stp;
                            }
                            c = min(c, cv.n_classes - 1u);
                            alb = cv.albedo[c];
                        }
                        ++cnt_ev;
                        if (ANALOG) {
                            if (y1 >= alb) { acc_absp += w; fate = 2; }          // alb = albedo threshold in analog mode
                        } else {
                            const uint32_t wn = mul_q31(w, alb);                 // Eq. 11 in expectation
                            acc_absp += w - wn; w = wn;
                        }
                        const float *M = cv.phase + c * cv.K1;
                        const uint32_t k = x2 >> cv.shiftK;
                        const float frac = __uint2float_rn(x2 - (k << cv.shiftK)) * cv.frac_scale;
                        const float m0 = M[k], m1 = M[k + 1u];
                        const float ct = fmaf(m1 - m0, frac, m0);                   // cos(theta) from D_K
                        const float cphi = __cosf(__int2float_rn((int)x3) * 1.46291807927e-9f);   // phi = 2 pi x3/2^32
                        const float sq = fast_sqrt(fmaxf((1.f - ct) * (1.f + ct) * (1.f - mu) * (1.f + mu), 0.f));
                        mu_new = fmaf(mu, ct, -cphi * sq);                           // z row of Eq. 16 (Eq. 17 at |mu| = 1)
                        mu_new = fminf(fmaxf(mu_new, -1.f), 1.f);
                        T = Tn;
                        if (fate < 0) ++n_sc;
                    }
                    if (fate < 0) {
                        vt = fmaf(0.5f * (mu_new - mu), v_here, vt);                 // Eq. 4
                        mu = mu_new;
                        ++flight;
                        if (P.max_events && n_sc >= P.max_events && w <= P.roulette_wcap) {   // Russian roulette
                            if (!ANALOG) {
                                uint32_t y2, y3;
                                philox4x32_10(id_lo, id_hi, ud.stream, 2u * flight - 1u, P.key0, P.key1, y0, y1, y2, y3);
                            }
                            if (y0 < P.roulette_thr) {
                                uint32_t wn = (uint32_t)__float2uint_rd(__uint2float_rd(w) * P.roulette_inv_p);
                                wn = max(min(wn, kWOne), w);
                                atomicAdd(&s_stats[ST_GAINED], (unsigned long long)(wn - w));
                                w = wn;
                            } else {
                                atomicAdd(&s_stats[ST_KILLED], (unsigned long long)w);
                                fate = 3;
                            }
                        }
                    }
                }
                if (fate >= 0) {                            // history over (step (7))
                    alive = false;
                    max_ev = max(max_ev, n_sc + n_refl);
                    if (TRACE) {
                        const unsigned long long idx = (((unsigned long long)id_hi << 32) | id_lo) - P.first_id;
                        pdv_trace_record r;
                        r.vt = vt; r.weight = (float)((double)w * kWScale); r.mu_exit = mu; r.fate = fate;
                        r.n_scatter = (int)n_sc; r.n_reflect = (int)n_refl;
                        P.trace[idx] = r;
                    }
                }
            }

            // ---------------- warp-aggregated tally into the block's private histogram (Eq. 19) ----------------
            const uint32_t tm = __ballot_sync(FULL_MASK, tally_bin >= 0);
            if (tm) {
                if (tally_bin >= 0) {
                    const uint32_t peers = __match_any_sync(tm, tally_bin);
                    unsigned long long sw = 0ull, sw2 = 0ull;
                    for (uint32_t m = peers; m; m &= m - 1u) {            // sum the weights of the lanes in my bin
                        const uint32_t wl = __shfl_sync(peers, tally_w, __ffs(m) - 1);
                        sw += wl;
                        sw2 += ((unsigned long long)wl * wl) >> 31;
                    }
                    if (lane == (uint32_t)(__ffs(peers) - 1)) {
                        atomicAdd(&s_hist[tally_bin], sw);
                        atomicAdd(&s_hist2[tally_bin], sw2);
                    }
                }
            }
        }

        // ---- block flush: per-thread counters -> warp -> shared -> global; histogram -> global ------------------
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc_esc += __shfl_xor_sync(FULL_MASK, acc_esc, o);
            acc_absp += __shfl_xor_sync(FULL_MASK, acc_absp, o);
            acc_abss += __shfl_xor_sync(FULL_MASK, acc_abss, o);
            cnt_hist += __shfl_xor_sync(FULL_MASK, cnt_hist, o);
            cnt_ev += __shfl_xor_sync(FULL_MASK, cnt_ev, o);
            cnt_refl += __shfl_xor_sync(FULL_MASK, cnt_refl, o);
            max_ev = max(max_ev, __shfl_xor_sync(FULL_MASK, max_ev, o));
        }
        if (lane == 0) {
            atomicAdd(&s_stats[ST_ESCAPED], acc_esc);
            atomicAdd(&s_stats[ST_ABS_PART], acc_absp);
            atomicAdd(&s_stats[ST_ABS_SURF], acc_abss);
            atomicAdd(&s_stats[ST_HISTORIES], (unsigned long long)cnt_hist);
            atomicAdd(&s_stats[ST_EVENTS], (unsigned long long)cnt_ev);
            atomicAdd(&s_stats[ST_REFLECT], (unsigned long long)cnt_refl);
            atomicMax(&s_stats[ST_MAXEV], (unsigned long long)max_ev);
        }
        __syncthreads();
        {
            unsigned long long *gh = P.hist + (size_t)u * P.n_bins, *gh2 = P.hist2 + (size_t)u * P.n_bins;
            unsigned long long det = 0ull;
            for (uint32_t i = tid; i < P.n_bins; i += blockDim.x) {
                const unsigned long long a = s_hist[i], b = s_hist2[i];
                if (a) { atomicAdd(gh + i, a); det += a; }
                if (b) atomicAdd(gh2 + i, b);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) det += __shfl_xor_sync(FULL_MASK, det, o);
            unsigned long long *gs = P.stats + (size_t)u * ST_COUNT;
            if (lane == 0 && det) atomicAdd(gs + ST_DETECTED, det);
            if (tid < ST_COUNT && tid != ST_DETECTED && s_stats[tid]) {
                if (tid == ST_MAXEV) atomicMax(gs + tid, s_stats[tid]);
                else atomicAdd(gs + tid, s_stats[tid]);
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------------------
template <bool POLY, bool ANALOG, bool TRACE>
static cudaError_t launch_t(const RunParams &rp, LaunchShape s, cudaStream_t st) {
    auto k = transport_kernel<POLY, ANALOG, TRACE>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, s.smem);
    if (e != cudaSuccess) return e;
    k<<<s.grid, s.block, s.smem, st>>>(rp);
    return cudaGetLastError();
}

template <bool POLY, bool ANALOG, bool TRACE>
static cudaError_t occ_t(int block, int smem, int *out) {
    auto k = transport_kernel<POLY, ANALOG, TRACE>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, k, block, smem);
}

#define PDV_DISPATCH(FN, ...)                                                      \
    do {                                                                           \
        if (trace) {                                                               \
            if (poly) return analog ? FN<true, true, true>(__VA_ARGS__) : FN<true, false, true>(__VA_ARGS__);    \
            return analog ? FN<false, true, true>(__VA_ARGS__) : FN<false, false, true>(__VA_ARGS__);            \
        }                                                                          \
        if (poly) return analog ? FN<true, true, false>(__VA_ARGS__) : FN<true, false, false>(__VA_ARGS__);      \
        return analog ? FN<false, true, false>(__VA_ARGS__) : FN<false, false, false>(__VA_ARGS__);              \
    } while (0)

cudaError_t launch_transport(const RunParams &rp, bool poly, bool analog, bool trace, LaunchShape shape, cudaStream_t st) {
    PDV_DISPATCH(launch_t, rp, shape, st);
}

cudaError_t transport_max_blocks_per_sm(bool poly, bool analog, bool trace, int block, int smem, int *out) {
    PDV_DISPATCH(occ_t, block, smem, out);
}

// ---- finalize: Q31 integers -> doubles (H12 input; stats) ------------------------------------------------------
__global__ void finalize_kernel(const unsigned long long *hist, const unsigned long long *hist2,
                                const unsigned long long *stats, uint32_t n_units, uint32_t n_bins,
                                double *out_hist, double *out_hist2, pdv_run_stats *out_stats) {
    const size_t n = (size_t)n_units * n_bins;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        out_hist[i] = (double)hist[i] * kWScale;
        if (out_hist2) out_hist2[i] = (double)hist2[i] * kWScale;
    }
    if (out_stats) {
        for (size_t u = blockIdx.x * (size_t)blockDim.x + threadIdx.x; u < n_units; u += (size_t)gridDim.x * blockDim.x) {
            const unsigned long long *s = stats + u * ST_COUNT;
            pdv_run_stats r;
            r.detected = (double)s[ST_DETECTED] * kWScale; r.underflow = (double)s[ST_UNDER] * kWScale;
            r.overflow = (double)s[ST_OVER] * kWScale; r.escaped = (double)s[ST_ESCAPED] * kWScale;
            r.absorbed_particles = (double)s[ST_ABS_PART] * kWScale; r.absorbed_surface = (double)s[ST_ABS_SURF] * kWScale;
            r.roulette_killed = (double)s[ST_KILLED] * kWScale; r.roulette_gained = (double)s[ST_GAINED] * kWScale;
            r.truncated = (double)s[ST_TRUNC] * kWScale;
            r.histories = s[ST_HISTORIES]; r.particle_events = s[ST_EVENTS]; r.surface_reflections = s[ST_REFLECT];
            r.max_events_in_history = s[ST_MAXEV];
            out_stats[u] = r;
        }
    }
}

cudaError_t launch_finalize(const unsigned long long *hist, const unsigned long long *hist2, const unsigned long long *stats,
                            uint32_t n_units, uint32_t n_bins, double *out_hist, double *out_hist2, pdv_run_stats *out_stats,
                            cudaStream_t st) {
    const size_t n = (size_t)n_units * n_bins;
    int grid = (int)((n + 255) / 256);
    if (grid < 1) grid = 1;
    if (grid > 1184) grid = 1184;
    finalize_kernel<<<grid, 256, 0, st>>>(hist, hist2, stats, n_units, n_bins, out_hist, out_hist2, out_stats);
    return cudaGetLastError();
}

// ---- spectrogram (H12): stack of instantaneous spectra, Eq. 19 --------------------------------------
__global__ void spectrogram_kernel(const double *hist, size_t n, double inv_n, double inv_dv, int scale, float floor_db,
                                   float *out) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double p = hist[i] * inv_n;
        float r;
        if (scale == 0) r = (float)p;
        else if (scale == 1) r = (float)(p * inv_dv);
        else r = p > 0.0 ? fmaxf(10.0f * log10f((float)p), floor_db) : floor_db;
        out[i] = r;
    }
}

cudaError_t launch_spectrogram(const double *hist, int n_snap, int n_bins, double inv_n, double inv_dv, int scale,
                               float floor_db, float *out, cudaStream_t st) {
    const size_t n = (size_t)n_snap * n_bins;
    if (n == 0) return cudaSuccess;
    int grid = (int)((n + 255) / 256);
    if (grid > 1184) grid = 1184;
    spectrogram_kernel<<<grid, 256, 0, st>>>(hist, n, inv_n, inv_dv, scale, floor_db, out);
    return cudaGetLastError();
}

// ---- issue-rate microbenchmarks: the FP32/SFU denominators of the roofline ---------------------
// Each thread runs 8 independent chains so the pipe, not the dependency latency, limits the rate.
__global__ void __launch_bounds__(512) ffma_peak_kernel(unsigned long long iters, float seed, float *sink,
                                                        unsigned long long *clk, unsigned long long *ns) {
    float a0 = seed, a1 = seed + 1.f, a2 = seed + 2.f, a3 = seed + 3.f, a4 = seed + 4.f, a5 = seed + 5.f, a6 = seed + 6.f,
          a7 = seed + 7.f;
    const float m = 0.999f + seed * 1e-9f, c = 1e-3f + seed;
    unsigned long long t0 = 0, g0 = 0;
    if (threadIdx.x == 0) { t0 = clock64(); asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0)); }
    for (unsigned long long i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            a0 = fmaf(a0, m, c); a1 = fmaf(a1, m, c); a2 = fmaf(a2, m, c); a3 = fmaf(a3, m, c);
            a4 = fmaf(a4, m, c); a5 = fmaf(a5, m, c); a6 = fmaf(a6, m, c); a7 = fmaf(a7, m, c);
        }
    }
    if (threadIdx.x == 0) {
        unsigned long long t1 = clock64(), g1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
        clk[blockIdx.x] = t1 - t0; ns[blockIdx.x] = g1 - g0;
    }
    const float r = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (r == 123.456f) sink[0] = r;
}

__global__ void __launch_bounds__(512) mufu_peak_kernel(unsigned long long iters, float seed, float *sink) {
    float a0 = seed + 1.5f, a1 = seed + 2.5f, a2 = seed + 3.5f, a3 = seed + 4.5f, a4 = seed + 5.5f, a5 = seed + 6.5f,
          a6 = seed + 7.5f, a7 = seed + 8.5f;
    for (unsigned long long i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            a0 = __log2f(a0) ; a1 = __log2f(a1); a2 = __log2f(a2); a3 = __log2f(a3);
            a4 = __log2f(a4); a5 = __log2f(a5); a6 = __log2f(a6); a7 = __log2f(a7);
            a0 = __cosf(a0); a1 = __cosf(a1); a2 = __cosf(a2); a3 = __cosf(a3);
            a4 = __cosf(a4); a5 = __cosf(a5); a6 = __cosf(a6); a7 = __cosf(a7);
        }
    }
    const float r = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (r == 123.456f) sink[0] = r;
}

cudaError_t launch_issue_peaks(double millis, double *ffma, double *mufu, double *mhz, int n_sm, cudaStream_t st) {
    float *sink = nullptr;
    unsigned long long *clk = nullptr, *ns = nullptr;
    const int grid = n_sm * 4, block = 512;
    cudaError_t e;
    if ((e = cudaMalloc(&sink, 4)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&clk, sizeof(unsigned long long) * grid * 2)) != cudaSuccess) { cudaFree(sink); return e; }
    ns = clk + grid;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    auto time_ffma = [&](unsigned long long it, float *ms) {
        cudaEventRecord(e0, st);
        ffma_peak_kernel<<<grid, block, 0, st>>>(it, 0.f, sink, clk, ns);
        cudaEventRecord(e1, st);
        cudaError_t r = cudaEventSynchronize(e1);
        if (r == cudaSuccess) cudaEventElapsedTime(ms, e0, e1);
        return r;
    };
    auto time_mufu = [&](unsigned long long it, float *ms) {
        cudaEventRecord(e0, st);
        mufu_peak_kernel<<<grid, block, 0, st>>>(it, 0.f, sink);
        cudaEventRecord(e1, st);
        cudaError_t r = cudaEventSynchronize(e1);
        if (r == cudaSuccess) cudaEventElapsedTime(ms, e0, e1);
        return r;
    };
    float ms = 0.f;
    unsigned long long it = 2000;
    e = time_ffma(it, &ms);                                   // warm-up + calibration
    if (e == cudaSuccess) e = time_ffma(it, &ms);
    if (e == cudaSuccess) {
        it = (unsigned long long)(it * millis / (ms > 1e-3f ? ms : 1e-3f)) + 1;
        e = time_ffma(it, &ms);
    }
    if (e == cudaSuccess) {
        if (ffma) *ffma = (double)grid * block * it * 128.0 / (ms * 1e-3);
        unsigned long long hc[2];
        cudaMemcpy(&hc[0], clk, 8, cudaMemcpyDeviceToHost);
        cudaMemcpy(&hc[1], ns, 8, cudaMemcpyDeviceToHost);
        if (mhz) *mhz = hc[1] ? (double)hc[0] / (double)hc[1] * 1e3 : 0.0;
        it = 500;
        e = time_mufu(it, &ms);
        if (e == cudaSuccess) e = time_mufu(it, &ms);
        if (e == cudaSuccess) {
            it = (unsigned long long)(it * millis / (ms > 1e-3f ? ms : 1e-3f)) + 1;
            e = time_mufu(it, &ms);
        }
        if (e == cudaSuccess && mufu) *mufu = (double)grid * block * it * 128.0 / (ms * 1e-3);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink); cudaFree(clk);
    return e;
}

}  // namespace pdv
