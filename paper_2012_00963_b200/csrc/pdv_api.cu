// pdv_api.cu -- the C-ABI of include/pdv.h: argument checking, cloud upload, workspace, launches, read-back.
// No arithmetic of the method lives here beyond packing the fp32/fixed-point device tables.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <mutex>
#include <new>
#include <string>
#include <thread>
#include <atomic>
#include <deque>
#include <vector>

#include "pdv_device.h"
#include "pdv_optics.hpp"

using namespace pdv;

struct pdv_cloud {
    HostCloud host;
    std::vector<unsigned char> blob;     // device image (host copy)
    mutable std::mutex mu;
    mutable unsigned char *d_blob = nullptr;
    mutable size_t d_bytes = 0;
    mutable int device = -1;
    // Recorded (by run_impl) behind every launch that reads d_blob.  It travels with the buffer into the cache when the cloud is
    // destroyed: the next cloud that takes the buffer waits for THIS event only -- i.e. for the runs that could still read the
    // old image -- instead of synchronising the whole device.  Created with the buffer, without timing.
    mutable cudaEvent_t last_read = nullptr;
    mutable bool read_pending = false;
    // Gas environment: the per-snapshot device images of this cloud for the snapshot times of its last run (host copies).  A
    // spectrogram that is run again for the same times (more histories, another seed: what bench.py's steps do) skips the host
    // build of its images (0.4 ms each); another list of times rebuilds them.  Guarded by mu.
    mutable std::vector<double> gas_t;
    mutable std::vector<std::vector<unsigned char>> gas_imgs;
};

namespace {

thread_local std::string g_err;

// Launch statistics and timing events of the last run of this host thread ON EACH STREAM it used (pdv_last_launch_info /
// pdv_launch_info_on_stream): two asynchronous runs on two streams keep their own events, so the first one's kernel time is not
// overwritten by the second.  A small table (the 16 most recently used streams of the thread); events are created once per slot.
struct LastLaunch {
    int n_kernels = 0; float ms = 0.f; int grid = 0, block = 0, smem = 0, variant = 0; bool pending = false;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int device = -1;
    cudaStream_t stream = nullptr;
    unsigned long long used = 0;                              // recency stamp; 0: slot never used
    // process teardown: the CUDA context may already be gone; the events are leaked rather than destroyed
};
thread_local LastLaunch g_launches[16];
thread_local unsigned long long g_launch_clock = 0;
thread_local LastLaunch *g_last_ptr = nullptr;                // the slot of the most recent run of this thread
#define g_last (*g_last_ptr)
#define g_ev (*g_last_ptr)

LastLaunch *launch_slot(cudaStream_t st, bool create) {
    LastLaunch *oldest = &g_launches[0];
    for (LastLaunch &l : g_launches) {
        if (l.used && l.stream == st) return &l;
        if (l.used < oldest->used) oldest = &l;
    }
    if (!create) return nullptr;
    oldest->stream = st;
    oldest->n_kernels = 0; oldest->ms = 0.f; oldest->pending = false; oldest->grid = oldest->block = oldest->smem = oldest->variant = 0;
    return oldest;                                            // its events, if any, are reused
}

// Pinned host staging buffer of this host thread for the read-back of a host-output run (one D2H copy at PCIe speed instead
// of several pageable ones); grown on demand, never shrunk.
struct PinnedStage {
    unsigned char *p = nullptr;
    size_t bytes = 0;
};
thread_local PinnedStage g_stage;

pdv_status fail(pdv_status s, const std::string &msg) { g_err = msg; return s; }
pdv_status cuda_fail(cudaError_t e, const char *what) {
    g_err = std::string(what) + ": " + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? PDV_E_NOMEM : PDV_E_CUDA;
}
#define CU(call, what) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, what); } while (0)

size_t align16(size_t v) { return (v + 15) & ~(size_t)15; }
uint32_t f2u(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }
float u2f(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }

uint32_t to_thr32(double p) {            // smallest integer t with t/2^32 >= p, clamped
    const double v = std::ceil(p * 4294967296.0);
    if (v <= 0.0) return 0u;
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    return (uint32_t)v;
}

// Device image of a cloud (gu == nullptr: the paper's vacuum, depth rows in v/2) or of one (cloud, snapshot) unit in a gas
// environment (gu: its tables; depth rows in the height zeta, per-bin class thresholds, per-class drag constants).
void build_blob(const HostCloud &h, std::vector<unsigned char> &blob, const GasUnit *gu = nullptr) {
    const int nc = h.n_classes, K = h.K, nd = h.n_depth;
    const std::vector<double> &T_src = gu ? gu->T_edge : h.T_edge;
    int steps = 0;
    while ((1 << steps) < nc) ++steps;
    const int n_pad = 1 << steps;
    // fp32 depth edges, T_0 = 0 at the cloud top ... T_nd = tau_ext at the free surface, non-decreasing
    // The device carries optical depths in units of ln 2: a flight is then  T' = T + mu lg2(xi)  -- the SFU's base-2 logarithm
    // without the multiplication by ln 2 (pdv_device.h).  Everything below (slopes, guide, tau_ext, closed form) is in those units.
    std::vector<float> Tf(nd + 1);
    for (int j = 0; j <= nd; ++j) Tf[j] = (float)(T_src[j] / 0.6931471805599453);
    Tf[0] = 0.f;
    for (int j = 1; j <= nd; ++j) if (Tf[j] < Tf[j - 1]) Tf[j] = Tf[j - 1];
    // depth rows (layout: pdv_device.h).  Half velocities: the Doppler update is  v~ += (mu' - mu) v/2  (Eq. 4).
    const double dv = (h.v_max - h.v_fs) / nd;
    std::vector<float> slope(nd + 1, 0.f);                    // d(v/2)/dT (gas: dzeta/dT) inside bin j; 0 for an empty bin
    for (int j = 0; j < nd; ++j) {
        const double dT = (double)Tf[j + 1] - (double)Tf[j];
        const double dy = gu ? gu->zeta_edge[j + 1] - gu->zeta_edge[j] : -0.5 * dv;
        slope[j] = dT > 0.0 ? (float)(dy / dT) : 0.f;
    }
    // guide over (float bits >> shift): the coarsest shift for which no cell straddles two bin edges
    float t_min = 0.f;
    for (int j = 1; j <= nd; ++j) if (Tf[j] > 0.f) { t_min = Tf[j]; break; }
    uint32_t base = 0, n_guide = 1, shift = 16, bisect = 0;
    std::vector<uint16_t> guide(1, (uint16_t)(nd - 1));       // tau_ext = 0: every lookup is at the surface
    if (t_min > 0.f) {
        bool ok = false;
        for (shift = 16; shift >= 10 && !ok; --shift) {
            const uint32_t top = f2u(Tf[nd]) >> shift;
            base = f2u(t_min) >> shift;
            n_guide = top - base + 1;
            if (n_guide > 16384u) break;
            guide.assign(n_guide, 0);
            int j = 0;
            ok = true;
            for (uint32_t i = 0; i < n_guide; ++i) {
                if (i > 0) {                                  // cell 0 also serves every T below it: j = 0
                    const float lo = u2f((base + i) << shift);
                    while (j + 1 <= nd - 1 && Tf[j + 1] <= lo) ++j;
                }
                guide[i] = (uint16_t)j;
                const float hi = u2f(((base + i + 1) << shift) - 1u);
                if (j + 2 < nd && !(Tf[j + 2] > hi)) ok = false;      // a second inner edge inside the cell (T_nd = tau_ext may be)
            }
            if (ok) break;
        }
        if (!ok) {                                            // pathological table: coarse guide unused, kernel bisects
            bisect = 1; shift = 16;
            base = f2u(t_min) >> shift;
            n_guide = (f2u(Tf[nd]) >> shift) - base + 1;
            guide.assign(n_guide, 0);
        }
    }
    DevCloudHeader hd;
    std::memset(&hd, 0, sizeof(hd));
    size_t off = sizeof(DevCloudHeader);
    // a one-class cloud carries its phase table and albedo twice: in a polydisperse launch without the class clamp (transport_kernel's
    // ALT) a class word of 0xffffffff picks "class 1" of such a cloud -- it must be the same class
    const int nc_tab = nc == 1 ? 2 : nc;
    hd.off_phase = (uint32_t)off;  off = align16(off + sizeof(float) * 2 * (size_t)nc_tab * K);
    off += 80;                                                // the block writes its Philox round keys in front of the rows (pdv_device.h)
    hd.off_rows = (uint32_t)off;   off = align16(off + sizeof(float) * 4 * (size_t)nd);
    hd.off_thr = (uint32_t)off;    off = align16(off + sizeof(uint32_t) * 2 * PDV_MAX_CLASSES);     // thr[32] | thr24[32] (pdv_device.h)
    hd.off_albedo = (uint32_t)off; off = align16(off + sizeof(float) * std::max(n_pad, 2));
    hd.off_albthr = (uint32_t)off; off = align16(off + sizeof(uint32_t) * std::max(n_pad, 2));
    hd.off_guide = (uint32_t)off;  off = align16(off + sizeof(uint16_t) * n_guide);
    // class thresholds first: the class guide is sized from them (layout: pdv_device.h)
    std::vector<uint32_t> thr_v(n_pad, 0xFFFFFFFFu);
    {
        double cum = 0.0;
        for (int c = 0; c < nc - 1; ++c) {
            cum += h.p_class[c];
            const double v = std::ceil(cum * 4294967296.0 - 0.5);     // x1 + 0.5 >= cum 2^32
            thr_v[c] = v <= 0.0 ? 0u : (v >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)v);
        }
    }
    auto cell_counts = [&](uint32_t sh, uint32_t g, int &below, int &inside) {
        const uint32_t first = g << sh, last = first | ((1u << sh) - 1u);
        below = inside = 0;
        for (int j = 0; j < nc - 1; ++j) {
            if (thr_v[j] <= first) ++below;
            else if (thr_v[j] <= last) ++inside;
        }
    };
    uint32_t cg_shift = 24;                                   // coarsest guide without a cell that holds two thresholds
    for (; cg_shift > 20; --cg_shift) {
        bool clean = true;
        for (uint32_t g = 0; g < (1u << (32 - cg_shift)) && clean; ++g) {
            int below, inside;
            cell_counts(cg_shift, g, below, inside);
            clean = inside <= 1;
        }
        if (clean) break;
    }
    const uint32_t n_cg = 1u << (32 - cg_shift);             // one class: 256 zeros (a polydisperse launch reads the guide of every cloud)
    hd.off_cguide = (uint32_t)off; off = align16(off + n_cg);
    hd.cguide_shift = cg_shift;
    if (gu) {
        hd.gas = 1; hd.gas_steps = (uint32_t)steps; hd.gas_inv_2t = (float)(0.5 / gu->t);
        hd.off_gthr = (uint32_t)off; off = align16(off + sizeof(uint32_t) * (size_t)nd * (n_pad + 1));      // rows of n_pad + 1 words
        hd.off_gcls = (uint32_t)off; off = align16(off + sizeof(float) * 2 * n_pad);
    }
    hd.blob_bytes = (uint32_t)off;
    hd.n_classes = nc; hd.K = K; hd.n_depth = nd; hd.n_guide = n_guide; hd.guide_base = base;
    hd.guide_shift = shift; hd.depth_bisect = bisect;
    if (h.depth_model == 1) {              // v/2 = v_fs/2 - (v_fs ln2 / (2 beta)) lg2(E + (1 - E) T / tau_ext)   (R26)
        const double E = std::exp(-h.beta * (h.v_max / h.v_fs - 1.0));
        hd.depth_bisect = 2;
        hd.an_c0 = (float)(0.5 * h.v_fs);
        hd.an_c1 = (float)(-0.5 * h.v_fs * 0.6931471805599453 / h.beta);
        hd.an_c2 = Tf[nd] > 0.f ? (float)E : 1.f;             // empty cloud: every event is at the surface, v = v_fs
        hd.an_c3 = Tf[nd] > 0.f ? (float)((1.0 - E) / (double)Tf[nd]) : 0.f;
    }
    hd.log2K = 0;
    while ((1 << hd.log2K) < K) ++hd.log2K;
    hd.tau_ext = Tf[nd]; hd.vh_fs = (float)(0.5 * h.v_fs);
    hd.R_f = (float)h.R;
    hd.omr_q31 = (float)((1.0 - (double)hd.R_f) * 2147483648.0);
    hd.R_thr = to_thr32(h.R);
    hd.surface_model = (uint32_t)h.surface_model;
    const uint32_t shiftK = 32u - hd.log2K;                   // K <= 4096: shiftK >= 20
    hd.frac_mask = 0xFFFu << (shiftK - 12u);
    blob.assign(off, 0);
    std::memcpy(blob.data(), &hd, sizeof(hd));
    float *ph = reinterpret_cast<float *>(blob.data() + hd.off_phase);
    std::vector<float> Mf(K + 1);
    for (int ct = 0; ct < nc_tab; ++ct) {
        const int c = ct < nc ? ct : 0;
        float prev = -1.f;
        for (int k = 0; k <= K; ++k) {
            float v = (float)h.phase[(size_t)c * (K + 1) + k];
            if (v < prev) v = prev;
            Mf[k] = v;
            prev = v;
        }
        for (int k = 0; k < K; ++k) {                         // (M[k], (M[k+1] - M[k]) 2^-shiftK): layout in pdv_device.h
            ph[2 * ((size_t)ct * K + k) + 0] = Mf[k];
            ph[2 * ((size_t)ct * K + k) + 1] = (float)std::ldexp((double)Mf[k + 1] - (double)Mf[k], -(int)shiftK);
        }
    }
    float *rows = reinterpret_cast<float *>(blob.data() + hd.off_rows);
    for (int j = 0; j < nd; ++j) {
        rows[4 * j + 0] = Tf[j + 1];
        rows[4 * j + 1] = gu ? (float)gu->zeta_edge[j + 1] : (j + 1 == nd ? hd.vh_fs : (float)(0.5 * (h.v_max - (j + 1) * dv)));
        rows[4 * j + 2] = slope[j];
        rows[4 * j + 3] = slope[j + 1];
    }
    uint32_t *thr = reinterpret_cast<uint32_t *>(blob.data() + hd.off_thr);
    float *alb = reinterpret_cast<float *>(blob.data() + hd.off_albedo);
    uint32_t *albt = reinterpret_cast<uint32_t *>(blob.data() + hd.off_albthr);
    for (int c = 0; c < PDV_MAX_CLASSES; ++c) {
        // thr24: for a class word whose low byte is replaced by 0x80 (first and second flight of a group, D2),
        //   thr <= (W & ~0xff | 0x80)   <=>   W >= 256 ceil((thr - 128) / 256),
        // so those flights compare the raw word W with thr24 and mask nothing
        const uint32_t t = c < n_pad ? thr_v[c] : 0xFFFFFFFFu;
        const uint64_t t24 = t < 128u ? 0u : ((uint64_t)t - 128u + 255u) / 256u;
        thr[c] = t;
        thr[PDV_MAX_CLASSES + c] = t24 >= (1u << 24) ? 0xFFFFFFFFu : (uint32_t)(t24 << 8);
    }
    for (int c = 0; c < n_pad; ++c) {
        const double om = c < nc ? h.k_sca[c] / h.k_ext[c] : 0.0;
        alb[c] = (float)std::min(std::max(om, 0.0), 1.0);
        albt[c] = to_thr32(om);
    }
    if (nc == 1) { alb[1] = alb[0]; albt[1] = albt[0]; }
    std::memcpy(blob.data() + hd.off_guide, guide.data(), sizeof(uint16_t) * n_guide);
    if (gu) {
        uint32_t *gt = reinterpret_cast<uint32_t *>(blob.data() + hd.off_gthr);
        for (int j = 0; j < nd; ++j)
            for (int c = 0; c < n_pad; ++c) {
                double v = 4294967295.0;
                if (c < nc - 1) v = std::ceil(gu->class_cum[(size_t)j * nc + c] * 4294967296.0 - 0.5);
                gt[(size_t)j * (n_pad + 1) + c] = v <= 0.0 ? 0u : (v >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)v);
            }
        float *gc = reinterpret_cast<float *>(blob.data() + hd.off_gcls);
        for (int c = 0; c < n_pad; ++c) {
            const double L = c < nc ? gu->L[c] : std::numeric_limits<double>::infinity();
            gc[2 * c + 0] = std::isinf(L) ? 0.f : (float)(0.5 * L / gu->t);
            gc[2 * c + 1] = std::isinf(L) ? 0.f : (float)(-1.0 / L);
        }
    }
    unsigned char *cg = blob.data() + hd.off_cguide;          // class guide (layout: pdv_device.h)
    for (uint32_t g = 0; nc > 1 && g < n_cg; ++g) {
        int below, inside;
        cell_counts(cg_shift, g, below, inside);
        // a cell above every threshold points at the LAST threshold (below it, so the compare is true and the class is nc - 1)
        // instead of at the padding behind it: the padding (0xffffffff) is then never compared, and the class needs no clamp
        if (below == nc - 1) below = nc - 2;
        cg[g] = (unsigned char)(below | (inside > 1 ? 0x80 : 0));
        if (inside > 1) ++hd.cguide_flagged;
    }
    std::memcpy(blob.data(), &hd, sizeof(hd));
}

// Device images of destroyed clouds are kept for the next cloud instead of going back to the driver: cudaFree was measured at
// 0.5 ... 750 ms for the 14 images of a sweep (it synchronises the device and may unmap memory).  Buffers come in power-of-two
// sizes from 64 KiB, so the image of one workload fits the buffer another left behind.  At most 256 buffers / 256 MiB; when
// that is full the OLDEST buffer goes back to the driver and the new one stays -- a loop that creates and destroys the same
// clouds never reaches cudaMalloc / cudaFree after its first turn, whatever ran before it (round 2: the 14-cloud sweep at the
// end of bench.py's default run took 426 ms per end-to-end step instead of 66, the cache being full of smaller buffers).
struct BlobCache {
    struct Entry { unsigned char *p; size_t bytes; int device; cudaEvent_t last_read; bool read_pending; };
    std::mutex mu;
    std::deque<Entry> free_list;                               // oldest first
    size_t total = 0;
    static size_t capacity_for(size_t bytes) {
        size_t cap = (size_t)64 << 10;
        while (cap < bytes) cap <<= 1;
        return cap;
    }
    bool take(size_t cap, int device, Entry &out) {           // a cached buffer of exactly this capacity; prefers one nobody reads any more
        std::lock_guard<std::mutex> lk(mu);
        long pick = -1;
        for (size_t i = free_list.size(); i-- > 0;)
            if (free_list[i].device == device && free_list[i].bytes == cap) {
                if (pick < 0) pick = (long)i;
                if (!free_list[i].read_pending || cudaEventQuery(free_list[i].last_read) == cudaSuccess) { pick = (long)i; break; }
            }
        if (pick < 0) { cudaGetLastError(); return false; }
        cudaGetLastError();                                   // cudaErrorNotReady of a query is not an error
        out = free_list[(size_t)pick];
        total -= cap;
        free_list.erase(free_list.begin() + pick);
        return true;
    }
    void give(const Entry &e) {
        std::vector<Entry> evict;
        {
            std::lock_guard<std::mutex> lk(mu);
            free_list.push_back(e);
            total += e.bytes;
            while (free_list.size() > 256 || total > ((size_t)256 << 20)) {
                evict.push_back(free_list.front());
                total -= free_list.front().bytes;
                free_list.pop_front();
            }
        }
        for (const Entry &q : evict) { cudaFree(q.p); if (q.last_read) cudaEventDestroy(q.last_read); }      // cudaFree waits for the device
    }
};
BlobCache g_blob_cache;

// Upload path of the cloud images: a pinned staging buffer per host thread and ONE library-owned non-blocking stream per device.
// pdv_cloud_create copies the image into the staging buffer, enqueues one cudaMemcpyAsync on that stream and waits for that
// stream only -- a kernel running on any other stream (a long pdv_mc_run with device outputs) neither delays the creation nor
// is delayed by it.  (Round 2: a blocking cudaMemcpy from pageable memory plus a cudaDeviceSynchronize on every reuse of a cached
// buffer: creating one cloud waited for every stream's work.)
thread_local PinnedStage g_upload_stage;
pdv_status upload_stream(int device, cudaStream_t *out) {
    static std::mutex mu;
    static cudaStream_t streams[64] = {nullptr};
    std::lock_guard<std::mutex> lk(mu);
    cudaStream_t &s = streams[device & 63];
    if (!s) CU(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking), "cudaStreamCreate(upload)");
    *out = s;
    return PDV_OK;
}

pdv_status ensure_on_device(const pdv_cloud *c, int device) {
    std::lock_guard<std::mutex> lk(c->mu);
    if (c->d_blob && c->device == device) return PDV_OK;
    if (c->d_blob) return fail(PDV_E_INVALID, "cloud was uploaded to another CUDA device");
    const size_t cap = BlobCache::capacity_for(c->blob.size());
    BlobCache::Entry e{nullptr, cap, device, nullptr, false};
    if (g_blob_cache.take(cap, device, e)) {
        // the buffer belonged to a destroyed cloud: the runs that may still read the old image (enqueued on any stream) must
        // be over before it is overwritten -- they end at the buffer's last_read event; nothing else is waited for
        if (e.read_pending) CU(cudaEventSynchronize(e.last_read), "cudaEventSynchronize(reuse of a cloud buffer)");
    } else {
        CU(cudaMalloc(&e.p, cap), "cudaMalloc(cloud tables)");
        cudaError_t ee = cudaEventCreateWithFlags(&e.last_read, cudaEventDisableTiming);
        if (ee != cudaSuccess) { cudaFree(e.p); return cuda_fail(ee, "cudaEventCreate(cloud buffer)"); }
    }
    auto give_back = [&]() { g_blob_cache.give(BlobCache::Entry{e.p, cap, device, e.last_read, false}); };
    cudaStream_t up = nullptr;
    pdv_status s = upload_stream(device, &up);
    if (s != PDV_OK) { give_back(); return s; }
    if (g_upload_stage.bytes < c->blob.size()) {
        if (g_upload_stage.p) cudaFreeHost(g_upload_stage.p);
        g_upload_stage.p = nullptr; g_upload_stage.bytes = 0;
        const size_t want = std::max(BlobCache::capacity_for(c->blob.size()), (size_t)1 << 18);
        cudaError_t ee = cudaMallocHost(&g_upload_stage.p, want);
        if (ee != cudaSuccess) { give_back(); return cuda_fail(ee, "cudaMallocHost(upload staging)"); }
        g_upload_stage.bytes = want;
    }
    std::memcpy(g_upload_stage.p, c->blob.data(), c->blob.size());
    cudaError_t ee = cudaMemcpyAsync(e.p, g_upload_stage.p, c->blob.size(), cudaMemcpyHostToDevice, up);
    if (ee == cudaSuccess) ee = cudaStreamSynchronize(up);    // the staging buffer is free again and the image is resident
    if (ee != cudaSuccess) { give_back(); return cuda_fail(ee, "cudaMemcpyAsync(cloud tables)"); }
    c->d_bytes = cap;                                         // capacity of the buffer (the image fills blob.size() of it)
    c->d_blob = e.p;
    c->last_read = e.last_read;
    c->read_pending = false;
    c->device = device;
    return PDV_OK;
}

// Device scratch of ONE call (tally workspace, unit table, output staging): allocated on the caller's stream from the device's
// stream-ordered pool and released, in stream order, behind the call's last kernel.  Two runs enqueued on different streams
// (output_on_device = 1) therefore never share cursors or tallies, and nothing a kernel in flight uses is ever freed or
// reused early.  The pool keeps its memory (release threshold = max), so after the first call this costs microseconds.
struct StreamScratch {
    unsigned char *p = nullptr;
    cudaStream_t st = nullptr;
    ~StreamScratch() { if (p) cudaFreeAsync(p, st); }
};
pdv_status scratch_alloc(size_t bytes, int device, cudaStream_t st, StreamScratch &out) {
    static std::mutex mu;
    static bool pool_ready[64] = {false};
    {
        std::lock_guard<std::mutex> lk(mu);
        if (!pool_ready[device & 63]) {
            cudaMemPool_t pool;
            CU(cudaDeviceGetDefaultMemPool(&pool, device), "cudaDeviceGetDefaultMemPool");
            unsigned long long keep = ~0ull;
            CU(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep), "cudaMemPoolSetAttribute");
            pool_ready[device & 63] = true;
        }
    }
    void *p = nullptr;
    CU(cudaMallocAsync(&p, std::max(bytes, (size_t)256), st), "cudaMallocAsync(workspace)");
    out.p = static_cast<unsigned char *>(p);
    out.st = st;
    return PDV_OK;
}

pdv_status ensure_events(int device, cudaStream_t st) {
    g_last_ptr = launch_slot(st, true);
    g_last.used = ++g_launch_clock;
    if (g_ev.e0 && g_ev.device != device) {
        cudaEventDestroy(g_ev.e0); cudaEventDestroy(g_ev.e1);
        g_ev.e0 = g_ev.e1 = nullptr;
    }
    if (!g_ev.e0) {
        CU(cudaEventCreate(&g_ev.e0), "cudaEventCreate");
        CU(cudaEventCreate(&g_ev.e1), "cudaEventCreate");
        g_ev.device = device;
    }
    return PDV_OK;
}

pdv_status stage_buffer(size_t bytes, unsigned char **out) {
    if (g_stage.bytes < bytes) {
        if (g_stage.p) cudaFreeHost(g_stage.p);
        g_stage.p = nullptr; g_stage.bytes = 0;
        const size_t want = std::max(bytes, (size_t)1 << 16);
        CU(cudaMallocHost(&g_stage.p, want), "cudaMallocHost(read-back staging)");
        g_stage.bytes = want;
    }
    *out = g_stage.p;
    return PDV_OK;
}

struct RunPlan {
    RunParams rp;
    LaunchShape shape;
    KernelVariant variant;
};

struct DeviceInfo { int n_sm = 0; size_t smem_optin = 0; bool valid = false; };
const DeviceInfo &device_info(int device) {           // cudaGetDeviceProperties costs milliseconds: ask once per device
    static std::mutex mu;
    static DeviceInfo info[64];
    std::lock_guard<std::mutex> lk(mu);
    DeviceInfo &d = info[device & 63];
    if (!d.valid) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, device) == cudaSuccess) d.n_sm = v;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, device) == cudaSuccess) d.smem_optin = (size_t)v;
        d.valid = d.n_sm > 0;
    }
    return d;
}

pdv_status check_opts(const pdv_run_opts *o) {
    if (!o) return fail(PDV_E_INVALID, "opts is NULL");
    if (o->struct_size != sizeof(pdv_run_opts)) return fail(PDV_E_INVALID, "opts->struct_size mismatch");
    if (o->n_bins < 1 || o->n_bins > PDV_MAX_BINS) return fail(PDV_E_INVALID, "n_bins out of range");
    if (!(o->v_hi > o->v_lo) || !std::isfinite(o->v_hi) || !std::isfinite(o->v_lo)) return fail(PDV_E_INVALID, "need v_hi > v_lo");
    if (!(o->aperture_sr > 0.0) || o->aperture_sr > 2.0 * 3.14159265358979323846 * (1 + 1e-12))
        return fail(PDV_E_INVALID, "aperture_sr not in (0, 2 pi]");
    if (o->mode != 0 && o->mode != 1) return fail(PDV_E_INVALID, "mode must be 0 or 1");
    if (o->max_events < 0) return fail(PDV_E_INVALID, "max_events < 0");
    if (o->max_events > 0 && !(o->roulette_survival > 0.0 && o->roulette_survival <= 1.0))
        return fail(PDV_E_INVALID, "roulette_survival not in (0,1]");
    if (o->threads_per_block < 0 || o->threads_per_block > 1024 || (o->threads_per_block % 32) != 0)
        return fail(PDV_E_INVALID, "threads_per_block must be a multiple of 32, <= 1024");
    if (o->launch_model != 0 && o->launch_model != 1) return fail(PDV_E_INVALID, "launch_model must be 0 or 1");
    if (o->blocks_per_sm < 0 || o->blocks_per_sm > 32) return fail(PDV_E_INVALID, "blocks_per_sm out of range");
    return PDV_OK;
}

// Estimated flights (particle events + reflections + the exit flight) of one history in a cloud of vertical optical thickness
// tau: only the RATIOS between the units of a launch matter (they place the blocks, see RunParams::block_start), and a wrong
// estimate costs a few more unit visits, never a wrong result.  Measured on the configs of BASELINE.json: 4.9 (tau 1.25), 9.8
// (1.87), 20 (4.1), 45 (9.3), 92 (18.7) -- the mean path of a slab grows linearly with its thickness.
double estimated_flights(double tau, double mean_albedo, const pdv_run_opts *o) {
    double f = 2.3 + 4.8 * tau;
    if (o->max_events > 0) { const double m = 1.25 * o->max_events; f = m * (1.0 - std::exp(-f / m)); }
    if (o->mode == 1) f = 1.0 / (1.0 / f + std::max(0.0, 1.0 - mean_albedo));      // analog histories end by absorption
    if (o->single_scatter_only) f = std::min(f, 3.0);
    return f;
}

// Fills the run parameters and the launch shape.  `ws` layout: next_id | hist | hist2 | stats | units.
pdv_status make_plan(const pdv_cloud *const *clouds, int n_clouds, int n_units, uint64_t n_photons, uint64_t seed,
                     const pdv_run_opts *o, bool trace, int device, RunPlan &plan, size_t max_blob) {
    RunParams &rp = plan.rp;
    std::memset(&rp, 0, sizeof(rp));
    rp.n_units = (uint32_t)n_units;
    rp.n_bins = (uint32_t)o->n_bins;
    rp.max_events = o->max_events > 0 ? (uint32_t)o->max_events : 0xFFFFFFFFu;
    const double p = o->max_events > 0 ? o->roulette_survival : 1.0;
    rp.roulette_thr = to_thr32(p);
    rp.roulette_p = (float)p;
    rp.roulette_inv_p = (float)(1.0 / p);
    rp.v_lo = (float)o->v_lo;
    rp.inv_dv = (float)((double)o->n_bins / (o->v_hi - o->v_lo));
    rp.mu_aperture = (float)(1.0 - o->aperture_sr / (2.0 * 3.14159265358979323846));
    rp.n_photons = n_photons;
    rp.first_id = o->first_photon_id;
    rp.launch_model = (uint32_t)o->launch_model;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) { rp.key0[r] = k0; rp.key1[r] = k1; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }

    KernelVariant &kv = plan.variant;
    kv.poly = false;
    for (int i = 0; i < n_clouds; ++i) kv.poly = kv.poly || clouds[i]->host.n_classes > 1;
    kv.analog = o->mode == 1;
    kv.sso = o->single_scatter_only != 0;
    kv.trace = trace;
    kv.roulette = o->max_events > 0;
    {   // long histories?  cost-weighted mean of the estimated flights per history over the clouds of the launch
        double sum = 0.0, sum2 = 0.0;
        for (int i = 0; i < n_clouds; ++i) {
            const HostCloud &h = clouds[i]->host;
            double om = 0.0;
            for (int c = 0; c < h.n_classes; ++c) om += h.p_class[c] * h.k_sca[c] / h.k_ext[c];
            const double f = estimated_flights(h.tau_ext, om, o);
            sum += f; sum2 += f * f;
        }
#ifndef PDV_ALT_MIN_FLIGHTS
#define PDV_ALT_MIN_FLIGHTS 22.0          /* experiment builds may override.  One 5 um cloud, 2e7 histories, plain / long-history kernel,
                                             ns per 1e3 flights at 9.8 / 14 / 18.5 / 23 / 32 / 46 / 93 flights per history:
                                             3.71 / 3.49 / 3.40 / 3.35 / 3.31 / 3.24 / 3.24  against  4.06 / 3.63 / 3.42 / 3.30 / 3.17 / 3.06 / 3.03 */
#endif
        kv.alt = sum > 0.0 && sum2 / sum >= PDV_ALT_MIN_FLIGHTS;
    }
    if (kv.poly) {       // several classes: alt = every class guide of the launch is clean
        kv.alt = true;
        for (int i = 0; i < n_clouds; ++i) {
            DevCloudHeader hd;
            std::memcpy(&hd, clouds[i]->blob.data(), sizeof(hd));
            kv.alt = kv.alt && hd.cguide_flagged == 0u;
        }
    }
    // dm 0: every cloud uses the one-probe depth table and the paper's surface law; 1: every cloud uses the closed-form
    // depth model and the paper's surface law; 2 (general kernel): anything else, decided per unit at run time
    {
        int n_closed = 0;
        bool odd = kv.sso || kv.trace || o->launch_model != 0;
        for (int i = 0; i < n_clouds; ++i) {
            DevCloudHeader hd;
            std::memcpy(&hd, clouds[i]->blob.data(), sizeof(hd));
            n_closed += hd.depth_bisect == 2u ? 1 : 0;
            odd = odd || hd.depth_bisect == 1u || hd.surface_model != 0u;
        }
        kv.dm = odd || (n_closed != 0 && n_closed != n_clouds) ? 2 : (n_closed ? 1 : 0);
        bool any_gas = false;
        for (int i = 0; i < n_clouds; ++i) any_gas = any_gas || clouds[i]->host.gas();
        if (any_gas) {                 // gas units: their own instantiations (dm 3), vacuum clouds of the launch ride along with L = infinity
            if (odd || n_closed) return fail(PDV_E_UNSUPPORTED, "a launch with a gas cloud supports neither single_scatter_only, pdv_mc_trace, launch_model 1, "
                                                                "surface_model 1, depth_model 1 nor a depth table that needs bisection");
            kv.dm = 3;
        }
    }

    const DeviceInfo &di = device_info(device);
    if (!di.valid) return fail(PDV_E_CUDA, "cannot query the CUDA device");
    const int smem = (int)(16 * (size_t)o->n_bins + max_blob);
    if ((size_t)smem > di.smem_optin)
        return fail(PDV_E_UNSUPPORTED, "cloud tables + histogram exceed the shared memory of one block");
    // 1024 resident threads per SM (64 registers each): two blocks of 512 when their shared memory fits twice, else one of 1024
    int block = o->threads_per_block, per_sm = 0;
    // polydisperse clouds: their tables leave room for one block per SM: PDV_LB_THREADS_POLY threads (pdv_device.h)
    if (kv.poly) block = block == 0 ? PDV_LB_THREADS_POLY : std::min(block, PDV_LB_THREADS_POLY);
    // one class: 1024 resident threads per SM either way.  Several units: two blocks of 512 when their shared memory fits twice
    // (finer grain where blocks move from unit to unit: config 4 123.9 ms against 135.3 with one block of 1024); ONE unit: one
    // block of 1024 (half as many stagings, flushes and warp pools: config 2 3.73 ms against 3.81)
    // long histories (the ALT instantiation of the production one-class kernel): PDV_LB_THREADS_LONG resident threads at 80 registers
    const int lb = !kv.poly && kv.alt && !kv.analog && !kv.sso && !kv.trace && kv.dm == 0 ? PDV_LB_THREADS_LONG : PDV_LB_THREADS;
    if (block == 0) block = (n_units > 1 && 2 * (size_t)(smem + 1024 + 18432) <= di.smem_optin + 1024) ? lb / 2 : lb;   // 18 KB: the kernel's static shared memory (warp queues)
    block = std::min(block, lb);
    // dynamic + STATIC shared memory (warp queues, keys, statistics: ~17 KB) must fit the opt-in limit of a block: without this
    // check a launch within 17 KB of the limit failed later, inside cudaFuncSetAttribute, with a misleading CUDA error
    size_t static_smem = 0;
    CU(transport_static_smem(kv, &static_smem), "cudaFuncGetAttributes(transport kernel)");
    if ((size_t)smem + static_smem > di.smem_optin) {
        char msg[200];
        std::snprintf(msg, sizeof(msg), "cloud tables + histogram (%d bytes) + the kernel's static shared memory (%zu) exceed the %zu bytes "
                      "of one block", smem, static_smem, di.smem_optin);
        return fail(PDV_E_UNSUPPORTED, msg);
    }
    {
        struct Key { KernelVariant v; int block, smem, device; };
        static std::mutex mu;
        static std::vector<std::pair<Key, int>> cache;       // occupancy queries are not free either
        std::lock_guard<std::mutex> lk(mu);
        for (const auto &e : cache)
            if (e.first.v.poly == kv.poly && e.first.v.analog == kv.analog && e.first.v.sso == kv.sso && e.first.v.trace == kv.trace && e.first.v.roulette == kv.roulette && e.first.v.dm == kv.dm && e.first.v.alt == kv.alt &&
                e.first.block == block && e.first.smem == smem && e.first.device == device) { per_sm = e.second; break; }
        if (per_sm == 0) {
            CU(transport_max_blocks_per_sm(kv, block, smem, &per_sm), "occupancy query");
            if (per_sm >= 1) cache.push_back({Key{kv, block, smem, device}, per_sm});
        }
    }
    if (per_sm < 1) return fail(PDV_E_UNSUPPORTED, "transport kernel does not fit on an SM with these tables");
    (void)static_smem;
    if (o->blocks_per_sm > 0) per_sm = std::min(per_sm, o->blocks_per_sm);
    long long grid = (long long)di.n_sm * per_sm;
    const unsigned long long total = n_photons * (unsigned long long)n_units;
    const long long useful = (long long)((total + block - 1) / block);       // one history per thread at least
    if (useful < grid) grid = std::max(1LL, useful);
    plan.shape.grid = (int)grid; plan.shape.block = block; plan.shape.smem = smem;
    return PDV_OK;
}

pdv_status run_impl(const pdv_cloud *const *clouds, int n_clouds, const double *t_snap, int n_snap, const uint32_t *unit_streams,
                    uint64_t n_photons, uint64_t seed, const pdv_run_opts *o, double *hist, double *hist2,
                    pdv_run_stats *stats, pdv_trace_record *records, void *cuda_stream) {
    const int n_units = n_clouds * n_snap;
    const bool trace = records != nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(PDV_E_CUDA, "no CUDA device available (this library has no CPU fallback)");
    }
    int device = 0;
    CU(cudaGetDevice(&device), "cudaGetDevice");
    size_t max_blob = 0;
    bool any_gas = false;
    for (int i = 0; i < n_clouds; ++i) {
        pdv_status s = ensure_on_device(clouds[i], device);
        if (s != PDV_OK) return s;
        max_blob = std::max(max_blob, clouds[i]->blob.size());
        any_gas = any_gas || clouds[i]->host.gas();
    }
    // Gas environment (R38): the depth tables depend on the snapshot time, so every (cloud, snapshot) unit gets its
    // own device image, built here and copied with the unit table
    std::vector<unsigned char> gas_images;
    std::vector<size_t> gas_off;
    if (any_gas) {
        if (!t_snap) return fail(PDV_E_UNSUPPORTED, "gas clouds need snapshot times (not available through pdv_mc_trace)");
        max_blob = 0;
        // the units are independent: built on parallel host threads (0.4 ms each; a 20-snapshot spectrogram 7.6 -> ~1 ms), and
        // kept with their cloud: the next run of the same cloud at the same snapshot times reuses them (pdv_cloud::gas_imgs)
        std::vector<const std::vector<unsigned char> *> imgs((size_t)n_units, nullptr);
        std::vector<std::unique_lock<std::mutex>> locks;      // the clouds' caches stay locked while this call reads them
        std::vector<int> todo;                                // units whose image must be built
        {
            std::vector<const pdv_cloud *> uniq(clouds, clouds + n_clouds);          // the same cloud may come twice in one launch
            std::sort(uniq.begin(), uniq.end());                                       // one lock order for every caller
            uniq.erase(std::unique(uniq.begin(), uniq.end()), uniq.end());
            for (const pdv_cloud *c : uniq) locks.emplace_back(c->mu);
            std::vector<const pdv_cloud *> seen;
            for (int i = 0; i < n_clouds; ++i) {
                const pdv_cloud *c = clouds[i];
                if (std::find(seen.begin(), seen.end(), c) != seen.end()) continue;
                seen.push_back(c);
                const bool hit = c->gas_t.size() == (size_t)n_snap && std::equal(c->gas_t.begin(), c->gas_t.end(), t_snap) &&
                                 c->gas_imgs.size() == (size_t)n_snap;
                if (!hit) {
                    c->gas_t.assign(t_snap, t_snap + n_snap);
                    c->gas_imgs.assign((size_t)n_snap, std::vector<unsigned char>());
                    for (int j = 0; j < n_snap; ++j) todo.push_back(i * n_snap + j);
                }
            }
            for (int u = 0; u < n_units; ++u) imgs[(size_t)u] = &clouds[u / n_snap]->gas_imgs[(size_t)(u % n_snap)];
        }
        if (!todo.empty()) {
            std::atomic<int> next{0};
            const int n_todo = (int)todo.size();
            auto work = [&]() {
                for (int k = next.fetch_add(1); k < n_todo; k = next.fetch_add(1)) {
                    const int u = todo[(size_t)k];
                    GasUnit gu;
                    build_gas_unit(clouds[u / n_snap]->host, t_snap[u % n_snap], gu);
                    build_blob(clouds[u / n_snap]->host, clouds[u / n_snap]->gas_imgs[(size_t)(u % n_snap)], &gu);
                }
            };
            const int n_thr = std::min(n_todo, (int)std::min(std::max(1u, std::thread::hardware_concurrency()), 16u));
            std::vector<std::thread> pool;
            for (int k = 1; k < n_thr; ++k) pool.emplace_back(work);
            work();
            for (auto &th : pool) th.join();
        }
        for (int u = 0; u < n_units; ++u) {
            const std::vector<unsigned char> &img = *imgs[(size_t)u];
            DevCloudHeader hd;
            std::memcpy(&hd, img.data(), sizeof(hd));
            if (hd.depth_bisect == 1u) return fail(PDV_E_UNSUPPORTED, "gas unit: depth table too irregular for the one-probe guide (use fewer n_depth_bins)");
            gas_off.push_back(gas_images.size());
            gas_images.insert(gas_images.end(), img.begin(), img.end());
            max_blob = std::max(max_blob, img.size());
        }
    }
    RunPlan plan;
    pdv_status s = make_plan(clouds, n_clouds, n_units, n_photons, seed, o, trace, device, plan, max_blob);
    if (s != PDV_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t nb = (size_t)o->n_bins;
    const int grid = plan.shape.grid;
    // scratch layout: [cursors | Q31 hist | Q31 hist2 | stats] (zeroed) [unit table | block starts] (one H2D copy)
    // [double hist | double hist2 | run stats] (host-output runs: one D2H copy)
    size_t off = 0;
    const size_t o_next = off;  off = align16(off + 8 * (size_t)n_units);
    const size_t o_hist = off;  off = align16(off + 8 * nb * n_units);
    const size_t o_hist2 = off; off = align16(off + 8 * nb * n_units);
    const size_t o_stats = off; off = align16(off + 8 * (size_t)ST_COUNT * n_units);
    const size_t zero_bytes = off;
    const size_t o_units = off; off = align16(off + sizeof(UnitDesc) * (size_t)n_units);
    const size_t o_start = off; off = align16(off + sizeof(uint32_t) * (size_t)grid);
    const size_t o_gas = off;   off = align16(off + gas_images.size());
    const size_t table_bytes = off - o_units;
    const size_t o_oh = off;    off = align16(off + 8 * nb * n_units);
    const size_t o_oh2 = off;   off = align16(off + (hist2 ? 8 * nb * n_units : 0));
    const size_t o_os = off;    off = align16(off + (stats ? sizeof(pdv_run_stats) * (size_t)n_units : 0));
    const size_t out_bytes = off - o_oh;
    StreamScratch scratch;
    if ((s = scratch_alloc(off, device, st, scratch)) != PDV_OK) return s;
    unsigned char *ws = scratch.p;
    if ((s = ensure_events(device, st)) != PDV_OK) return s;

    // ---- unit table: visiting order (descending estimated cost), where each block starts, guided chunk sizes per unit ----
    std::vector<unsigned char> table(table_bytes, 0);
    UnitDesc *units = reinterpret_cast<UnitDesc *>(table.data());
    uint32_t *block_start = reinterpret_cast<uint32_t *>(table.data() + (o_start - o_units));
    {
        std::vector<double> cost(n_units);
        for (int i = 0; i < n_clouds; ++i) {
            const HostCloud &h = clouds[i]->host;
            double om = 0.0;
            for (int c = 0; c < h.n_classes; ++c) om += h.p_class[c] * h.k_sca[c] / h.k_ext[c];
            const double f = estimated_flights(h.tau_ext, om, o);
            for (int j = 0; j < n_snap; ++j) cost[(size_t)i * n_snap + j] = f;
        }
        std::vector<uint32_t> ord(n_units);
        for (int k = 0; k < n_units; ++k) ord[k] = (uint32_t)k;
        std::stable_sort(ord.begin(), ord.end(), [&](uint32_t x, uint32_t y) { return cost[x] > cost[y]; });   // equal clouds keep their order
        double total = 0.0;
        for (int k = 0; k < n_units; ++k) total += cost[k];
        for (int i = 0; i < n_clouds; ++i)
            for (int j = 0; j < n_snap; ++j) {
                const size_t k = (size_t)i * n_snap + j;
                UnitDesc &u = units[k];
                u.cloud_blob = any_gas ? ws + o_gas + gas_off[k] : clouds[i]->d_blob;
                u.stream = unit_streams ? unit_streams[k] : (uint32_t)k;
                // threads expected on this unit: its share of the grid, at least one block
                const double threads = std::max(1.0, cost[k] / total * grid) * plan.shape.block;
                u.chunk = (uint32_t)std::min(std::max(std::floor((double)n_photons / (threads * 4.0)), 1.0), 128.0);
                u.chunk_per_remaining = (float)(1.0 / (2.0 * threads));
            }
        for (int k = 0; k < n_units; ++k) units[k].visit = ord[k];
        double cum = 0.0;                                          // cost line: unit ord[k] covers [cum, cum + cost)
        int k = 0;
        for (int b = 0; b < grid; ++b) {
            const double x = (b + 0.5) / grid * total;
            while (k + 1 < n_units && cum + cost[ord[k]] <= x) { cum += cost[ord[k]]; ++k; }
            block_start[b] = (uint32_t)k;
        }
    }
    if (any_gas) std::memcpy(table.data() + (o_gas - o_units), gas_images.data(), gas_images.size());
    pdv_trace_record *d_trace = nullptr;
    if (trace && n_photons) CU(cudaMalloc(&d_trace, sizeof(pdv_trace_record) * n_photons), "cudaMalloc(trace)");
    auto cleanup = [&]() { if (d_trace) cudaFree(d_trace); };
#define CUX(call, what) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { cleanup(); return cuda_fail(e_, what); } } while (0)

    CUX(cudaMemsetAsync(ws, 0, zero_bytes, st), "cudaMemsetAsync(workspace)");
    CUX(cudaMemcpyAsync(ws + o_units, table.data(), table_bytes, cudaMemcpyHostToDevice, st), "copy unit table");
    RunParams &rp = plan.rp;
    rp.units = reinterpret_cast<const UnitDesc *>(ws + o_units);
    rp.block_start = reinterpret_cast<const uint32_t *>(ws + o_start);
    rp.next_id = reinterpret_cast<unsigned long long *>(ws + o_next);
    rp.hist = reinterpret_cast<unsigned long long *>(ws + o_hist);
    rp.hist2 = reinterpret_cast<unsigned long long *>(ws + o_hist2);
    rp.stats = reinterpret_cast<unsigned long long *>(ws + o_stats);
    rp.trace = d_trace;

    g_last.n_kernels = 0; g_last.ms = 0.f; g_last.pending = false;
    g_last.grid = plan.shape.grid; g_last.block = plan.shape.block; g_last.smem = plan.shape.smem;
    {
        const KernelVariant &v = plan.variant;
        const bool alt = v.alt && !v.analog && !v.sso && !v.trace && v.dm == 0;          // the ALT instantiation exists and was launched
        g_last.variant = (v.poly ? 1 : 0) | (v.analog ? 2 : 0) | (v.sso ? 4 : 0) | (v.trace ? 8 : 0) | (v.roulette ? 16 : 0) | (alt ? 32 : 0) |
                         ((v.sso || v.trace ? 2 : v.dm) << 8);
    }
    CUX(cudaEventRecord(g_ev.e0, st), "cudaEventRecord");
    if (n_photons > 0) {
        CUX(launch_transport(rp, plan.variant, plan.shape, st), "transport kernel launch");
        g_last.n_kernels += 1;
    }
    CUX(cudaEventRecord(g_ev.e1, st), "cudaEventRecord");
    g_last.pending = true;               // elapsed time is read when the events have completed
    if (n_photons > 0)                   // whoever reuses a cloud's buffer after its destruction waits for this launch (ensure_on_device)
        for (int i = 0; i < n_clouds; ++i) {
            std::lock_guard<std::mutex> lk(clouds[i]->mu);
            if (clouds[i]->last_read && cudaEventRecord(clouds[i]->last_read, st) == cudaSuccess) clouds[i]->read_pending = true;
        }

    const bool dev_out = o->output_on_device != 0;
    double *oh = dev_out ? hist : reinterpret_cast<double *>(ws + o_oh);
    double *oh2 = hist2 ? (dev_out ? hist2 : reinterpret_cast<double *>(ws + o_oh2)) : nullptr;
    pdv_run_stats *os = stats ? (dev_out ? stats : reinterpret_cast<pdv_run_stats *>(ws + o_os)) : nullptr;
    CUX(launch_finalize(rp.hist, rp.hist2, rp.stats, (uint32_t)n_units, (uint32_t)nb, oh, oh2, os, st), "finalize kernel launch");
    g_last.n_kernels += 1;
    if (!dev_out) {
        // one D2H copy into this thread's pinned staging buffer; the caller's buffers are written only after everything
        // has succeeded, so they stay untouched on failure
        unsigned char *stage = nullptr;
        if ((s = stage_buffer(out_bytes, &stage)) != PDV_OK) { cleanup(); return s; }
        CUX(cudaMemcpyAsync(stage, ws + o_oh, out_bytes, cudaMemcpyDeviceToHost, st), "read back tallies");
        CUX(cudaStreamSynchronize(st), "transport kernel execution");
        if (trace && n_photons) CUX(cudaMemcpy(records, d_trace, sizeof(pdv_trace_record) * n_photons, cudaMemcpyDeviceToHost), "read back trace");
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, g_ev.e0, g_ev.e1) == cudaSuccess) g_last.ms = ms;
        g_last.pending = false;
        std::memcpy(hist, stage, 8 * nb * n_units);
        if (hist2) std::memcpy(hist2, stage + (o_oh2 - o_oh), 8 * nb * n_units);
        if (stats) std::memcpy(stats, stage + (o_os - o_oh), sizeof(pdv_run_stats) * n_units);
    } else if (trace) {
        CUX(cudaStreamSynchronize(st), "transport kernel execution");
        if (n_photons) CUX(cudaMemcpy(records, d_trace, sizeof(pdv_trace_record) * n_photons, cudaMemcpyDeviceToHost), "read back trace");
    }
    cleanup();
#undef CUX
    return PDV_OK;
}

// ---- pdv_mc_run_static: the workspace of a run as a fixed array inside the library (include/pdv.h) -----------------------------
// For host programs that cannot let this library allocate device memory (all HBM already belongs to their own arena, or their
// footprint must be fixed at load time).  The array is part of this module's device image: every GPU that loads the library
// holds PDV_STATIC_SCRATCH_BYTES of it until the process exits.
//
// `g_static_scratch` below is, in HOST code, only a handle for the runtime's symbol table -- not a device address.  Handing it
// to a kernel would make the kernel fault (or, on a system where the GPU can reach host memory, scribble over host data).  The
// device address is looked up once per device with cudaGetSymbolAddress while that device is current, and that pointer is
// what the kernels get.
}  // namespace
static __device__ __align__(256) unsigned char g_static_scratch[PDV_STATIC_SCRATCH_BYTES];
namespace {

pdv_status static_scratch_address(int device, unsigned char **out) {
    static std::mutex mu;
    static unsigned char *addr[64] = {nullptr};
    if (device < 0 || device >= 64) return fail(PDV_E_UNSUPPORTED, "pdv_mc_run_static: device ordinal above 63");
    std::lock_guard<std::mutex> lk(mu);
    if (!addr[device]) {                                      // set-up, once per device; `device` is the current device here
        void *p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_static_scratch), "cudaGetSymbolAddress(static scratch)");
        if (!p) return fail(PDV_E_CUDA, "cudaGetSymbolAddress(static scratch) returned a null address");
        addr[device] = static_cast<unsigned char *>(p);
    }
    *out = addr[device];
    return PDV_OK;
}

// Same work as run_impl for a vacuum launch with device outputs, with every device allocation taken out: the clouds must be
// resident already, the workspace is the static array, no timing events, no pinned staging.
pdv_status run_static_impl(const pdv_cloud *const *clouds, int n_clouds, int n_snap, const uint32_t *unit_streams,
                           uint64_t n_photons, uint64_t seed, const pdv_run_opts *o, double *hist, double *hist2,
                           pdv_run_stats *stats, void *cuda_stream) {
    const int n_units = n_clouds * n_snap;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(PDV_E_CUDA, "no CUDA device available (this library has no CPU fallback)");
    }
    int device = 0;
    CU(cudaGetDevice(&device), "cudaGetDevice");
    size_t max_blob = 0;
    for (int i = 0; i < n_clouds; ++i) {
        if (clouds[i]->host.gas())
            return fail(PDV_E_UNSUPPORTED, "pdv_mc_run_static: a cloud in a gas environment needs per-snapshot images that are uploaded per call; use pdv_mc_run");
        std::lock_guard<std::mutex> lk(clouds[i]->mu);
        if (!clouds[i]->d_blob || clouds[i]->device != device)
            return fail(PDV_E_INVALID, "pdv_mc_run_static: every cloud must already be resident on the current device "
                                       "(create it with pdv_cloud_create while this device is current; this call uploads nothing)");
        max_blob = std::max(max_blob, clouds[i]->blob.size());
    }
    RunPlan plan;
    pdv_status s = make_plan(clouds, n_clouds, n_units, n_photons, seed, o, false, device, plan, max_blob);
    if (s != PDV_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t nb = (size_t)o->n_bins;
    const int grid = plan.shape.grid;
    // layout inside the array: [cursors | Q31 hist | Q31 hist2 | stats] (cleared by every call) [unit table | block starts]
    size_t off = 0;
    const size_t o_next = off;  off = align16(off + 8 * (size_t)n_units);
    const size_t o_hist = off;  off = align16(off + 8 * nb * n_units);
    const size_t o_hist2 = off; off = align16(off + 8 * nb * n_units);
    const size_t o_stats = off; off = align16(off + 8 * (size_t)ST_COUNT * n_units);
    const size_t zero_bytes = off;
    const size_t o_units = off; off = align16(off + sizeof(UnitDesc) * (size_t)n_units);
    const size_t o_start = off; off = align16(off + sizeof(uint32_t) * (size_t)grid);
    const size_t table_bytes = off - o_units;
    if (off > (size_t)PDV_STATIC_SCRATCH_BYTES) {
        char msg[256];
        std::snprintf(msg, sizeof(msg), "pdv_mc_run_static: %d units x %d bins need %zu bytes of workspace, the static array holds %u "
                      "(split the run into fewer units per call, or use pdv_mc_run)", n_units, o->n_bins, off, (unsigned)PDV_STATIC_SCRATCH_BYTES);
        return fail(PDV_E_UNSUPPORTED, msg);
    }
    unsigned char *ws = nullptr;
    if ((s = static_scratch_address(device, &ws)) != PDV_OK) return s;

    // unit table: visiting order by descending estimated cost, block starts along the cost line, guided chunk sizes -- as
    // run_impl builds it.  It only schedules: no result depends on it.
    std::vector<unsigned char> table(table_bytes, 0);
    UnitDesc *units = reinterpret_cast<UnitDesc *>(table.data());
    uint32_t *block_start = reinterpret_cast<uint32_t *>(table.data() + (o_start - o_units));
    {
        std::vector<double> cost(n_units);
        for (int i = 0; i < n_clouds; ++i) {
            const HostCloud &h = clouds[i]->host;
            double om = 0.0;
            for (int c = 0; c < h.n_classes; ++c) om += h.p_class[c] * h.k_sca[c] / h.k_ext[c];
            const double f = estimated_flights(h.tau_ext, om, o);
            for (int j = 0; j < n_snap; ++j) cost[(size_t)i * n_snap + j] = f;
        }
        std::vector<uint32_t> ord(n_units);
        for (int k = 0; k < n_units; ++k) ord[k] = (uint32_t)k;
        std::stable_sort(ord.begin(), ord.end(), [&](uint32_t x, uint32_t y) { return cost[x] > cost[y]; });
        double total = 0.0;
        for (int k = 0; k < n_units; ++k) total += cost[k];
        for (int i = 0; i < n_clouds; ++i)
            for (int j = 0; j < n_snap; ++j) {
                const size_t k = (size_t)i * n_snap + j;
                UnitDesc &u = units[k];
                u.cloud_blob = clouds[i]->d_blob;
                u.stream = unit_streams ? unit_streams[k] : (uint32_t)k;
                const double threads = std::max(1.0, cost[k] / total * grid) * plan.shape.block;
                u.chunk = (uint32_t)std::min(std::max(std::floor((double)n_photons / (threads * 4.0)), 1.0), 128.0);
                u.chunk_per_remaining = (float)(1.0 / (2.0 * threads));
            }
        for (int k = 0; k < n_units; ++k) units[k].visit = ord[k];
        double cum = 0.0;
        int k = 0;
        for (int b = 0; b < grid; ++b) {
            const double x = (b + 0.5) / grid * total;
            while (k + 1 < n_units && cum + cost[ord[k]] <= x) { cum += cost[ord[k]]; ++k; }
            block_start[b] = (uint32_t)k;
        }
    }
    // the array still holds the previous call's cursors and tallies: clear them in stream order, then upload the table
    CU(cudaMemsetAsync(ws, 0, zero_bytes, st), "cudaMemsetAsync(static workspace)");
    CU(cudaMemcpyAsync(ws + o_units, table.data(), table_bytes, cudaMemcpyHostToDevice, st), "copy unit table");
    RunParams &rp = plan.rp;
    rp.units = reinterpret_cast<const UnitDesc *>(ws + o_units);
    rp.block_start = reinterpret_cast<const uint32_t *>(ws + o_start);
    rp.next_id = reinterpret_cast<unsigned long long *>(ws + o_next);
    rp.hist = reinterpret_cast<unsigned long long *>(ws + o_hist);
    rp.hist2 = reinterpret_cast<unsigned long long *>(ws + o_hist2);
    rp.stats = reinterpret_cast<unsigned long long *>(ws + o_stats);
    rp.trace = nullptr;
    if (n_photons > 0) {
        CU(launch_transport(rp, plan.variant, plan.shape, st), "transport kernel launch");
        for (int i = 0; i < n_clouds; ++i) {                  // recording an existing event allocates nothing
            std::lock_guard<std::mutex> lk(clouds[i]->mu);
            if (clouds[i]->last_read && cudaEventRecord(clouds[i]->last_read, st) == cudaSuccess) clouds[i]->read_pending = true;
        }
    }
    CU(launch_finalize(rp.hist, rp.hist2, rp.stats, (uint32_t)n_units, (uint32_t)nb, hist, hist2, stats, st), "finalize kernel launch");
    return PDV_OK;
}

}  // namespace

// =================================================================================================================
extern "C" {

const char *pdv_last_error(void) { return g_err.c_str(); }
const char *pdv_version(void) { return "pdv_b200 0.1 (sm_100a)"; }

pdv_status pdv_lognormal_classes(double d_median, double sigma_ln, int32_t n, double *diameter, double *weight,
                                 int32_t *n_out) {
    g_err.clear();
    int no = 0;
    pdv_status s = lognormal_classes(d_median, sigma_ln, n, diameter, weight, &no);
    if (s != PDV_OK) return fail(s, "pdv_lognormal_classes: need d_median > 0, sigma_ln >= 0, n >= 1, non-NULL outputs");
    if (n_out) *n_out = no;
    return PDV_OK;
}

pdv_status pdv_cloud_create(const pdv_cloud_params *params, pdv_cloud **out) {
    g_err.clear();
    if (!params || !out) return fail(PDV_E_INVALID, "params / out is NULL");
    if (params->struct_size != sizeof(pdv_cloud_params)) return fail(PDV_E_INVALID, "params->struct_size mismatch");
    pdv_cloud *c = new (std::nothrow) pdv_cloud;
    if (!c) return fail(PDV_E_NOMEM, "out of host memory");
    std::string err;
    pdv_status s;
    try {
        s = build_host_cloud(*params, c->host, err);
        if (s == PDV_OK) build_blob(c->host, c->blob);
    } catch (const std::bad_alloc &) {
        delete c;
        return fail(PDV_E_NOMEM, "out of host memory");
    }
    if (s != PDV_OK) { delete c; return fail(s, err); }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) == cudaSuccess && ndev > 0) {
        int device = 0;
        if (cudaGetDevice(&device) == cudaSuccess) {
            s = ensure_on_device(c, device);
            if (s != PDV_OK) { delete c; return s; }
        }
    } else {
        cudaGetLastError();          // host-only cloud: tables can be inspected, pdv_mc_run will refuse
    }
    *out = c;
    return PDV_OK;
}

void pdv_cloud_destroy(pdv_cloud *c) {
    if (!c) return;
    if (c->d_blob) g_blob_cache.give(BlobCache::Entry{c->d_blob, c->d_bytes, c->device, c->last_read, c->read_pending});
    delete c;
}

pdv_status pdv_cloud_get_info(const pdv_cloud *c, pdv_cloud_info *out) {
    g_err.clear();
    if (!c || !out) return fail(PDV_E_INVALID, "cloud / out is NULL");
    if (out->struct_size != sizeof(pdv_cloud_info)) return fail(PDV_E_INVALID, "out->struct_size mismatch");
    const HostCloud &h = c->host;
    out->n_classes = h.n_classes; out->n_phase_bins = h.K; out->n_depth_bins = h.n_depth;
    out->on_device = c->d_blob ? 1 : 0;
    out->tau_ext = h.tau_ext; out->kappa = h.kappa; out->sauter_diameter = h.sauter; out->v_fs = h.v_fs; out->v_max = h.v_max;
    double om = 0.0, gs = 0.0;
    for (int i = 0; i < h.n_classes; ++i) {
        const double a = h.k_sca[i] / h.k_ext[i];
        om += h.p_class[i] * a;
        gs += h.p_class[i] * a * h.g[i];
    }
    out->mean_albedo = om;
    out->mean_g = om > 0.0 ? gs / om : 0.0;
    return PDV_OK;
}

pdv_status pdv_estimated_flights(const pdv_cloud *c, const void *opts, double *out) {
    g_err.clear();
    if (!c || !out) return fail(PDV_E_INVALID, "cloud / out is NULL");
    pdv_run_opts o;
    std::memset(&o, 0, sizeof(o));
    if (opts) {
        const pdv_run_opts *in = static_cast<const pdv_run_opts *>(opts);
        if (in->struct_size != sizeof(pdv_run_opts)) return fail(PDV_E_INVALID, "opts->struct_size mismatch");
        o = *in;
        if (o.max_events > 0 && !(o.roulette_survival > 0.0 && o.roulette_survival <= 1.0)) return fail(PDV_E_INVALID, "roulette_survival not in (0,1]");
    }
    const HostCloud &h = c->host;
    double om = 0.0;
    for (int i = 0; i < h.n_classes; ++i) om += h.p_class[i] * h.k_sca[i] / h.k_ext[i];
    *out = estimated_flights(h.tau_ext, om, &o);
    return PDV_OK;
}

pdv_status pdv_cloud_get_tables(const pdv_cloud *c, double *k_ext, double *k_sca, double *g, double *p_class,
                                double *phase, double *T_edge) {
    g_err.clear();
    if (!c) return fail(PDV_E_INVALID, "cloud is NULL");
    const HostCloud &h = c->host;
    const size_t n = (size_t)h.n_classes;
    if (k_ext) std::memcpy(k_ext, h.k_ext.data(), 8 * n);
    if (k_sca) std::memcpy(k_sca, h.k_sca.data(), 8 * n);
    if (g) std::memcpy(g, h.g.data(), 8 * n);
    if (p_class) std::memcpy(p_class, h.p_class.data(), 8 * n);
    if (phase) std::memcpy(phase, h.phase.data(), 8 * h.phase.size());
    if (T_edge) std::memcpy(T_edge, h.T_edge.data(), 8 * h.T_edge.size());
    return PDV_OK;
}

pdv_status pdv_cloud_get_image(const pdv_cloud *c, pdv_image_layout *lay, unsigned char *image, size_t capacity) {
    g_err.clear();
    if (!c || !lay) return fail(PDV_E_INVALID, "cloud / layout is NULL");
    if (lay->struct_size != sizeof(pdv_image_layout)) return fail(PDV_E_INVALID, "layout->struct_size mismatch");
    if (c->host.gas()) return fail(PDV_E_INVALID, "a cloud in a gas environment has one image per snapshot, built by pdv_mc_run");
    DevCloudHeader hd;
    std::memcpy(&hd, c->blob.data(), sizeof(hd));
    lay->image_bytes = hd.blob_bytes; lay->n_classes = hd.n_classes; lay->n_phase_bins = hd.K; lay->log2_phase_bins = hd.log2K;
    lay->n_depth_bins = hd.n_depth; lay->off_phase = hd.off_phase; lay->off_rows = hd.off_rows; lay->off_thr = hd.off_thr;
    lay->off_thr24 = hd.off_thr + 4u * PDV_MAX_CLASSES; lay->off_albedo = hd.off_albedo; lay->off_guide = hd.off_guide;
    lay->n_guide = hd.n_guide; lay->guide_base = hd.guide_base; lay->guide_shift = hd.guide_shift; lay->depth_bisect = hd.depth_bisect;
    lay->off_cguide = hd.off_cguide; lay->cguide_cells = 1u << (32u - hd.cguide_shift); lay->cguide_shift = hd.cguide_shift;
    lay->cguide_flagged = hd.cguide_flagged; lay->frac_mask = hd.frac_mask;
    lay->tau_ext_ln2 = hd.tau_ext; lay->half_v_fs = hd.vh_fs; lay->surface_reflectivity = hd.R_f;
    if (image) std::memcpy(image, c->blob.data(), std::min(capacity, c->blob.size()));
    return PDV_OK;
}

pdv_status pdv_cloud_gas_tables(const pdv_cloud *c, double t, double *zeta_edge, double *T_edge, double *class_cum, double *drag_length) {
    g_err.clear();
    if (!c) return fail(PDV_E_INVALID, "cloud is NULL");
    if (!c->host.gas()) return fail(PDV_E_INVALID, "the cloud is in vacuum (gas_density = 0): it has no per-snapshot tables");
    if (!(t > 0.0) || !std::isfinite(t)) return fail(PDV_E_INVALID, "t must be > 0");
    GasUnit gu;
    build_gas_unit(c->host, t, gu);
    if (zeta_edge) std::memcpy(zeta_edge, gu.zeta_edge.data(), 8 * gu.zeta_edge.size());
    if (T_edge) std::memcpy(T_edge, gu.T_edge.data(), 8 * gu.T_edge.size());
    if (class_cum) std::memcpy(class_cum, gu.class_cum.data(), 8 * gu.class_cum.size());
    if (drag_length) std::memcpy(drag_length, gu.L.data(), 8 * gu.L.size());
    return PDV_OK;
}

pdv_status pdv_mc_run(const pdv_cloud *const *clouds, int32_t n_clouds, const double *t_snap, int32_t n_snap,
                      uint64_t n_photons, uint64_t seed, const pdv_run_opts *opts,
                      double *hist, double *hist2, pdv_run_stats *stats, void *cuda_stream) {
    g_err.clear();
    if (!clouds || n_clouds < 1) return fail(PDV_E_INVALID, "need at least one cloud");
    if (!t_snap || n_snap < 1) return fail(PDV_E_INVALID, "need at least one snapshot time");
    if (!hist) return fail(PDV_E_INVALID, "hist is NULL");
    pdv_status s = check_opts(opts);
    if (s != PDV_OK) return s;
    for (int i = 0; i < n_clouds; ++i) if (!clouds[i]) return fail(PDV_E_INVALID, "clouds[i] is NULL");
    for (int j = 0; j < n_snap; ++j) if (!(t_snap[j] > 0.0) || !std::isfinite(t_snap[j])) return fail(PDV_E_INVALID, "snapshot times must be > 0");
    if ((long long)n_clouds * n_snap > (1 << 20)) return fail(PDV_E_INVALID, "too many (cloud, snapshot) units");
    if (n_photons >= (1ull << 33)) return fail(PDV_E_INVALID, "n_photons per unit must be below 2^33: a Q31 tally in 64 bits wraps at the weight of 2^33 photons (split the run into id ranges)");
    if (opts->first_photon_id > (1ull << 62)) return fail(PDV_E_INVALID, "photon ids must stay below 2^63");
    return run_impl(clouds, n_clouds, t_snap, n_snap, opts->unit_streams, n_photons, seed, opts, hist, hist2, stats, nullptr, cuda_stream);
}

pdv_status pdv_mc_run_static(const pdv_cloud *const *clouds, int32_t n_clouds, const double *t_snap, int32_t n_snap,
                             uint64_t n_photons, uint64_t seed, const pdv_run_opts *opts,
                             double *hist, double *hist2, pdv_run_stats *stats, void *cuda_stream) {
    g_err.clear();
    if (!clouds || n_clouds < 1) return fail(PDV_E_INVALID, "need at least one cloud");
    if (!t_snap || n_snap < 1) return fail(PDV_E_INVALID, "need at least one snapshot time");
    if (!hist) return fail(PDV_E_INVALID, "hist is NULL");
    pdv_status s = check_opts(opts);
    if (s != PDV_OK) return s;
    if (!opts->output_on_device) return fail(PDV_E_INVALID, "pdv_mc_run_static writes device buffers only: set output_on_device = 1");
    for (int i = 0; i < n_clouds; ++i) if (!clouds[i]) return fail(PDV_E_INVALID, "clouds[i] is NULL");
    for (int j = 0; j < n_snap; ++j) if (!(t_snap[j] > 0.0) || !std::isfinite(t_snap[j])) return fail(PDV_E_INVALID, "snapshot times must be > 0");
    if ((long long)n_clouds * n_snap > (1 << 20)) return fail(PDV_E_INVALID, "too many (cloud, snapshot) units");
    if (n_photons >= (1ull << 33)) return fail(PDV_E_INVALID, "n_photons per unit must be below 2^33: a Q31 tally in 64 bits wraps at the weight of 2^33 photons (split the run into id ranges)");
    if (opts->first_photon_id > (1ull << 62)) return fail(PDV_E_INVALID, "photon ids must stay below 2^63");
    return run_static_impl(clouds, n_clouds, n_snap, opts->unit_streams, n_photons, seed, opts, hist, hist2, stats, cuda_stream);
}

pdv_status pdv_mc_trace(const pdv_cloud *cloud, uint32_t unit, uint64_t n_photons, uint64_t seed,
                        const pdv_run_opts *opts, double *hist, double *hist2, pdv_run_stats *stats,
                        pdv_trace_record *records, void *cuda_stream) {
    g_err.clear();
    if (!cloud || !hist || !records) return fail(PDV_E_INVALID, "cloud / hist / records is NULL");
    pdv_status s = check_opts(opts);
    if (s != PDV_OK) return s;
    if (opts->output_on_device) return fail(PDV_E_INVALID, "pdv_mc_trace writes host buffers only");
    if (n_photons > (1ull << 28)) return fail(PDV_E_INVALID, "pdv_mc_trace: at most 2^28 histories");
    const pdv_cloud *cl[1] = {cloud};
    return run_impl(cl, 1, nullptr, 1, &unit, n_photons, seed, opts, hist, hist2, stats, records, cuda_stream);
}

pdv_status pdv_spectrogram(const double *hist, int32_t n_snap, int32_t n_bins, uint64_t n_photons,
                           double v_lo, double v_hi, int32_t scale, float floor_db, float *out,
                           int32_t on_device, void *cuda_stream) {
    g_err.clear();
    if (!hist || !out) return fail(PDV_E_INVALID, "hist / out is NULL");
    if (n_snap < 0 || n_bins < 1 || n_photons == 0) return fail(PDV_E_INVALID, "need n_snap >= 0, n_bins >= 1, n_photons > 0");
    if (!(v_hi > v_lo)) return fail(PDV_E_INVALID, "need v_hi > v_lo");
    if (scale < 0 || scale > 2) return fail(PDV_E_INVALID, "scale must be 0, 1 or 2");
    if (n_snap == 0) return PDV_OK;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(PDV_E_CUDA, "no CUDA device available (this library has no CPU fallback)");
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)n_snap * n_bins;
    const double inv_n = 1.0 / (double)n_photons, inv_dv = (double)n_bins / (v_hi - v_lo);
    if (on_device) {
        CU(launch_spectrogram(hist, n_snap, n_bins, inv_n, inv_dv, scale, floor_db, out, st), "spectrogram kernel launch");
        return PDV_OK;
    }
    int device = 0;
    CU(cudaGetDevice(&device), "cudaGetDevice");
    StreamScratch scratch;
    pdv_status s = scratch_alloc(align16(8 * n) + 4 * n, device, st, scratch);
    if (s != PDV_OK) return s;
    unsigned char *ws = scratch.p;
    double *dh = reinterpret_cast<double *>(ws);
    float *dout = reinterpret_cast<float *>(ws + align16(8 * n));
    std::vector<float> tmp(n);
    CU(cudaMemcpyAsync(dh, hist, 8 * n, cudaMemcpyHostToDevice, st), "copy hist");
    CU(launch_spectrogram(dh, n_snap, n_bins, inv_n, inv_dv, scale, floor_db, dout, st), "spectrogram kernel launch");
    CU(cudaMemcpyAsync(tmp.data(), dout, 4 * n, cudaMemcpyDeviceToHost, st), "read back spectrogram");
    CU(cudaStreamSynchronize(st), "spectrogram kernel execution");
    std::memcpy(out, tmp.data(), 4 * n);
    return PDV_OK;
}

pdv_status pdv_spectrum_peaks(const double *hist, int32_t n_units, int32_t n_bins, uint64_t n_photons, double v_lo, double v_hi,
                              const double *v_fs, const pdv_peak_opts *opts, pdv_peak *out, int32_t on_device, void *cuda_stream) {
    g_err.clear();
    if (!hist || !v_fs || !out || !opts) return fail(PDV_E_INVALID, "hist / v_fs / opts / out is NULL");
    if (opts->struct_size != sizeof(pdv_peak_opts)) return fail(PDV_E_INVALID, "opts->struct_size mismatch");
    if (n_units < 0 || n_bins < 1 || n_bins > PDV_MAX_BINS) return fail(PDV_E_INVALID, "need n_units >= 0, 1 <= n_bins <= PDV_MAX_BINS");
    if (!(v_hi > v_lo) || !std::isfinite(v_hi) || !std::isfinite(v_lo)) return fail(PDV_E_INVALID, "need v_hi > v_lo");
    if (opts->smooth_half < 0 || opts->smooth_passes < 0 || opts->fit_half < 1 || opts->smooth_half > PDV_MAX_BINS ||
        opts->smooth_passes > 16 || opts->fit_half > PDV_MAX_BINS)
        return fail(PDV_E_INVALID, "need 0 <= smooth_half, 0 <= smooth_passes <= 16, 1 <= fit_half (windows at most PDV_MAX_BINS)");
    if (!(opts->x_max >= opts->x_min)) return fail(PDV_E_INVALID, "need x_max >= x_min");
    if (n_units == 0) return PDV_OK;
    if (!on_device)
        for (int i = 0; i < n_units; ++i)
            if (!(v_fs[i] > 0.0) || !std::isfinite(v_fs[i])) return fail(PDV_E_INVALID, "v_fs must be > 0");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(PDV_E_CUDA, "no CUDA device available (this library has no CPU fallback)");
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (on_device) {
        CU(launch_peaks(hist, n_units, n_bins, (double)n_photons, v_lo, v_hi, v_fs, *opts, out, st), "peak kernel launch");
        return PDV_OK;
    }
    int device = 0;
    CU(cudaGetDevice(&device), "cudaGetDevice");
    const size_t n = (size_t)n_units * n_bins;
    const size_t off_v = align16(8 * n), off_o = align16(off_v + 8 * (size_t)n_units);
    StreamScratch scratch;
    pdv_status s = scratch_alloc(off_o + sizeof(pdv_peak) * (size_t)n_units, device, st, scratch);
    if (s != PDV_OK) return s;
    unsigned char *ws = scratch.p;
    std::vector<pdv_peak> tmp(n_units);
    CU(cudaMemcpyAsync(ws, hist, 8 * n, cudaMemcpyHostToDevice, st), "copy hist");
    CU(cudaMemcpyAsync(ws + off_v, v_fs, 8 * (size_t)n_units, cudaMemcpyHostToDevice, st), "copy v_fs");
    CU(launch_peaks(reinterpret_cast<double *>(ws), n_units, n_bins, (double)n_photons, v_lo, v_hi,
                    reinterpret_cast<double *>(ws + off_v), *opts, reinterpret_cast<pdv_peak *>(ws + off_o), st), "peak kernel launch");
    CU(cudaMemcpyAsync(tmp.data(), ws + off_o, sizeof(pdv_peak) * (size_t)n_units, cudaMemcpyDeviceToHost, st), "read back peaks");
    CU(cudaStreamSynchronize(st), "peak kernel execution");
    std::memcpy(out, tmp.data(), sizeof(pdv_peak) * (size_t)n_units);
    return PDV_OK;
}

pdv_status pdv_phase_sampling_check(const pdv_cloud *cloud, int32_t class_index, uint64_t n_samples, uint64_t seed, int32_t n_bins,
                                    uint64_t *hist_table, uint64_t *hist_exact, pdv_phase_check *info, void *cuda_stream) {
    g_err.clear();
    if (!cloud || !hist_table || !hist_exact) return fail(PDV_E_INVALID, "cloud / hist_table / hist_exact is NULL");
    const HostCloud &h = cloud->host;
    if (class_index < 0 || class_index >= h.n_classes) return fail(PDV_E_INVALID, "class_index out of range");
    if (n_bins < 1 || n_bins > 4096) return fail(PDV_E_INVALID, "n_bins must be in [1, 4096]");
    if (h.phase_model != 0) return fail(PDV_E_UNSUPPORTED, "the cloud samples an isotropic phase function: there is no Mie function to reject on");
    // Mie series of the class (Eq. 12-14), coefficients premultiplied by (2n+1)/(n(n+1))
    const double x = 3.14159265358979323846 * h.diameter[class_index] / h.wavelength;
    std::vector<double> a_re, a_im, b_re, b_im;
    mie_coefficients(x, h.m_re, h.m_im, a_re, a_im, b_re, b_im);
    const int n_terms = (int)a_re.size();
    if (n_terms > 1024) return fail(PDV_E_UNSUPPORTED, "more than 1024 Mie terms");
    std::vector<float> coef(4 * (size_t)n_terms);
    std::vector<double> fa_re(n_terms), fa_im(n_terms), fb_re(n_terms), fb_im(n_terms);
    for (int n = 1; n <= n_terms; ++n) {
        const double f = (2.0 * n + 1.0) / (n * (n + 1.0));
        fa_re[n - 1] = f * a_re[n - 1]; fa_im[n - 1] = f * a_im[n - 1]; fb_re[n - 1] = f * b_re[n - 1]; fb_im[n - 1] = f * b_im[n - 1];
        coef[4 * (n - 1) + 0] = (float)fa_re[n - 1]; coef[4 * (n - 1) + 1] = (float)fa_im[n - 1];
        coef[4 * (n - 1) + 2] = (float)fb_re[n - 1]; coef[4 * (n - 1) + 3] = (float)fb_im[n - 1];
    }
    double i_max = 0.0;                                       // bound of the rejection: maximum over 20001 angles, plus 2 %
    const int n_grid = 20000;
    for (int i = 0; i <= n_grid; ++i) {
        const double mu = std::cos(3.14159265358979323846 * i / n_grid);
        double pp = 0.0, pc = 1.0, s1r = 0, s1i = 0, s2r = 0, s2i = 0;
        for (int n = 1; n <= n_terms; ++n) {
            const double tau = n * mu * pc - (n + 1.0) * pp;
            s1r += fa_re[n - 1] * pc + fb_re[n - 1] * tau; s1i += fa_im[n - 1] * pc + fb_im[n - 1] * tau;
            s2r += fa_re[n - 1] * tau + fb_re[n - 1] * pc; s2i += fa_im[n - 1] * tau + fb_im[n - 1] * pc;
            const double pn = ((2.0 * n + 1.0) * mu * pc - (n + 1.0) * pp) / n;
            pp = pc; pc = pn;
        }
        i_max = std::max(i_max, s1r * s1r + s1i * s1i + s2r * s2r + s2i * s2i);
    }
    i_max *= 1.02;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(PDV_E_CUDA, "no CUDA device available (this library has no CPU fallback)");
    }
    int device = 0;
    CU(cudaGetDevice(&device), "cudaGetDevice");
    pdv_status s = ensure_on_device(cloud, device);
    if (s != PDV_OK) return s;
    const DeviceInfo &di = device_info(device);
    if (!di.valid) return fail(PDV_E_CUDA, "cannot query the CUDA device");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t o_hist = align16(16 * (size_t)n_terms), o_sum = align16(o_hist + 16 * (size_t)n_bins), o_cnt = o_sum + 16;
    StreamScratch scratch;
    if ((s = scratch_alloc(o_cnt + 16, device, st, scratch)) != PDV_OK) return s;
    unsigned char *ws = scratch.p;
    DevCloudHeader hd;
    std::memcpy(&hd, cloud->blob.data(), sizeof(hd));
    const float2 *phase = reinterpret_cast<const float2 *>(cloud->d_blob + hd.off_phase) + (size_t)class_index * hd.K;
    CU(cudaMemcpyAsync(ws, coef.data(), 16 * (size_t)n_terms, cudaMemcpyHostToDevice, st), "copy Mie coefficients");
    CU(cudaMemsetAsync(ws + o_hist, 0, o_cnt + 16 - o_hist, st), "cudaMemsetAsync(sampling check)");
    CU(launch_phase_check(phase, hd.K, hd.log2K, hd.frac_mask, reinterpret_cast<const float4 *>(ws), n_terms, (float)i_max,
                          n_samples, seed, n_bins, reinterpret_cast<unsigned long long *>(ws + o_hist),
                          reinterpret_cast<double *>(ws + o_sum), reinterpret_cast<unsigned long long *>(ws + o_cnt), di.n_sm, st),
       "sampling-check kernel launch");
    std::vector<unsigned long long> hh(2 * (size_t)n_bins);
    double sums[2];
    unsigned long long cnts[2];
    CU(cudaMemcpyAsync(hh.data(), ws + o_hist, 16 * (size_t)n_bins, cudaMemcpyDeviceToHost, st), "read back counts");
    CU(cudaMemcpyAsync(sums, ws + o_sum, 16, cudaMemcpyDeviceToHost, st), "read back sums");
    CU(cudaMemcpyAsync(cnts, ws + o_cnt, 16, cudaMemcpyDeviceToHost, st), "read back counters");
    CU(cudaStreamSynchronize(st), "sampling-check kernel execution");
    for (int i = 0; i < n_bins; ++i) { hist_table[i] = hh[i]; hist_exact[i] = hh[(size_t)n_bins + i]; }
    if (info) {
        info->sum_cos_table = sums[0]; info->sum_cos_exact = sums[1]; info->i_max = (double)(float)i_max;
        info->n_trials = cnts[0]; info->n_bound_violations = cnts[1];
    }
    return PDV_OK;
}

pdv_status pdv_philox_blocks(const uint32_t *counters, int32_t n, uint64_t seed, uint32_t *out_static, uint32_t *out_shared,
                             uint32_t *out_param) {
    g_err.clear();
    if (n < 0 || n > (1 << 20) || (n > 0 && (!counters || !out_static || !out_shared || !out_param)))
        return fail(PDV_E_INVALID, "pdv_philox_blocks: need 0 <= n <= 2^20 and non-NULL buffers");
    if (n == 0) return PDV_OK;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(PDV_E_CUDA, "no CUDA device available (this library has no CPU fallback)");
    }
    uint32_t key0[10], key1[10];                              // the round keys as make_plan derives them from the seed
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) { key0[r] = k0; key1[r] = k1; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    const size_t bytes = 16 * (size_t)n;
    unsigned char *d = nullptr;
    CU(cudaMalloc(&d, 4 * bytes), "cudaMalloc(philox check)");
    cudaError_t e = cudaMemcpy(d, counters, bytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = launch_philox_check(key0, key1, reinterpret_cast<const uint4 *>(d), n, reinterpret_cast<uint4 *>(d + bytes),
                                                  reinterpret_cast<uint4 *>(d + 2 * bytes), reinterpret_cast<uint4 *>(d + 3 * bytes), nullptr);
    if (e == cudaSuccess) e = cudaMemcpy(out_static, d + bytes, bytes, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(out_shared, d + 2 * bytes, bytes, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(out_param, d + 3 * bytes, bytes, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(e, "philox check kernel");
    return PDV_OK;
}

pdv_status pdv_issue_peaks(double millis, double *ffma, double *mufu, double *mhz, int32_t *n_sm, void *cuda_stream) {
    g_err.clear();
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(PDV_E_CUDA, "no CUDA device available");
    }
    if (!(millis > 0.0) || millis > 5000.0) return fail(PDV_E_INVALID, "millis must be in (0, 5000]");
    int device = 0;
    CU(cudaGetDevice(&device), "cudaGetDevice");
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, device), "cudaGetDeviceProperties");
    if (n_sm) *n_sm = prop.multiProcessorCount;
    CU(launch_issue_peaks(millis, ffma, mufu, mhz, prop.multiProcessorCount, (cudaStream_t)cuda_stream), "issue-peak kernels");
    return PDV_OK;
}

static pdv_status launch_info_of(LastLaunch *l, int32_t *n_kernels, float *transport_ms, int32_t *grid, int32_t *block, int32_t *smem_bytes,
                                 int32_t *variant) {
    static const LastLaunch none;
    if (!l) l = const_cast<LastLaunch *>(&none);
    if (l->pending && l->e0 && l->e1) {          // output_on_device run: wait for that run's transport kernel only
        float ms = 0.f;
        if (cudaEventSynchronize(l->e1) == cudaSuccess && cudaEventElapsedTime(&ms, l->e0, l->e1) == cudaSuccess)
            l->ms = ms;
        else
            cudaGetLastError();
        l->pending = false;
    }
    if (n_kernels) *n_kernels = l->n_kernels;
    if (transport_ms) *transport_ms = l->ms;
    if (grid) *grid = l->grid;
    if (block) *block = l->block;
    if (smem_bytes) *smem_bytes = l->smem;
    if (variant) *variant = l->variant;
    return PDV_OK;
}

pdv_status pdv_last_launch_info(int32_t *n_kernels, float *transport_ms, int32_t *grid, int32_t *block, int32_t *smem_bytes, int32_t *variant) {
    return launch_info_of(g_last_ptr, n_kernels, transport_ms, grid, block, smem_bytes, variant);
}

pdv_status pdv_launch_info_on_stream(void *cuda_stream, int32_t *n_kernels, float *transport_ms, int32_t *grid, int32_t *block,
                                     int32_t *smem_bytes, int32_t *variant) {
    return launch_info_of(launch_slot((cudaStream_t)cuda_stream, false), n_kernels, transport_ms, grid, block, smem_bytes, variant);
}

}  // extern "C"
