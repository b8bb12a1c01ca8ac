// mi_api.cu -- the C-ABI boundary (include/mi.h) and the host runtime behind it: context,
// argument validation, transform generation (step a2), chunked launch planning, copy-back.
// No step of the path runs on the CPU except a2 (12 numbers per transform, in double).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <unordered_map>
#include <vector>

#include "mi_internal.h"

struct mi_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int32_t fd[3] = {0, 0, 0}, md[3] = {0, 0, 0};
    double fs[3] = {1, 1, 1}, ms[3] = {1, 1, 1};
    int nb = 0;
    float flo = 0, fhi = 1, mlo = 0, mhi = 1, fscale = 1, mscale = 1;
    int64_t nf = 0, nm = 0;
    uint8_t* d_fbins = nullptr;         // fixed bins (CANON-5), as mi_get_bins returns them
    uint8_t* d_fbins_ranked = nullptr;  // fixed bins replaced by their population rank
    uint8_t* d_rank = nullptr;          // 256: fixed bin -> rank
    int* d_rank_inv = nullptr;          // 256: rank -> fixed bin
    float* d_moving_pad = nullptr;      // replicate-padded moving volume (mx+2, my+2, mz+2)
    float4* d_moving_quad = nullptr;    // its yz-quads (generic kernel, trilinear): 16 bytes per padded voxel
    uint8_t* d_mbins = nullptr;
    uint32_t* d_mbins_quad = nullptr;   // yz-quads of the replicate-padded moving bins (partial-volume interpolation)
    int hot_mbin = 0;                   // most populated moving bin (partial-volume kernel's register-summed cell)
    uint16_t* d_fbins16_ranked = nullptr; // nbins > 256: fixed bins replaced by their population rank
    int* d_wrank_inv = nullptr;          // nbins > 256: rank -> fixed bin (kMaxBinsWide entries)
    uint8_t* d_wrow_used = nullptr;      // nbins > 256: 1 where a fixed bin holds voxels (rows the entropy pass reads)
    uint32_t* d_mask_bits = nullptr;    // NULL, or one bit per fixed voxel (mi_set_fixed_mask)
    unsigned rare_cap = 0;              // rare voxels without a mask (upper bound of n_rare)
    unsigned rare_alloc = 0;            // entries d_rare was allocated for
    bool wide = false;                  // nbins > 256: uint16 bins, global-memory histograms, generic kernel only
    uint16_t* d_fbins16 = nullptr;
    uint16_t* d_mbins16 = nullptr;
    int rows_smem = 0;                  // generic kernel: ranked fixed-bin rows in shared memory
    int gpitch = 0;                     // generic kernel: words per shared histogram row
    int ty_log2 = 3;                    // generic kernel: row tile = 8 (y) x 4 (z)
    // separable path (diagonal-matrix families)
    uint8_t* d_fb_pitched = nullptr;    // ranked fixed bins, [fnz][colpitch]
    int colpitch = 0;                   // fny*fnx rounded up to a multiple of kZColAlign
    int zpitch = 0;                     // words per shared histogram row of the z kernel
    int bin_mode = mi::kBinGeneral;     // moving-side binning variant of the z kernel (mi_internal.h)
    bool fuse_entropy = true;           // step a5 as the z kernel's epilogue when possible
    int zrows_smem = 0;                 // shared-memory histogram rows of the z kernel (dump row included)
    int zrows_real = 0;                 // fixed ranks counted in shared memory; ranks >= this are "rare"
    uint2* d_rare = nullptr;            // rare voxels (col, iz | rank << 16)
    unsigned n_rare = 0;
    void* d_X = nullptr;        size_t cap_X = 0;      // bytes
    void* d_XY = nullptr;       size_t cap_XY = 0;     // bytes
    uint8_t* d_colvalid = nullptr; size_t cap_cv = 0;
    float2* d_axis = nullptr;   size_t cap_axis = 0;   // 3 axes x nmax (scale, offset)
    size_t xy_budget = (size_t)12 << 30;               // bytes of xy-plane scratch per batch
    size_t sep_hist_budget = (size_t)3 << 30;          // bytes of histogram scratch per batch
    int tsallis_form = MI_TSALLIS_ADDITIVE;
    bool use_separable = true;
    bool separable_ok = true;                          // false: nbins > 256, or a fixed volume the z kernel cannot index
    int num_sms = 0;                                   // queried in mi_create
    size_t smem_optin = 48 * 1024;
    size_t hist_budget = (size_t)1 << 30;  // bytes of global histogram scratch per chunk
    // mi_set_option state (defaults = the measured optimum)
    int opt_zpad = 9, opt_zrows_max = 0, opt_bin_mode_max = mi::kBinFastPrescaled;
    int opt_gpad = 5, opt_gsmem_kb = 196, opt_unroll = 0, opt_match_any = 0, opt_gather = 1, opt_gthreads = 1024, opt_slab_mb = 16;
    unsigned long long* d_red_count = nullptr;         // histogram updates issued by the z kernel (last call)
    long long last_reds = 0;
    bool generic_has_rare = true;                      // a populated fixed-bin rank has no shared row in the generic kernel
    int bin_mode_natural = mi::kBinGeneral;            // what the data allows (mi_create)
    unsigned long long h_counts[256] = {};             // fixed-bin populations and ranks (nbins <= 256)
    uint8_t h_rank[256] = {};

    // scratch, grown on demand
    float* d_M = nullptr;      size_t cap_M = 0;       // transforms
    float* h_M = nullptr;      size_t cap_hM = 0;      // pinned staging
    uint32_t* d_hist = nullptr; size_t cap_hist = 0;   // bytes
    double* d_mi = nullptr;    size_t cap_mi = 0;      // doubles
    int64_t* d_nvalid = nullptr; size_t cap_nv = 0;
    double* d_q = nullptr;     size_t cap_q = 0;
    double* d_map = nullptr;   size_t cap_map = 0;
    int64_t* d_argmax = nullptr; size_t cap_am = 0;
    cudaEvent_t ev_staging = nullptr;  // h_M may be reused once this has completed
    bool staging_busy = false;

    std::string err;
    int last_path = 0;                  // 0 generic kernel, 1 separable kernels, 2 wide-histogram kernel (last call)
    float last_ms[5] = {0, 0, 0, 0, 0};
    int64_t last_launches[5] = {0, 0, 0, 0, 0};
};

namespace mi {

// Device memory comes from one library-level stream-ordered pool per device whose release threshold
// is unbounded: what a destroyed context frees stays cached for the next one (the multi-GB scratch of
// a map would otherwise be mapped and unmapped by the driver on every mi_create / mi_destroy cycle),
// until mi_release_cached_memory() trims it.
std::mutex g_pool_mutex;
cudaMemPool_t g_pools[64] = {};

cudaError_t device_pool(int dev, cudaMemPool_t* out) {
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    if (g_pools[dev] == nullptr) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        cudaError_t e = cudaMemPoolCreate(&pool, &props);
        if (e != cudaSuccess) return e;
        unsigned long long keep = ~0ULL;
        e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        if (e != cudaSuccess) { cudaMemPoolDestroy(pool); return e; }
        g_pools[dev] = pool;
    }
    *out = g_pools[dev];
    return cudaSuccess;
}

// Stream-ordered allocation on the context's stream (every use of the memory is ordered on it too).
// Sizes are rounded up to 2 MB, so every buffer starts on a 2 MB boundary whatever was allocated before it.
// This is a measured requirement, not tidiness: the z kernel streams three pitched arrays (xy planes, fixed bins,
// column flags) and its time depends on where they sit relative to each other -- one extra 8-byte allocation
// early in mi_create, which shifted everything behind it by 512 bytes, cost 21 % of the headline step (773 ms
// against 636 ms, the CTAs on three SMs running 8-22 % longer, round 2).
//
// In front of the pool sits an exact-size cache: a freed block is parked under (device, stream, bytes) and handed
// back to the next request with the same key; only a miss goes to the pool.  Why: the pool keeps freed memory, but
// it satisfies a request of a new size by splitting a bigger free block, and it rebuilds a big block later by
// re-mapping physical memory into a fresh virtual range -- measured at about 250 ms for the 12 GB of a C5 map's
// scratch, every create / map / destroy cycle, as soon as mi_create's allocation sequence no longer matched the
// previous cycle's frees by luck (round 3).  A create / map / destroy loop asks for the same
// sizes every time, so exact-size reuse never splits anything.  Reuse on the SAME stream needs no event: the
// block's earlier uses precede its new ones in stream order.  A pool allocation that fails with out-of-memory
// returns the parked blocks of that device to the pool and is retried; mi_release_cached_memory does the same.
struct ParkedBlock { void* p; size_t bytes; cudaStream_t s; };
struct LiveBlock { size_t bytes; int dev; };
std::mutex g_cache_mutex;
std::vector<ParkedBlock> g_parked[64];
std::unordered_map<void*, LiveBlock> g_live;

void unpark_all_locked(int dev) {   // g_cache_mutex held
    for (const ParkedBlock& b : g_parked[dev]) {
        if (cudaFreeAsync(b.p, b.s) != cudaSuccess) {   // the caller's stream may be gone by now
            cudaGetLastError();
            cudaFree(b.p);
        }
    }
    g_parked[dev].clear();
}
void unpark_all(int dev) {
    if (dev < 0 || dev >= 64) return;
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    unpark_all_locked(dev);
}

// Pinned staging buffers are parked the same way (by exact size): cudaMallocHost / cudaFreeHost map and unmap
// the buffer on the device and synchronise it, which a create / map / destroy loop should not pay every cycle.
// A buffer is parked only when no copy from it is in flight (mi_destroy synchronises the stream first).
struct ParkedHost { void* p; size_t bytes; };
std::vector<ParkedHost> g_parked_host;
cudaError_t pinned_alloc(void** p, size_t bytes) {
    {
        std::lock_guard<std::mutex> lock(g_cache_mutex);
        for (size_t i = g_parked_host.size(); i-- > 0;) {
            if (g_parked_host[i].bytes == bytes) {
                *p = g_parked_host[i].p;
                g_parked_host.erase(g_parked_host.begin() + (long)i);
                return cudaSuccess;
            }
        }
    }
    return cudaMallocHost(p, bytes);
}
void pinned_free(void* p, size_t bytes) {
    if (!p) return;
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    g_parked_host.push_back(ParkedHost{p, bytes});
}
void unpark_pinned() {
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    for (const ParkedHost& b : g_parked_host) cudaFreeHost(b.p);
    g_parked_host.clear();
}

cudaError_t dev_alloc(void** p, size_t bytes, int dev, cudaStream_t s) {
    cudaMemPool_t pool = nullptr;
    cudaError_t e = device_pool(dev, &pool);
    if (e != cudaSuccess) return e;
    constexpr size_t kGranule = (size_t)2 << 20;
    bytes = ((bytes ? bytes : 1) + kGranule - 1) / kGranule * kGranule;
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    std::vector<ParkedBlock>& parked = g_parked[dev];
    for (size_t i = parked.size(); i-- > 0;) {
        if (parked[i].bytes == bytes && parked[i].s == s) {
            *p = parked[i].p;
            parked.erase(parked.begin() + (long)i);
            g_live[*p] = LiveBlock{bytes, dev};
            return cudaSuccess;
        }
    }
    e = cudaMallocFromPoolAsync(p, bytes, pool, s);
    if (e == cudaErrorMemoryAllocation && !parked.empty()) {
        cudaGetLastError();
        unpark_all_locked(dev);
        cudaDeviceSynchronize();   // the frees were queued on their own streams
        e = cudaMallocFromPoolAsync(p, bytes, pool, s);
    }
    if (e == cudaSuccess) g_live[*p] = LiveBlock{bytes, dev};
    return e;
}
void dev_free(void* p, cudaStream_t s) {
    if (!p) return;
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    const auto it = g_live.find(p);
    if (it == g_live.end()) {   // not from dev_alloc: cannot happen inside the library
        cudaFreeAsync(p, s);
        return;
    }
    g_parked[it->second.dev].push_back(ParkedBlock{p, it->second.bytes, s});
    g_live.erase(it);
}

int sm_count() {
    static int cached[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return 1; }
    if (cached[dev] == 0) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v < 1) { cudaGetLastError(); return 1; }
        cached[dev] = v;
    }
    return cached[dev];
}

thread_local std::string g_thread_error;
void set_thread_error(const std::string& msg) { g_thread_error = msg; }
bool is_host_pointer(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        cudaGetLastError();
        return true;
    }
    return !(at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged);
}

}  // namespace mi

namespace {

using mi::dev_alloc;
using mi::dev_free;

struct DeviceGuard {
    int prev = -1;
    bool ok = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; cudaGetLastError(); }
        ok = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

mi_status fail(mi_ctx* c, mi_status s, const std::string& msg) {
    if (c) c->err = msg; else mi::set_thread_error(msg);
    return s;
}
mi_status cuda_fail(mi_ctx* c, cudaError_t e, const char* where) {
    cudaGetLastError();
    const mi_status s = (e == cudaErrorMemoryAllocation) ? MI_ERR_OUT_OF_MEMORY : MI_ERR_CUDA;
    return fail(c, s, std::string(where) + ": " + cudaGetErrorString(e));
}
#define MI_CUDA(ctx, call)                                           \
    do {                                                             \
        cudaError_t e__ = (call);                                    \
        if (e__ != cudaSuccess) return cuda_fail((ctx), e__, #call); \
    } while (0)

bool is_host_ptr(const void* p) { return mi::is_host_pointer(p); }

template <typename T>
mi_status grow(mi_ctx* c, T** p, size_t* cap, size_t need) {
    if (need <= *cap) return MI_OK;
    if (*p) { dev_free(*p, c->stream); *p = nullptr; *cap = 0; }
    MI_CUDA(c, dev_alloc(reinterpret_cast<void**>(p), need * sizeof(T), c->device, c->stream));
    *cap = need;
    return MI_OK;
}

// interpolation argument of the compute entry points; partial volume needs the shared-memory path
mi_status validate_interp(mi_ctx* c, int interp) {
    if (interp != MI_INTERP_NEAREST && interp != MI_INTERP_TRILINEAR && interp != MI_INTERP_PARTIAL_VOLUME)
        return fail(c, MI_ERR_INVALID_ARG, "unknown interpolation");
    if (interp == MI_INTERP_PARTIAL_VOLUME && c->wide)
        return fail(c, MI_ERR_UNSUPPORTED, "partial-volume interpolation needs nbins <= 256");
    return MI_OK;
}

bool finite3(const double v[3]) { return std::isfinite(v[0]) && std::isfinite(v[1]) && std::isfinite(v[2]); }

struct EventTimer {
    // accumulates device time per class over a call; events are recorded on the context's stream
    struct Span { cudaEvent_t a, b; int cls; };
    std::vector<Span> spans;
    std::vector<size_t> open;   // spans may nest (class 4 inside class 1)
    cudaStream_t s;
    explicit EventTimer(cudaStream_t st) : s(st) {}
    void begin(int cls) {
        Span sp{nullptr, nullptr, cls};
        cudaEventCreate(&sp.a);
        cudaEventCreate(&sp.b);
        cudaEventRecord(sp.a, s);
        open.push_back(spans.size());
        spans.push_back(sp);
    }
    void end() {
        cudaEventRecord(spans[open.back()].b, s);
        open.pop_back();
    }
    void collect(float ms[5]) {
        for (auto& sp : spans) {
            float t = 0.f;
            if (cudaEventSynchronize(sp.b) == cudaSuccess && cudaEventElapsedTime(&t, sp.a, sp.b) == cudaSuccess)
                ms[sp.cls] += t;
            cudaEventDestroy(sp.a);
            cudaEventDestroy(sp.b);
        }
        spans.clear();
        cudaGetLastError();
    }
    ~EventTimer() {
        for (auto& sp : spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
    }
};

mi_status validate_q(mi_ctx* c, const double* q, int32_t nq) {
    if (nq < 0) return fail(c, MI_ERR_INVALID_ARG, "nq < 0");
    if (nq > 0 && q == nullptr) return fail(c, MI_ERR_INVALID_ARG, "q is NULL but nq > 0");
    // q <= 32: the kernels accumulate sum c^q = sum exp(q ln c) over integer counts c < 2^31 and scale by
    // N^-q afterwards; 32 ln 2^31 = 687.6 stays below the double overflow threshold (709.78) with room for
    // the 2^16 terms of a histogram, so no q in range can overflow (include/mi.h documents the bound)
    for (int i = 0; i < nq; ++i)
        if (!(std::isfinite(q[i]) && q[i] > 0.0 && q[i] <= 32.0)) return fail(c, MI_ERR_INVALID_ARG, "q must be finite, > 0 and <= 32");
    return MI_OK;
}

// Launch layout derived from the options (mi_set_option) and the data: shared-memory rows and row
// pitches of both histogram kernels, the z kernel's binning variant and -- for the separable path --
// the pitched fixed bins with the rare-voxel list, which depend on the row count and on the
// fixed-voxel mask.  Called by mi_create, mi_set_option and mi_set_fixed_mask; the device is current.
// The quad copies of the moving side are big -- 16 B per padded voxel for the float yz-quads the generic trilinear
// kernels gather from, 4 B for the bin quads of partial volume -- and a context that only ever runs separable
// (translation / scale) maps or nearest-neighbour needs neither.  They are built on the first call that does.
mi_status ensure_moving_quads(mi_ctx* c, bool float_quads, bool bin_quads) {
    cudaStream_t s = c->stream;
    const size_t npad = ((size_t)c->md[0] + 2) * ((size_t)c->md[1] + 2) * ((size_t)c->md[2] + 2);
    if (float_quads && c->d_moving_quad == nullptr) {
        cudaError_t e = dev_alloc((void**)&c->d_moving_quad, npad * sizeof(float4), c->device, s);
        if (e != cudaSuccess) { c->d_moving_quad = nullptr; return cuda_fail(c, e, "cudaMalloc moving quads"); }
        e = mi::launch_quad_build(c->d_moving_pad, c->d_moving_quad, c->md[0], c->md[1], c->md[2], s);
        if (e != cudaSuccess) { dev_free(c->d_moving_quad, s); c->d_moving_quad = nullptr; return cuda_fail(c, e, "build moving quads"); }
    }
    if (bin_quads && c->d_mbins_quad == nullptr) {
        cudaError_t e = dev_alloc((void**)&c->d_mbins_quad, npad * sizeof(uint32_t), c->device, s);
        if (e != cudaSuccess) { c->d_mbins_quad = nullptr; return cuda_fail(c, e, "cudaMalloc moving bin quads"); }
        e = mi::launch_bins_quad_build(c->d_mbins, c->d_mbins_quad, c->md[0], c->md[1], c->md[2], s);
        if (e != cudaSuccess) { dev_free(c->d_mbins_quad, s); c->d_mbins_quad = nullptr; return cuda_fail(c, e, "build moving bin quads"); }
    }
    return MI_OK;
}

mi_status plan_layout(mi_ctx* c) {
    cudaStream_t s = c->stream;
    // generic kernel: the gathers live in L1, which is what the shared histogram leaves of the SM's
    // 256 KB; above 196 KB of shared memory the next carve-out step leaves only 28 KB
    size_t gsmem = (size_t)c->opt_gsmem_kb << 10;
    if (gsmem > c->smem_optin) gsmem = c->smem_optin;
    c->gpitch = c->nb + c->opt_gpad;
    c->rows_smem = mi::hist_rows_in_smem(c->nb, c->gpitch, gsmem);
    if (c->rows_smem < 1) return fail(c, MI_ERR_UNSUPPORTED, "device has too little shared memory");
    if (c->wide) return MI_OK;
    c->generic_has_rare = false;
    for (int a = 0; a < 256; ++a)
        if ((int)c->h_rank[a] >= c->rows_smem && c->h_counts[a] > 0) c->generic_has_rare = true;
    c->bin_mode = c->bin_mode_natural < c->opt_bin_mode_max ? c->bin_mode_natural : c->opt_bin_mode_max;
    // bank of histogram word (a, b) = (a*pad + b) mod 32: an odd pad walks the rows over all banks
    c->zpitch = c->nb + c->opt_zpad;
    c->zrows_smem = mi::zhist_rows_in_smem(c->nb, c->zpitch, c->fd[2], c->md[2] + 2, c->smem_optin);
    if (c->opt_zrows_max >= 2 && c->opt_zrows_max < c->zrows_smem) c->zrows_smem = c->opt_zrows_max;
    if (!c->separable_ok || c->zrows_smem < 2) return MI_OK;
    // the separable path keeps ranks < zrows_real in shared memory; if not every bin fits, the last
    // shared row becomes a dump row and the voxels of the rare ranks go to a list
    c->zrows_real = c->zrows_smem > c->nb ? c->nb : c->zrows_smem - 1;
    unsigned long long n_rare = 0;
    for (int a = 0; a < 256; ++a)
        if ((int)c->h_rank[a] >= c->zrows_real) n_rare += c->h_counts[a];
    if (c->d_rare == nullptr || n_rare > c->rare_alloc) {
        dev_free(c->d_rare, s);
        c->d_rare = nullptr;
        MI_CUDA(c, dev_alloc((void**)&c->d_rare, (size_t)(n_rare + 1) * sizeof(uint2), c->device, s));
        c->rare_alloc = (unsigned)n_rare;
    }
    c->rare_cap = (unsigned)n_rare;
    unsigned* d_count = nullptr;
    MI_CUDA(c, dev_alloc((void**)&d_count, sizeof(unsigned), c->device, s));
    unsigned h_count = 0;
    cudaError_t e = cudaMemsetAsync(d_count, 0, sizeof(unsigned), s);
    if (e == cudaSuccess)
        e = mi::launch_pitch_bins(c->d_fbins_ranked, c->d_mask_bits, c->fd[0] * c->fd[1], c->colpitch, c->fd[2], c->zrows_real,
                                  c->d_fb_pitched, c->d_rare, d_count, c->rare_cap, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h_count, d_count, sizeof(unsigned), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    dev_free(d_count, s);
    if (e != cudaSuccess) return cuda_fail(c, e, "pitch fixed bins");
    c->n_rare = h_count < c->rare_cap ? h_count : c->rare_cap;
    return MI_OK;
}

// A map whose index-space matrices are all diagonal with per-axis parameters: transform
// (k0,k1,k2) has c_x = fma(ax[k0].x, ix, ax[k0].y) and likewise for y (k1) and z (k2).
struct SeparablePlan {
    int n[3];
    std::vector<float2> axis[3];
};

// Decide whether the grid of index-space matrices hM (p0 fastest) is separable and extract the
// per-axis (scale, offset) tables.  Every transform is checked bit for bit against the tables.
bool make_separable_plan(const std::vector<float>& hM, const int32_t n[3], SeparablePlan* plan) {
    const int64_t N = (int64_t)n[0] * n[1] * n[2];
    const int diag[3] = {0, 5, 10}, off[3] = {3, 7, 11};
    for (int d = 0; d < 3; ++d) {
        plan->n[d] = n[d];
        plan->axis[d].resize(n[d]);
    }
    auto at = [&](int k0, int k1, int k2) { return hM.data() + (((int64_t)k2 * n[1] + k1) * n[0] + k0) * 12; };
    for (int k = 0; k < n[0]; ++k) plan->axis[0][k] = make_float2(at(k, 0, 0)[diag[0]], at(k, 0, 0)[off[0]]);
    for (int k = 0; k < n[1]; ++k) plan->axis[1][k] = make_float2(at(0, k, 0)[diag[1]], at(0, k, 0)[off[1]]);
    for (int k = 0; k < n[2]; ++k) plan->axis[2][k] = make_float2(at(0, 0, k)[diag[2]], at(0, 0, k)[off[2]]);
    // the z kernel walks the moving planes upwards: c_z must not decrease with iz
    for (int k = 0; k < n[2]; ++k)
        if (!(plan->axis[2][k].x >= 0.0f)) return false;
    for (int64_t t = 0; t < N; ++t) {
        const float* M = hM.data() + t * 12;
        const int k[3] = {(int)(t % n[0]), (int)((t / n[0]) % n[1]), (int)(t / ((int64_t)n[0] * n[1]))};
        if (M[1] != 0.f || M[2] != 0.f || M[4] != 0.f || M[6] != 0.f || M[8] != 0.f || M[9] != 0.f) return false;
        for (int d = 0; d < 3; ++d) {
            const float2 e = plan->axis[d][k[d]];
            if (std::memcmp(&e.x, &M[diag[d]], 4) != 0 || std::memcmp(&e.y, &M[off[d]], 4) != 0) return false;
        }
    }
    return true;
}

// Steps a3 + a4 of a separable map: for groups of p0 values run the x-pass, the y-pass for every
// (p0,p1) pair of the group, then one z-lerp + histogram item per transform, then the entropy
// kernel (a5) writing straight into map order.  Results land in c->d_mi / c->d_nvalid; the joint
// histograms, if asked for (hist_out: host or device, map order), are copied out item by item.
// When even one (p0,p1) pair does not fit the scratch budgets the function returns kSepFallback and
// the caller takes the generic kernel (same arithmetic, no scratch).
constexpr mi_status kSepFallback = static_cast<mi_status>(-1);

mi_status run_separable(mi_ctx* c, const SeparablePlan& sp, int32_t nq, int interp, EventTimer& timer,
                        uint32_t* hist_out) {
    cudaStream_t s = c->stream;
    const bool nn = interp == MI_INTERP_NEAREST;
    const int n0 = sp.n[0], n1 = sp.n[1], n2 = sp.n[2];
    const size_t nbins2 = (size_t)c->nb * c->nb;
    const int fnx = c->fd[0], cols = c->fd[0] * c->fd[1], fnz = c->fd[2];
    const int planes = nn ? c->md[2] : c->md[2] + 2;
    const int prows = nn ? c->md[1] : c->md[1] + 2;
    const size_t elem = nn ? 1 : sizeof(float);
    const size_t x_bytes_per_a = (size_t)planes * prows * fnx * elem;
    const size_t xy_bytes_per_pair = (size_t)planes * c->colpitch * elem;
    // fused: step a5 runs as the z kernel's epilogue and no histogram leaves the SM
    const bool fused = c->fuse_entropy && c->n_rare == 0 && nq <= mi::kMaxQPerPass && hist_out == nullptr;
    const size_t hist_bytes_per_pair = fused ? 1 : (size_t)n2 * nbins2 * sizeof(uint32_t);

    // Batch = ga values of p0 x gb values of p1.  Whole p0 slabs (gb = n1) when the scratch budgets
    // allow, as many as minimise idle SM-waves; otherwise one p0 at a time in chunks of p1.
    size_t max_pairs = c->xy_budget / xy_bytes_per_pair;
    if (!fused && c->sep_hist_budget / hist_bytes_per_pair < max_pairs)   // fused: no histogram leaves the SM
        max_pairs = c->sep_hist_budget / hist_bytes_per_pair;
    if (max_pairs > 65535) max_pairs = 65535;  // gridDim.y of the y-pass
    if (max_pairs < 1) return kSepFallback;
    int ga = 1, gb = n1;
    if (max_pairs >= (size_t)n1) {
        int ga_max = (int)(max_pairs / (size_t)n1);
        if (ga_max > n0) ga_max = n0;
        long long best_waves = -1;
        for (int g = 1; g <= ga_max; ++g) {
            const long long per = ((long long)g * n1 * n2 + c->num_sms - 1) / c->num_sms;
            const int rem = n0 % g;
            long long waves = (long long)(n0 / g) * per;
            if (rem) waves += ((long long)rem * n1 * n2 + c->num_sms - 1) / c->num_sms;
            if (best_waves < 0 || waves <= best_waves) { best_waves = waves; ga = g; }
        }
    } else {
        gb = (int)max_pairs;
    }

    mi_status st;
    const int nmax = n0 > n1 ? (n0 > n2 ? n0 : n2) : (n1 > n2 ? n1 : n2);
    if ((st = grow(c, &c->d_axis, &c->cap_axis, (size_t)3 * nmax)) != MI_OK) return st;
    if ((st = grow(c, reinterpret_cast<uint8_t**>(&c->d_X), &c->cap_X, (size_t)ga * x_bytes_per_a)) != MI_OK) return st;
    if ((st = grow(c, reinterpret_cast<uint8_t**>(&c->d_XY), &c->cap_XY, (size_t)ga * gb * xy_bytes_per_pair)) != MI_OK) return st;
    if ((st = grow(c, &c->d_colvalid, &c->cap_cv, (size_t)ga * gb * c->colpitch)) != MI_OK) return st;
    if (!fused && (st = grow(c, reinterpret_cast<uint8_t**>(&c->d_hist), &c->cap_hist, (size_t)ga * gb * hist_bytes_per_pair)) != MI_OK) return st;
    const float prescale = (!nn && c->bin_mode == mi::kBinFastPrescaled) ? c->mscale : 1.0f;
    for (int d = 0; d < 3; ++d)
        MI_CUDA(c, cudaMemcpyAsync(c->d_axis + (size_t)d * nmax, sp.axis[d].data(), sp.axis[d].size() * sizeof(float2),
                                   cudaMemcpyHostToDevice, s));
    const float2* ax = c->d_axis;
    const float2* ay = c->d_axis + nmax;
    const float2* az = c->d_axis + 2 * (size_t)nmax;

    for (int a0 = 0; a0 < n0; a0 += ga) {
        const int na = (n0 - a0 < ga) ? (n0 - a0) : ga;
        for (int b0 = 0; b0 < n1; b0 += gb) {
            const int nbc = (n1 - b0 < gb) ? (n1 - b0) : gb;
            const int npairs = na * nbc;
            const long long items = (long long)npairs * n2;
            const mi::OutMap om{1, n0, n1, n2, a0, b0, nbc};
            timer.begin(1);
            if (b0 == 0) {   // the x-lerped rows of a p0 group serve all of its p1 chunks
                if (nn)
                    MI_CUDA(c, mi::launch_xpass(true, c->d_mbins, c->md[0], c->md[2] * c->md[1], c->md[0], ax, a0, na, fnx, c->d_X, s));
                else
                    MI_CUDA(c, mi::launch_xpass(false, c->d_moving_pad, c->md[0] + 2, planes * prows, c->md[0], ax, a0, na, fnx, c->d_X, s));
                c->last_launches[1] += 1;
            }
            MI_CUDA(c, mi::launch_ypass(nn, c->d_X, planes, prows, c->md[0], c->md[1], ax, ay, a0, b0, nbc, npairs, fnx, cols,
                                        c->colpitch, prescale, c->d_XY, c->d_colvalid, s));
            mi::ZHistArgs z;
            z.xy = c->d_XY;
            z.colvalid = c->d_colvalid;
            z.fb = c->d_fb_pitched;
            z.rank_inv = c->d_rank_inv;
            z.az = az;
            z.hist = c->d_hist;
            z.fnz = fnz;
            z.colpitch = c->colpitch;
            z.planes = planes;
            z.mnz = c->md[2];
            z.nb = c->nb;
            z.rows_smem = c->zrows_smem;
            z.pitch = c->zpitch;
            z.bin_mode = c->bin_mode;
            z.rows_real = c->zrows_real;
            z.rare = c->d_rare;
            z.n_rare = c->n_rare;
            z.mlo = c->mlo;
            z.mscale = c->mscale;
            z.n_pairs = npairs;
            z.n2 = n2;
            z.fused = fused ? 1 : 0;
            z.q = c->d_q;
            z.nq = nq;
            z.nq_total = nq;
            z.form = c->tsallis_form;
            z.mi_out = c->d_mi;
            z.nvalid = c->d_nvalid;
            z.om = om;
            z.match_any = c->opt_match_any;
            z.red_count = c->d_red_count;
            timer.begin(4);
            MI_CUDA(c, mi::launch_zhist(nn, z, c->num_sms, s));
            timer.end();
            c->last_launches[1] += 2 + (c->n_rare > 0 ? 1 : 0);
            c->last_launches[4] += 1;
            timer.end();
            if (fused) continue;

            timer.begin(2);
            int q_off = 0;
            do {
                MI_CUDA(c, mi::launch_entropy(c->d_hist, c->nb, (int)items, c->d_q, nq, q_off, c->tsallis_form, c->d_mi,
                                              c->d_nvalid, om, s));
                c->last_launches[2] += 1;
                q_off += mi::kMaxQPerPass;
            } while (q_off < nq);
            timer.end();
            if (hist_out != nullptr)
                for (long long item = 0; item < items; ++item)
                    MI_CUDA(c, cudaMemcpyAsync(hist_out + om.dst(item) * nbins2, c->d_hist + (size_t)item * nbins2,
                                               nbins2 * sizeof(uint32_t), cudaMemcpyDefault, s));
        }
    }
    return MI_OK;
}

// CTAs per transform of the generic kernels: one when there are many transforms; otherwise the volume is split
// into slabs of 32-row tiles so that about 16 waves of CTAs exist (each slab keeps >= 2 tiles).  The quad-gather
// kernel orders its items slab-major, so for it the slabs are also made small enough that a slab's share of the
// 16-byte-per-voxel quad volume (plus the margin a rotation adds) stays in L2 while all SMs work on it.
int generic_nslabs(const mi_ctx* c, int64_t cnt, int interp) {
    const int rows_total = c->fd[1] * c->fd[2];
    const int cap = rows_total / 64 > 1 ? rows_total / 64 : 1;
    int nslabs = 1;
    const int64_t want = 16LL * c->num_sms;
    if (cnt < want) {
        nslabs = (int)((want + cnt - 1) / cnt);
        if (nslabs > cap) nslabs = cap;
    }
    if (interp == MI_INTERP_TRILINEAR && c->opt_gather == 1 && c->opt_slab_mb > 0) {
        const size_t quad_bytes = (size_t)(c->md[0] + 2) * (c->md[1] + 2) * (c->md[2] + 2) * sizeof(float4);
        const int by_l2 = (int)((quad_bytes + ((size_t)c->opt_slab_mb << 20) - 1) / ((size_t)c->opt_slab_mb << 20));
        if (by_l2 > nslabs) nslabs = by_l2 < cap ? by_l2 : cap;
    }
    return nslabs;
}

// The shared core of mi_eval_batch and mi_map.  hM: N x 12 index-space fp32 transforms in host
// memory.  If map_out != NULL the result is assembled channel-major (step a6) instead of being
// returned transform-major.  If sep != NULL the histograms are built by the separable path.
mi_status eval_core(mi_ctx* c, const std::vector<float>& hM, int64_t N, const double* q, int32_t nq,
                    int interp, double* mi_out, void* hist_out_v, int64_t* nvalid_out,
                    double* map_out, int64_t* argmax_out, const SeparablePlan* sep = nullptr) {
    const int nch = 1 + nq;
    const size_t nbins2 = (size_t)c->nb * c->nb;
    // partial-volume histograms hold uint64 weight units, the others uint32 counts
    const bool pv = interp == MI_INTERP_PARTIAL_VOLUME;
    const size_t helem = pv ? sizeof(unsigned long long) : sizeof(uint32_t);
    uint32_t* const hist_out = static_cast<uint32_t*>(hist_out_v);
    if (pv) sep = nullptr;
    cudaStream_t s = c->stream;
    for (int k = 0; k < 5; ++k) { c->last_ms[k] = 0.f; c->last_launches[k] = 0; }
    EventTimer timer(s);

    // ---- setup: scratch + upload of transforms and q -------------------------------------------
    timer.begin(0);
    mi_status st;
    if ((st = grow(c, &c->d_M, &c->cap_M, (size_t)N * 12)) != MI_OK) return st;
    if ((st = grow(c, &c->d_mi, &c->cap_mi, (size_t)N * nch)) != MI_OK) return st;
    if ((st = grow(c, &c->d_nvalid, &c->cap_nv, (size_t)N)) != MI_OK) return st;
    if ((st = grow(c, &c->d_q, &c->cap_q, (size_t)(nq > 0 ? nq : 1))) != MI_OK) return st;
    if (c->staging_busy) { MI_CUDA(c, cudaEventSynchronize(c->ev_staging)); c->staging_busy = false; }
    if ((size_t)N * 12 > c->cap_hM) {
        if (c->h_M) {
            mi::pinned_free(c->h_M, c->cap_hM * sizeof(float));
            c->h_M = nullptr; c->cap_hM = 0;
        }
        MI_CUDA(c, mi::pinned_alloc(reinterpret_cast<void**>(&c->h_M), (size_t)N * 12 * sizeof(float)));
        c->cap_hM = (size_t)N * 12;
    }
    std::memcpy(c->h_M, hM.data(), (size_t)N * 12 * sizeof(float));
    MI_CUDA(c, cudaMemcpyAsync(c->d_M, c->h_M, (size_t)N * 12 * sizeof(float), cudaMemcpyHostToDevice, s));
    MI_CUDA(c, cudaEventRecord(c->ev_staging, s));
    c->staging_busy = true;
    if (nq > 0) MI_CUDA(c, cudaMemcpyAsync(c->d_q, q, (size_t)nq * sizeof(double), cudaMemcpyDefault, s));
    timer.end();

    // ---- chunk plan --------------------------------------------------------------------------------
    const bool hist_to_user_dev = hist_out != nullptr && !is_host_ptr(hist_out);
    int64_t chunk = (int64_t)(c->hist_budget / (nbins2 * helem));
    if (chunk < 1) chunk = 1;
    if (chunk > N) chunk = N;
    if (c->wide && chunk > 65535) chunk = 65535;   // the wide entropy pass puts the transform on gridDim.y
    c->last_reds = -1;   // -1: not counted (only the z kernel of the separable path counts its updates)
    if (sep != nullptr) {
        MI_CUDA(c, cudaMemsetAsync(c->d_red_count, 0, sizeof(unsigned long long), s));
        st = run_separable(c, *sep, nq, interp, timer, hist_out);
        if (st == kSepFallback) sep = nullptr;   // one (p0,p1) pair exceeds the scratch budgets: generic kernel
        else if (st != MI_OK) return st;
    }
    c->last_path = sep != nullptr ? 1 : (pv ? 3 : (c->wide ? 2 : 0));
    if (!hist_to_user_dev && sep == nullptr) {
        if ((st = grow(c, reinterpret_cast<uint8_t**>(&c->d_hist), &c->cap_hist,
                       (size_t)chunk * nbins2 * helem)) != MI_OK)
            return st;
    }
    if (sep == nullptr &&
        (st = ensure_moving_quads(c, interp == MI_INTERP_TRILINEAR && c->opt_gather == 1, pv)) != MI_OK)
        return st;
    for (int64_t off = 0; sep == nullptr && off < N; off += chunk) {
        const int64_t cnt = (N - off < chunk) ? (N - off) : chunk;
        uint32_t* hist = hist_to_user_dev
            ? reinterpret_cast<uint32_t*>(static_cast<char*>(hist_out_v) + (size_t)off * nbins2 * helem) : c->d_hist;

        timer.begin(1);
        MI_CUDA(c, cudaMemsetAsync(hist, 0, (size_t)cnt * nbins2 * helem, s));
        mi::ResampleArgs a;
        a.fbins_ranked = c->d_fbins_ranked;
        a.rank_inv = c->d_rank_inv;
        a.mask_bits = c->d_mask_bits;
        a.moving_pad = c->d_moving_pad;
        a.moving_quad = c->d_moving_quad;
        a.gather = c->opt_gather;
        a.threads = c->opt_gthreads;
        a.has_rare = c->generic_has_rare ? 1 : 0;
        a.sink = nullptr;
        a.mbins = c->d_mbins;
        a.rows_smem = c->rows_smem;
        a.pitch = c->gpitch;
        a.ty_log2 = c->ty_log2;
        a.unroll = c->opt_unroll;
        a.M = c->d_M + (size_t)off * 12;
        a.hist = hist;
        a.f = {c->fd[0], c->fd[1], c->fd[2]};
        a.m = {c->md[0], c->md[1], c->md[2]};
        a.nb = c->nb;
        a.mlo = c->mlo;
        a.mscale = c->mscale;
        a.n_transforms = (int)cnt;
        const int nslabs = generic_nslabs(c, cnt, interp);
        a.nslabs = nslabs;
        timer.begin(4);
        if (pv) {
            mi::PvArgs pa;
            pa.fbins_ranked = c->d_fbins_ranked;
            pa.rank_inv = c->d_rank_inv;
            pa.mask_bits = c->d_mask_bits;
            pa.mbins_quad = c->d_mbins_quad;
            pa.M = a.M;
            pa.hist = reinterpret_cast<unsigned long long*>(hist);
            pa.rows_smem = c->rows_smem;
            pa.pitch = c->gpitch;
            pa.f = a.f;
            pa.m = a.m;
            pa.nb = c->nb;
            pa.n_transforms = (int)cnt;
            pa.nchunks = 0;
            pa.rows_per_chunk = 0;
            pa.hot_b = c->hot_mbin;
            MI_CUDA(c, mi::launch_resample_hist_pv(pa, c->num_sms, s));
        } else if (c->wide) {
            mi::WideArgs w;
            w.fbins = c->d_fbins16;
            w.mbins = c->d_mbins16;
            w.mask_bits = c->d_mask_bits;
            w.moving_pad = c->d_moving_pad;
            w.M = a.M;
            w.hist = hist;
            w.f = a.f;
            w.m = a.m;
            w.nb = c->nb;
            w.mlo = c->mlo;
            w.mscale = c->mscale;
            w.n_transforms = (int)cnt;
            w.nslabs = nslabs;
            w.moving_quad = c->d_moving_quad;
            w.fbins_ranked = c->d_fbins16_ranked;
            w.rank_inv = c->d_wrank_inv;
            w.rows_smem = c->rows_smem;
            w.pitch = c->gpitch;
            w.version = c->opt_gather == 1 ? 2 : 1;
            w.unroll = c->opt_unroll;
            MI_CUDA(c, mi::launch_resample_hist_wide(w, interp, c->num_sms, s));
        } else {
            MI_CUDA(c, mi::launch_resample_hist(a, interp, c->num_sms, s));
        }
        timer.end();
        c->last_launches[1] += 1;
        c->last_launches[4] += 1;
        timer.end();

        timer.begin(2);
        int q_off = 0;
        do {
            if (pv)
                MI_CUDA(c, mi::launch_entropy_pv(reinterpret_cast<const unsigned long long*>(hist), c->nb, (int)cnt, c->d_q, nq,
                                                 q_off, c->tsallis_form, c->d_mi + (size_t)off * nch, c->d_nvalid + off,
                                                 mi::OutMap{0, 0, 0, 0, 0, 0, 0}, s));
            else
            MI_CUDA(c, mi::launch_entropy(hist, c->nb, (int)cnt, c->d_q, nq, q_off, c->tsallis_form,
                                          c->d_mi + (size_t)off * nch, c->d_nvalid + off, mi::OutMap{0, 0, 0, 0, 0, 0, 0}, s,
                                          c->d_wrow_used));
            c->last_launches[2] += 1;
            q_off += mi::kMaxQPerPass;
        } while (q_off < nq);
        timer.end();

        if (hist_out != nullptr && !hist_to_user_dev)
            MI_CUDA(c, cudaMemcpyAsync(static_cast<char*>(hist_out_v) + (size_t)off * nbins2 * helem, hist,
                                       (size_t)cnt * nbins2 * helem, cudaMemcpyDeviceToHost, s));
    }

    // ---- outputs -----------------------------------------------------------------------------------
    bool host_out = false;
    if (map_out != nullptr) {
        timer.begin(3);
        const bool map_dev = !is_host_ptr(map_out);
        const bool am_dev = argmax_out != nullptr && !is_host_ptr(argmax_out);
        double* dmap = map_out;
        if (!map_dev) {
            if ((st = grow(c, &c->d_map, &c->cap_map, (size_t)N * nch)) != MI_OK) return st;
            dmap = c->d_map;
        }
        if ((st = grow(c, &c->d_argmax, &c->cap_am, (size_t)nch)) != MI_OK) return st;
        int64_t* dam = am_dev ? argmax_out : c->d_argmax;
        MI_CUDA(c, mi::launch_map_assemble(c->d_mi, N, nch, dmap, dam, s));
        c->last_launches[3] += 1;
        timer.end();
        if (!map_dev) {
            MI_CUDA(c, cudaMemcpyAsync(map_out, dmap, (size_t)N * nch * sizeof(double), cudaMemcpyDeviceToHost, s));
            host_out = true;
        }
        if (argmax_out != nullptr && !am_dev) {
            MI_CUDA(c, cudaMemcpyAsync(argmax_out, dam, (size_t)nch * sizeof(int64_t), cudaMemcpyDeviceToHost, s));
            host_out = true;
        }
    }
    if (mi_out != nullptr) {
        MI_CUDA(c, cudaMemcpyAsync(mi_out, c->d_mi, (size_t)N * nch * sizeof(double), cudaMemcpyDefault, s));
        host_out |= is_host_ptr(mi_out);
    }
    if (nvalid_out != nullptr) {
        MI_CUDA(c, cudaMemcpyAsync(nvalid_out, c->d_nvalid, (size_t)N * sizeof(int64_t), cudaMemcpyDefault, s));
        host_out |= is_host_ptr(nvalid_out);
    }
    if (hist_out != nullptr && !hist_to_user_dev) host_out = true;
    // Host outputs must be complete on return.  The per-class timings need the events anyway, so
    // the call always drains its own work; device outputs stay ordered on the stream.
    unsigned long long h_reds = 0;
    if (sep != nullptr) MI_CUDA(c, cudaMemcpyAsync(&h_reds, c->d_red_count, sizeof(h_reds), cudaMemcpyDeviceToHost, s));
    MI_CUDA(c, cudaStreamSynchronize(s));
    if (sep != nullptr) c->last_reds = (long long)h_reds;
    (void)host_out;
    timer.collect(c->last_ms);
    return MI_OK;
}

}  // namespace

extern "C" {

const char* mi_version(void) { return "mi-b200 0.1 (sm_100a)"; }

const char* mi_last_error(const mi_ctx* ctx) { return ctx ? ctx->err.c_str() : mi::g_thread_error.c_str(); }

mi_status mi_family_matrix(mi_family family, const double p[3], double T_out[12]) {
    if (p == nullptr || T_out == nullptr) return MI_ERR_INVALID_ARG;
    if (!finite3(p)) return MI_ERR_INVALID_ARG;
    return mi::family_matrix((int)family, p, T_out) == 0 ? MI_OK : MI_ERR_INVALID_ARG;
}

mi_status mi_index_affine(const double T[12], const int32_t fixed_dims[3], const double fixed_spacing[3],
                          const int32_t moving_dims[3], const double moving_spacing[3], float M_out[12]) {
    if (!T || !fixed_dims || !fixed_spacing || !moving_dims || !moving_spacing || !M_out)
        return MI_ERR_INVALID_ARG;
    for (int i = 0; i < 12; ++i)
        if (!std::isfinite(T[i])) return MI_ERR_INVALID_ARG;
    for (int d = 0; d < 3; ++d) {
        if (fixed_dims[d] < 1 || moving_dims[d] < 1) return MI_ERR_INVALID_ARG;
        if (!(std::isfinite(fixed_spacing[d]) && fixed_spacing[d] > 0.0)) return MI_ERR_INVALID_ARG;
        if (!(std::isfinite(moving_spacing[d]) && moving_spacing[d] > 0.0)) return MI_ERR_INVALID_ARG;
    }
    mi::index_affine(T, fixed_dims, fixed_spacing, moving_dims, moving_spacing, M_out);
    return MI_OK;
}

mi_status mi_create(mi_ctx** out, const float* fixed, const int32_t fixed_dims[3],
                    const double fixed_spacing[3], const float* moving, const int32_t moving_dims[3],
                    const double moving_spacing[3], int32_t nbins, float fixed_lo, float fixed_hi,
                    float moving_lo, float moving_hi, int32_t device, void* cuda_stream) {
    if (out == nullptr) return fail(nullptr, MI_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!fixed || !moving || !fixed_dims || !moving_dims || !fixed_spacing || !moving_spacing)
        return fail(nullptr, MI_ERR_INVALID_ARG, "NULL argument");
    int64_t nf = 1, nm = 1;
    for (int d = 0; d < 3; ++d) {
        if (fixed_dims[d] < 1 || moving_dims[d] < 1) return fail(nullptr, MI_ERR_INVALID_ARG, "volume dim < 1");
        if (!(std::isfinite(fixed_spacing[d]) && fixed_spacing[d] > 0.0) ||
            !(std::isfinite(moving_spacing[d]) && moving_spacing[d] > 0.0))
            return fail(nullptr, MI_ERR_INVALID_ARG, "spacing must be finite and > 0");
        nf *= fixed_dims[d];
        nm *= moving_dims[d];
        if (nf > 0x7FFFFFFFLL || nm > 0x7FFFFFFFLL)
            return fail(nullptr, MI_ERR_UNSUPPORTED, "volume has more than 2^31-1 voxels");
        if (moving_dims[d] > 4194302)  // the kernels' floor trick needs |index| < 2^22
            return fail(nullptr, MI_ERR_UNSUPPORTED, "moving volume dimension > 4194302");
    }
    const int64_t npad = ((int64_t)moving_dims[0] + 2) * ((int64_t)moving_dims[1] + 2) * ((int64_t)moving_dims[2] + 2);
    if (npad > 0x7FFFFFFFLL) return fail(nullptr, MI_ERR_UNSUPPORTED, "padded moving volume has more than 2^31-1 voxels");
    if (nbins < 2) return fail(nullptr, MI_ERR_INVALID_ARG, "nbins < 2");
    if (nbins > mi::kMaxBinsWide) return fail(nullptr, MI_ERR_UNSUPPORTED, "nbins > 4096 is not supported");
    if (!(std::isfinite(fixed_lo) && std::isfinite(fixed_hi) && fixed_lo < fixed_hi) ||
        !(std::isfinite(moving_lo) && std::isfinite(moving_hi) && moving_lo < moving_hi))
        return fail(nullptr, MI_ERR_INVALID_ARG, "intensity range must be finite with lo < hi");

    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceCount");
    if (device < 0 || device >= ndev) return fail(nullptr, MI_ERR_INVALID_ARG, "no such CUDA device");

    mi_ctx* c = new (std::nothrow) mi_ctx();
    if (!c) return fail(nullptr, MI_ERR_OUT_OF_MEMORY, "host allocation failed");
    c->device = device;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    DeviceGuard guard(device);
    mi_status st = MI_OK;
    float* d_tmp = nullptr;
    float* d_mov = nullptr;
    unsigned long long* d_counts = nullptr;
    do {
        if (!guard.ok) { st = fail(nullptr, MI_ERR_CUDA, "cudaSetDevice failed"); break; }
        int v = 0;
        if ((e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) { st = cuda_fail(nullptr, e, "attr"); break; }
        c->num_sms = v;
        if ((e = cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, device)) != cudaSuccess) { st = cuda_fail(nullptr, e, "attr"); break; }
        c->smem_optin = (size_t)v;
        for (int d = 0; d < 3; ++d) {
            c->fd[d] = fixed_dims[d]; c->md[d] = moving_dims[d];
            c->fs[d] = fixed_spacing[d]; c->ms[d] = moving_spacing[d];
        }
        c->nb = nbins; c->nf = nf; c->nm = nm;
        c->flo = fixed_lo; c->fhi = fixed_hi; c->mlo = moving_lo; c->mhi = moving_hi;
        c->fscale = mi::bin_scale(nbins, fixed_lo, fixed_hi);
        c->mscale = mi::bin_scale(nbins, moving_lo, moving_hi);
        // +16 bytes of slack so 16-byte vector stores of the last partial group stay inside
        if ((e = dev_alloc((void**)&c->d_fbins, (size_t)nf + 16, device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc fixed bins"); break; }
        if ((e = dev_alloc((void**)&c->d_mbins, (size_t)nm + 16, device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc moving bins"); break; }
        if ((e = dev_alloc((void**)&c->d_fbins_ranked, (size_t)nf + 16, device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc ranked bins"); break; }
        if ((e = dev_alloc((void**)&c->d_rank, 256, device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc rank"); break; }
        if ((e = dev_alloc((void**)&c->d_rank_inv, 256 * sizeof(int), device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc rank_inv"); break; }
        if ((e = dev_alloc((void**)&d_counts, mi::kMaxBinsWide * sizeof(unsigned long long), device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc counts"); break; }
        if ((e = dev_alloc((void**)&c->d_moving_pad, (size_t)npad * sizeof(float), device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc padded moving"); break; }
        if ((e = dev_alloc((void**)&d_mov, (size_t)nm * sizeof(float), device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc moving"); break; }
        if ((e = dev_alloc((void**)&d_tmp, (size_t)nf * sizeof(float), device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc staging"); break; }
        c->colpitch = (int)(((int64_t)fixed_dims[0] * fixed_dims[1] + mi::kZColAlign - 1) / mi::kZColAlign * mi::kZColAlign);
        if ((e = dev_alloc((void**)&c->d_fb_pitched, (size_t)c->colpitch * fixed_dims[2] + 16, device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc pitched bins"); break; }
        c->separable_ok = nbins <= 256 && fixed_dims[2] <= 65535;   // the rare list packs iz into 16 bits
        if ((e = dev_alloc((void**)&c->d_red_count, sizeof(unsigned long long), device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc counter"); break; }
        if ((e = cudaEventCreateWithFlags(&c->ev_staging, cudaEventDisableTiming)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaEventCreate"); break; }
        cudaStream_t s = c->stream;
        if ((e = cudaMemcpyAsync(d_tmp, fixed, (size_t)nf * sizeof(float), cudaMemcpyDefault, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "copy fixed"); break; }
        if ((e = cudaMemcpyAsync(d_mov, moving, (size_t)nm * sizeof(float), cudaMemcpyDefault, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "copy moving"); break; }
        if ((e = cudaMemsetAsync(d_counts, 0, 256 * sizeof(unsigned long long), s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "memset"); break; }
        c->wide = nbins > 256;
        if (c->wide) {
            if ((e = dev_alloc((void**)&c->d_fbins16, (size_t)nf * sizeof(uint16_t), device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc wide fixed bins"); break; }
            if ((e = dev_alloc((void**)&c->d_mbins16, (size_t)nm * sizeof(uint16_t), device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc wide moving bins"); break; }
            if ((e = mi::launch_prebin16(d_tmp, c->d_fbins16, nf, c->flo, c->fscale, nbins, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "prebin fixed (wide)"); break; }
            if ((e = mi::launch_prebin16(d_mov, c->d_mbins16, nm, c->mlo, c->mscale, nbins, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "prebin moving (wide)"); break; }
            {   // rank the fixed bins by population (host: 4096 counts) and remap them: the most populated fixed
                // bins get resample_wide_kernel's shared-memory rows
                std::vector<unsigned long long> h_c(mi::kMaxBinsWide);
                if ((e = mi::launch_bin_count16(c->d_fbins16, nf, d_counts, s)) != cudaSuccess ||
                    (e = cudaMemcpyAsync(h_c.data(), d_counts, h_c.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s)) != cudaSuccess ||
                    (e = cudaStreamSynchronize(s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "count wide bins"); break; }
                std::vector<int> order(mi::kMaxBinsWide);
                for (int b = 0; b < mi::kMaxBinsWide; ++b) order[b] = b;
                std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return h_c[x] > h_c[y]; });
                std::vector<uint16_t> h_rank(mi::kMaxBinsWide);
                for (int r = 0; r < mi::kMaxBinsWide; ++r) h_rank[order[r]] = (uint16_t)r;
                std::vector<uint8_t> h_used(mi::kMaxBinsWide);
                for (int b = 0; b < mi::kMaxBinsWide; ++b) h_used[b] = h_c[b] > 0 ? 1 : 0;
                uint16_t* d_wrank = nullptr;
                if ((e = dev_alloc((void**)&d_wrank, mi::kMaxBinsWide * sizeof(uint16_t), device, c->stream)) != cudaSuccess) { st = cuda_fail(nullptr, e, "cudaMalloc wide ranks"); break; }
                bool failed = false;
                if ((e = dev_alloc((void**)&c->d_wrank_inv, mi::kMaxBinsWide * sizeof(int), device, c->stream)) != cudaSuccess ||
                    (e = dev_alloc((void**)&c->d_fbins16_ranked, (size_t)nf * sizeof(uint16_t), device, c->stream)) != cudaSuccess ||
                    (e = cudaMemcpyAsync(d_wrank, h_rank.data(), h_rank.size() * sizeof(uint16_t), cudaMemcpyHostToDevice, s)) != cudaSuccess ||
                    (e = cudaMemcpyAsync(c->d_wrank_inv, order.data(), order.size() * sizeof(int), cudaMemcpyHostToDevice, s)) != cudaSuccess ||
                    (e = dev_alloc((void**)&c->d_wrow_used, mi::kMaxBinsWide, device, c->stream)) != cudaSuccess ||
                    (e = cudaMemcpyAsync(c->d_wrow_used, h_used.data(), h_used.size(), cudaMemcpyHostToDevice, s)) != cudaSuccess ||
                    (e = mi::launch_remap16(c->d_fbins16, c->d_fbins16_ranked, nf, d_wrank, s)) != cudaSuccess ||
                    (e = cudaStreamSynchronize(s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "rank wide fixed bins"); failed = true; }
                dev_free(d_wrank, c->stream);
                if (failed) break;
            }
        } else {
            if ((e = mi::launch_prebin(d_tmp, c->d_fbins, nf, c->flo, c->fscale, nbins, nullptr, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "prebin fixed"); break; }
            if ((e = mi::launch_prebin(d_mov, c->d_mbins, nm, c->mlo, c->mscale, nbins, reinterpret_cast<unsigned*>(d_counts), s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "prebin moving"); break; }
            {
                unsigned h_flag = 1;
                if ((e = cudaMemcpyAsync(&h_flag, d_counts, sizeof(unsigned), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "copy flag"); break; }
                if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "sync flag"); break; }
                // kBinFast*: no clamps needed (mi_internal.h); prescaled when the bin scale is a power of two
                // (so that scaling commutes with every rounding; 2^-100 < scale keeps products normal)
                int ex = 0;
                const bool pow2 = std::frexp(c->mscale, &ex) == 0.5f && ex > -100 && ex < 100;
                c->bin_mode_natural = (h_flag == 0 && c->mlo == 0.0f) ? (pow2 ? mi::kBinFastPrescaled : mi::kBinFast) : mi::kBinGeneral;
            }
            if ((e = mi::launch_rank_fixed_bins(c->d_fbins, nf, d_counts, c->d_rank, c->d_rank_inv, c->d_fbins_ranked, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "rank fixed bins"); break; }
            if ((e = cudaMemcpyAsync(c->h_counts, d_counts, sizeof(c->h_counts), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "copy counts"); break; }
            if ((e = cudaMemcpyAsync(c->h_rank, c->d_rank, sizeof(c->h_rank), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "copy ranks"); break; }
            if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "sync ranks"); break; }
        }
        if ((st = plan_layout(c)) != MI_OK) { mi::set_thread_error(c->err); break; }
        if (!c->wide) {
            {   // the most populated moving bin (d_counts is free again: the fixed counts are on the host)
                unsigned long long h_mcounts[256];
                if ((e = mi::launch_bin_count(c->d_mbins, nm, d_counts, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "count moving bins"); break; }
                if ((e = cudaMemcpyAsync(h_mcounts, d_counts, sizeof(h_mcounts), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "copy moving counts"); break; }
                if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "sync moving counts"); break; }
                c->hot_mbin = 0;
                for (int b = 1; b < nbins; ++b)
                    if (h_mcounts[b] > h_mcounts[c->hot_mbin]) c->hot_mbin = b;
            }
        }
        if ((e = mi::launch_pad_replicate(d_mov, c->d_moving_pad, moving_dims[0], moving_dims[1], moving_dims[2], s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "pad moving"); break; }
        // the yz-quad copies (float4 / u32 per padded voxel) are built by the first call that gathers from them
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { st = cuda_fail(nullptr, e, "mi_create sync"); break; }
    } while (false);
    dev_free(d_tmp, c->stream);
    dev_free(d_mov, c->stream);
    dev_free(d_counts, c->stream);
    if (st != MI_OK) {
        mi_destroy(c);
        return st;
    }
    *out = c;
    return MI_OK;
}

void mi_destroy(mi_ctx* c) {
    if (!c) return;
    DeviceGuard guard(c->device);
    if (guard.ok) {
        void* bufs[] = {c->d_fbins, c->d_fbins_ranked, c->d_rank, c->d_rank_inv, c->d_moving_pad, c->d_mask_bits, c->d_fbins16, c->d_mbins16, c->d_mbins,
                        c->d_mbins_quad, c->d_moving_quad, c->d_fbins16_ranked, c->d_wrank_inv, c->d_wrow_used, c->d_red_count, c->d_fb_pitched, c->d_rare, c->d_X, c->d_XY, c->d_colvalid, c->d_axis, c->d_M, c->d_hist,
                        c->d_mi, c->d_nvalid, c->d_q, c->d_map, c->d_argmax};
        for (void* b : bufs) dev_free(b, c->stream);
        cudaStreamSynchronize(c->stream);
        mi::pinned_free(c->h_M, c->cap_hM * sizeof(float));
        if (c->ev_staging) cudaEventDestroy(c->ev_staging);
        cudaGetLastError();
    }
    delete c;
}

mi_status mi_release_cached_memory(int32_t device) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess) { cudaGetLastError(); return MI_ERR_CUDA; }
    if (device < 0 || device >= ndev || device >= 64) return MI_ERR_INVALID_ARG;
    {
        DeviceGuard guard(device);
        if (!guard.ok) return MI_ERR_CUDA;
        mi::unpark_all(device);
        mi::unpark_pinned();
        if (cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); return MI_ERR_CUDA; }
    }
    std::lock_guard<std::mutex> lock(mi::g_pool_mutex);
    if (mi::g_pools[device] == nullptr) return MI_OK;
    if (cudaMemPoolTrimTo(mi::g_pools[device], 0) != cudaSuccess) { cudaGetLastError(); return MI_ERR_CUDA; }
    return MI_OK;
}

mi_status mi_set_fixed_mask(mi_ctx* c, const uint8_t* mask) {
    if (!c) return MI_ERR_INVALID_ARG;
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(c, MI_ERR_CUDA, "cudaSetDevice failed");
    cudaStream_t s = c->stream;
    uint8_t* d_mask = nullptr;
    mi_status st = MI_OK;
    do {
        cudaError_t e;
        if (mask != nullptr) {
            if ((e = dev_alloc((void**)&d_mask, (size_t)c->nf, c->device, s)) != cudaSuccess) { st = cuda_fail(c, e, "cudaMalloc mask"); break; }
            if ((e = cudaMemcpyAsync(d_mask, mask, (size_t)c->nf, cudaMemcpyDefault, s)) != cudaSuccess) { st = cuda_fail(c, e, "copy mask"); break; }
            if (c->d_mask_bits == nullptr &&
                (e = dev_alloc((void**)&c->d_mask_bits, (size_t)((c->nf + 31) / 32) * sizeof(uint32_t), c->device, s)) != cudaSuccess) { st = cuda_fail(c, e, "cudaMalloc mask bits"); break; }
            if ((e = mi::launch_mask_bits(d_mask, c->nf, c->d_mask_bits, s)) != cudaSuccess) { st = cuda_fail(c, e, "mask bits"); break; }
        } else if (c->d_mask_bits != nullptr) {
            dev_free(c->d_mask_bits, s);
            c->d_mask_bits = nullptr;
        }
        // the separable path reads the mask through its pitched fixed bins: rebuild them (and the rare list)
        st = plan_layout(c);
        if (st == MI_OK && (e = cudaStreamSynchronize(s)) != cudaSuccess) st = cuda_fail(c, e, "sync");
    } while (false);
    dev_free(d_mask, s);
    return st;
}

mi_status mi_set_tsallis_form(mi_ctx* c, mi_tsallis_form form) {
    if (!c) return MI_ERR_INVALID_ARG;
    if (form != MI_TSALLIS_ADDITIVE && form != MI_TSALLIS_PSEUDO_ADDITIVE)
        return fail(c, MI_ERR_INVALID_ARG, "unknown Tsallis form");
    c->tsallis_form = (int)form;
    return MI_OK;
}

mi_status mi_set_option(mi_ctx* c, mi_option key, int64_t v) {
    if (!c) return MI_ERR_INVALID_ARG;
    bool relayout = false;
    // the options plan_layout reads: restored if the new value gives a layout the device cannot hold
    const int old_bin_mode_max = c->opt_bin_mode_max, old_zrows_max = c->opt_zrows_max, old_zpad = c->opt_zpad,
              old_gpad = c->opt_gpad, old_gsmem_kb = c->opt_gsmem_kb;
    auto bad = [&]() { return fail(c, MI_ERR_INVALID_ARG, "mi_set_option: value out of range"); };
    switch (key) {
    case MI_OPT_SEPARABLE: c->use_separable = v != 0; break;
    case MI_OPT_FUSE_ENTROPY: c->fuse_entropy = v != 0; break;
    case MI_OPT_BIN_MODE_MAX:
        if (v < mi::kBinGeneral || v > mi::kBinFastPrescaled) return bad();
        c->opt_bin_mode_max = (int)v; relayout = true; break;
    case MI_OPT_ZHIST_ROWS_MAX:
        if (v != 0 && (v < 2 || v > 257)) return bad();
        c->opt_zrows_max = (int)v; relayout = true; break;
    case MI_OPT_ZHIST_PAD:
        if (v < 1 || v > 64) return bad();
        c->opt_zpad = (int)v; relayout = true; break;
    case MI_OPT_XY_BUDGET_MB:
        if (v < 0 || v > (1 << 20)) return bad();
        c->xy_budget = (size_t)v << 20; break;
    case MI_OPT_SEP_HIST_BUDGET_MB:
        if (v < 0 || v > (1 << 20)) return bad();
        c->sep_hist_budget = (size_t)v << 20; break;
    case MI_OPT_HIST_BUDGET_MB:
        if (v < 1 || v > (1 << 20)) return bad();
        c->hist_budget = (size_t)v << 20; break;
    case MI_OPT_GENERIC_PAD:
        if (v < 0 || v > 64) return bad();
        c->opt_gpad = (int)v; relayout = true; break;
    case MI_OPT_GENERIC_SMEM_KB:
        if (v < 8 || v > (int64_t)(c->smem_optin >> 10)) return bad();
        c->opt_gsmem_kb = (int)v; relayout = true; break;
    case MI_OPT_GENERIC_TY_LOG2:
        if (v < 0 || v > 5) return bad();
        c->ty_log2 = (int)v; break;
    case MI_OPT_GENERIC_UNROLL:
        if (v < 0 || v > 4) return bad();
        c->opt_unroll = (int)v; break;
    case MI_OPT_ZHIST_MATCH_ANY: c->opt_match_any = v != 0; break;
    case MI_OPT_GENERIC_GATHER:
        if (v < 0 || v > 1) return bad();
        c->opt_gather = (int)v;
        if (v == 0 && c->d_moving_quad != nullptr) {   // 16 B per padded voxel nobody reads any more
            dev_free(c->d_moving_quad, c->stream);
            c->d_moving_quad = nullptr;
        }
        break;
    case MI_OPT_GENERIC_THREADS:
        if (v != 512 && v != 768 && v != 1024) return bad();
        c->opt_gthreads = (int)v; break;
    case MI_OPT_GENERIC_SLAB_MB:
        if (v < 0 || v > (1 << 20)) return bad();
        c->opt_slab_mb = (int)v; break;
    default:
        return fail(c, MI_ERR_INVALID_ARG, "mi_set_option: unknown or read-only key");
    }
    if (!relayout) return MI_OK;
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(c, MI_ERR_CUDA, "cudaSetDevice failed");
    const mi_status st = plan_layout(c);
    if (st != MI_OK) {
        // the context keeps working with the layout it had: put the old values back and plan again
        const std::string why = c->err;
        c->opt_bin_mode_max = old_bin_mode_max; c->opt_zrows_max = old_zrows_max; c->opt_zpad = old_zpad;
        c->opt_gpad = old_gpad; c->opt_gsmem_kb = old_gsmem_kb;
        if (plan_layout(c) != MI_OK) return st;
        return fail(c, st, "mi_set_option: value rejected, option unchanged (" + why + ")");
    }
    return MI_OK;
}

mi_status mi_get_option(const mi_ctx* c, mi_option key, int64_t* out) {
    if (!c || !out) return MI_ERR_INVALID_ARG;
    switch (key) {
    case MI_OPT_SEPARABLE: *out = c->use_separable; break;
    case MI_OPT_FUSE_ENTROPY: *out = c->fuse_entropy; break;
    case MI_OPT_BIN_MODE_MAX: *out = c->opt_bin_mode_max; break;
    case MI_OPT_ZHIST_ROWS_MAX: *out = c->opt_zrows_max; break;
    case MI_OPT_ZHIST_PAD: *out = c->opt_zpad; break;
    case MI_OPT_XY_BUDGET_MB: *out = (int64_t)(c->xy_budget >> 20); break;
    case MI_OPT_SEP_HIST_BUDGET_MB: *out = (int64_t)(c->sep_hist_budget >> 20); break;
    case MI_OPT_HIST_BUDGET_MB: *out = (int64_t)(c->hist_budget >> 20); break;
    case MI_OPT_GENERIC_PAD: *out = c->opt_gpad; break;
    case MI_OPT_GENERIC_SMEM_KB: *out = c->opt_gsmem_kb; break;
    case MI_OPT_GENERIC_TY_LOG2: *out = c->ty_log2; break;
    case MI_OPT_GENERIC_UNROLL: *out = c->opt_unroll; break;
    case MI_OPT_ZHIST_MATCH_ANY: *out = c->opt_match_any; break;
    case MI_OPT_GENERIC_GATHER: *out = c->opt_gather; break;
    case MI_OPT_GENERIC_THREADS: *out = c->opt_gthreads; break;
    case MI_OPT_GENERIC_SLAB_MB: *out = c->opt_slab_mb; break;
    case MI_INFO_LAST_UPDATES_ISSUED: *out = c->last_reds; break;
    case MI_INFO_QUADS_BUILT: *out = (c->d_moving_quad ? 1 : 0) | (c->d_mbins_quad ? 2 : 0); break;
    case MI_INFO_NUM_SMS: *out = c->num_sms; break;
    case MI_INFO_BIN_MODE: *out = c->bin_mode; break;
    case MI_INFO_ZHIST_ROWS: *out = c->wide ? 0 : c->zrows_real; break;
    case MI_INFO_RARE_VOXELS: *out = c->wide ? 0 : (int64_t)c->n_rare; break;
    case MI_INFO_GENERIC_ROWS: *out = c->rows_smem; break;
    case MI_INFO_LAST_PATH: *out = c->last_path; break;
    default: return MI_ERR_INVALID_ARG;
    }
    return MI_OK;
}

static mi_status eval_batch_impl(mi_ctx* c, const double* T, int64_t N, const double* q, int32_t nq, int interp,
                                 double* mi_out, void* hist_out, int64_t* nvalid_out) {
    if (!c) return MI_ERR_INVALID_ARG;
    if (N < 0) return fail(c, MI_ERR_INVALID_ARG, "N < 0");
    mi_status st = validate_interp(c, interp);
    if (st != MI_OK) return st;
    st = validate_q(c, q, nq);
    if (st != MI_OK) return st;
    if (N == 0) return MI_OK;
    if (T == nullptr || mi_out == nullptr) return fail(c, MI_ERR_INVALID_ARG, "NULL argument");
    if (N > 0x7FFFFFFFLL / 16) return fail(c, MI_ERR_UNSUPPORTED, "too many transforms in one call");
    std::vector<float> hM;
    try {
        hM.resize((size_t)N * 12);
    } catch (const std::bad_alloc&) {
        return fail(c, MI_ERR_OUT_OF_MEMORY, "host allocation failed");
    }
    for (int64_t t = 0; t < N; ++t) {
        const double* Tt = T + t * 12;
        for (int i = 0; i < 12; ++i)
            if (!std::isfinite(Tt[i])) return fail(c, MI_ERR_INVALID_ARG, "non-finite matrix entry");
        mi::index_affine(Tt, c->fd, c->fs, c->md, c->ms, hM.data() + t * 12);
    }
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(c, MI_ERR_CUDA, "cudaSetDevice failed");
    return eval_core(c, hM, N, q, nq, interp, mi_out, hist_out, nvalid_out, nullptr, nullptr);
}

mi_status mi_eval_batch(mi_ctx* c, const double* T, int64_t N, const double* q, int32_t nq,
                        mi_interp interp, double* mi_out, uint32_t* hist_out, int64_t* nvalid_out) {
    if (c && interp == MI_INTERP_PARTIAL_VOLUME && hist_out != nullptr)
        return fail(c, MI_ERR_INVALID_ARG, "partial-volume histograms are uint64: use mi_eval_batch_pv");
    return eval_batch_impl(c, T, N, q, nq, (int)interp, mi_out, hist_out, nvalid_out);
}

mi_status mi_eval_batch_pv(mi_ctx* c, const double* T, int64_t N, const double* q, int32_t nq,
                           double* mi_out, uint64_t* hist_out, int64_t* nvalid_out) {
    return eval_batch_impl(c, T, N, q, nq, MI_INTERP_PARTIAL_VOLUME, mi_out, hist_out, nvalid_out);
}

mi_status mi_seed_from_map(mi_family family, const double lo[3], const double hi[3], const int32_t n[3],
                           int64_t index, double p_out[9]) {
    if (!lo || !hi || !n || !p_out) return MI_ERR_INVALID_ARG;
    if (!finite3(lo) || !finite3(hi) || n[0] < 1 || n[1] < 1 || n[2] < 1) return MI_ERR_INVALID_ARG;
    const int64_t total = (int64_t)n[0] * n[1] * n[2];
    if (index < 0 || index >= total) return MI_ERR_INVALID_ARG;
    const int64_t k[3] = {index % n[0], (index / n[0]) % n[1], index / ((int64_t)n[0] * n[1])};
    double p[3];
    for (int d = 0; d < 3; ++d) p[d] = n[d] == 1 ? lo[d] : lo[d] + (double)k[d] * (hi[d] - lo[d]) / (double)(n[d] - 1);
    return mi::seed_from_node((int)family, p, p_out) == 0 ? MI_OK : MI_ERR_INVALID_ARG;
}

mi_status mi_compose_matrix(const double p[9], double T_out[12]) {
    if (p == nullptr || T_out == nullptr) return MI_ERR_INVALID_ARG;
    for (int i = 0; i < 9; ++i)
        if (!std::isfinite(p[i])) return MI_ERR_INVALID_ARG;
    mi::compose_matrix(p, T_out);
    return MI_OK;
}

}  // extern "C"

namespace {

// One multi-metric gradient (arguments already validated; the device is current).
mi_status gradient_core(mi_ctx* c, const double p[9], const double delta[9], double q, int interp,
                        double grad_out[9], double value_out[2]) {
    mi_status st;
    // transform 0 = p; then p + d_k e_k, p - d_k e_k for every parameter with d_k > 0
    int slot[9];
    int64_t N = 1;
    for (int k = 0; k < 9; ++k) {
        slot[k] = delta[k] > 0.0 ? (int)N : -1;
        if (delta[k] > 0.0) N += 2;
    }
    std::vector<float> hM((size_t)N * 12);
    auto put = [&](int64_t t, const double pk[9]) {
        double T[12];
        mi::compose_matrix(pk, T);
        mi::index_affine(T, c->fd, c->fs, c->md, c->ms, hM.data() + t * 12);
    };
    put(0, p);
    for (int k = 0; k < 9; ++k) {
        if (slot[k] < 0) continue;
        double pk[9];
        for (int i = 0; i < 9; ++i) pk[i] = p[i];
        pk[k] = p[k] + delta[k];
        put(slot[k], pk);
        pk[k] = p[k] - delta[k];
        put(slot[k] + 1, pk);
    }
    std::vector<double> vals((size_t)N * 2);
    st = eval_core(c, hM, N, &q, 1, interp, vals.data(), nullptr, nullptr, nullptr, nullptr);
    if (st != MI_OK) return st;
    for (int k = 0; k < 9; ++k) {
        grad_out[k] = 0.0;
        if (slot[k] < 0) continue;
        const int ch = k < 3 ? 1 : 0;   // Tsallis for the translation parameters, Shannon for the rest
        grad_out[k] = (vals[(size_t)slot[k] * 2 + ch] - vals[(size_t)(slot[k] + 1) * 2 + ch]) / (2.0 * delta[k]);
    }
    if (value_out) { value_out[0] = vals[0]; value_out[1] = vals[1]; }
    return MI_OK;
}

// Smallest finite-difference steps under partial-volume interpolation.  PV rounds each axis' fraction to 1/32
// voxel (reading A21), so MI is piecewise constant in the transform: a step must move the sample points by at
// least one quantisation step or both arms of the central difference see the same histogram.
//   translation k     one step of moving axis k: s_m[k] / 32 mm
//   rotation, scale   a point at distance r from the centre moves r * angle (r * factor change); the reference
//                     radius is a quarter of the smallest fixed extent (not below one fixed voxel), so that every
//                     voxel farther out than that moves at least one step of the coarsest moving axis
void pv_min_delta(const mi_ctx* c, double out[9]) {
    double step_mm = 0.0, extent = 0.0, smin = c->fs[0];
    for (int k = 0; k < 3; ++k) {
        out[k] = c->ms[k] / 32.0;
        if (out[k] > step_mm) step_mm = out[k];
        const double e = c->fs[k] * (double)(c->fd[k] - 1);
        if (k == 0 || e < extent) extent = e;
        if (c->fs[k] < smin) smin = c->fs[k];
    }
    double r_ref = 0.25 * extent;
    if (r_ref < smin) r_ref = smin;
    for (int k = 0; k < 3; ++k) {
        out[3 + k] = step_mm / r_ref * (180.0 / 3.14159265358979323846);
        out[6 + k] = step_mm / r_ref;
    }
}

mi_status validate_gradient_args(mi_ctx* c, const double* p, const double* delta, double q, int interp) {
    if (!p || !delta) return fail(c, MI_ERR_INVALID_ARG, "NULL argument");
    mi_status st = validate_interp(c, interp);
    if (st != MI_OK) return st;
    st = validate_q(c, &q, 1);
    if (st != MI_OK) return st;
    for (int i = 0; i < 9; ++i)
        if (!std::isfinite(p[i]) || !std::isfinite(delta[i])) return fail(c, MI_ERR_INVALID_ARG, "non-finite parameter");
    if (interp == MI_INTERP_PARTIAL_VOLUME) {
        double dmin[9];
        pv_min_delta(c, dmin);
        for (int i = 0; i < 9; ++i)
            if (delta[i] > 0.0 && delta[i] < dmin[i])
                return fail(c, MI_ERR_INVALID_ARG,
                            "delta[" + std::to_string(i) + "] = " + std::to_string(delta[i]) + " is below " +
                                std::to_string(dmin[i]) + ", the smallest step partial-volume interpolation resolves "
                                "(weights are quantised to 1/32 voxel; see mi_pv_min_delta)");
    }
    return MI_OK;
}

}  // namespace

extern "C" {

mi_status mi_pv_min_delta(const mi_ctx* c, double delta_min_out[9]) {
    if (!c || !delta_min_out) return MI_ERR_INVALID_ARG;
    pv_min_delta(c, delta_min_out);
    return MI_OK;
}

mi_status mi_multimetric_gradient(mi_ctx* c, const double p[9], const double delta[9], double q, mi_interp interp,
                                  double grad_out[9], double value_out[2]) {
    if (!c) return MI_ERR_INVALID_ARG;
    if (!grad_out) return fail(c, MI_ERR_INVALID_ARG, "NULL argument");
    mi_status st = validate_gradient_args(c, p, delta, q, (int)interp);
    if (st != MI_OK) return st;
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(c, MI_ERR_CUDA, "cudaSetDevice failed");
    return gradient_core(c, p, delta, q, (int)interp, grad_out, value_out);
}

mi_status mi_register(mi_ctx* c, const double p0[9], const double delta[9], const double step0[3],
                      const double step_min[3], int32_t max_iter, double q, mi_interp interp, double p_out[9],
                      double* trace_out, mi_register_info* info_out) {
    if (!c) return MI_ERR_INVALID_ARG;
    if (!step0 || !step_min || !p_out) return fail(c, MI_ERR_INVALID_ARG, "NULL argument");
    mi_status st = validate_gradient_args(c, p0, delta, q, (int)interp);
    if (st != MI_OK) return st;
    if (max_iter < 0) return fail(c, MI_ERR_INVALID_ARG, "max_iter < 0");
    for (int g = 0; g < 3; ++g)
        if (!std::isfinite(step0[g]) || !std::isfinite(step_min[g])) return fail(c, MI_ERR_INVALID_ARG, "non-finite step");
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(c, MI_ERR_CUDA, "cudaSetDevice failed");
    double p[9], L[3], prev[3][3], vals[2] = {0.0, 0.0};
    bool have_prev[3] = {false, false, false};
    for (int i = 0; i < 9; ++i) p[i] = p0[i];
    for (int g = 0; g < 3; ++g) L[g] = step0[g];
    if (trace_out) for (int i = 0; i < 9; ++i) trace_out[i] = p[i];
    int it = 0;
    while (it < max_iter) {
        double grad[9];
        st = gradient_core(c, p, delta, q, (int)interp, grad, vals);
        if (st != MI_OK) return st;
        bool moved = false;
        for (int g = 0; g < 3; ++g) {
            if (!(L[g] >= step_min[g] && L[g] > 0.0)) continue;
            const double* gg = grad + 3 * g;
            const double norm = std::sqrt(gg[0] * gg[0] + gg[1] * gg[1] + gg[2] * gg[2]);
            if (norm == 0.0) continue;
            const double d[3] = {gg[0] / norm, gg[1] / norm, gg[2] / norm};
            if (have_prev[g] && d[0] * prev[g][0] + d[1] * prev[g][1] + d[2] * prev[g][2] < 0.0) L[g] = L[g] / 2.0;
            for (int i = 0; i < 3; ++i) prev[g][i] = d[i];
            have_prev[g] = true;
            if (L[g] >= step_min[g]) {
                for (int i = 0; i < 3; ++i) p[3 * g + i] = p[3 * g + i] + L[g] * d[i];
                moved = true;
            }
        }
        ++it;
        if (trace_out) for (int i = 0; i < 9; ++i) trace_out[(size_t)it * 9 + i] = p[i];
        if (!moved) break;
    }
    for (int i = 0; i < 9; ++i) p_out[i] = p[i];
    if (info_out) {
        info_out->iterations = it;
        for (int g = 0; g < 3; ++g) info_out->steps[g] = L[g];
        info_out->values[0] = vals[0];
        info_out->values[1] = vals[1];
    }
    return MI_OK;
}

mi_status mi_map_range(mi_ctx* c, mi_family family, const double lo[3], const double hi[3], const int32_t n[3],
                       const int32_t begin[3], const int32_t end[3], const double* q, int32_t nq, mi_interp interp,
                       double* map_out, int64_t* argmax_out, uint32_t* hist_out) {
    if (!c) return MI_ERR_INVALID_ARG;
    if (!lo || !hi || !n || !map_out) return fail(c, MI_ERR_INVALID_ARG, "NULL argument");
    mi_status st = validate_interp(c, (int)interp);
    if (st != MI_OK) return st;
    if (interp == MI_INTERP_PARTIAL_VOLUME && hist_out != nullptr)
        return fail(c, MI_ERR_INVALID_ARG, "partial-volume histograms are uint64: use mi_eval_batch_pv");
    if ((int)family < 0 || (int)family > MI_FAMILY_SCALE_LOG) return fail(c, MI_ERR_INVALID_ARG, "unknown family");
    if (!finite3(lo) || !finite3(hi)) return fail(c, MI_ERR_INVALID_ARG, "non-finite grid bound");
    int32_t kb[3], m[3];   // first node and node count of the sub-box per axis
    int64_t N = 1;
    for (int d = 0; d < 3; ++d) {
        if (n[d] < 1) return fail(c, MI_ERR_INVALID_ARG, "grid n < 1");
        kb[d] = begin ? begin[d] : 0;
        const int32_t ke = end ? end[d] : n[d];
        if (kb[d] < 0 || ke > n[d] || ke <= kb[d]) return fail(c, MI_ERR_INVALID_ARG, "empty or out-of-grid node range");
        m[d] = ke - kb[d];
        N *= m[d];
        if (N > 0x7FFFFFFFLL / 16) return fail(c, MI_ERR_UNSUPPORTED, "too many transforms in one call");
    }
    st = validate_q(c, q, nq);
    if (st != MI_OK) return st;
    std::vector<float> hM;
    try {
        hM.resize((size_t)N * 12);
    } catch (const std::bad_alloc&) {
        return fail(c, MI_ERR_OUT_OF_MEMORY, "host allocation failed");
    }
    // step a2: one transform per node of the sub-box, p0 fastest.  Node k of axis d has the parameter
    // of the WHOLE grid, lo + k (hi - lo)/(n - 1): a slab computed here is bit-identical to the same
    // nodes of the full map.
    for (int j2 = 0; j2 < m[2]; ++j2)
        for (int j1 = 0; j1 < m[1]; ++j1)
            for (int j0 = 0; j0 < m[0]; ++j0) {
                const int kk[3] = {kb[0] + j0, kb[1] + j1, kb[2] + j2};
                double p[3], T[12];
                for (int d = 0; d < 3; ++d)
                    p[d] = n[d] == 1 ? lo[d] : lo[d] + (double)kk[d] * (hi[d] - lo[d]) / (double)(n[d] - 1);
                mi::family_matrix((int)family, p, T);
                for (int i = 0; i < 12; ++i)
                    if (!std::isfinite(T[i])) return fail(c, MI_ERR_INVALID_ARG, "non-finite matrix entry");
                const int64_t t = ((int64_t)j2 * m[1] + j1) * m[0] + j0;
                mi::index_affine(T, c->fd, c->fs, c->md, c->ms, hM.data() + t * 12);
            }
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(c, MI_ERR_CUDA, "cudaSetDevice failed");
    // translation / scale maps have diagonal matrices: separable fast path (same arithmetic)
    SeparablePlan plan;
    const bool diag_family = family == MI_FAMILY_TRANSLATION || family == MI_FAMILY_SCALE || family == MI_FAMILY_SCALE_LOG;
    const bool sep = diag_family && interp != MI_INTERP_PARTIAL_VOLUME && c->use_separable && c->separable_ok &&
                     c->zrows_smem >= 2 && make_separable_plan(hM, m, &plan);
    return eval_core(c, hM, N, q, nq, (int)interp, nullptr, hist_out, nullptr, map_out, argmax_out,
                     sep ? &plan : nullptr);
}

mi_status mi_map(mi_ctx* c, mi_family family, const double lo[3], const double hi[3], const int32_t n[3],
                 const double* q, int32_t nq, mi_interp interp, double* map_out, int64_t* argmax_out) {
    return mi_map_range(c, family, lo, hi, n, nullptr, nullptr, q, nq, interp, map_out, argmax_out, nullptr);
}

mi_status mi_get_bins(mi_ctx* c, int32_t which, void* out) {
    if (!c || !out) return MI_ERR_INVALID_ARG;
    if (which != 0 && which != 1) return fail(c, MI_ERR_INVALID_ARG, "which must be 0 or 1");
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(c, MI_ERR_CUDA, "cudaSetDevice failed");
    const size_t n = (size_t)(which == 0 ? c->nf : c->nm);
    if (c->wide) {   // two bytes per voxel
        const uint16_t* src16 = which == 0 ? c->d_fbins16 : c->d_mbins16;
        MI_CUDA(c, cudaMemcpyAsync(out, src16, n * sizeof(uint16_t), cudaMemcpyDefault, c->stream));
        MI_CUDA(c, cudaStreamSynchronize(c->stream));
        return MI_OK;
    }
    const uint8_t* src = which == 0 ? c->d_fbins : c->d_mbins;
    MI_CUDA(c, cudaMemcpyAsync(out, src, n, cudaMemcpyDefault, c->stream));
    MI_CUDA(c, cudaStreamSynchronize(c->stream));
    return MI_OK;
}

mi_status mi_last_timing(const mi_ctx* c, float ms[5], int64_t launches[5]) {
    if (!c) return MI_ERR_INVALID_ARG;
    for (int k = 0; k < 5; ++k) {
        if (ms) ms[k] = c->last_ms[k];
        if (launches) launches[k] = c->last_launches[k];
    }
    return MI_OK;
}

mi_status mi_probe_gather_rate(mi_ctx* c, const double* T, int32_t n_transforms, int32_t reps, double* samples_per_s) {
    if (!c) return MI_ERR_INVALID_ARG;
    if (!T || !samples_per_s || n_transforms < 1 || n_transforms > (1 << 20) || reps < 1)
        return fail(c, MI_ERR_INVALID_ARG, "mi_probe_gather_rate: bad argument");
    if (c->wide) return fail(c, MI_ERR_UNSUPPORTED, "mi_probe_gather_rate needs nbins <= 256");
    std::vector<float> hM((size_t)n_transforms * 12);
    for (int t = 0; t < n_transforms; ++t) {
        for (int i = 0; i < 12; ++i)
            if (!std::isfinite(T[(size_t)t * 12 + i])) return fail(c, MI_ERR_INVALID_ARG, "non-finite matrix entry");
        mi::index_affine(T + (size_t)t * 12, c->fd, c->fs, c->md, c->ms, hM.data() + (size_t)t * 12);
    }
    DeviceGuard guard(c->device);
    if (!guard.ok) return fail(c, MI_ERR_CUDA, "cudaSetDevice failed");
    cudaStream_t s = c->stream;
    mi_status st;
    if ((st = grow(c, &c->d_M, &c->cap_M, (size_t)n_transforms * 12)) != MI_OK) return st;
    MI_CUDA(c, cudaMemcpyAsync(c->d_M, hM.data(), hM.size() * sizeof(float), cudaMemcpyHostToDevice, s));
    MI_CUDA(c, cudaMemsetAsync(c->d_red_count, 0, sizeof(unsigned long long), s));
    if ((st = ensure_moving_quads(c, c->opt_gather == 1, false)) != MI_OK) return st;
    mi::ResampleArgs a;
    a.fbins_ranked = c->d_fbins_ranked;
    a.rank_inv = c->d_rank_inv;
    a.mask_bits = c->d_mask_bits;
    a.moving_pad = c->d_moving_pad;
    a.moving_quad = c->d_moving_quad;
    a.gather = c->opt_gather;
    a.threads = c->opt_gthreads;
    a.has_rare = c->generic_has_rare ? 1 : 0;
    a.sink = reinterpret_cast<unsigned*>(c->d_red_count);
    a.mbins = c->d_mbins;
    a.rows_smem = c->rows_smem;      // the probe keeps the kernel's shared-memory size: same L1 carve-out
    a.pitch = c->gpitch;
    a.ty_log2 = c->ty_log2;
    a.unroll = c->opt_unroll;
    a.M = c->d_M;
    a.hist = nullptr;
    a.f = {c->fd[0], c->fd[1], c->fd[2]};
    a.m = {c->md[0], c->md[1], c->md[2]};
    a.nb = c->nb;
    a.mlo = c->mlo;
    a.mscale = c->mscale;
    a.n_transforms = n_transforms;
    a.nslabs = generic_nslabs(c, n_transforms, MI_INTERP_TRILINEAR);   // the launch shape mi_eval_batch / mi_map use
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    MI_CUDA(c, cudaEventCreate(&e0));
    cudaError_t e = cudaEventCreate(&e1);
    if (e != cudaSuccess) {
        cudaEventDestroy(e0);
        return cuda_fail(c, e, "cudaEventCreate");
    }
    float best = 1e30f;
    for (int rep = 0; rep <= reps && e == cudaSuccess; ++rep) {   // the first run warms up
        cudaEventRecord(e0, s);
        e = mi::launch_resample_hist(a, MI_INTERP_TRILINEAR, c->num_sms, s);
        cudaEventRecord(e1, s);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return cuda_fail(c, e, "gather probe");
    *samples_per_s = (double)c->nf * n_transforms / (best * 1e-3);
    return MI_OK;
}

mi_status mi_probe_shared_atomic_rate(int32_t device, int32_t nbins, int32_t pattern, int32_t iters,
                                      double* updates_per_s) {
    if (!updates_per_s || nbins < 8 || nbins > 256 || pattern < 0 || pattern > 6 || iters < 1)
        return MI_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess) { cudaGetLastError(); return MI_ERR_CUDA; }
    if (device < 0 || device >= ndev) return MI_ERR_INVALID_ARG;
    DeviceGuard guard(device);
    if (!guard.ok) return MI_ERR_CUDA;
    int sms = 0, smem = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return MI_ERR_CUDA;
    if (cudaDeviceGetAttribute(&smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, device) != cudaSuccess) return MI_ERR_CUDA;
    const cudaError_t e = mi::run_shared_atomic_probe(nbins, pattern, iters, sms, (size_t)smem, updates_per_s);
    if (e != cudaSuccess) { cudaGetLastError(); return MI_ERR_CUDA; }
    return MI_OK;
}

}  // extern "C"
