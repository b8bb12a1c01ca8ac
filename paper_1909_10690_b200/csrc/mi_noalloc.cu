// mi_noalloc.cu -- mi_eval_noalloc: one transform's joint histogram and MI with no device allocation.
//
// Who this is for.  Every other compute entry point of the library takes device memory from the
// library's stream-ordered pool (mi_create, and the scratch each call grows on demand).  Some callers
// cannot live with that:
//   * a host application that has handed the whole device to its own allocator (a tensor framework's
//     caching allocator, a renderer, a process running under a fixed MPS / MIG memory limit), so that a
//     cudaMalloc made behind its back fails or starves it;
//   * a latency-critical loop (an intra-operative registration step, a real-time viewer) where the
//     device-wide synchronisation that cudaMalloc / cudaFree imply is not acceptable.
// For them this file holds the ONE piece of scratch the generic path cannot do without -- the
// nbins x nbins joint histogram in global memory that the resample kernel fills and the entropy kernel
// reads -- in a file-scope __device__ array, g_noalloc_scratch below.  The caller passes the two volumes
// and the outputs as DEVICE pointers it already owns; nothing here calls cudaMalloc, cudaFree,
// cudaMallocAsync or any other allocating routine.
//
// What it costs.  kScratchBytes (256 KB + 256 B) of device memory on every GPU on which this library's
// module is loaded, held until the process exits, whether or not this entry point is ever called.
//
// Rules that follow from one shared array (see include/mi.h for the user-facing statement):
//   * sizes: nbins <= 256, nq <= 8, one transform per call; anything larger is rejected with
//     MI_ERR_UNSUPPORTED and a message, never truncated;
//   * the array keeps what the previous call left in it, so every call clears the cells it is about to
//     use (noalloc_prepare_kernel) on the caller's stream before the histogram kernel runs;
//   * two calls that are in flight on the same GPU at the same time (two streams, two host threads, two
//     contexts of one process) use the SAME cells and corrupt each other: order them on one stream or
//     with events;
//   * the device address of the array is looked up once per device by the first call on that device
//     (cudaGetSymbolAddress with that device current), together with the shared-memory opt-in of the
//     kernel; make that first call during set-up, before any stream capture is begun.
//
// The arithmetic is DESIGN.md's CANON-2..5 restated for volumes that have not been pre-processed: the
// fixed voxel is binned on the fly, the moving neighbours are fetched from the caller's unpadded volume
// with the edge clamp written out, and the entropy reduction is the library's existing kernel reading
// the static histogram.  Results are bit-identical to mi_eval_batch's (tests/test_zz_no_alloc.py).
#include <cmath>
#include <mutex>
#include <string>

#include "mi_device.cuh"
#include "mi_internal.h"

namespace {

constexpr int kNoAllocMaxBins = 256;                 // largest nbins this entry point accepts
constexpr int kNoAllocMaxQ = mi::kMaxQPerPass;       // Tsallis orders per call (one entropy pass)
constexpr size_t kHeaderBytes = 256;                 // the q values live in front of the histogram
constexpr size_t kHistBytes = (size_t)kNoAllocMaxBins * kNoAllocMaxBins * sizeof(uint32_t);
constexpr size_t kScratchBytes = kHeaderBytes + kHistBytes;
constexpr int kThreads = 512;
constexpr size_t kSmemBudget = 200 * 1024;           // shared histogram rows per CTA (1 CTA per SM)

// The scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device
// address and must never be handed to a kernel or to cudaMemsetAsync as if it were one.
static __device__ __align__(256) unsigned char g_noalloc_scratch[kScratchBytes];

struct QList {
    double q[kNoAllocMaxQ];
};

struct NoAllocArgs {
    const float* fixed;      // [fz][fy][fx], caller's device memory
    const float* moving;     // [mz][my][mx], caller's device memory
    uint32_t* hist;          // the static histogram (device address from cudaGetSymbolAddress)
    float M[12];             // index-space affine (CANON-1), row-major [M | m0]
    int fnx, fny, fnz, mnx, mny, mnz;
    int nb, rows_smem;       // fixed-bin rows below rows_smem are counted in shared memory
    float flo, fscale, mlo, mscale;
};

// Clears the nb*nb histogram cells this call will use and stores the q values in the header.
__global__ void __launch_bounds__(256) noalloc_prepare_kernel(unsigned char* __restrict__ scratch, QList ql, int nq,
                                                              int ncells) {
    uint32_t* __restrict__ hist = reinterpret_cast<uint32_t*>(scratch + kHeaderBytes);
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < ncells; i += gridDim.x * blockDim.x) hist[i] = 0u;
    if (blockIdx.x == 0 && threadIdx.x < kNoAllocMaxQ)
        reinterpret_cast<double*>(scratch)[threadIdx.x] = threadIdx.x < nq ? ql.q[threadIdx.x] : 1.0;
}

// CANON-5: t = (v - lo) * scale with both roundings, floor, clamp to [0, nb-1].
__device__ __forceinline__ int canon_bin(float v, float lo, float scale, int nb) {
    const float t = __fmul_rn(__fsub_rn(v, lo), scale);
    return (int)fminf(fmaxf(floorf(t), 0.0f), (float)(nb - 1));
}
__device__ __forceinline__ float canon_lerp(float p, float q, float f) { return __fmaf_rn(f, __fsub_rn(q, p), p); }

// a3 + a4 for one transform.  A warp takes one fixed row (iy, iz) at a time, its lanes walk x.
// Counts of fixed bins below rows_smem are collected in this CTA's shared memory and merged into the
// static histogram when the CTA is done; the other rows (only when nb*nb*4 B exceeds the shared budget)
// go to the static histogram directly.
template <int INTERP>
__global__ void __launch_bounds__(kThreads, 1) noalloc_hist_kernel(const __grid_constant__ NoAllocArgs a) {
    extern __shared__ uint32_t sh_hist[];
    const int nb = a.nb;
    const int ncells_sh = a.rows_smem * nb;
    for (int i = threadIdx.x; i < ncells_sh; i += kThreads) sh_hist[i] = 0u;
    __syncthreads();

    const int lane = threadIdx.x & 31;
    const int warps_per_cta = kThreads / 32;
    const long long nrows = (long long)a.fny * a.fnz;
    const float fmx = (float)a.mnx, fmy = (float)a.mny, fmz = (float)a.mnz;
    for (long long row = (long long)blockIdx.x * warps_per_cta + (threadIdx.x >> 5); row < nrows;
         row += (long long)gridDim.x * warps_per_cta) {
        const int iz = (int)(row / a.fny), iy = (int)(row - (long long)iz * a.fny);
        const float fy = (float)iy, fz = (float)iz;
        // CANON-2: the part of the coordinate that is constant along the row
        const float rx = __fmaf_rn(a.M[1], fy, __fmaf_rn(a.M[2], fz, a.M[3]));
        const float ry = __fmaf_rn(a.M[5], fy, __fmaf_rn(a.M[6], fz, a.M[7]));
        const float rz = __fmaf_rn(a.M[9], fy, __fmaf_rn(a.M[10], fz, a.M[11]));
        const float* __restrict__ frow = a.fixed + (size_t)row * a.fnx;
        for (int ix = lane; ix < a.fnx; ix += 32) {
            const float fx = (float)ix;
            const float cx = __fmaf_rn(a.M[0], fx, rx), cy = __fmaf_rn(a.M[4], fx, ry), cz = __fmaf_rn(a.M[8], fx, rz);
            float v;
            if (INTERP == MI_INTERP_NEAREST) {
                // CANON-3: round half up, validity decided on the rounded float
                const float qx = floorf(__fadd_rn(cx, 0.5f)), qy = floorf(__fadd_rn(cy, 0.5f)),
                            qz = floorf(__fadd_rn(cz, 0.5f));
                if (!(qx >= 0.0f && qx < fmx && qy >= 0.0f && qy < fmy && qz >= 0.0f && qz < fmz)) continue;
                v = __ldg(a.moving + ((size_t)(int)qz * a.mny + (int)qy) * a.mnx + (int)qx);
            } else {
                // CANON-4: region [-0.5, n-0.5), neighbours clamped to the volume, x- then y- then z-lerps
                if (!(cx >= -0.5f && cx < fmx - 0.5f && cy >= -0.5f && cy < fmy - 0.5f && cz >= -0.5f && cz < fmz - 0.5f))
                    continue;
                const float gx = floorf(cx), gy = floorf(cy), gz = floorf(cz);
                const float wx = __fsub_rn(cx, gx), wy = __fsub_rn(cy, gy), wz = __fsub_rn(cz, gz);
                const int x0 = max((int)gx, 0), x1 = min((int)gx + 1, a.mnx - 1);
                const int y0 = max((int)gy, 0), y1 = min((int)gy + 1, a.mny - 1);
                const int z0 = max((int)gz, 0), z1 = min((int)gz + 1, a.mnz - 1);
                const float* __restrict__ p00 = a.moving + ((size_t)z0 * a.mny + y0) * a.mnx;
                const float* __restrict__ p10 = a.moving + ((size_t)z0 * a.mny + y1) * a.mnx;
                const float* __restrict__ p01 = a.moving + ((size_t)z1 * a.mny + y0) * a.mnx;
                const float* __restrict__ p11 = a.moving + ((size_t)z1 * a.mny + y1) * a.mnx;
                const float v00 = canon_lerp(__ldg(p00 + x0), __ldg(p00 + x1), wx);
                const float v10 = canon_lerp(__ldg(p10 + x0), __ldg(p10 + x1), wx);
                const float v01 = canon_lerp(__ldg(p01 + x0), __ldg(p01 + x1), wx);
                const float v11 = canon_lerp(__ldg(p11 + x0), __ldg(p11 + x1), wx);
                v = canon_lerp(canon_lerp(v00, v10, wy), canon_lerp(v01, v11, wy), wz);
            }
            const int fa = canon_bin(__ldg(frow + ix), a.flo, a.fscale, nb);
            const int mb = canon_bin(v, a.mlo, a.mscale, nb);
            if (fa < a.rows_smem) atomicAdd(&sh_hist[fa * nb + mb], 1u);   // CANON-6
            else atomicAdd(&a.hist[fa * nb + mb], 1u);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < ncells_sh; i += kThreads) {
        const uint32_t c = sh_hist[i];
        if (c != 0u) atomicAdd(&a.hist[i], c);
    }
}

// ---- per-device set-up ----------------------------------------------------------------------------
struct DeviceState {
    bool ready = false;
    unsigned char* scratch = nullptr;   // DEVICE address of g_noalloc_scratch on this device
    int num_sms = 0;
    size_t smem_optin = 0;
};
std::mutex g_setup_mutex;
DeviceState g_devices[64];

// Runs with `device` current.  cudaGetSymbolAddress is what turns the host-side stand-in of the array
// into the address the kernels may dereference; it differs from device to device.
cudaError_t device_setup(int device, const DeviceState** out) {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    DeviceState& d = g_devices[device];
    if (!d.ready) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (p == nullptr) return cudaErrorInvalidSymbol;
        int v = 0;
        if ((e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) return e;
        d.num_sms = v;
        if ((e = cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, device)) != cudaSuccess) return e;
        d.smem_optin = (size_t)v;
        const int optin = (int)(d.smem_optin < kSmemBudget ? d.smem_optin : kSmemBudget);
        if ((e = cudaFuncSetAttribute(noalloc_hist_kernel<MI_INTERP_NEAREST>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      optin)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(noalloc_hist_kernel<MI_INTERP_TRILINEAR>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      optin)) != cudaSuccess) return e;
        d.scratch = static_cast<unsigned char*>(p);
        d.ready = true;
    }
    *out = &d;
    return cudaSuccess;
}

struct ScopedDevice {
    int prev = -1;
    bool ok = false;
    explicit ScopedDevice(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; cudaGetLastError(); }
        ok = cudaSetDevice(dev) == cudaSuccess;
    }
    ~ScopedDevice() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

mi_status na_fail(mi_status s, const std::string& msg) {
    mi::set_thread_error("mi_eval_noalloc: " + msg);
    return s;
}
mi_status na_cuda_fail(cudaError_t e, const char* where) {
    cudaGetLastError();
    return na_fail(MI_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

}  // namespace

extern "C" mi_status mi_eval_noalloc(const float* fixed_dev, const int32_t fixed_dims[3], const double fixed_spacing[3],
                                     const float* moving_dev, const int32_t moving_dims[3],
                                     const double moving_spacing[3], int32_t nbins, float fixed_lo, float fixed_hi,
                                     float moving_lo, float moving_hi, const double T[12], const double* q, int32_t nq,
                                     mi_interp interp, mi_tsallis_form form, double* mi_out_dev, uint32_t* hist_out_dev,
                                     int64_t* nvalid_out_dev, int32_t device, void* cuda_stream) {
    if (!fixed_dev || !moving_dev || !fixed_dims || !moving_dims || !fixed_spacing || !moving_spacing || !T || !mi_out_dev)
        return na_fail(MI_ERR_INVALID_ARG, "NULL argument");
    if (nq < 0 || (nq > 0 && q == nullptr)) return na_fail(MI_ERR_INVALID_ARG, "nq < 0, or nq > 0 with q == NULL");
    if (nbins < 2) return na_fail(MI_ERR_INVALID_ARG, "nbins < 2");
    if (nbins > kNoAllocMaxBins)
        return na_fail(MI_ERR_UNSUPPORTED, "nbins = " + std::to_string(nbins) + " exceeds the static scratch (nbins <= " +
                                               std::to_string(kNoAllocMaxBins) + "); use mi_create + mi_eval_batch");
    if (nq > kNoAllocMaxQ)
        return na_fail(MI_ERR_UNSUPPORTED, "nq = " + std::to_string(nq) + " exceeds the limit of " +
                                               std::to_string(kNoAllocMaxQ) + " orders per call");
    if (interp != MI_INTERP_NEAREST && interp != MI_INTERP_TRILINEAR)
        return na_fail(MI_ERR_UNSUPPORTED, "interp must be MI_INTERP_NEAREST or MI_INTERP_TRILINEAR");
    if (form != MI_TSALLIS_ADDITIVE && form != MI_TSALLIS_PSEUDO_ADDITIVE) return na_fail(MI_ERR_INVALID_ARG, "unknown Tsallis form");
    int64_t nf = 1, nm = 1;
    for (int d = 0; d < 3; ++d) {
        if (fixed_dims[d] < 1 || moving_dims[d] < 1) return na_fail(MI_ERR_INVALID_ARG, "volume dim < 1");
        if (!(std::isfinite(fixed_spacing[d]) && fixed_spacing[d] > 0.0) ||
            !(std::isfinite(moving_spacing[d]) && moving_spacing[d] > 0.0))
            return na_fail(MI_ERR_INVALID_ARG, "spacing must be finite and > 0");
        nf *= fixed_dims[d];
        nm *= moving_dims[d];
        if (nf > 0x7FFFFFFFLL || nm > 0x7FFFFFFFLL) return na_fail(MI_ERR_UNSUPPORTED, "volume has more than 2^31-1 voxels");
    }
    if (!(std::isfinite(fixed_lo) && std::isfinite(fixed_hi) && fixed_lo < fixed_hi) ||
        !(std::isfinite(moving_lo) && std::isfinite(moving_hi) && moving_lo < moving_hi))
        return na_fail(MI_ERR_INVALID_ARG, "intensity range must be finite with lo < hi");
    for (int i = 0; i < 12; ++i)
        if (!std::isfinite(T[i])) return na_fail(MI_ERR_INVALID_ARG, "non-finite matrix entry");
    QList ql;
    for (int k = 0; k < kNoAllocMaxQ; ++k) ql.q[k] = 1.0;
    for (int k = 0; k < nq; ++k) {
        if (!(std::isfinite(q[k]) && q[k] > 0.0 && q[k] <= 32.0)) return na_fail(MI_ERR_INVALID_ARG, "q must be finite, > 0 and <= 32");
        ql.q[k] = q[k];
    }

    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess) return na_cuda_fail(e, "cudaGetDeviceCount");
    if (device < 0 || device >= ndev || device >= 64) return na_fail(MI_ERR_INVALID_ARG, "no such CUDA device");
    ScopedDevice guard(device);
    if (!guard.ok) return na_fail(MI_ERR_CUDA, "cudaSetDevice failed");
    // Host data cannot be staged without a device buffer, and there is none to stage it in.
    if (mi::is_host_pointer(fixed_dev) || mi::is_host_pointer(moving_dev) || mi::is_host_pointer(mi_out_dev) ||
        (hist_out_dev && mi::is_host_pointer(hist_out_dev)) || (nvalid_out_dev && mi::is_host_pointer(nvalid_out_dev)))
        return na_fail(MI_ERR_INVALID_ARG, "volumes and outputs must be device pointers (nothing can be staged without allocating)");

    const DeviceState* dev = nullptr;
    if ((e = device_setup(device, &dev)) != cudaSuccess) return na_cuda_fail(e, "set-up of the static scratch");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);

    NoAllocArgs a;
    a.fixed = fixed_dev;
    a.moving = moving_dev;
    a.hist = reinterpret_cast<uint32_t*>(dev->scratch + kHeaderBytes);
    mi::index_affine(T, fixed_dims, fixed_spacing, moving_dims, moving_spacing, a.M);
    a.fnx = fixed_dims[0]; a.fny = fixed_dims[1]; a.fnz = fixed_dims[2];
    a.mnx = moving_dims[0]; a.mny = moving_dims[1]; a.mnz = moving_dims[2];
    a.nb = nbins;
    a.flo = fixed_lo; a.fscale = mi::bin_scale(nbins, fixed_lo, fixed_hi);
    a.mlo = moving_lo; a.mscale = mi::bin_scale(nbins, moving_lo, moving_hi);
    const size_t budget = dev->smem_optin < kSmemBudget ? dev->smem_optin : kSmemBudget;
    const size_t row_bytes = (size_t)nbins * sizeof(uint32_t);
    a.rows_smem = (int)(budget / row_bytes < (size_t)nbins ? budget / row_bytes : (size_t)nbins);
    const size_t smem = (size_t)a.rows_smem * row_bytes;

    const int ncells = nbins * nbins;
    noalloc_prepare_kernel<<<(ncells + 255) / 256, 256, 0, s>>>(dev->scratch, ql, nq, ncells);
    if ((e = cudaGetLastError()) != cudaSuccess) return na_cuda_fail(e, "noalloc_prepare_kernel");

    const long long nrows = (long long)a.fny * a.fnz;
    long long grid = (nrows + kThreads / 32 - 1) / (kThreads / 32);
    if (grid > dev->num_sms) grid = dev->num_sms;   // one CTA per SM, each keeps its own shared histogram
    if (grid < 1) grid = 1;
    if (interp == MI_INTERP_NEAREST) noalloc_hist_kernel<MI_INTERP_NEAREST><<<(unsigned)grid, kThreads, smem, s>>>(a);
    else noalloc_hist_kernel<MI_INTERP_TRILINEAR><<<(unsigned)grid, kThreads, smem, s>>>(a);
    if ((e = cudaGetLastError()) != cudaSuccess) return na_cuda_fail(e, "noalloc_hist_kernel");

    // a5 from the static histogram with the library's entropy kernel (no scratch of its own at nbins <= 256)
    mi::OutMap om = {};
    e = mi::launch_entropy(a.hist, nbins, 1, reinterpret_cast<const double*>(dev->scratch), nq, 0, (int)form, mi_out_dev,
                           nvalid_out_dev, om, s);
    if (e != cudaSuccess) return na_cuda_fail(e, "entropy_kernel");
    if (hist_out_dev != nullptr) {
        e = cudaMemcpyAsync(hist_out_dev, a.hist, (size_t)ncells * sizeof(uint32_t), cudaMemcpyDeviceToDevice, s);
        if (e != cudaSuccess) return na_cuda_fail(e, "copy of the histogram");
    }
    return MI_OK;
}
