// mi_analysis.cu -- capture-range analysis of an exhaustive map: the paper reads
// its maps through the paths a gradient descent takes on them and the regions that converge to the
// ground truth (Figs. 2-5).  Two exact, parameter-free read-outs (A17):
//   gradient_kernel   finite-difference gradient field in parameter units
//   basin_*_kernel    discrete steepest ascent / descent: best-neighbour pointers, pointer doubling
//                     to the extremum each node reaches (+ path lengths), arg max, statistics
// Everything is integer / compare work on doubles or IEEE double subtract + divide: the results are
// reproducible bit for bit on any IEEE machine.
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include <cmath>
#include <string>

#include "mi_internal.h"

namespace mi {
namespace {

struct Grid3 {
    int n0, n1, n2;
};

// ---- gradient -----------------------------------------------------------------------------------
// One thread per node; component d = (M[k+1] - M[k-1]) / (2 h_d) inside, one-sided on the faces.
// The map is read through L1/L2 (7 reads per node, 6 of them neighbours), the field is streamed out.
__global__ void __launch_bounds__(256) gradient_kernel(const double* __restrict__ m, Grid3 g, double h0, double h1,
                                                       double h2, double* __restrict__ out) {
    const int64_t total = (int64_t)g.n0 * g.n1 * g.n2;
    const int64_t s1 = g.n0, s2 = (int64_t)g.n0 * g.n1;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
        const int k0 = (int)(t % g.n0);
        const int64_t r = t / g.n0;
        const int k1 = (int)(r % g.n1), k2 = (int)(r / g.n1);
        auto diff = [&](int k, int n, int64_t stride, double h) -> double {
            if (n == 1) return 0.0;
            if (k == 0) return __ddiv_rn(__dsub_rn(m[t + stride], m[t]), h);
            if (k == n - 1) return __ddiv_rn(__dsub_rn(m[t], m[t - stride]), h);
            return __ddiv_rn(__dsub_rn(m[t + stride], m[t - stride]), __dmul_rn(2.0, h));
        };
        out[t] = diff(k0, g.n0, 1, h0);
        out[total + t] = diff(k1, g.n1, s1, h1);
        out[2 * total + t] = diff(k2, g.n2, s2, h2);
    }
}

// ---- basins -------------------------------------------------------------------------------------
// next[t]: neighbours are visited in increasing linear index; a candidate replaces the best so far
// only if strictly better, so the node itself wins ties and among neighbours the lowest index does.
// dist[t] = 1 if the node moves, else 0.
__global__ void __launch_bounds__(256) basin_next_kernel(const double* __restrict__ m, Grid3 g, double sign,
                                                         int conn, int* __restrict__ next, int* __restrict__ dist) {
    const int total = g.n0 * g.n1 * g.n2;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < total; t += gridDim.x * blockDim.x) {
        const int k0 = t % g.n0;
        const int r = t / g.n0;
        const int k1 = r % g.n1, k2 = r / g.n1;
        double best = sign * m[t];
        int bi = t;
        for (int d2 = -1; d2 <= 1; ++d2) {
            const int q2 = k2 + d2;
            if (q2 < 0 || q2 >= g.n2) continue;
            for (int d1 = -1; d1 <= 1; ++d1) {
                const int q1 = k1 + d1;
                if (q1 < 0 || q1 >= g.n1) continue;
                for (int d0 = -1; d0 <= 1; ++d0) {
                    const int q0 = k0 + d0;
                    if (q0 < 0 || q0 >= g.n0) continue;
                    const int nz = (d2 != 0) + (d1 != 0) + (d0 != 0);
                    if (nz == 0 || (conn == 6 && nz != 1)) continue;
                    const int q = (q2 * g.n1 + q1) * g.n0 + q0;
                    const double v = sign * m[q];
                    if (v > best) { best = v; bi = q; }
                }
            }
        }
        next[t] = bi;
        dist[t] = bi != t ? 1 : 0;
    }
}

// One round of pointer doubling (ping-pong buffers): ptr'[t] = ptr[ptr[t]], dist'[t] = dist[t] +
// dist[ptr[t]] (dist[t] is the number of moves from t to ptr[t]).  *changed is set if any pointer moved.
__global__ void __launch_bounds__(256) basin_jump_kernel(const int* __restrict__ ptr, const int* __restrict__ dist,
                                                         int total, int* __restrict__ ptr_out,
                                                         int* __restrict__ dist_out, int* __restrict__ changed) {
    bool any = false;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < total; t += gridDim.x * blockDim.x) {
        const int p = ptr[t];
        const int pp = ptr[p];
        ptr_out[t] = pp;
        dist_out[t] = dist[t] + dist[p];
        any |= pp != p;
    }
    if (__any_sync(0xffffffffu, any) && (threadIdx.x & 31) == 0) atomicOr(changed, 1);
}

// Global extremum of sign*m, lowest index on ties (one CTA).
__global__ void __launch_bounds__(1024) basin_argmax_kernel(const double* __restrict__ m, int total, double sign,
                                                            int* __restrict__ out) {
    __shared__ double sv[1024];
    __shared__ int si[1024];
    double best = -CUDART_INF;
    int bi = total;
    for (int t = threadIdx.x; t < total; t += blockDim.x) {
        const double v = sign * m[t];
        if (v > best || bi == total) { best = v; bi = t; }   // t ascends per thread: first maximum kept
    }
    sv[threadIdx.x] = best;
    si[threadIdx.x] = bi;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            const double v2 = sv[threadIdx.x + o];
            const int i2 = si[threadIdx.x + o];
            const bool take = i2 < total && (si[threadIdx.x] == total || v2 > sv[threadIdx.x] ||
                                             (v2 == sv[threadIdx.x] && i2 < si[threadIdx.x]));
            if (take) { sv[threadIdx.x] = v2; si[threadIdx.x] = i2; }
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = si[0] < total ? si[0] : 0;
}

// stats[0] = extrema (next[t] == t), stats[1] = captured (label[t] == label[target]), stats[2] = max steps;
// also widens the labels to int64 for the caller.
__global__ void __launch_bounds__(256) basin_stats_kernel(const int* __restrict__ next, const int* __restrict__ label,
                                                          const int* __restrict__ steps, int total,
                                                          const int* __restrict__ target, int64_t* __restrict__ label64,
                                                          unsigned long long* __restrict__ stats) {
    const int tl = label[target[0]];
    unsigned ext = 0, cap = 0;
    int mx = 0;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < total; t += gridDim.x * blockDim.x) {
        const int l = label[t];
        ext += next[t] == t;
        cap += l == tl;
        mx = max(mx, steps[t]);
        if (label64 != nullptr) label64[t] = (int64_t)l;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ext += __shfl_xor_sync(0xffffffffu, ext, o);
        cap += __shfl_xor_sync(0xffffffffu, cap, o);
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((threadIdx.x & 31) == 0) {
        if (ext) atomicAdd(&stats[0], (unsigned long long)ext);
        if (cap) atomicAdd(&stats[1], (unsigned long long)cap);
        atomicMax(&stats[2], (unsigned long long)mx);
        if (blockIdx.x == 0 && threadIdx.x == 0) stats[3] = (unsigned long long)tl;
    }
}

unsigned grid_for(int64_t total, int block) {
    int64_t b = (total + block - 1) / block;
    if (b < 1) b = 1;
    if (b > sm_count() * 8) b = sm_count() * 8;
    return (unsigned)b;
}

}  // namespace
}  // namespace mi

// ---- C ABI --------------------------------------------------------------------------------------
namespace {

struct Guard {   // device switch + scratch owned by one call
    int prev = -1;
    bool ok = false;
    cudaStream_t s = nullptr;
    void* bufs[12];
    int nbufs = 0;
    Guard(int dev, cudaStream_t st) : s(st) {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; cudaGetLastError(); }
        ok = cudaSetDevice(dev) == cudaSuccess;
    }
    cudaError_t alloc(void** p, size_t bytes, int dev) {
        cudaError_t e = mi::dev_alloc(p, bytes, dev, s);
        if (e == cudaSuccess) bufs[nbufs++] = *p;
        return e;
    }
    ~Guard() {
        if (ok) {
            for (int i = 0; i < nbufs; ++i) mi::dev_free(bufs[i], s);
            cudaStreamSynchronize(s);
            cudaGetLastError();
        }
        if (prev >= 0) cudaSetDevice(prev);
    }
};

mi_status bad(mi_status st, const std::string& msg) {
    mi::set_thread_error(msg);
    return st;
}
mi_status cuda_bad(cudaError_t e, const char* where) {
    cudaGetLastError();
    mi::set_thread_error(std::string(where) + ": " + cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? MI_ERR_OUT_OF_MEMORY : MI_ERR_CUDA;
}
#define AN_CUDA(call)                                           \
    do {                                                        \
        cudaError_t e__ = (call);                               \
        if (e__ != cudaSuccess) return cuda_bad(e__, #call);    \
    } while (0)

mi_status check_common(const double* map, const int32_t n[3], int32_t device, int64_t* total) {
    if (map == nullptr || n == nullptr) return bad(MI_ERR_INVALID_ARG, "NULL argument");
    int64_t t = 1;
    for (int d = 0; d < 3; ++d) {
        if (n[d] < 1) return bad(MI_ERR_INVALID_ARG, "grid n < 1");
        t *= n[d];
        if (t > 0x7FFFFFFFLL) return bad(MI_ERR_UNSUPPORTED, "map has more than 2^31-1 nodes");
    }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess) return cuda_bad(e, "cudaGetDeviceCount");
    if (device < 0 || device >= ndev) return bad(MI_ERR_INVALID_ARG, "no such CUDA device");
    *total = t;
    return MI_OK;
}

}  // namespace

extern "C" {

mi_status mi_map_gradient(const double* map, const int32_t n[3], const double lo[3], const double hi[3],
                          double* grad_out, int32_t device, void* cuda_stream) {
    if (lo == nullptr || hi == nullptr || grad_out == nullptr) return bad(MI_ERR_INVALID_ARG, "NULL argument");
    int64_t total = 0;
    mi_status st = check_common(map, n, device, &total);
    if (st != MI_OK) return st;
    double h[3];
    for (int d = 0; d < 3; ++d) {
        if (!std::isfinite(lo[d]) || !std::isfinite(hi[d])) return bad(MI_ERR_INVALID_ARG, "non-finite grid bound");
        h[d] = n[d] == 1 ? 1.0 : (hi[d] - lo[d]) / (double)(n[d] - 1);
        if (n[d] > 1 && !(h[d] != 0.0 && std::isfinite(h[d]))) return bad(MI_ERR_INVALID_ARG, "grid step is zero");
    }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    Guard g(device, s);
    if (!g.ok) return bad(MI_ERR_CUDA, "cudaSetDevice failed");
    const double* dmap = map;
    if (mi::is_host_pointer(map)) {
        void* p = nullptr;
        AN_CUDA(g.alloc(&p, (size_t)total * sizeof(double), device));
        AN_CUDA(cudaMemcpyAsync(p, map, (size_t)total * sizeof(double), cudaMemcpyHostToDevice, s));
        dmap = static_cast<const double*>(p);
    }
    double* dout = grad_out;
    const bool out_host = mi::is_host_pointer(grad_out);
    if (out_host) {
        void* p = nullptr;
        AN_CUDA(g.alloc(&p, (size_t)total * 3 * sizeof(double), device));
        dout = static_cast<double*>(p);
    }
    mi::gradient_kernel<<<mi::grid_for(total, 256), 256, 0, s>>>(dmap, mi::Grid3{n[0], n[1], n[2]}, h[0], h[1], h[2], dout);
    AN_CUDA(cudaGetLastError());
    if (out_host) AN_CUDA(cudaMemcpyAsync(grad_out, dout, (size_t)total * 3 * sizeof(double), cudaMemcpyDeviceToHost, s));
    AN_CUDA(cudaStreamSynchronize(s));
    return MI_OK;
}

mi_status mi_map_basins(const double* map, const int32_t n[3], int32_t direction, int32_t connectivity,
                        int64_t target, int64_t* label_out, int32_t* steps_out, mi_basin_stats* stats_out,
                        int32_t device, void* cuda_stream) {
    int64_t total64 = 0;
    mi_status st = check_common(map, n, device, &total64);
    if (st != MI_OK) return st;
    if (direction != 1 && direction != -1) return bad(MI_ERR_INVALID_ARG, "direction must be +1 or -1");
    if (connectivity != 6 && connectivity != 26) return bad(MI_ERR_INVALID_ARG, "connectivity must be 6 or 26");
    if (target < -1 || target >= total64) return bad(MI_ERR_INVALID_ARG, "target is not a node of the map");
    const int total = (int)total64;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    Guard g(device, s);
    if (!g.ok) return bad(MI_ERR_CUDA, "cudaSetDevice failed");
    const double* dmap = map;
    if (mi::is_host_pointer(map)) {
        void* p = nullptr;
        AN_CUDA(g.alloc(&p, (size_t)total * sizeof(double), device));
        AN_CUDA(cudaMemcpyAsync(p, map, (size_t)total * sizeof(double), cudaMemcpyHostToDevice, s));
        dmap = static_cast<const double*>(p);
    }
    int *next = nullptr, *ptr[2] = {nullptr, nullptr}, *dist[2] = {nullptr, nullptr}, *flags = nullptr;
    unsigned long long* stats = nullptr;
    AN_CUDA(g.alloc((void**)&next, (size_t)total * sizeof(int), device));
    for (int k = 0; k < 2; ++k) {
        AN_CUDA(g.alloc((void**)&ptr[k], (size_t)total * sizeof(int), device));
        AN_CUDA(g.alloc((void**)&dist[k], (size_t)total * sizeof(int), device));
    }
    AN_CUDA(g.alloc((void**)&flags, 64 * sizeof(int), device));     // [0] target node, [1 + it] changed in round it
    AN_CUDA(g.alloc((void**)&stats, 4 * sizeof(unsigned long long), device));
    AN_CUDA(cudaMemsetAsync(flags, 0, 64 * sizeof(int), s));
    AN_CUDA(cudaMemsetAsync(stats, 0, 4 * sizeof(unsigned long long), s));

    const mi::Grid3 grid{n[0], n[1], n[2]};
    const unsigned blocks = mi::grid_for(total, 256);
    mi::basin_next_kernel<<<blocks, 256, 0, s>>>(dmap, grid, (double)direction, connectivity, next, dist[0]);
    AN_CUDA(cudaGetLastError());
    AN_CUDA(cudaMemcpyAsync(ptr[0], next, (size_t)total * sizeof(int), cudaMemcpyDeviceToDevice, s));
    if (target < 0) {
        mi::basin_argmax_kernel<<<1, 1024, 0, s>>>(dmap, total, (double)direction, flags);
        AN_CUDA(cudaGetLastError());
    } else {
        const int t32 = (int)target;
        AN_CUDA(cudaMemcpyAsync(flags, &t32, sizeof(int), cudaMemcpyHostToDevice, s));
        AN_CUDA(cudaStreamSynchronize(s));   // t32 lives on this stack frame
    }
    // pointer doubling: after round r every pointer has advanced 2^r moves (or reached its extremum);
    // paths are shorter than 2^31 nodes, so 32 rounds always suffice.  Rounds are launched four at a
    // time between looks at the "changed" flags.
    int cur = 0, rounds = 0;
    bool done = false;
    while (!done && rounds < 32) {
        const int first = rounds;
        for (int k = 0; k < 4 && rounds < 32; ++k, ++rounds) {
            mi::basin_jump_kernel<<<blocks, 256, 0, s>>>(ptr[cur], dist[cur], total, ptr[cur ^ 1], dist[cur ^ 1],
                                                        flags + 1 + rounds);
            AN_CUDA(cudaGetLastError());
            cur ^= 1;
        }
        int h_changed[4] = {0, 0, 0, 0};
        AN_CUDA(cudaMemcpyAsync(h_changed, flags + 1 + first, (size_t)(rounds - first) * sizeof(int),
                                cudaMemcpyDeviceToHost, s));
        AN_CUDA(cudaStreamSynchronize(s));
        for (int k = 0; k < rounds - first; ++k)
            if (!h_changed[k]) done = true;
    }
    int64_t* dlabel = label_out;
    const bool label_host = label_out != nullptr && mi::is_host_pointer(label_out);
    if (label_host) AN_CUDA(g.alloc((void**)&dlabel, (size_t)total * sizeof(int64_t), device));
    mi::basin_stats_kernel<<<blocks, 256, 0, s>>>(next, ptr[cur], dist[cur], total, flags, dlabel, stats);
    AN_CUDA(cudaGetLastError());
    if (label_host)
        AN_CUDA(cudaMemcpyAsync(label_out, dlabel, (size_t)total * sizeof(int64_t), cudaMemcpyDeviceToHost, s));
    if (steps_out != nullptr)
        AN_CUDA(cudaMemcpyAsync(steps_out, dist[cur], (size_t)total * sizeof(int32_t), cudaMemcpyDefault, s));
    unsigned long long h_stats[4] = {0, 0, 0, 0};
    int h_target = 0;
    AN_CUDA(cudaMemcpyAsync(h_stats, stats, sizeof(h_stats), cudaMemcpyDeviceToHost, s));
    AN_CUDA(cudaMemcpyAsync(&h_target, flags, sizeof(int), cudaMemcpyDeviceToHost, s));
    AN_CUDA(cudaStreamSynchronize(s));
    if (stats_out != nullptr) {
        stats_out->n_extrema = (int64_t)h_stats[0];
        stats_out->captured = (int64_t)h_stats[1];
        stats_out->max_steps = (int32_t)h_stats[2];
        stats_out->target_label = (int64_t)h_stats[3];
        stats_out->target = (int64_t)h_target;
        stats_out->capture_fraction = (double)h_stats[1] / (double)total;
        stats_out->iterations = rounds;
    }
    return MI_OK;
}

}  // extern "C"
