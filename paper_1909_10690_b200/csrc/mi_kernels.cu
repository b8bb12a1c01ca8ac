// mi_kernels.cu -- the CUDA kernels of the exhaustive-MI-map hot path (sm_100a).
//
//   a1 prebin_kernel          fixed/moving float32 -> uint8 bin indices (HBM streaming, 16-byte vectors)
//   a3+a4 resample_hist_kernel  per transform: continuous index of every fixed voxel, trilinear or
//                             nearest sample of the moving volume, CTA-private joint histogram in
//                             shared memory, merge to global
//   a5 entropy_kernel         joint histogram -> marginals, sum c ln c, sum c^q -> Shannon and
//                             Tsallis MI (eq. 1-2; "same histogram" PAPER.md:199)
//   a6 map_assemble_kernel    channel-major 3D parameter image + arg max (eq. 3)
//
// Every fp32 operation that decides a voxel or a bin uses an explicitly rounded intrinsic
// (__fmaf_rn, __fadd_rn, __fsub_rn, __fmul_rn) so -fmad contraction cannot change it; the sequence
// is DESIGN.md CANON-2..5.
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "mi_internal.h"

namespace mi {

// ------------------------------------------------------------------------------------------------
// a1: pre-binning (DESIGN.md CANON-5)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int bin_index(float v, float lo, float scale, float top) {
    const float t = __fmul_rn(__fsub_rn(v, lo), scale);
    const float f = fminf(fmaxf(floorf(t), 0.0f), top);
    return __float2int_rz(f);
}

// Each thread turns 16 consecutive floats (4 x 16-byte loads) into one 16-byte store.
__global__ void __launch_bounds__(256) prebin_kernel(const float* __restrict__ vol,
                                                     uint8_t* __restrict__ bins, int64_t n, float lo,
                                                     float scale, float top) {
    const int64_t nvec = n >> 4;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const float4* src = reinterpret_cast<const float4*>(vol) + i * 4;
        float4 v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = __ldcs(src + k);
        uint32_t w[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            w[k] = (uint32_t)bin_index(v[k].x, lo, scale, top) |
                   ((uint32_t)bin_index(v[k].y, lo, scale, top) << 8) |
                   ((uint32_t)bin_index(v[k].z, lo, scale, top) << 16) |
                   ((uint32_t)bin_index(v[k].w, lo, scale, top) << 24);
        }
        reinterpret_cast<uint4*>(bins)[i] = make_uint4(w[0], w[1], w[2], w[3]);
    }
    // ragged tail (< 16 voxels), one thread each
    const int64_t tail0 = nvec << 4;
    const int64_t j = tail0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) bins[j] = (uint8_t)bin_index(vol[j], lo, scale, top);
}

cudaError_t launch_prebin(const float* vol, uint8_t* bins, int64_t n, float lo, float scale, int nb,
                          cudaStream_t s) {
    if (n <= 0) return cudaSuccess;
    const int64_t nvec = n >> 4;
    int64_t blocks = (nvec + 255) / 256;
    if (blocks < 1) blocks = 1;
    if (blocks > 148 * 16) blocks = 148 * 16;
    prebin_kernel<<<(unsigned)blocks, 256, 0, s>>>(vol, bins, n, lo, scale, (float)(nb - 1));
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a3 + a4: resample + joint histogram
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned warp_sum(unsigned v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// CANON-4 lerp: L(p,q,f) = fma(f, q - p, p) with q - p rounded first.
__device__ __forceinline__ float lerp_rn(float p, float q, float f) {
    return __fmaf_rn(f, __fsub_rn(q, p), p);
}

struct MovingView {
    const float* __restrict__ vol;
    const uint8_t* __restrict__ bins;
    int nx, ny, nz;
    float fx, fy, fz;  // (float)n
    float lo, scale, top;
};

// Moving bin of the sample at continuous index (cx,cy,cz), or -1 if it is outside the volume.
// All loads use clamped (always in-bounds) addresses so they can be issued before the validity
// test resolves.
template <int INTERP>
__device__ __forceinline__ int sample_bin(const MovingView& mv, float cx, float cy, float cz) {
    if (INTERP == MI_INTERP_NEAREST) {
        // CANON-3: round half up, validity tested in float.
        const float rx = floorf(__fadd_rn(cx, 0.5f));
        const float ry = floorf(__fadd_rn(cy, 0.5f));
        const float rz = floorf(__fadd_rn(cz, 0.5f));
        const bool ok = rx >= 0.0f && rx < mv.fx && ry >= 0.0f && ry < mv.fy && rz >= 0.0f && rz < mv.fz;
        const int jx = min(max(__float2int_rz(rx), 0), mv.nx - 1);
        const int jy = min(max(__float2int_rz(ry), 0), mv.ny - 1);
        const int jz = min(max(__float2int_rz(rz), 0), mv.nz - 1);
        const int b = __ldg(mv.bins + ((jz * mv.ny + jy) * mv.nx + jx));
        return ok ? b : -1;
    } else {
        // CANON-4: region [-0.5, n-0.5), edge clamp, x-lerps then y-lerps then the z-lerp.
        const bool ok = cx >= -0.5f && cx < __fsub_rn(mv.fx, 0.5f) && cy >= -0.5f &&
                        cy < __fsub_rn(mv.fy, 0.5f) && cz >= -0.5f && cz < __fsub_rn(mv.fz, 0.5f);
        const float gx = floorf(cx), gy = floorf(cy), gz = floorf(cz);
        const float tx = __fsub_rn(cx, gx), ty = __fsub_rn(cy, gy), tz = __fsub_rn(cz, gz);
        const int jx = __float2int_rz(gx), jy = __float2int_rz(gy), jz = __float2int_rz(gz);
        const int x0 = min(max(jx, 0), mv.nx - 1), x1 = max(min(jx + 1, mv.nx - 1), 0);
        const int y0 = min(max(jy, 0), mv.ny - 1), y1 = max(min(jy + 1, mv.ny - 1), 0);
        const int z0 = min(max(jz, 0), mv.nz - 1), z1 = max(min(jz + 1, mv.nz - 1), 0);
        const int r00 = (z0 * mv.ny + y0) * mv.nx, r10 = (z0 * mv.ny + y1) * mv.nx;
        const int r01 = (z1 * mv.ny + y0) * mv.nx, r11 = (z1 * mv.ny + y1) * mv.nx;
        const float a000 = __ldg(mv.vol + r00 + x0), a100 = __ldg(mv.vol + r00 + x1);
        const float a010 = __ldg(mv.vol + r10 + x0), a110 = __ldg(mv.vol + r10 + x1);
        const float a001 = __ldg(mv.vol + r01 + x0), a101 = __ldg(mv.vol + r01 + x1);
        const float a011 = __ldg(mv.vol + r11 + x0), a111 = __ldg(mv.vol + r11 + x1);
        const float v00 = lerp_rn(a000, a100, tx);
        const float v10 = lerp_rn(a010, a110, tx);
        const float v01 = lerp_rn(a001, a101, tx);
        const float v11 = lerp_rn(a011, a111, tx);
        const float w0 = lerp_rn(v00, v10, ty);
        const float w1 = lerp_rn(v01, v11, ty);
        const float v = lerp_rn(w0, w1, tz);
        const int b = bin_index(v, mv.lo, mv.scale, mv.top);
        return ok ? b : -1;
    }
}

// CTA-private histogram update.  PACK16: two 16-bit counters per word (256 bins -> 128 KB); a
// counter that reaches 2^15 is drained to the global histogram by the thread whose add set bit 15,
// so counters never carry into their neighbour (at most 1024 adds can land before the drain).
template <bool PACK16>
__device__ __forceinline__ void hist_add(uint32_t* sh, uint32_t* gh, int idx) {
    if (PACK16) {
        const unsigned shift = (idx & 1) << 4;
        const unsigned old = atomicAdd(&sh[idx >> 1], 1u << shift);
        if (((old >> shift) & 0xFFFFu) == 0x7FFFu) {
            atomicSub(&sh[idx >> 1], 0x8000u << shift);
            atomicAdd(&gh[idx], 0x8000u);
        }
    } else {
        atomicAdd(&sh[idx], 1u);
    }
}

template <int INTERP, bool PACK16, int UNROLL>
__global__ void __launch_bounds__(kHistThreads, 1)
resample_hist_kernel(const __grid_constant__ ResampleArgs a) {
    extern __shared__ __align__(16) uint32_t sh_hist[];
    const int nb = a.nb;
    const int nbins2 = nb * nb;
    const int words = PACK16 ? (nbins2 + 1) / 2 : nbins2;
    for (int w = threadIdx.x; w < words; w += blockDim.x) sh_hist[w] = 0u;
    __syncthreads();

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    const int fnx = a.f.nx;
    const int rows_total = a.f.ny * a.f.nz;

    MovingView mv;
    mv.vol = a.moving;
    mv.bins = a.mbins;
    mv.nx = a.m.nx; mv.ny = a.m.ny; mv.nz = a.m.nz;
    mv.fx = (float)a.m.nx; mv.fy = (float)a.m.ny; mv.fz = (float)a.m.nz;
    mv.lo = a.mlo; mv.scale = a.mscale; mv.top = (float)(nb - 1);

    const long long nitems = (long long)a.n_transforms * a.nslabs;
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int t = (int)(item / a.nslabs);
        const int slab = (int)(item - (long long)t * a.nslabs);
        const int row_lo = (int)((long long)rows_total * slab / a.nslabs);
        const int row_hi = (int)((long long)rows_total * (slab + 1) / a.nslabs);
        float m[12];
#pragma unroll
        for (int i = 0; i < 12; ++i) m[i] = __ldg(a.M + (size_t)t * 12 + i);
        uint32_t* gh = a.hist + (size_t)t * nbins2;
        unsigned cnt0 = 0;  // private count of bin (0,0): the background-on-background hot spot

        for (int row = row_lo + warp; row < row_hi; row += nwarps) {
            const int iz = row / a.f.ny;
            const int iy = row - iz * a.f.ny;
            const float fy = (float)iy, fz = (float)iz;
            // CANON-2: row terms, then one fma per voxel and axis
            const float rx = __fmaf_rn(m[1], fy, __fmaf_rn(m[2], fz, m[3]));
            const float ry = __fmaf_rn(m[5], fy, __fmaf_rn(m[6], fz, m[7]));
            const float rz = __fmaf_rn(m[9], fy, __fmaf_rn(m[10], fz, m[11]));
            const uint8_t* __restrict__ frow = a.fbins + (size_t)row * fnx;
            for (int ix0 = lane; ix0 < fnx; ix0 += 32 * UNROLL) {
                int idx[UNROLL];
#pragma unroll
                for (int u = 0; u < UNROLL; ++u) {
                    const int ix = ix0 + 32 * u;
                    idx[u] = -1;
                    if (ix < fnx) {
                        const float fx = (float)ix;
                        const float cx = __fmaf_rn(m[0], fx, rx);
                        const float cy = __fmaf_rn(m[4], fx, ry);
                        const float cz = __fmaf_rn(m[8], fx, rz);
                        const int b = sample_bin<INTERP>(mv, cx, cy, cz);
                        const int fa = __ldg(frow + ix);
                        idx[u] = b >= 0 ? fa * nb + b : -1;
                    }
                }
#pragma unroll
                for (int u = 0; u < UNROLL; ++u) {
                    if (idx[u] == 0) ++cnt0;
                    else if (idx[u] > 0) hist_add<PACK16>(sh_hist, gh, idx[u]);
                }
            }
        }
        cnt0 = warp_sum(cnt0);
        if (lane == 0 && cnt0) atomicAdd(gh, cnt0);
        __syncthreads();
        // merge the CTA-private histogram into the transform's global histogram and re-zero it
        for (int w = threadIdx.x; w < words; w += blockDim.x) {
            const uint32_t v = sh_hist[w];
            if (v) {
                sh_hist[w] = 0u;
                if (PACK16) {
                    if (v & 0xFFFFu) atomicAdd(&gh[2 * w], v & 0xFFFFu);
                    if (v >> 16) atomicAdd(&gh[2 * w + 1], v >> 16);
                } else {
                    atomicAdd(&gh[w], v);
                }
            }
        }
        __syncthreads();
    }
}

template <int INTERP, bool PACK16, int UNROLL>
static cudaError_t launch_resample_t(const ResampleArgs& a, int num_sms, size_t smem_optin,
                                     cudaStream_t s) {
    const size_t nbins2 = (size_t)a.nb * a.nb;
    const size_t smem = (PACK16 ? (nbins2 + 1) / 2 : nbins2) * sizeof(uint32_t);
    if (smem > smem_optin) return cudaErrorInvalidConfiguration;
    auto kern = resample_hist_kernel<INTERP, PACK16, UNROLL>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long nitems = (long long)a.n_transforms * a.nslabs;
    long long grid = nitems < num_sms ? nitems : num_sms;
    if (grid < 1) return cudaSuccess;
    kern<<<(unsigned)grid, kHistThreads, smem, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_resample_hist(const ResampleArgs& a, int interp, int num_sms, size_t smem_optin,
                                 cudaStream_t s) {
    const bool pack16 = (size_t)a.nb * a.nb * sizeof(uint32_t) > 96 * 1024;
    if (interp == MI_INTERP_NEAREST) {
        return pack16 ? launch_resample_t<MI_INTERP_NEAREST, true, 4>(a, num_sms, smem_optin, s)
                      : launch_resample_t<MI_INTERP_NEAREST, false, 4>(a, num_sms, smem_optin, s);
    }
    return pack16 ? launch_resample_t<MI_INTERP_TRILINEAR, true, 2>(a, num_sms, smem_optin, s)
                  : launch_resample_t<MI_INTERP_TRILINEAR, false, 2>(a, num_sms, smem_optin, s);
}

// ------------------------------------------------------------------------------------------------
// a5: entropy reduction (DESIGN.md CANON-7)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// One CTA per transform.  With c the integer counts and N their total:
//   H = -sum (c/N) ln (c/N) = ln N - (sum c ln c)/N,      sum p^q = exp(-q ln N) * sum c^q.
// Accumulators per distribution X in {A, B, AB}: L_X = sum c ln c and P_X[k] = sum c^q_k.
__global__ void __launch_bounds__(kEntropyThreads)
entropy_kernel(const uint32_t* __restrict__ hist, int nb, const double* __restrict__ q, int nq_total,
               int q_off, int nq_pass, int form, double* __restrict__ mi_out,
               int64_t* __restrict__ nvalid) {
    constexpr int NW = kEntropyThreads / 32;
    constexpr int NACC = 3 * (1 + kMaxQPerPass);
    __shared__ unsigned sh_pa[256], sh_pb[256];
    __shared__ double sh_red[NACC][NW];
    __shared__ unsigned long long sh_n[NW];
    const int t = blockIdx.x;
    const uint32_t* __restrict__ h = hist + (size_t)t * nb * nb;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    double qv[kMaxQPerPass];
#pragma unroll
    for (int k = 0; k < kMaxQPerPass; ++k) qv[k] = k < nq_pass ? q[q_off + k] : 1.0;

    for (int i = threadIdx.x; i < 256; i += kEntropyThreads) { sh_pa[i] = 0u; sh_pb[i] = 0u; }
    __syncthreads();

    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = 0.0;

    // joint terms + marginal counts
    for (int r = warp; r < nb; r += NW) {
        unsigned rowsum = 0;
        for (int c = lane; c < nb; c += 32) {
            const unsigned v = h[r * nb + c];
            if (v) {
                rowsum += v;
                atomicAdd(&sh_pb[c], v);
                const double dv = (double)v;
                const double lc = log(dv);
                acc[2] += dv * lc;
#pragma unroll
                for (int k = 0; k < kMaxQPerPass; ++k)
                    if (k < nq_pass) acc[3 + 3 * k + 2] += exp(qv[k] * lc);
            }
        }
        rowsum = warp_sum(rowsum);
        if (lane == 0) sh_pa[r] = rowsum;
    }
    __syncthreads();

    // marginal terms
    unsigned long long n_local = 0;
    for (int i = threadIdx.x; i < nb; i += kEntropyThreads) {
        const unsigned ca = sh_pa[i], cb = sh_pb[i];
        n_local += ca;
        if (ca) {
            const double dv = (double)ca, lc = log(dv);
            acc[0] += dv * lc;
#pragma unroll
            for (int k = 0; k < kMaxQPerPass; ++k)
                if (k < nq_pass) acc[3 + 3 * k + 0] += exp(qv[k] * lc);
        }
        if (cb) {
            const double dv = (double)cb, lc = log(dv);
            acc[1] += dv * lc;
#pragma unroll
            for (int k = 0; k < kMaxQPerPass; ++k)
                if (k < nq_pass) acc[3 + 3 * k + 1] += exp(qv[k] * lc);
        }
    }
#pragma unroll
    for (int i = 0; i < NACC; ++i) {
        const double s = warp_sum_d(acc[i]);
        if (lane == 0) sh_red[i][warp] = s;
    }
    {
        unsigned lo = (unsigned)n_local, hi = (unsigned)(n_local >> 32);
        lo = warp_sum(lo);  // n_local < 2^32 per thread and the total fits in 32 bits (N_f < 2^31)
        hi = warp_sum(hi);
        if (lane == 0) sh_n[warp] = ((unsigned long long)hi << 32) + lo;
    }
    __syncthreads();

    if (threadIdx.x == 0) {
        double tot[NACC];
        for (int i = 0; i < NACC; ++i) {
            double s = 0.0;
            for (int w = 0; w < NW; ++w) s += sh_red[i][w];
            tot[i] = s;
        }
        unsigned long long n = 0;
        for (int w = 0; w < NW; ++w) n += sh_n[w];
        double* out = mi_out + (size_t)t * (1 + nq_total);
        if (nvalid != nullptr) nvalid[t] = (int64_t)n;
        if (n == 0) {
            out[0] = 0.0;
            for (int k = 0; k < nq_pass; ++k) out[1 + q_off + k] = 0.0;
        } else {
            const double N = (double)n, lnN = log(N);
            const double HA = lnN - tot[0] / N, HB = lnN - tot[1] / N, HAB = lnN - tot[2] / N;
            const double I = HA + HB - HAB;  // eq. 2
            out[0] = I;
            for (int k = 0; k < nq_pass; ++k) {
                const double qq = qv[k];
                double val;
                if (qq == 1.0) {
                    val = I;
                } else {
                    const double sc = exp(-qq * lnN);
                    const double SA = (1.0 - tot[3 + 3 * k + 0] * sc) / (qq - 1.0);
                    const double SB = (1.0 - tot[3 + 3 * k + 1] * sc) / (qq - 1.0);
                    const double SAB = (1.0 - tot[3 + 3 * k + 2] * sc) / (qq - 1.0);
                    val = SA + SB - SAB;
                    if (form == MI_TSALLIS_PSEUDO_ADDITIVE) val += (1.0 - qq) * SA * SB;
                }
                out[1 + q_off + k] = val;
            }
        }
    }
}

cudaError_t launch_entropy(const uint32_t* hist, int nb, int n_transforms, const double* q_dev, int nq,
                           int q_off, int form, double* mi_out, int64_t* nvalid, cudaStream_t s) {
    if (n_transforms <= 0) return cudaSuccess;
    int nq_pass = nq - q_off;
    if (nq_pass > kMaxQPerPass) nq_pass = kMaxQPerPass;
    if (nq_pass < 0) nq_pass = 0;
    entropy_kernel<<<n_transforms, kEntropyThreads, 0, s>>>(hist, nb, q_dev, nq, q_off, nq_pass, form,
                                                           mi_out, nvalid);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a6: map assembly + arg max (one CTA per channel)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) map_assemble_kernel(const double* __restrict__ mi, int64_t n,
                                                           int nch, double* __restrict__ map_out,
                                                           int64_t* __restrict__ argmax_out) {
    __shared__ double sh_v[256];
    __shared__ int64_t sh_i[256];
    const int ch = blockIdx.x;
    double best = -CUDART_INF;
    int64_t bi = n;  // sentinel: nothing better than -inf seen
    for (int64_t t = threadIdx.x; t < n; t += blockDim.x) {
        const double v = mi[t * nch + ch];
        map_out[(int64_t)ch * n + t] = v;
        if (v > best) { best = v; bi = t; }  // t ascends per thread: first maximum is kept
    }
    sh_v[threadIdx.x] = best;
    sh_i[threadIdx.x] = bi;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            const double v2 = sh_v[threadIdx.x + o];
            const int64_t i2 = sh_i[threadIdx.x + o];
            if (v2 > sh_v[threadIdx.x] || (v2 == sh_v[threadIdx.x] && i2 < sh_i[threadIdx.x])) {
                sh_v[threadIdx.x] = v2;
                sh_i[threadIdx.x] = i2;
            }
        }
        __syncthreads();
    }
    if (threadIdx.x == 0 && argmax_out != nullptr) argmax_out[ch] = sh_i[0] < n ? sh_i[0] : 0;
}

cudaError_t launch_map_assemble(const double* mi, int64_t n, int nch, double* map_out,
                                int64_t* argmax_out, cudaStream_t s) {
    if (n <= 0 || nch <= 0) return cudaSuccess;
    map_assemble_kernel<<<nch, 256, 0, s>>>(mi, n, nch, map_out, argmax_out);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Roofline probe: shared-memory atomicAdd rate on an nbins x nbins table
// ------------------------------------------------------------------------------------------------
template <bool PACK16>
__global__ void __launch_bounds__(kHistThreads, 1)
atomic_probe_kernel(int nbins2, int pattern, int iters, unsigned* __restrict__ sink) {
    extern __shared__ __align__(16) uint32_t sh_tab[];
    const int words = PACK16 ? (nbins2 + 1) / 2 : nbins2;
    for (int w = threadIdx.x; w < words; w += blockDim.x) sh_tab[w] = 0u;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned state = (blockIdx.x * 1024u + threadIdx.x) * 2654435761u + 12345u;
    const unsigned mask_rows = (unsigned)(nbins2 / 32 > 0 ? nbins2 / 32 : 1);
    for (int it = 0; it < iters; ++it) {
        int idx;
        if (pattern == 0) {
            // lane-distinct banks: consecutive (packed: every other) bins of one 32-word row
            const unsigned row = (warp * 7u + (unsigned)it * 13u) % (PACK16 ? mask_rows / 2 : mask_rows);
            idx = PACK16 ? (int)(row * 64u + 2u * lane) : (int)(row * 32u + lane);
        } else if (pattern == 1) {
            state = state * 1664525u + 1013904223u;
            idx = (int)(((unsigned long long)(state >> 8) * (unsigned)nbins2) >> 24);
        } else {
            idx = (int)(sink[0] & 1u) + 2;  // one address, not provably uniform at compile time
        }
        if (idx >= nbins2) idx = nbins2 - 1;
        if (PACK16) {
            const unsigned shift = (idx & 1) << 4;
            const unsigned old = atomicAdd(&sh_tab[idx >> 1], 1u << shift);
            if (((old >> shift) & 0xFFFFu) == 0x7FFFu) atomicSub(&sh_tab[idx >> 1], 0x8000u << shift);
        } else {
            atomicAdd(&sh_tab[idx], 1u);
        }
    }
    __syncthreads();
    unsigned s = 0;
    for (int w = threadIdx.x; w < words; w += blockDim.x) s += sh_tab[w];
    if (s == 0xFFFFFFFFu) sink[1] = s;  // keep the table live
}

cudaError_t run_shared_atomic_probe(int nbins, int pattern, int iters, int num_sms, size_t smem_optin,
                                    double* updates_per_s) {
    const int nbins2 = nbins * nbins;
    const bool pack16 = (size_t)nbins2 * sizeof(uint32_t) > 96 * 1024;
    const size_t smem = (pack16 ? (size_t)(nbins2 + 1) / 2 : (size_t)nbins2) * sizeof(uint32_t);
    if (smem > smem_optin) return cudaErrorInvalidConfiguration;
    unsigned* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, 2 * sizeof(unsigned));
    if (e != cudaSuccess) return e;
    cudaMemset(sink, 0, 2 * sizeof(unsigned));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best_ms = 1e30f;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {
        cudaEventRecord(e0, 0);
        if (pack16) {
            cudaFuncSetAttribute(atomic_probe_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            atomic_probe_kernel<true><<<num_sms, kHistThreads, smem, 0>>>(nbins2, pattern, iters, sink);
        } else {
            cudaFuncSetAttribute(atomic_probe_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            atomic_probe_kernel<false><<<num_sms, kHistThreads, smem, 0>>>(nbins2, pattern, iters, sink);
        }
        cudaEventRecord(e1, 0);
        e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (e != cudaSuccess) return e;
    *updates_per_s = (double)iters * kHistThreads * num_sms / (best_ms * 1e-3);
    return cudaSuccess;
}

}  // namespace mi
