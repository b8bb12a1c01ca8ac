// mi_pv.cu -- partial-volume interpolation (reading A21): the joint histogram
// of Maes et al. (the paper's ref. [5]), which interpolates no intensity -- "we start to see
// the effects of interpolation", PAPER.md:214 -- but lets the eight neighbours n_i of a sample point each
// add their trilinear weight to the cell (bin u(x), bin v(n_i)).
//
// Arithmetic (reading A21): coordinates, validity, floor / fraction and edge clamp are CANON-2 / CANON-4;
// the fraction of each axis is rounded to 1/32 voxel, u = floor(32 f + 0.5), and a neighbour's weight is the
// integer product of (u or 32 - u) over the axes, so a sample adds exactly 2^15 units and every histogram is an
// integer table that does not depend on the order of the updates.  Neighbour bins come from the yz-quads of the
// pre-binned, replicate-padded moving volume (two 4-byte gathers, no lerps).
//
//   resample_hist_pv_kernel   CTA-private u32 histogram in shared memory, one (transform, chunk of rows) item
//                             at a time; a chunk holds at most 131040 voxels so that no counter can pass
//                             2^32 (131040 * 2^15 < 2^32); merged into the transform's uint64 histogram
//   entropy_pv_kernel         step a5 on uint64 counts (unit 2^-15 voxel; probabilities are unit-free)
#include <cuda_runtime.h>
#include <stdint.h>

#include "mi_device.cuh"
#include "mi_internal.h"

namespace mi {

namespace {

constexpr int kPvChunkVoxels = 131040;   // multiple of 32; 131040 * 32768 = 4293918720 < 2^32

// yz-quads of the replicate-padded moving BIN volume: entry (x,y,z) of the padded grid holds the bins of the padded
// voxels (x,y,z), (x,y+1,z), (x,y,z+1), (x,y+1,z+1) in bytes 0..3 -- the entries x and x+1 are the eight neighbours of
// a sample, two 4-byte loads instead of eight 1-byte gathers (the load/store unit writes 4 bytes per lane into the
// register file whatever the access size, profiles/r2c_ncu.md section 6).
__global__ void __launch_bounds__(256) bins_quad_build_kernel(const uint8_t* __restrict__ src, uint32_t* __restrict__ dst,
                                                              int nx, int ny, int nz) {
    const int px = nx + 2, py = ny + 2, pz = nz + 2;
    const int64_t total = (int64_t)px * py * pz;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % px);
        const int64_t r = i / px;
        const int y = (int)(r % py), z = (int)(r / py);
        const int sx = min(max(x - 1, 0), nx - 1);
        const int sy0 = min(max(y - 1, 0), ny - 1), sy1 = min(max(y, 0), ny - 1);   // padded y and y+1
        const int sz0 = min(max(z - 1, 0), nz - 1), sz1 = min(max(z, 0), nz - 1);   // padded z and z+1
        const uint32_t b00 = src[((int64_t)sz0 * ny + sy0) * nx + sx], b10 = src[((int64_t)sz0 * ny + sy1) * nx + sx];
        const uint32_t b01 = src[((int64_t)sz1 * ny + sy0) * nx + sx], b11 = src[((int64_t)sz1 * ny + sy1) * nx + sx];
        dst[i] = b00 | (b10 << 8) | (b01 << 16) | (b11 << 24);
    }
}

// One axis: validity (CANON-4 region), the raw float bits of magic + floor(c) and the weight pair (32 - u, u).
struct PvAxis {
    bool ok;
    unsigned tbits;
    unsigned w0, w1;
};
__device__ __forceinline__ PvAxis pv_axis(float c, float half_hi) {
    PvAxis a;
    a.ok = c >= -0.5f && c < half_hi;
    const float t = __fadd_rd(c, kFloorMagic);
    a.tbits = __float_as_uint(t);
    const float f = __fsub_rn(c, __fsub_rn(t, kFloorMagic));
    const int u = __float2int_rd(__fadd_rn(__fmul_rn(f, 32.0f), 0.5f));
    a.w1 = (unsigned)u;
    a.w0 = 32u - (unsigned)u;
    return a;
}

// One (transform, chunk of fixed rows) item per CTA at a time; a warp takes whole rows, a lane the voxels
// ix = lane + 32 j of its row, kPvUnroll of them per trip with all their loads issued first.
constexpr int kPvUnroll = 2;

template <bool MASK>
__global__ void __launch_bounds__(kHistThreads, 1) resample_hist_pv_kernel(const __grid_constant__ PvArgs a) {
    extern __shared__ __align__(16) uint32_t sh_hist[];
    const int nb = a.nb, pitch = a.pitch, rows_smem = a.rows_smem;
    const int words = rows_smem * pitch;
    for (int w = threadIdx.x; w < words; w += blockDim.x) sh_hist[w] = 0u;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int fnx = a.f.nx, fny = a.f.ny;
    const int rows_total = a.f.ny * a.f.nz;
    const unsigned pnx = (unsigned)a.m.nx + 2u, pny = (unsigned)a.m.ny + 2u;
    // padded index of cell (jx+1, jy+1, jz+1) from the raw float bits T_k = magic + j_k (as in resample_quad_kernel)
    const unsigned fold = (unsigned)(kFloorMagicBits - 1) * (pny * pnx + pnx + 1u);
    const float hx = __fsub_rn((float)a.m.nx, 0.5f), hy = __fsub_rn((float)a.m.ny, 0.5f), hz = __fsub_rn((float)a.m.nz, 0.5f);
    const uint32_t* __restrict__ quad = a.mbins_quad;
    const float flane = (float)lane;
    const long long nitems = (long long)a.n_transforms * a.nchunks;
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int t = (int)(item / a.nchunks);
        const int chunk = (int)(item - (long long)t * a.nchunks);
        const int row_lo = chunk * a.rows_per_chunk;
        const int row_hi = min(row_lo + a.rows_per_chunk, rows_total);
        float m[12];
#pragma unroll
        for (int i = 0; i < 12; ++i) m[i] = __ldg(a.M + (size_t)t * 12 + i);
        unsigned long long* gh = a.hist + (size_t)t * nb * nb;
        // The weighted updates are ATOMS.ADD with a data operand; on real volumes a quarter of a background warp's
        // lanes hit the cell (most populated fixed bin, most populated moving bin) and cost a crossbar pass each
        // (6.9 passes per warp-wide update measured, against 3 for distinct cells).  That one cell is summed in a
        // register per lane and added once per item: at most 131 040 voxels x 2^15 < 2^32 per chunk, as for the row.
        unsigned hot_acc = 0u;
        const unsigned hot_b = (unsigned)a.hot_b;
        for (int row = row_lo + warp; row < row_hi; row += nwarps) {
            const int iz = row / fny, iy = row - iz * fny;
            const float fy = (float)iy, fz = (float)iz;
            // CANON-2: row terms, then one fma per voxel and axis
            const float rx = __fmaf_rn(m[1], fy, __fmaf_rn(m[2], fz, m[3]));
            const float ry = __fmaf_rn(m[5], fy, __fmaf_rn(m[6], fz, m[7]));
            const float rz = __fmaf_rn(m[9], fy, __fmaf_rn(m[10], fz, m[11]));
            const uint8_t* __restrict__ frow = a.fbins_ranked + (size_t)row * (unsigned)fnx;
            float fx0 = flane;
            for (unsigned ix0 = (unsigned)lane; ix0 < (unsigned)fnx; ix0 += 32u * kPvUnroll, fx0 += (float)(32 * kPvUnroll)) {
                PvAxis ax[kPvUnroll], ay[kPvUnroll], az[kPvUnroll];
                unsigned idx[kPvUnroll];
                bool ok[kPvUnroll];
#pragma unroll
                for (int u = 0; u < kPvUnroll; ++u) {
                    const float fx = fx0 + (float)(32 * u);
                    ax[u] = pv_axis(__fmaf_rn(m[0], fx, rx), hx);
                    ay[u] = pv_axis(__fmaf_rn(m[4], fx, ry), hy);
                    az[u] = pv_axis(__fmaf_rn(m[8], fx, rz), hz);
                    bool v = ax[u].ok && ay[u].ok && az[u].ok && (ix0 + 32u * u < (unsigned)fnx);
                    if (MASK) {
                        const unsigned vi = (unsigned)row * (unsigned)fnx + min(ix0 + 32u * u, (unsigned)fnx - 1u);
                        v = v && ((__ldg(a.mask_bits + (vi >> 5)) >> (vi & 31u)) & 1u);
                    }
                    const unsigned i = (az[u].tbits * pny + ay[u].tbits) * pnx + ax[u].tbits - fold;
                    idx[u] = v ? i : 0u;
                    ok[u] = v;
                }
                uint32_t q0[kPvUnroll], q1[kPvUnroll];
                unsigned fa[kPvUnroll];
#pragma unroll
                for (int u = 0; u < kPvUnroll; ++u) {
                    q0[u] = __ldg(quad + idx[u]);
                    q1[u] = __ldg(quad + idx[u] + 1);
                    fa[u] = ok[u] ? (unsigned)__ldg(frow + ix0 + 32u * u) : 0u;
                }
#pragma unroll
                for (int u = 0; u < kPvUnroll; ++u) {
                    if (!ok[u]) continue;
                    const unsigned wy0z0 = ay[u].w0 * az[u].w0, wy1z0 = ay[u].w1 * az[u].w0;
                    const unsigned wy0z1 = ay[u].w0 * az[u].w1, wy1z1 = ay[u].w1 * az[u].w1;
                    // neighbour (dx,dy,dz): byte dy + 2 dz of entry x + dx, x fastest
                    const unsigned bins[8] = {q0[u] & 0xFFu, q1[u] & 0xFFu, (q0[u] >> 8) & 0xFFu, (q1[u] >> 8) & 0xFFu,
                                              (q0[u] >> 16) & 0xFFu, (q1[u] >> 16) & 0xFFu, q0[u] >> 24, q1[u] >> 24};
                    const unsigned wts[8] = {ax[u].w0 * wy0z0, ax[u].w1 * wy0z0, ax[u].w0 * wy1z0, ax[u].w1 * wy1z0,
                                             ax[u].w0 * wy0z1, ax[u].w1 * wy0z1, ax[u].w0 * wy1z1, ax[u].w1 * wy1z1};
                    if ((int)fa[u] < rows_smem) {
                        uint32_t* row_ptr = sh_hist + fa[u] * pitch;
                        const unsigned hot_key = fa[u] == 0u ? hot_b : 0xFFFFFFFFu;   // rank 0 always has a shared row
#pragma unroll
                        for (int k = 0; k < 8; ++k) {
                            const bool hot = bins[k] == hot_key;
                            hot_acc += hot ? wts[k] : 0u;
                            if (wts[k] != 0u && !hot) atomicAdd(row_ptr + bins[k], wts[k]);
                        }
                    } else {
                        unsigned long long* grow = gh + (size_t)__ldg(a.rank_inv + fa[u]) * nb;
#pragma unroll
                        for (int k = 0; k < 8; ++k)
                            if (wts[k]) atomicAdd(grow + bins[k], (unsigned long long)wts[k]);
                    }
                }
            }
        }
        {
            unsigned h = hot_acc;                                  // <= 128 voxels x 2^15 per lane: no overflow
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) h += __shfl_xor_sync(0xffffffffu, h, o);
            if (lane == 0 && h) atomicAdd(sh_hist + hot_b, h);
        }
        __syncthreads();
        for (int r = warp; r < rows_smem; r += nwarps) {
            unsigned long long* grow = gh + (size_t)__ldg(a.rank_inv + r) * nb;
            for (int b = lane; b < nb; b += 32) {
                const uint32_t c = sh_hist[r * pitch + b];
                if (c) {
                    sh_hist[r * pitch + b] = 0u;
                    atomicAdd(grow + b, (unsigned long long)c);
                }
            }
        }
        __syncthreads();
    }
}

// Step a5 on a uint64 histogram whose unit is 2^-15 voxel: counts are scaled back to voxels (an exact
// division by a power of two), so sum c^q keeps the range argument of include/mi.h (q <= 32).
__global__ void __launch_bounds__(kEntropyThreads)
entropy_pv_kernel(const unsigned long long* __restrict__ hist, int nb, const double* __restrict__ q, int nq_total,
                  int q_off, int nq_pass, int form, double* __restrict__ mi_out, int64_t* __restrict__ nvalid,
                  const OutMap om) {
    constexpr int NW = kEntropyThreads / 32;
    constexpr int NACC = 3 * (1 + kMaxQPerPass);
    constexpr double kUnit = 1.0 / 32768.0;
    __shared__ unsigned long long sh_pa[256], sh_pb[256];
    __shared__ double sh_red[NACC][NW];
    __shared__ unsigned long long sh_n[NW];
    const int t = blockIdx.x;
    const unsigned long long* __restrict__ h = hist + (size_t)t * nb * nb;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double qv[kMaxQPerPass];
#pragma unroll
    for (int k = 0; k < kMaxQPerPass; ++k) qv[k] = k < nq_pass ? q[q_off + k] : 1.0;
    for (int i = threadIdx.x; i < 256; i += kEntropyThreads) { sh_pa[i] = 0ull; sh_pb[i] = 0ull; }
    __syncthreads();
    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
    auto add_terms = [&](unsigned long long c, int which) {
        const double dv = (double)c * kUnit, lc = log(dv);
        acc[which] += dv * lc;
#pragma unroll
        for (int k = 0; k < kMaxQPerPass; ++k)
            if (k < nq_pass) acc[3 + 3 * k + which] += exp(qv[k] * lc);
    };
    for (int r = warp; r < nb; r += NW) {
        unsigned long long rowsum = 0ull;
        for (int c = lane; c < nb; c += 32) {
            const unsigned long long v = h[(size_t)r * nb + c];
            if (v) {
                rowsum += v;
                atomicAdd(&sh_pb[c], v);
                add_terms(v, 2);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) rowsum += __shfl_xor_sync(0xffffffffu, rowsum, o);
        if (lane == 0) sh_pa[r] = rowsum;
    }
    __syncthreads();
    unsigned long long n_local = 0ull;
    for (int i = threadIdx.x; i < nb; i += kEntropyThreads) {
        const unsigned long long ca = sh_pa[i], cb = sh_pb[i];
        n_local += ca;
        if (ca) add_terms(ca, 0);
        if (cb) add_terms(cb, 1);
    }
#pragma unroll
    for (int i = 0; i < NACC; ++i) {
        const double s = warp_sum_d(acc[i]);
        if (lane == 0) sh_red[i][warp] = s;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) n_local += __shfl_xor_sync(0xffffffffu, n_local, o);
    if (lane == 0) sh_n[warp] = n_local;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot[NACC];
        for (int i = 0; i < NACC; ++i) {
            double s = 0.0;
            for (int w = 0; w < NW; ++w) s += sh_red[i][w];
            tot[i] = s;
        }
        unsigned long long n = 0ull;
        for (int w = 0; w < NW; ++w) n += sh_n[w];
        entropy_finish(tot, (double)n * kUnit, (long long)(n >> 15), t, qv, nq_pass, q_off, nq_total, form, mi_out,
                       nvalid, om);
    }
}

}  // namespace

cudaError_t launch_bins_quad_build(const uint8_t* src, uint32_t* dst, int nx, int ny, int nz, cudaStream_t s) {
    const int64_t total = (int64_t)(nx + 2) * (ny + 2) * (nz + 2);
    int64_t blocks = (total + 255) / 256;
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    bins_quad_build_kernel<<<(unsigned)blocks, 256, 0, s>>>(src, dst, nx, ny, nz);
    return cudaGetLastError();
}

cudaError_t launch_resample_hist_pv(PvArgs a, int num_sms, cudaStream_t s) {
    if (a.rows_smem < 1 || a.pitch < a.nb || a.nb > 256) return cudaErrorInvalidConfiguration;
    // a chunk holds whole fixed rows and at most kPvChunkVoxels voxels: no u32 counter of the shared histogram can
    // pass 2^32 before the chunk is merged (a row longer than that is split by the voxel count of one row only
    // when fnx > kPvChunkVoxels, which mi_create's 2^31-voxel limit and this check exclude)
    if (a.f.nx > kPvChunkVoxels) return cudaErrorInvalidConfiguration;
    const int rows_total = a.f.ny * a.f.nz;
    a.rows_per_chunk = kPvChunkVoxels / a.f.nx;
    a.nchunks = (rows_total + a.rows_per_chunk - 1) / a.rows_per_chunk;
    const long long nitems = (long long)a.n_transforms * a.nchunks;
    if (nitems < 1) return cudaSuccess;
    const size_t smem = (size_t)a.rows_smem * a.pitch * sizeof(uint32_t);
    auto launch = [&](auto kern) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        const long long grid = nitems < num_sms ? nitems : num_sms;
        kern<<<(unsigned)grid, kHistThreads, smem, s>>>(a);
        return cudaGetLastError();
    };
    return a.mask_bits != nullptr ? launch(resample_hist_pv_kernel<true>) : launch(resample_hist_pv_kernel<false>);
}

cudaError_t launch_entropy_pv(const unsigned long long* hist, int nb, int n_transforms, const double* q_dev, int nq,
                              int q_off, int form, double* mi_out, int64_t* nvalid, OutMap om, cudaStream_t s) {
    if (n_transforms <= 0) return cudaSuccess;
    if (nb > 256) return cudaErrorInvalidConfiguration;
    int nq_pass = nq - q_off;
    if (nq_pass > kMaxQPerPass) nq_pass = kMaxQPerPass;
    if (nq_pass < 0) nq_pass = 0;
    entropy_pv_kernel<<<n_transforms, kEntropyThreads, 0, s>>>(hist, nb, q_dev, nq, q_off, nq_pass, form, mi_out, nvalid, om);
    return cudaGetLastError();
}

}  // namespace mi
