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

#include "mi_device.cuh"
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
// `flag` (may be NULL) is set when a voxel is negative, not finite, or lands above the last bin
// edge ((v - lo)*scale > nb): while it stays 0 and lo == 0 the z-histogram kernel may skip both
// clamps of CANON-5 (mi_internal.h, kBinFast).
__device__ __forceinline__ bool plain_inrange(float v, float lo, float scale, float top) {
    return v >= 0.0f && __fmul_rn(__fsub_rn(v, lo), scale) <= top + 1.0f;
}

__global__ void __launch_bounds__(256) prebin_kernel(const float* __restrict__ vol,
                                                     uint8_t* __restrict__ bins, int64_t n, float lo,
                                                     float scale, float top, unsigned* __restrict__ flag) {
    const int64_t nvec = n >> 4;
    bool odd = false;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const float4* src = reinterpret_cast<const float4*>(vol) + i * 4;
        float4 v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            v[k] = __ldcs(src + k);
            odd |= !(plain_inrange(v[k].x, lo, scale, top) && plain_inrange(v[k].y, lo, scale, top) &&
                     plain_inrange(v[k].z, lo, scale, top) && plain_inrange(v[k].w, lo, scale, top));
        }
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
    if (j < n) {
        bins[j] = (uint8_t)bin_index(vol[j], lo, scale, top);
        odd |= !plain_inrange(vol[j], lo, scale, top);
    }
    if (flag != nullptr && __any_sync(0xffffffffu, odd) && (threadIdx.x & 31) == 0) atomicOr(flag, 1u);
}

cudaError_t launch_prebin(const float* vol, uint8_t* bins, int64_t n, float lo, float scale, int nb,
                          unsigned* flag, cudaStream_t s) {
    if (n <= 0) return cudaSuccess;
    const int64_t nvec = n >> 4;
    int64_t blocks = (nvec + 255) / 256;
    if (blocks < 1) blocks = 1;
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    prebin_kernel<<<(unsigned)blocks, 256, 0, s>>>(vol, bins, n, lo, scale, (float)(nb - 1), flag);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a1b: helpers run once per context: replicate-padded moving volume, fixed-bin population ranks
// ------------------------------------------------------------------------------------------------
// pm has dims (nx+2, ny+2, nz+2); pm[z][y][x] = moving[clamp(z-1)][clamp(y-1)][clamp(x-1)].
// Reading the 2x2x2 cell at padded index (jx+1, jy+1, jz+1), jk = floor(c_k) in [-1, n_k-1], gives
// exactly the edge-clamped neighbours of CANON-4 (i0 = max(j,0), i1 = min(j+1, n-1)).
__global__ void __launch_bounds__(256) pad_replicate_kernel(const float* __restrict__ src,
                                                            float* __restrict__ dst, int nx, int ny, int nz) {
    const int px = nx + 2, py = ny + 2, pz = nz + 2;
    const int64_t total = (int64_t)px * py * pz;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % px);
        const int64_t r = i / px;
        const int y = (int)(r % py), z = (int)(r / py);
        const int sx = min(max(x - 1, 0), nx - 1), sy = min(max(y - 1, 0), ny - 1), sz = min(max(z - 1, 0), nz - 1);
        dst[i] = src[((int64_t)sz * ny + sy) * nx + sx];
    }
}

cudaError_t launch_pad_replicate(const float* src, float* dst, int nx, int ny, int nz, cudaStream_t s) {
    const int64_t total = (int64_t)(nx + 2) * (ny + 2) * (nz + 2);
    int64_t blocks = (total + 255) / 256;
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    pad_replicate_kernel<<<(unsigned)blocks, 256, 0, s>>>(src, dst, nx, ny, nz);
    return cudaGetLastError();
}

// yz-quads of the padded moving volume: quad[z][y][x] = {pad[z][y][x], pad[z][y+1][x], pad[z+1][y][x],
// pad[z+1][y+1][x]} (indices clamped to the padded volume: the last row / plane is never a cell's base).  The
// 2x2x2 cell at padded base index i is then quad[i] (its x = jx face) and quad[i + 1] (its x = jx + 1 face): two
// adjacent 16-byte loads instead of eight 4-byte gathers -- the four values of a face travel together, and the
// 32 lanes of a warp (consecutive x) read 512 contiguous bytes per load when the row stays in one moving row.
__global__ void __launch_bounds__(256) quad_build_kernel(const float* __restrict__ pad, float4* __restrict__ quad,
                                                         int px, int py, int pz) {
    const int64_t total = (int64_t)px * py * pz;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % px);
        const int64_t r = i / px;
        const int y = (int)(r % py), z = (int)(r / py);
        const int y1 = min(y + 1, py - 1), z1 = min(z + 1, pz - 1);
        quad[i] = make_float4(pad[((int64_t)z * py + y) * px + x], pad[((int64_t)z * py + y1) * px + x],
                              pad[((int64_t)z1 * py + y) * px + x], pad[((int64_t)z1 * py + y1) * px + x]);
    }
}

cudaError_t launch_quad_build(const float* pad, float4* quad, int nx, int ny, int nz, cudaStream_t s) {
    const int64_t total = (int64_t)(nx + 2) * (ny + 2) * (nz + 2);
    int64_t blocks = (total + 255) / 256;
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    quad_build_kernel<<<(unsigned)blocks, 256, 0, s>>>(pad, quad, nx + 2, ny + 2, nz + 2);
    return cudaGetLastError();
}

// One bit per voxel from a byte mask (bit i of word i/32 = mask[i] != 0).
__global__ void __launch_bounds__(256) mask_bits_kernel(const uint8_t* __restrict__ mask, int64_t n,
                                                        uint32_t* __restrict__ bits) {
    const int64_t nwords = (n + 31) >> 5;
    const int lane = threadIdx.x & 31;
    for (int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; w < nwords;
         w += ((int64_t)gridDim.x * blockDim.x) >> 5) {
        const int64_t i = (w << 5) + lane;
        const unsigned word = __ballot_sync(0xffffffffu, i < n && mask[i] != 0);
        if (lane == 0) bits[w] = word;
    }
}

cudaError_t launch_mask_bits(const uint8_t* mask, int64_t n, uint32_t* bits, cudaStream_t s) {
    int64_t blocks = (n + 255) / 256;
    if (blocks < 1) blocks = 1;
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    mask_bits_kernel<<<(unsigned)blocks, 256, 0, s>>>(mask, n, bits);
    return cudaGetLastError();
}

// 256-bin population count of a uint8 volume (CTA-private shared histogram, merged with atomics).
__global__ void __launch_bounds__(256) bin_count_kernel(const uint8_t* __restrict__ bins, int64_t n,
                                                        unsigned long long* __restrict__ counts) {
    __shared__ unsigned sh[256];
    sh[threadIdx.x] = 0u;
    __syncthreads();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        atomicAdd(&sh[bins[i]], 1u);
    __syncthreads();
    if (sh[threadIdx.x]) atomicAdd(&counts[threadIdx.x], (unsigned long long)sh[threadIdx.x]);
}

// rank[a] = position of fixed bin a when bins are sorted by falling population (ties: lower bin
// first); inv[rank[a]] = a.  One CTA of 256 threads; counts has 256 entries.
__global__ void __launch_bounds__(256) bin_rank_kernel(const unsigned long long* __restrict__ counts,
                                                       uint8_t* __restrict__ rank, int* __restrict__ inv) {
    __shared__ unsigned long long c[256];
    c[threadIdx.x] = counts[threadIdx.x];
    __syncthreads();
    const unsigned long long mine = c[threadIdx.x];
    int r = 0;
    for (int j = 0; j < 256; ++j) r += (c[j] > mine) || (c[j] == mine && j < (int)threadIdx.x);
    rank[threadIdx.x] = (uint8_t)r;
    inv[r] = (int)threadIdx.x;
}

__global__ void __launch_bounds__(256) remap_bins_kernel(const uint8_t* __restrict__ in,
                                                         uint8_t* __restrict__ out, int64_t n,
                                                         const uint8_t* __restrict__ rank) {
    __shared__ uint8_t lut[256];
    lut[threadIdx.x] = rank[threadIdx.x];
    __syncthreads();
    const int64_t nvec = n >> 4;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        uint4 v = reinterpret_cast<const uint4*>(in)[i];
        uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int k = 0; k < 4; ++k)
            w[k] = (uint32_t)lut[w[k] & 0xFF] | ((uint32_t)lut[(w[k] >> 8) & 0xFF] << 8) |
                   ((uint32_t)lut[(w[k] >> 16) & 0xFF] << 16) | ((uint32_t)lut[w[k] >> 24] << 24);
        reinterpret_cast<uint4*>(out)[i] = make_uint4(w[0], w[1], w[2], w[3]);
    }
    const int64_t j = (nvec << 4) + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) out[j] = lut[in[j]];
}

cudaError_t launch_bin_count(const uint8_t* bins, int64_t n, unsigned long long* counts, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(counts, 0, 256 * sizeof(unsigned long long), s);
    if (e != cudaSuccess) return e;
    int64_t blocks = (n + 255) / 256;
    if (blocks < 1) blocks = 1;
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    bin_count_kernel<<<(unsigned)blocks, 256, 0, s>>>(bins, n, counts);
    return cudaGetLastError();
}

cudaError_t launch_rank_fixed_bins(const uint8_t* bins, int64_t n, unsigned long long* counts_scratch,
                                   uint8_t* rank, int* inv, uint8_t* ranked_bins, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(counts_scratch, 0, 256 * sizeof(unsigned long long), s);
    if (e != cudaSuccess) return e;
    int64_t blocks = (n + 255) / 256;
    if (blocks < 1) blocks = 1;
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    bin_count_kernel<<<(unsigned)blocks, 256, 0, s>>>(bins, n, counts_scratch);
    bin_rank_kernel<<<1, 256, 0, s>>>(counts_scratch, rank, inv);
    remap_bins_kernel<<<(unsigned)blocks, 256, 0, s>>>(bins, ranked_bins, n, rank);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a3 + a4: resample + joint histogram (generic affine)
// ------------------------------------------------------------------------------------------------
// CANON-4 lerp: L(p,q,f) = fma(f, q - p, p) with q - p rounded first.
__device__ __forceinline__ float lerp_rn(float p, float q, float f) {
    return __fmaf_rn(f, __fsub_rn(q, p), p);
}

struct Sample {
    bool ok;   // inside the moving volume (CANON-3/4 validity)
    int b;     // moving bin (meaningless if !ok)
};

struct MovingView {
    const float* __restrict__ pad;     // replicate-padded float volume, dims (nx+2, ny+2, nz+2)
    const float* __restrict__ pad_y;   // pad + (nx+2)
    const float* __restrict__ pad_z;   // pad + (nx+2)*(ny+2)
    const float* __restrict__ pad_yz;  // pad + (nx+2)*(ny+2) + (nx+2)
    const float4* __restrict__ quad;   // yz-quads of the padded volume (quad_build_kernel)
    const uint8_t* __restrict__ bins;  // unpadded bin volume (nearest neighbour)
    int nx, ny;                        // unpadded dims (nearest neighbour indexing)
    int pnx, pny;                      // padded dims
    unsigned fold;                     // index constant folding the magic bits and the +1 padding
    float fx, fy, fz;                  // (float)n
    float hx, hy, hz;                  // (float)n - 0.5f
    float lo, scale;
    int top;                           // nb - 1
};

// GATHER (trilinear): kGatherScalar = eight 4-byte loads from the padded volume; kGatherQuad = two adjacent
// 16-byte loads from the yz-quad volume (same eight floats, same lerp sequence).
enum { kGatherScalar = 0, kGatherQuad = 1 };

template <int INTERP, int GATHER>
__device__ __forceinline__ Sample sample_bin(const MovingView& mv, float cx, float cy, float cz) {
    Sample s;
    if (INTERP == MI_INTERP_NEAREST) {
        // CANON-3: r = floor(c + 0.5) (round half up), validity tested on r in float.
        const float tx = __fadd_rd(__fadd_rn(cx, 0.5f), kFloorMagic);
        const float ty = __fadd_rd(__fadd_rn(cy, 0.5f), kFloorMagic);
        const float tz = __fadd_rd(__fadd_rn(cz, 0.5f), kFloorMagic);
        const float rx = __fsub_rn(tx, kFloorMagic), ry = __fsub_rn(ty, kFloorMagic), rz = __fsub_rn(tz, kFloorMagic);
        s.ok = rx >= 0.0f && rx < mv.fx && ry >= 0.0f && ry < mv.fy && rz >= 0.0f && rz < mv.fz;
        const int jx = __float_as_int(tx) - kFloorMagicBits, jy = __float_as_int(ty) - kFloorMagicBits,
                  jz = __float_as_int(tz) - kFloorMagicBits;
        unsigned idx = ((unsigned)jz * (unsigned)mv.ny + (unsigned)jy) * (unsigned)mv.nx + (unsigned)jx;
        idx = s.ok ? idx : 0u;
        s.b = __ldg(mv.bins + idx);
    } else {
        // CANON-4: region [-0.5, n-0.5), edge clamp (via the padded copy), x- then y- then z-lerps.
        s.ok = cx >= -0.5f && cx < mv.hx && cy >= -0.5f && cy < mv.hy && cz >= -0.5f && cz < mv.hz;
        const float tx = __fadd_rd(cx, kFloorMagic), ty = __fadd_rd(cy, kFloorMagic), tz = __fadd_rd(cz, kFloorMagic);
        const float wx = __fsub_rn(cx, __fsub_rn(tx, kFloorMagic));
        const float wy = __fsub_rn(cy, __fsub_rn(ty, kFloorMagic));
        const float wz = __fsub_rn(cz, __fsub_rn(tz, kFloorMagic));
        unsigned idx = (__float_as_uint(tz) * (unsigned)mv.pny + __float_as_uint(ty)) * (unsigned)mv.pnx +
                       __float_as_uint(tx) - mv.fold;
        idx = s.ok ? idx : 0u;
        float a000, a100, a010, a110, a001, a101, a011, a111;
        if (GATHER == kGatherQuad) {
            const float4 q0 = __ldg(mv.quad + idx), q1 = __ldg(mv.quad + idx + 1);
            a000 = q0.x; a010 = q0.y; a001 = q0.z; a011 = q0.w;
            a100 = q1.x; a110 = q1.y; a101 = q1.z; a111 = q1.w;
        } else {
            a000 = __ldg(mv.pad + idx); a100 = __ldg(mv.pad + idx + 1);
            a010 = __ldg(mv.pad_y + idx); a110 = __ldg(mv.pad_y + idx + 1);
            a001 = __ldg(mv.pad_z + idx); a101 = __ldg(mv.pad_z + idx + 1);
            a011 = __ldg(mv.pad_yz + idx); a111 = __ldg(mv.pad_yz + idx + 1);
        }
        const float v00 = lerp_rn(a000, a100, wx);
        const float v10 = lerp_rn(a010, a110, wx);
        const float v01 = lerp_rn(a001, a101, wx);
        const float v11 = lerp_rn(a011, a111, wx);
        const float w0 = lerp_rn(v00, v10, wy);
        const float w1 = lerp_rn(v01, v11, wy);
        const float v = lerp_rn(w0, w1, wz);
        // CANON-5 with the floor/clamp done on the integer side (same result for finite v)
        const float t = __fmul_rn(__fsub_rn(v, mv.lo), mv.scale);
        s.b = min(max(__float2int_rd(t), 0), mv.top);
    }
    return s;
}

// One CTA works on one (transform, row slab) item at a time.  The joint histogram lives in shared
// memory as u32 counters updated with result-less atomics (the fastest shared atomic on sm_100a,
// see profiles/).  Fixed bins arrive RANKED by population: the `rows_smem` most populated fixed-bin
// rows are in shared memory, the rare tail (only when nb*nb*4 B exceeds shared memory, i.e. 256
// bins) is added straight to the global histogram.
// HIST = false is the roofline probe (mi_probe_gather_rate): the same kernel without the histogram updates --
// the moving bins are summed into a.sink instead -- i.e. the rate at which L1TEX delivers the samples.
template <int INTERP, int UNROLL, int GATHER, bool HIST>
__global__ void __launch_bounds__(kHistThreads, 1)
resample_hist_kernel(const __grid_constant__ ResampleArgs a) {
    extern __shared__ __align__(16) uint32_t sh_hist[];
    const int nb = a.nb;
    const int nbins2 = nb * nb;
    const int rows_smem = a.rows_smem;
    const int pitch = a.pitch;   // words per shared row; bank = (a*(pitch-nb) + b) mod 32
    const int words = rows_smem * pitch;
    for (int w = threadIdx.x; w < words; w += blockDim.x) sh_hist[w] = 0u;
    __syncthreads();

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    const int fnx = a.f.nx;
    // The 32 warps of the CTA take the rows of one (2^ty_log2 y) x (32 >> ty_log2 z) tile of fixed rows
    // at a time, so that the 2x2x2 stencils of neighbouring rows in y AND z hit the same L1 sectors.
    const int ty_log2 = a.ty_log2;
    const int wy = warp & ((1 << ty_log2) - 1), wz = warp >> ty_log2;
    const int tiles_y = (a.f.ny + (1 << ty_log2) - 1) >> ty_log2;
    const int tz_rows = 32 >> ty_log2;
    const int tiles_total = tiles_y * ((a.f.nz + tz_rows - 1) / tz_rows);

    MovingView mv;
    mv.pnx = a.m.nx + 2; mv.pny = a.m.ny + 2;
    mv.pad = a.moving_pad;
    mv.pad_y = a.moving_pad + mv.pnx;
    mv.pad_z = a.moving_pad + (size_t)mv.pnx * mv.pny;
    mv.pad_yz = mv.pad_z + mv.pnx;
    mv.quad = a.moving_quad;
    mv.bins = a.mbins;
    mv.nx = a.m.nx; mv.ny = a.m.ny;
    // padded index of cell (jx+1, jy+1, jz+1) from the raw float bits T_k = magic + j_k:
    // ((Tz*pny + Ty)*pnx + Tx) - (magic-1)*(pny*pnx + pnx + 1), all modulo 2^32.
    mv.fold = (unsigned)(kFloorMagicBits - 1) * (unsigned)(mv.pny * mv.pnx + mv.pnx + 1);
    mv.fx = (float)a.m.nx; mv.fy = (float)a.m.ny; mv.fz = (float)a.m.nz;
    mv.hx = __fsub_rn(mv.fx, 0.5f); mv.hy = __fsub_rn(mv.fy, 0.5f); mv.hz = __fsub_rn(mv.fz, 0.5f);
    mv.lo = a.mlo; mv.scale = a.mscale; mv.top = nb - 1;

    unsigned probe_acc = 0u;
    const long long nitems = (long long)a.n_transforms * a.nslabs;
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int slab = (int)(item / a.n_transforms);                   // slab-major (see resample_quad_kernel)
        const int t = (int)(item - (long long)slab * a.n_transforms);
        const int tile_lo = (int)((long long)tiles_total * slab / a.nslabs);
        const int tile_hi = (int)((long long)tiles_total * (slab + 1) / a.nslabs);
        float m[12];
#pragma unroll
        for (int i = 0; i < 12; ++i) m[i] = __ldg(a.M + (size_t)t * 12 + i);
        uint32_t* gh = a.hist + (size_t)t * nbins2;

        for (int tile = tile_lo; tile < tile_hi; ++tile) {
            const int tz = tile / tiles_y;
            const int iy = ((tile - tz * tiles_y) << ty_log2) + wy;
            const int iz = tz * tz_rows + wz;
            if (iy >= a.f.ny || iz >= a.f.nz) continue;
            const int row = iz * a.f.ny + iy;
            const float fy = (float)iy, fz = (float)iz;
            // CANON-2: row terms, then one fma per voxel and axis
            const float rx = __fmaf_rn(m[1], fy, __fmaf_rn(m[2], fz, m[3]));
            const float ry = __fmaf_rn(m[5], fy, __fmaf_rn(m[6], fz, m[7]));
            const float rz = __fmaf_rn(m[9], fy, __fmaf_rn(m[10], fz, m[11]));
            const uint8_t* __restrict__ frow = a.fbins_ranked + (size_t)row * fnx;
            for (int ix0 = lane; ix0 < fnx; ix0 += 32 * UNROLL) {
                Sample smp[UNROLL];
                int fa[UNROLL];
#pragma unroll
                for (int u = 0; u < UNROLL; ++u) {
                    const int ix = min(ix0 + 32 * u, fnx - 1);   // clamped: always a legal voxel
                    const float fx = (float)ix;
                    const float cx = __fmaf_rn(m[0], fx, rx);
                    const float cy = __fmaf_rn(m[4], fx, ry);
                    const float cz = __fmaf_rn(m[8], fx, rz);
                    smp[u] = sample_bin<INTERP, GATHER>(mv, cx, cy, cz);
                    smp[u].ok = smp[u].ok && (ix0 + 32 * u < fnx);
                    if (a.mask_bits != nullptr) {
                        const unsigned vi = (unsigned)row * (unsigned)fnx + (unsigned)ix;
                        smp[u].ok = smp[u].ok && ((__ldg(a.mask_bits + (vi >> 5)) >> (vi & 31u)) & 1u);
                    }
                    fa[u] = __ldg(frow + ix);
                }
#pragma unroll
                for (int u = 0; u < UNROLL; ++u) {
                    if (smp[u].ok) {
                        if (!HIST) probe_acc += (unsigned)(fa[u] * pitch + smp[u].b);
                        else if (fa[u] < rows_smem) atomicAdd(&sh_hist[fa[u] * pitch + smp[u].b], 1u);
                        else atomicAdd(&gh[__ldg(a.rank_inv + fa[u]) * nb + smp[u].b], 1u);
                    }
                }
            }
        }
        if (!HIST) continue;
        __syncthreads();
        // merge the CTA-private rows into the transform's global histogram (un-ranking the fixed
        // bin) and re-zero them for the next item
        for (int r = warp; r < rows_smem; r += nwarps) {
            uint32_t* grow = gh + (size_t)__ldg(a.rank_inv + r) * nb;
            for (int b = lane; b < nb; b += 32) {
                const uint32_t v = sh_hist[r * pitch + b];
                if (v) {
                    sh_hist[r * pitch + b] = 0u;
                    atomicAdd(&grow[b], v);
                }
            }
        }
        __syncthreads();
    }
    if (!HIST) {
        probe_acc = warp_sum(probe_acc);
        if (lane == 0) atomicAdd(a.sink, probe_acc);
    }
}

template <int INTERP, int UNROLL, int GATHER, bool HIST>
static cudaError_t launch_resample_t(const ResampleArgs& a, int num_sms, cudaStream_t s) {
    const size_t smem = (size_t)a.rows_smem * a.pitch * sizeof(uint32_t);
    auto kern = resample_hist_kernel<INTERP, UNROLL, GATHER, HIST>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    // leave the rest of the SM's 256 KB to L1 (the gathers live there)
    // (a hint in percent of 228 KB, rounded down: the driver picks the smallest carve-out that still
    // holds the CTA's shared memory + 1 KB)
    int carve = (int)((smem + 1024) * 100 / (228 * 1024));
    if (carve > 100) carve = 100;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, carve);
    if (e != cudaSuccess) return e;
    const long long nitems = (long long)a.n_transforms * a.nslabs;
    long long grid = nitems < num_sms ? nitems : num_sms;
    if (grid < 1) return cudaSuccess;
    kern<<<(unsigned)grid, kHistThreads, smem, s>>>(a);
    return cudaGetLastError();
}


// ------------------------------------------------------------------------------------------------
// a3 + a4, trilinear, yz-quad gathers: the kernel rotations (and every other non-diagonal transform) take.
// Same arithmetic as resample_hist_kernel<TRILINEAR> (CANON-2, CANON-4, CANON-5), organised so that the loads
// of several samples are in flight per lane (the first version waited on memory with one pair in flight; as
// committed the L1TEX data pipe is 92 % busy and the issue slots 83 %, profiles/r2c_ncu.md section 6) --
//   * every trip first resolves the cells of its U samples per lane and issues all 2U 16-byte loads (and the
//     U fixed-bin loads), then lerps, bins and counts: U independent load pairs are in flight per lane (the
//     64-register budget of a 1024-thread CTA made the compiler reuse one register set for all samples, i.e.
//     one pair in flight; THREADS < 1024 buys the registers);
//   * items are ordered SLAB-major (all transforms of a z slab of the fixed volume before the next slab), so
//     the SMs work on one region of the 16-byte-per-voxel quad volume at a time and it stays L2-resident
//     (launch_resample_hist picks the slab count from the quad volume's size);
//   * shared-memory updates use a 32-bit shared address computed once (RED.shared), tiles advance by counters
//     instead of a division per row.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void red_shared_inc32(unsigned addr) {
    asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory");
}

template <int THREADS, int U, bool HIST, bool MASK, bool RARE>
__global__ void __launch_bounds__(THREADS, 1) resample_quad_kernel(const __grid_constant__ ResampleArgs a) {
    extern __shared__ __align__(16) uint32_t sh_hist[];
    constexpr int NW = THREADS / 32;
    constexpr int TZ = NW / 8;                 // the CTA's warps cover 8 (y) x TZ (z) fixed rows at a time
    const int nb = a.nb, pitch = a.pitch, rows_smem = a.rows_smem;
    const int words = rows_smem * pitch;
    for (int w = threadIdx.x; w < words; w += THREADS) sh_hist[w] = 0u;
    __syncthreads();
    unsigned sbase = (unsigned)__cvta_generic_to_shared(sh_hist);
    asm volatile("" : "+r"(sbase));            // keep the shared base in a register (else it is re-derived per update)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wy = warp & 7, wz = warp >> 3;
    const int fnx = a.f.nx, fny = a.f.ny, fnz = a.f.nz;
    const int tiles_y = (fny + 7) >> 3;
    const int tiles_total = tiles_y * ((fnz + TZ - 1) / TZ);
    const unsigned pnx = (unsigned)a.m.nx + 2u, pny = (unsigned)a.m.ny + 2u;
    // padded index of cell (jx+1, jy+1, jz+1) from the raw float bits T_k = magic + j_k (see MovingView::fold)
    const unsigned fold = (unsigned)(kFloorMagicBits - 1) * (pny * pnx + pnx + 1u);
    const float hx = __fsub_rn((float)a.m.nx, 0.5f), hy = __fsub_rn((float)a.m.ny, 0.5f), hz = __fsub_rn((float)a.m.nz, 0.5f);
    const float mlo = a.mlo, mscale = a.mscale;
    const int top = nb - 1;
    const float4* __restrict__ quad = a.moving_quad;
    const float flane = (float)lane;
    unsigned probe_acc = 0u;

    const long long nitems = (long long)a.n_transforms * a.nslabs;
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int slab = (int)(item / a.n_transforms);                   // slab-major: neighbours in time share a slab
        const int t = (int)(item - (long long)slab * a.n_transforms);
        const int tile_lo = (int)((long long)tiles_total * slab / a.nslabs);
        const int tile_hi = (int)((long long)tiles_total * (slab + 1) / a.nslabs);
        float m[12];
#pragma unroll
        for (int i = 0; i < 12; ++i) m[i] = __ldg(a.M + (size_t)t * 12 + i);
        uint32_t* gh = a.hist + (size_t)t * nb * nb;

        int tz = tile_lo / tiles_y, ty = tile_lo - tz * tiles_y;
        for (int tile = tile_lo; tile < tile_hi; ++tile, ++ty) {
            if (ty == tiles_y) { ty = 0; ++tz; }
            const int iy = (ty << 3) + wy, iz = tz * TZ + wz;
            if (iy >= fny || iz >= fnz) continue;
            const unsigned row = (unsigned)(iz * fny + iy);
            const float fy = (float)iy, fz = (float)iz;
            // CANON-2: row terms, then one fma per voxel and axis
            const float rx = __fmaf_rn(m[1], fy, __fmaf_rn(m[2], fz, m[3]));
            const float ry = __fmaf_rn(m[5], fy, __fmaf_rn(m[6], fz, m[7]));
            const float rz = __fmaf_rn(m[9], fy, __fmaf_rn(m[10], fz, m[11]));
            const uint8_t* __restrict__ frow = a.fbins_ranked + (size_t)row * (unsigned)fnx;
            float fx0 = flane;                                           // (float)ix0, advanced by exact float adds
            for (unsigned ix0 = (unsigned)lane; ix0 < (unsigned)fnx; ix0 += 32u * U, fx0 += (float)(32 * U)) {
                // ---- phase 1: cells of the U samples, all loads issued ----
                unsigned idx[U];
                float wxs[U], wys[U], wzs[U];
                bool ok[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    // voxels past the row end get coordinates too (just numbers) and are marked invalid
                    const float fx = fx0 + (float)(32 * u);              // exact: small integers
                    const float cx = __fmaf_rn(m[0], fx, rx), cy = __fmaf_rn(m[4], fx, ry), cz = __fmaf_rn(m[8], fx, rz);
                    // CANON-4: region [-0.5, n-0.5), edge clamp (via the padded copy)
                    bool v = cx >= -0.5f && cx < hx && cy >= -0.5f && cy < hy && cz >= -0.5f && cz < hz &&
                             (ix0 + 32u * u < (unsigned)fnx);
                    if (MASK) {
                        const unsigned vi = row * (unsigned)fnx + min(ix0 + 32u * u, (unsigned)fnx - 1u);
                        v = v && ((__ldg(a.mask_bits + (vi >> 5)) >> (vi & 31u)) & 1u);
                    }
                    const float tx = __fadd_rd(cx, kFloorMagic), ty2 = __fadd_rd(cy, kFloorMagic), tz2 = __fadd_rd(cz, kFloorMagic);
                    wxs[u] = __fsub_rn(cx, __fsub_rn(tx, kFloorMagic));
                    wys[u] = __fsub_rn(cy, __fsub_rn(ty2, kFloorMagic));
                    wzs[u] = __fsub_rn(cz, __fsub_rn(tz2, kFloorMagic));
                    const unsigned i = (__float_as_uint(tz2) * pny + __float_as_uint(ty2)) * pnx + __float_as_uint(tx) - fold;
                    idx[u] = v ? i : 0u;
                    ok[u] = v;
                }
                float4 q0[U], q1[U];
                unsigned fa[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    q0[u] = __ldg(quad + idx[u]);
                    q1[u] = __ldg(quad + idx[u] + 1);
                    fa[u] = ok[u] ? (unsigned)__ldg(frow + ix0 + 32u * u) : 0u;
                }
                // ---- phase 2: x-, y-, z-lerps (CANON-4 order), binning (CANON-5), one update ----
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const float v00 = lerp_rn(q0[u].x, q1[u].x, wxs[u]);
                    const float v10 = lerp_rn(q0[u].y, q1[u].y, wxs[u]);
                    const float v01 = lerp_rn(q0[u].z, q1[u].z, wxs[u]);
                    const float v11 = lerp_rn(q0[u].w, q1[u].w, wxs[u]);
                    const float w0 = lerp_rn(v00, v10, wys[u]);
                    const float w1 = lerp_rn(v01, v11, wys[u]);
                    const float v = lerp_rn(w0, w1, wzs[u]);
                    const float tt = __fmul_rn(__fsub_rn(v, mlo), mscale);
                    const unsigned b = (unsigned)min(max(__float2int_rd(tt), 0), top);
                    const unsigned cell = fa[u] * (unsigned)pitch + b;
                    if (!HIST) {
                        if (ok[u]) probe_acc += cell;
                    } else if (!RARE) {
                        if (ok[u]) red_shared_inc32(sbase + cell * 4u);
                    } else {
                        const bool in_smem = (int)fa[u] < rows_smem;
                        if (ok[u] && in_smem) red_shared_inc32(sbase + cell * 4u);
                        if (ok[u] && !in_smem) atomicAdd(&gh[__ldg(a.rank_inv + fa[u]) * nb + b], 1u);
                    }
                }
            }
        }
        if (!HIST) continue;
        __syncthreads();
        // merge the CTA-private rows into the transform's global histogram (un-ranking the fixed bin) and
        // re-zero them for the next item
        for (int r = warp; r < rows_smem; r += NW) {
            uint32_t* grow = gh + (size_t)__ldg(a.rank_inv + r) * nb;
            for (int b = lane; b < nb; b += 32) {
                const uint32_t v = sh_hist[r * pitch + b];
                if (v) {
                    sh_hist[r * pitch + b] = 0u;
                    atomicAdd(&grow[b], v);
                }
            }
        }
        __syncthreads();
    }
    if (!HIST) {
        probe_acc = warp_sum(probe_acc);
        if (lane == 0) atomicAdd(a.sink, probe_acc);
    }
}

template <int THREADS, int U, bool HIST, bool MASK, bool RARE>
static cudaError_t launch_quad_t(const ResampleArgs& a, int num_sms, cudaStream_t s) {
    const size_t smem = (size_t)a.rows_smem * a.pitch * sizeof(uint32_t);
    auto kern = resample_quad_kernel<THREADS, U, HIST, MASK, RARE>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int carve = (int)((smem + 1024) * 100 / (228 * 1024));
    if (carve > 100) carve = 100;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, carve);
    if (e != cudaSuccess) return e;
    const long long nitems = (long long)a.n_transforms * a.nslabs;
    long long grid = nitems < num_sms ? nitems : num_sms;
    if (grid < 1) return cudaSuccess;
    kern<<<(unsigned)grid, THREADS, smem, s>>>(a);
    return cudaGetLastError();
}

template <int THREADS>
static cudaError_t launch_quad_threads(const ResampleArgs& a, int unroll, int num_sms, cudaStream_t s) {
    const bool probe = a.sink != nullptr, mask = a.mask_bits != nullptr;
    // RARE: some populated fixed-bin rank has no shared row (its updates go to the global histogram)
#define MI_QUAD(UU)                                                                                   \
    do {                                                                                              \
        if (probe) return launch_quad_t<THREADS, UU, false, false, false>(a, num_sms, s);             \
        if (mask) return launch_quad_t<THREADS, UU, true, true, true>(a, num_sms, s);                 \
        if (a.has_rare) return launch_quad_t<THREADS, UU, true, false, true>(a, num_sms, s);          \
        return launch_quad_t<THREADS, UU, true, false, false>(a, num_sms, s);                         \
    } while (0)
    if (unroll == 1) MI_QUAD(1);
    if (unroll == 2) MI_QUAD(2);
    if (unroll == 3) MI_QUAD(3);
    MI_QUAD(4);
#undef MI_QUAD
}

// ------------------------------------------------------------------------------------------------
// a3 + a4, nearest neighbour, arbitrary 3x4: resample_quad_kernel's organisation (cells of the U samples of a lane
// resolved first, all loads issued, then the updates through a 32-bit shared address) with CANON-3 sampling: the
// moving bin is one byte of the pre-binned volume.  Same tiles, same slab-major item order.
// ------------------------------------------------------------------------------------------------
template <int U, bool MASK, bool RARE>
__global__ void __launch_bounds__(kHistThreads, 1) resample_nn_kernel(const __grid_constant__ ResampleArgs a) {
    extern __shared__ __align__(16) uint32_t sh_hist[];
    constexpr int NW = kHistThreads / 32;
    constexpr int TZ = NW / 8;
    const int nb = a.nb, pitch = a.pitch, rows_smem = a.rows_smem;
    const int words = rows_smem * pitch;
    for (int w = threadIdx.x; w < words; w += kHistThreads) sh_hist[w] = 0u;
    __syncthreads();
    unsigned sbase = (unsigned)__cvta_generic_to_shared(sh_hist);
    asm volatile("" : "+r"(sbase));
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wy = warp & 7, wz = warp >> 3;
    const int fnx = a.f.nx, fny = a.f.ny, fnz = a.f.nz;
    const int tiles_y = (fny + 7) >> 3;
    const int tiles_total = tiles_y * ((fnz + TZ - 1) / TZ);
    const unsigned mnx = (unsigned)a.m.nx, mny = (unsigned)a.m.ny;
    const float fmx = (float)a.m.nx, fmy = (float)a.m.ny, fmz = (float)a.m.nz;
    // voxel index (jz*ny + jy)*nx + jx from the raw float bits T_k = magic + j_k, modulo 2^32
    const unsigned fold = (unsigned)kFloorMagicBits * (mny * mnx + mnx + 1u);
    const uint8_t* __restrict__ mbins = a.mbins;
    const float flane = (float)lane;

    const long long nitems = (long long)a.n_transforms * a.nslabs;
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int slab = (int)(item / a.n_transforms);
        const int t = (int)(item - (long long)slab * a.n_transforms);
        const int tile_lo = (int)((long long)tiles_total * slab / a.nslabs);
        const int tile_hi = (int)((long long)tiles_total * (slab + 1) / a.nslabs);
        float m[12];
#pragma unroll
        for (int i = 0; i < 12; ++i) m[i] = __ldg(a.M + (size_t)t * 12 + i);
        uint32_t* gh = a.hist + (size_t)t * nb * nb;

        int tz = tile_lo / tiles_y, ty = tile_lo - tz * tiles_y;
        for (int tile = tile_lo; tile < tile_hi; ++tile, ++ty) {
            if (ty == tiles_y) { ty = 0; ++tz; }
            const int iy = (ty << 3) + wy, iz = tz * TZ + wz;
            if (iy >= fny || iz >= fnz) continue;
            const unsigned row = (unsigned)(iz * fny + iy);
            const float fy = (float)iy, fz = (float)iz;
            // CANON-2: row terms, then one fma per voxel and axis
            const float rx = __fmaf_rn(m[1], fy, __fmaf_rn(m[2], fz, m[3]));
            const float ry = __fmaf_rn(m[5], fy, __fmaf_rn(m[6], fz, m[7]));
            const float rz = __fmaf_rn(m[9], fy, __fmaf_rn(m[10], fz, m[11]));
            const uint8_t* __restrict__ frow = a.fbins_ranked + (size_t)row * (unsigned)fnx;
            float fx0 = flane;
            for (unsigned ix0 = (unsigned)lane; ix0 < (unsigned)fnx; ix0 += 32u * U, fx0 += (float)(32 * U)) {
                unsigned idx[U];
                bool ok[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const float fx = fx0 + (float)(32 * u);
                    const float cx = __fmaf_rn(m[0], fx, rx), cy = __fmaf_rn(m[4], fx, ry), cz = __fmaf_rn(m[8], fx, rz);
                    // CANON-3: r = floor(c + 0.5) (round half up), validity tested on r in float
                    const float tx = __fadd_rd(__fadd_rn(cx, 0.5f), kFloorMagic);
                    const float ty2 = __fadd_rd(__fadd_rn(cy, 0.5f), kFloorMagic);
                    const float tz2 = __fadd_rd(__fadd_rn(cz, 0.5f), kFloorMagic);
                    const float qx = __fsub_rn(tx, kFloorMagic), qy = __fsub_rn(ty2, kFloorMagic), qz = __fsub_rn(tz2, kFloorMagic);
                    bool v = qx >= 0.0f && qx < fmx && qy >= 0.0f && qy < fmy && qz >= 0.0f && qz < fmz &&
                             (ix0 + 32u * u < (unsigned)fnx);
                    if (MASK) {
                        const unsigned vi = row * (unsigned)fnx + min(ix0 + 32u * u, (unsigned)fnx - 1u);
                        v = v && ((__ldg(a.mask_bits + (vi >> 5)) >> (vi & 31u)) & 1u);
                    }
                    const unsigned i = (__float_as_uint(tz2) * mny + __float_as_uint(ty2)) * mnx + __float_as_uint(tx) - fold;
                    idx[u] = v ? i : 0u;
                    ok[u] = v;
                }
                unsigned mb[U], fa[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    mb[u] = (unsigned)__ldg(mbins + idx[u]);
                    fa[u] = ok[u] ? (unsigned)__ldg(frow + ix0 + 32u * u) : 0u;
                }
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const unsigned cell = fa[u] * (unsigned)pitch + mb[u];
                    if (!RARE) {
                        if (ok[u]) red_shared_inc32(sbase + cell * 4u);
                    } else {
                        const bool in_smem = (int)fa[u] < rows_smem;
                        if (ok[u] && in_smem) red_shared_inc32(sbase + cell * 4u);
                        if (ok[u] && !in_smem) atomicAdd(&gh[__ldg(a.rank_inv + fa[u]) * nb + mb[u]], 1u);
                    }
                }
            }
        }
        __syncthreads();
        for (int r = warp; r < rows_smem; r += NW) {
            uint32_t* grow = gh + (size_t)__ldg(a.rank_inv + r) * nb;
            for (int b = lane; b < nb; b += 32) {
                const uint32_t v = sh_hist[r * pitch + b];
                if (v) {
                    sh_hist[r * pitch + b] = 0u;
                    atomicAdd(&grow[b], v);
                }
            }
        }
        __syncthreads();
    }
}

template <int U, bool MASK, bool RARE>
static cudaError_t launch_nn_t(const ResampleArgs& a, int num_sms, cudaStream_t s) {
    const size_t smem = (size_t)a.rows_smem * a.pitch * sizeof(uint32_t);
    auto kern = resample_nn_kernel<U, MASK, RARE>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int carve = (int)((smem + 1024) * 100 / (228 * 1024));
    if (carve > 100) carve = 100;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, carve);
    if (e != cudaSuccess) return e;
    const long long nitems = (long long)a.n_transforms * a.nslabs;
    long long grid = nitems < num_sms ? nitems : num_sms;
    if (grid < 1) return cudaSuccess;
    kern<<<(unsigned)grid, kHistThreads, smem, s>>>(a);
    return cudaGetLastError();
}

static cudaError_t launch_nn(const ResampleArgs& a, int unroll, int num_sms, cudaStream_t s) {
    const bool mask = a.mask_bits != nullptr;
#define MI_NN(UU)                                                                          \
    do {                                                                                   \
        if (mask) return launch_nn_t<UU, true, true>(a, num_sms, s);                       \
        if (a.has_rare) return launch_nn_t<UU, false, true>(a, num_sms, s);                \
        return launch_nn_t<UU, false, false>(a, num_sms, s);                               \
    } while (0)
    if (unroll == 1) MI_NN(1);
    if (unroll == 2) MI_NN(2);
    if (unroll == 3) MI_NN(3);
    MI_NN(4);
#undef MI_NN
}

int hist_rows_in_smem(int nb, int pitch, size_t smem_bytes) {
    const size_t reserve = 1024;  // static shared memory + alignment slack
    size_t rows = (smem_bytes > reserve ? smem_bytes - reserve : 0) / ((size_t)pitch * sizeof(uint32_t));
    if (rows > (size_t)nb) rows = (size_t)nb;
    return (int)rows;
}

cudaError_t launch_resample_hist(const ResampleArgs& a, int interp, int num_sms, cudaStream_t s) {
    if (a.rows_smem < 1 || a.pitch < a.nb || a.ty_log2 < 0 || a.ty_log2 > 5) return cudaErrorInvalidConfiguration;
    // Voxels in flight per lane: a row is ceil(fnx/32) warp-chunks and a lane takes `unroll` of them per
    // trip, so the last trip of a row idles (trips*unroll - chunks) chunks: pick the unroll in 1..4 that
    // wastes the fewest, the larger one on ties (260 voxels = 9 chunks -> 3).
    int unroll = a.unroll;
    if (unroll < 1 || unroll > 4) {
        const int chunks = (a.f.nx + 31) / 32;
        int best_waste = 1 << 30;
        for (int u = 1; u <= 4; ++u) {
            const int waste = (chunks + u - 1) / u * u - chunks;
            if (waste <= best_waste) { best_waste = waste; unroll = u; }
        }
    }
    if (interp == MI_INTERP_NEAREST) {
        if (a.sink != nullptr) return cudaErrorInvalidConfiguration;
        if (a.gather == kGatherQuad) return launch_nn(a, unroll, num_sms, s);   // MI_OPT_GENERIC_GATHER = 0: round 1's kernel
        if (unroll == 1) return launch_resample_t<MI_INTERP_NEAREST, 1, kGatherScalar, true>(a, num_sms, s);
        if (unroll == 2) return launch_resample_t<MI_INTERP_NEAREST, 2, kGatherScalar, true>(a, num_sms, s);
        if (unroll == 3) return launch_resample_t<MI_INTERP_NEAREST, 3, kGatherScalar, true>(a, num_sms, s);
        return launch_resample_t<MI_INTERP_NEAREST, 4, kGatherScalar, true>(a, num_sms, s);
    }
#define MI_TRI(G, H)                                                                                  \
    do {                                                                                              \
        if (unroll == 1) return launch_resample_t<MI_INTERP_TRILINEAR, 1, G, H>(a, num_sms, s);       \
        if (unroll == 2) return launch_resample_t<MI_INTERP_TRILINEAR, 2, G, H>(a, num_sms, s);       \
        if (unroll == 3) return launch_resample_t<MI_INTERP_TRILINEAR, 3, G, H>(a, num_sms, s);       \
        return launch_resample_t<MI_INTERP_TRILINEAR, 4, G, H>(a, num_sms, s);                        \
    } while (0)
    if (a.gather == kGatherQuad && a.moving_quad != nullptr) {
        if (a.threads == 512) return launch_quad_threads<512>(a, unroll, num_sms, s);
        if (a.threads == 768) return launch_quad_threads<768>(a, unroll, num_sms, s);
        return launch_quad_threads<1024>(a, unroll, num_sms, s);
    }
    if (a.sink != nullptr) MI_TRI(kGatherScalar, false);   // roofline probe: no histogram
    MI_TRI(kGatherScalar, true);
#undef MI_TRI
}

// ------------------------------------------------------------------------------------------------
// a5: entropy reduction (DESIGN.md CANON-7)
// ------------------------------------------------------------------------------------------------
// One CTA per transform.  With c the integer counts and N their total:
//   H = -sum (c/N) ln (c/N) = ln N - (sum c ln c)/N,      sum p^q = exp(-q ln N) * sum c^q.
// Accumulators per distribution X in {A, B, AB}: L_X = sum c ln c and P_X[k] = sum c^q_k.
template <int MAXB>
__global__ void __launch_bounds__(kEntropyThreads)
entropy_kernel(const uint32_t* __restrict__ hist, int nb, const double* __restrict__ q, int nq_total,
               int q_off, int nq_pass, int form, double* __restrict__ mi_out,
               int64_t* __restrict__ nvalid, const OutMap om) {
    constexpr int NW = kEntropyThreads / 32;
    constexpr int NACC = 3 * (1 + kMaxQPerPass);
    __shared__ unsigned sh_pa[MAXB], sh_pb[MAXB];
    __shared__ double sh_red[NACC][NW];
    __shared__ unsigned long long sh_n[NW];
    const int t = blockIdx.x;
    const uint32_t* __restrict__ h = hist + (size_t)t * nb * nb;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    double qv[kMaxQPerPass];
#pragma unroll
    for (int k = 0; k < kMaxQPerPass; ++k) qv[k] = k < nq_pass ? q[q_off + k] : 1.0;

    for (int i = threadIdx.x; i < MAXB; i += kEntropyThreads) { sh_pa[i] = 0u; sh_pb[i] = 0u; }
    __syncthreads();

    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = 0.0;

    // joint terms + marginal counts.  The table is mostly zeros and streams from DRAM: all MAXB/32 loads of a lane's
    // share of a row are issued first, then the non-zero ones are visited one by one so that the double-precision
    // terms are compiled once (inlined per load they spill; one load at a time the kernel waits on memory).
    constexpr int NV = MAXB / 32;
    for (int r = warp; r < nb; r += NW) {
        unsigned rowsum = 0;
        unsigned v[NV];
        unsigned nz = 0u;
#pragma unroll
        for (int u = 0; u < NV; ++u) {
            const int c = lane + 32 * u;
            v[u] = c < nb ? __ldg(h + (size_t)r * nb + c) : 0u;
        }
#pragma unroll
        for (int u = 0; u < NV; ++u) nz |= (v[u] != 0u ? 1u : 0u) << u;
        while (nz) {
            const int u = __ffs(nz) - 1;
            nz &= nz - 1u;
            unsigned val = v[0];
#pragma unroll
            for (int k = 1; k < NV; ++k) val = u == k ? v[k] : val;
            rowsum += val;
            atomicAdd(&sh_pb[lane + 32 * u], val);
            const double dv = (double)val;
            const double lc = log(dv);
            acc[2] += dv * lc;
#pragma unroll
            for (int k = 0; k < kMaxQPerPass; ++k)
                if (k < nq_pass) acc[3 + 3 * k + 2] += exp(qv[k] * lc);
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
        entropy_finish(tot, (double)n, (long long)n, t, qv, nq_pass, q_off, nq_total, form, mi_out, nvalid, om);
    }
}

// Wide histograms (nb > 256) are tens of megabytes each: the rows of one histogram are split over
// gridDim.x CTAs.  Pass 1: every CTA takes a row range of transform blockIdx.y -- joint terms into
// per-CTA partial sums, row sums (fixed marginal) stored, column sums (moving marginal) added to pb
// with integer atomics (order-free, so the result is reproducible).  Pass 2: one CTA per transform
// adds the marginal terms and the partial sums in a fixed order and finishes.
constexpr int kWideLoads = 16;   // loads in flight per lane
__global__ void __launch_bounds__(kEntropyThreads)
entropy_wide_partial_kernel(const uint32_t* __restrict__ hist, int nb, const double* __restrict__ q, int q_off,
                            int nq_pass, unsigned* __restrict__ pa, unsigned* __restrict__ pb,
                            double* __restrict__ partial /* [t][split][1 + kMaxQPerPass] */,
                            const uint8_t* __restrict__ row_used /* NULL, or nb flags: fixed bin holds voxels */) {
    constexpr int NW = kEntropyThreads / 32;
    constexpr int NA = 1 + kMaxQPerPass;
    __shared__ unsigned sh_pb[kMaxBinsWide];
    __shared__ double sh_red[NA][NW];
    const int t = blockIdx.y, split = blockIdx.x, nsplit = gridDim.x;
    const int r0 = (int)((long long)nb * split / nsplit), r1 = (int)((long long)nb * (split + 1) / nsplit);
    const uint32_t* __restrict__ h = hist + (size_t)t * nb * nb;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double qv[kMaxQPerPass];
#pragma unroll
    for (int k = 0; k < kMaxQPerPass; ++k) qv[k] = k < nq_pass ? q[q_off + k] : 1.0;
    for (int i = threadIdx.x; i < nb; i += kEntropyThreads) sh_pb[i] = 0u;
    __syncthreads();
    double acc[NA];
#pragma unroll
    for (int i = 0; i < NA; ++i) acc[i] = 0.0;
    for (int r = r0 + warp; r < r1; r += NW) {
        // a fixed bin without voxels has an all-zero row (pa is zero on entry): at 4096 bins most rows
        if (row_used != nullptr && __ldg(row_used + r) == 0) continue;
        const uint32_t* __restrict__ row = h + (size_t)r * nb;
        unsigned rowsum = 0;
        for (int c0 = lane; c0 < nb; c0 += 32 * kWideLoads) {   // kWideLoads loads in flight per lane
            unsigned v[kWideLoads];
#pragma unroll
            for (int u = 0; u < kWideLoads; ++u) v[u] = c0 + 32 * u < nb ? __ldg(row + c0 + 32 * u) : 0u;
            unsigned nz = 0u;
#pragma unroll
            for (int u = 0; u < kWideLoads; ++u) nz |= (v[u] != 0u ? 1u : 0u) << u;
            while (nz) {                                      // the non-zero ones, one by one: the terms are compiled once
                const int u = __ffs(nz) - 1;
                nz &= nz - 1u;
                unsigned val = v[0];
#pragma unroll
                for (int k = 1; k < kWideLoads; ++k) val = u == k ? v[k] : val;
                rowsum += val;
                atomicAdd(&sh_pb[c0 + 32 * u], val);
                const double dv = (double)val, lc = log(dv);
                acc[0] += dv * lc;
#pragma unroll
                for (int k = 0; k < kMaxQPerPass; ++k)
                    if (k < nq_pass) acc[1 + k] += exp(qv[k] * lc);
            }
        }
        rowsum = warp_sum(rowsum);
        if (lane == 0) pa[(size_t)t * nb + r] = rowsum;
    }
#pragma unroll
    for (int i = 0; i < NA; ++i) {
        const double sum = warp_sum_d(acc[i]);
        if (lane == 0) sh_red[i][warp] = sum;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nb; i += kEntropyThreads)
        if (sh_pb[i]) atomicAdd(&pb[(size_t)t * nb + i], sh_pb[i]);
    if (threadIdx.x < NA) {
        double sum = 0.0;
        for (int w = 0; w < NW; ++w) sum += sh_red[threadIdx.x][w];
        partial[((size_t)t * nsplit + split) * NA + threadIdx.x] = sum;
    }
}

__global__ void __launch_bounds__(kEntropyThreads)
entropy_wide_final_kernel(int nb, const double* __restrict__ q, int nq_total, int q_off, int nq_pass, int form,
                          const unsigned* __restrict__ pa, const unsigned* __restrict__ pb,
                          const double* __restrict__ partial, int nsplit, double* __restrict__ mi_out,
                          int64_t* __restrict__ nvalid, const OutMap om) {
    constexpr int NW = kEntropyThreads / 32;
    constexpr int NA = 1 + kMaxQPerPass;
    constexpr int NACC = 3 * NA;
    __shared__ double sh_red[2 * NA][NW];
    __shared__ unsigned long long sh_n[NW];
    const int t = blockIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double qv[kMaxQPerPass];
#pragma unroll
    for (int k = 0; k < kMaxQPerPass; ++k) qv[k] = k < nq_pass ? q[q_off + k] : 1.0;
    double acc[2 * NA];      // [0..NA) fixed marginal, [NA..2NA) moving marginal: sum c ln c, sum c^q_k
#pragma unroll
    for (int i = 0; i < 2 * NA; ++i) acc[i] = 0.0;
    unsigned long long n_local = 0;
    for (int i = threadIdx.x; i < nb; i += kEntropyThreads) {
        const unsigned cnt[2] = {pa[(size_t)t * nb + i], pb[(size_t)t * nb + i]};
        n_local += cnt[0];
#pragma unroll
        for (int d = 0; d < 2; ++d)
            if (cnt[d]) {
                const double dv = (double)cnt[d], lc = log(dv);
                acc[d * NA] += dv * lc;
#pragma unroll
                for (int k = 0; k < kMaxQPerPass; ++k)
                    if (k < nq_pass) acc[d * NA + 1 + k] += exp(qv[k] * lc);
            }
    }
#pragma unroll
    for (int i = 0; i < 2 * NA; ++i) {
        const double sum = warp_sum_d(acc[i]);
        if (lane == 0) sh_red[i][warp] = sum;
    }
    {
        unsigned lo = (unsigned)n_local, hi = (unsigned)(n_local >> 32);
        lo = warp_sum(lo);
        hi = warp_sum(hi);
        if (lane == 0) sh_n[warp] = ((unsigned long long)hi << 32) + lo;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot[NACC];
        for (int i = 0; i < NA; ++i) {
            double sa = 0.0, sb = 0.0, sab = 0.0;
            for (int w = 0; w < NW; ++w) { sa += sh_red[i][w]; sb += sh_red[NA + i][w]; }
            for (int sp = 0; sp < nsplit; ++sp) sab += partial[((size_t)t * nsplit + sp) * NA + i];
            const int base = i == 0 ? 0 : 3 + 3 * (i - 1);
            tot[base + 0] = sa; tot[base + 1] = sb; tot[base + 2] = sab;
        }
        unsigned long long n = 0;
        for (int w = 0; w < NW; ++w) n += sh_n[w];
        entropy_finish(tot, (double)n, (long long)n, t, qv, nq_pass, q_off, nq_total, form, mi_out, nvalid, om);
    }
}

cudaError_t launch_entropy(const uint32_t* hist, int nb, int n_transforms, const double* q_dev, int nq,
                           int q_off, int form, double* mi_out, int64_t* nvalid, OutMap om, cudaStream_t s,
                           const uint8_t* row_used) {
    if (n_transforms <= 0) return cudaSuccess;
    int nq_pass = nq - q_off;
    if (nq_pass > kMaxQPerPass) nq_pass = kMaxQPerPass;
    if (nq_pass < 0) nq_pass = 0;
    if (nb <= 256) {
        entropy_kernel<256><<<n_transforms, kEntropyThreads, 0, s>>>(hist, nb, q_dev, nq, q_off, nq_pass, form,
                                                                    mi_out, nvalid, om);
        return cudaGetLastError();
    }
    // wide: rows of every histogram split over about four waves of CTAs
    int nsplit = (4 * sm_count() + n_transforms - 1) / n_transforms;
    if (nsplit < 1) nsplit = 1;
    if (nsplit > 64) nsplit = 64;
    if (nsplit > nb) nsplit = nb;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    constexpr int NA = 1 + kMaxQPerPass;
    unsigned* pab = nullptr;
    double* partial = nullptr;
    const size_t cnt_words = (size_t)n_transforms * nb * 2;
    if ((e = dev_alloc((void**)&pab, cnt_words * sizeof(unsigned), dev, s)) != cudaSuccess) return e;
    if ((e = dev_alloc((void**)&partial, (size_t)n_transforms * nsplit * NA * sizeof(double), dev, s)) != cudaSuccess) {
        dev_free(pab, s);
        return e;
    }
    unsigned* pa = pab;
    unsigned* pb = pab + (size_t)n_transforms * nb;
    e = cudaMemsetAsync(pab, 0, cnt_words * sizeof(unsigned), s);
    if (e == cudaSuccess) {
        entropy_wide_partial_kernel<<<dim3(nsplit, n_transforms), kEntropyThreads, 0, s>>>(hist, nb, q_dev, q_off, nq_pass,
                                                                                         pa, pb, partial, row_used);
        entropy_wide_final_kernel<<<n_transforms, kEntropyThreads, 0, s>>>(nb, q_dev, nq, q_off, nq_pass, form, pa, pb,
                                                                          partial, nsplit, mi_out, nvalid, om);
        e = cudaGetLastError();
    }
    dev_free(pab, s);
    dev_free(partial, s);
    return e;
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
// Roofline probe: shared-memory atomicAdd(u32) rate; result-less adds, four
// independent updates per loop trip; pattern 6 keeps all index arithmetic out of the timed loop.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kHistThreads, 1)
atomic_probe_kernel(int words_log2, int pattern, int iters, unsigned* __restrict__ sink) {
    extern __shared__ __align__(16) uint32_t sh_tab[];
    const int words = 1 << words_log2;
    for (int w = threadIdx.x; w < words; w += blockDim.x) sh_tab[w] = 0u;
    __syncthreads();
    const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned mask = (unsigned)words - 1u;
    const unsigned tid = blockIdx.x * 1024u + threadIdx.x;
    unsigned state = tid * 2654435761u + 12345u;
    const unsigned same = (sink[0] & 1u) + 2u;  // one address, not provably uniform at compile time
    if (pattern == 6) {
        // pattern 1's statistics with NO index arithmetic in the timed loop: eight bins per thread, hashed once
        // (independent between the lanes of a warp), then only the updates.  Pattern 1 spends about a dozen
        // integer instructions per update on its hash and stops near 95 % of the crossbar bound; this one shows
        // what the crossbar itself sustains for lane-independent bins.
        unsigned pre[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            unsigned x = tid * 0x9E3779B9u + (unsigned)u * 0x85EBCA6Bu;
            x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;
            pre[u] = x & mask;
        }
        for (int it = 0; it < iters; it += 8) {
#pragma unroll
            for (int u = 0; u < 8; ++u) atomicAdd(&sh_tab[pre[u]], 1u);
        }
        iters = 0;
    }
    for (int it = 0; it < iters; it += 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            unsigned idx;
            if (pattern == 0) {
                idx = (((warp * 37u + (unsigned)(it + u) * 11u) << 5) + lane) & mask;  // lane-distinct banks
            } else if (pattern == 1) {
                // uniform random bins, INDEPENDENT between the lanes of a warp: a 32-bit integer hash of
                // (thread, update number).  32 independent lanes over 32 banks load the fullest bank with
                // 3.53 addresses on average -- the cost of a histogram update whose bin is data.
                unsigned x = tid * 0x9E3779B9u + (unsigned)(it + u) * 0x85EBCA6Bu;
                x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;
                idx = x & mask;
            } else if (pattern == 3) {
                // round 1's "random" pattern, kept for the record: one LCG per thread seeded linearly in the
                // thread index, so the 32 lanes of a warp form an arithmetic progression modulo 2^32 in every
                // round -- bins that look random in time but are evenly spread ACROSS the lanes (2.70
                // wavefronts per update instead of 3.53)
                state = state * 1664525u + 1013904223u;
                idx = (state >> 10) & mask;
            } else if (pattern == 5) {
                unsigned x = tid * 0x9E3779B9u + (unsigned)(it + u) * 0x85EBCA6Bu;      // as pattern 1
                x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;
                idx = x & mask;
            } else {
                idx = same;
            }
            // patterns 4 and 5 add a per-lane VALUE (the partial-volume kernel's weighted update, SASS ATOMS.ADD
            // instead of ATOMS.POPC.INC)
            if (pattern >= 4) atomicAdd(&sh_tab[idx], lane | 1u);
            else atomicAdd(&sh_tab[idx], 1u);
        }
    }
    __syncthreads();
    unsigned s = 0;
    for (int w = threadIdx.x; w < words; w += blockDim.x) s += sh_tab[w];
    if (s == 0xFFFFFFFFu) sink[1] = s;  // keep the table live
}

cudaError_t run_shared_atomic_probe(int nbins, int pattern, int iters, int num_sms, size_t smem_optin,
                                    double* updates_per_s) {
    // largest power-of-two table of u32 counters that is <= nbins^2 and fits in shared memory
    int words_log2 = 5;
    while ((1 << (words_log2 + 1)) <= nbins * nbins && ((size_t)4 << (words_log2 + 1)) <= smem_optin - 1024)
        ++words_log2;
    const size_t smem = (size_t)4 << words_log2;
    iters = (iters + 7) & ~7;
    unsigned* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, 2 * sizeof(unsigned));
    if (e != cudaSuccess) return e;
    cudaMemset(sink, 0, 2 * sizeof(unsigned));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best_ms = 1e30f;
    cudaFuncSetAttribute(atomic_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    for (int rep = 0; rep < 6 && e == cudaSuccess; ++rep) {
        cudaEventRecord(e0, 0);
        atomic_probe_kernel<<<num_sms, kHistThreads, smem, 0>>>(words_log2, pattern, iters, sink);
        cudaEventRecord(e1, 0);
        e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 1 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (e != cudaSuccess) return e;
    *updates_per_s = (double)iters * kHistThreads * num_sms / (best_ms * 1e-3);
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------
// Wide histograms, 256 < nbins <= kMaxBinsWide ("uses all the voxels and produces a
// full histogram"): uint16 bin indices, the joint histogram (nb*nb*4 bytes: 64 MB at 4096
// bins) lives in global memory and is updated with L2 reductions.  The lanes of a warp that hit the
// same counter are merged first (__match_any_sync): the background bin alone takes a quarter of all
// updates, and the L2 serialises updates of one address.  Same CANON-2..5 arithmetic as above.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) prebin16_kernel(const float* __restrict__ vol, uint16_t* __restrict__ bins,
                                                       int64_t n, float lo, float scale, float top) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        bins[i] = (uint16_t)bin_index(__ldcs(vol + i), lo, scale, top);
}

cudaError_t launch_prebin16(const float* vol, uint16_t* bins, int64_t n, float lo, float scale, int nb, cudaStream_t s) {
    if (n <= 0) return cudaSuccess;
    int64_t blocks = (n + 255) / 256;
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    prebin16_kernel<<<(unsigned)blocks, 256, 0, s>>>(vol, bins, n, lo, scale, (float)(nb - 1));
    return cudaGetLastError();
}

template <int INTERP>
__global__ void __launch_bounds__(512) resample_hist_wide_kernel(const __grid_constant__ WideArgs a) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int fnx = a.f.nx, nb = a.nb;
    const int rows_total = a.f.ny * a.f.nz;
    const int pnx = a.m.nx + 2, pny = a.m.ny + 2;
    const float fxm = (float)a.m.nx, fym = (float)a.m.ny, fzm = (float)a.m.nz;
    const float hx = __fsub_rn(fxm, 0.5f), hy = __fsub_rn(fym, 0.5f), hz = __fsub_rn(fzm, 0.5f);
    const long long nitems = (long long)a.n_transforms * a.nslabs;
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int t = (int)(item / a.nslabs);
        const int slab = (int)(item - (long long)t * a.nslabs);
        const int row_lo = (int)((long long)rows_total * slab / a.nslabs);
        const int row_hi = (int)((long long)rows_total * (slab + 1) / a.nslabs);
        float m[12];
#pragma unroll
        for (int i = 0; i < 12; ++i) m[i] = __ldg(a.M + (size_t)t * 12 + i);
        uint32_t* gh = a.hist + (size_t)t * nb * nb;
        for (int row = row_lo + warp; row < row_hi; row += nwarps) {
            const int iz = row / a.f.ny, iy = row - iz * a.f.ny;
            const float fy = (float)iy, fz = (float)iz;
            const float rx = __fmaf_rn(m[1], fy, __fmaf_rn(m[2], fz, m[3]));
            const float ry = __fmaf_rn(m[5], fy, __fmaf_rn(m[6], fz, m[7]));
            const float rz = __fmaf_rn(m[9], fy, __fmaf_rn(m[10], fz, m[11]));
            const uint16_t* __restrict__ frow = a.fbins + (size_t)row * fnx;
            for (int ix0 = 0; ix0 < fnx; ix0 += 32) {          // the whole warp stays in the loop (match_any)
                const int ix = ix0 + lane;
                bool ok = ix < fnx;
                unsigned key = 0xFFFFFFFFu;
                if (ok) {
                    const float fx = (float)ix;
                    const float cx = __fmaf_rn(m[0], fx, rx), cy = __fmaf_rn(m[4], fx, ry), cz = __fmaf_rn(m[8], fx, rz);
                    int b = 0;
                    if (INTERP == MI_INTERP_NEAREST) {
                        const float qx = floorf(__fadd_rn(cx, 0.5f)), qy = floorf(__fadd_rn(cy, 0.5f)), qz = floorf(__fadd_rn(cz, 0.5f));
                        ok = qx >= 0.0f && qx < fxm && qy >= 0.0f && qy < fym && qz >= 0.0f && qz < fzm;
                        if (ok) b = __ldg(a.mbins + ((size_t)(int)qz * a.m.ny + (int)qy) * a.m.nx + (int)qx);
                    } else {
                        ok = cx >= -0.5f && cx < hx && cy >= -0.5f && cy < hy && cz >= -0.5f && cz < hz;
                        if (ok) {
                            const float gx = floorf(cx), gy = floorf(cy), gz = floorf(cz);
                            const float wx = __fsub_rn(cx, gx), wy = __fsub_rn(cy, gy), wz = __fsub_rn(cz, gz);
                            const float* __restrict__ p = a.moving_pad + ((size_t)((int)gz + 1) * pny + ((int)gy + 1)) * pnx + ((int)gx + 1);
                            const float* __restrict__ pz = p + (size_t)pnx * pny;
                            const float v00 = lerp_rn(__ldg(p), __ldg(p + 1), wx), v10 = lerp_rn(__ldg(p + pnx), __ldg(p + pnx + 1), wx);
                            const float v01 = lerp_rn(__ldg(pz), __ldg(pz + 1), wx), v11 = lerp_rn(__ldg(pz + pnx), __ldg(pz + pnx + 1), wx);
                            const float v = lerp_rn(lerp_rn(v00, v10, wy), lerp_rn(v01, v11, wy), wz);
                            const float tt = __fmul_rn(__fsub_rn(v, a.mlo), a.mscale);
                            b = min(max(__float2int_rd(tt), 0), nb - 1);
                        }
                    }
                    if (ok && a.mask_bits != nullptr) {
                        const unsigned vi = (unsigned)row * (unsigned)fnx + (unsigned)ix;
                        ok = (__ldg(a.mask_bits + (vi >> 5)) >> (vi & 31u)) & 1u;
                    }
                    if (ok) key = (unsigned)__ldg(frow + ix) * (unsigned)nb + (unsigned)b;
                }
                // one reduction per distinct counter of the warp
                const unsigned peers = __match_any_sync(0xffffffffu, key);
                if (ok && lane == __ffs(peers) - 1) atomicAdd(&gh[key], (unsigned)__popc(peers));
            }
        }
    }
}

// 4096-bin population count of a uint16 volume (CTA-private shared histogram, merged with atomics): finds the
// most populated fixed and moving bins of a wide context (resample_wide_kernel's register-summed cell).
__global__ void __launch_bounds__(256) bin_count16_kernel(const uint16_t* __restrict__ bins, int64_t n,
                                                          unsigned long long* __restrict__ counts) {
    __shared__ unsigned sh[kMaxBinsWide];
    for (int i = threadIdx.x; i < kMaxBinsWide; i += 256) sh[i] = 0u;
    __syncthreads();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        atomicAdd(&sh[bins[i] & (kMaxBinsWide - 1)], 1u);
    __syncthreads();
    for (int i = threadIdx.x; i < kMaxBinsWide; i += 256)
        if (sh[i]) atomicAdd(&counts[i], (unsigned long long)sh[i]);
}

cudaError_t launch_bin_count16(const uint16_t* bins, int64_t n, unsigned long long* counts, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(counts, 0, kMaxBinsWide * sizeof(unsigned long long), s);
    if (e != cudaSuccess) return e;
    int64_t blocks = (n + 255) / 256;
    if (blocks < 1) blocks = 1;
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    bin_count16_kernel<<<(unsigned)blocks, 256, 0, s>>>(bins, n, counts);
    return cudaGetLastError();
}

// fixed bins -> population ranks (uint16): the most populated fixed bins get the shared-memory rows of
// resample_wide_kernel
__global__ void __launch_bounds__(256) remap16_kernel(const uint16_t* __restrict__ bins, uint16_t* __restrict__ ranked,
                                                      int64_t n, const uint16_t* __restrict__ rank) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        ranked[i] = __ldg(rank + (bins[i] & (kMaxBinsWide - 1)));
}

cudaError_t launch_remap16(const uint16_t* bins, uint16_t* ranked, int64_t n, const uint16_t* rank, cudaStream_t s) {
    int64_t blocks = (n + 255) / 256;
    if (blocks < 1) blocks = 1;
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    remap16_kernel<<<(unsigned)blocks, 256, 0, s>>>(bins, ranked, n, rank);
    return cudaGetLastError();
}

// Wide histograms, second version: resample_quad_kernel's organisation (rows of an 8 x 4 tile per CTA pass, the cells
// of U samples per lane resolved first, all loads issued -- two 16-byte yz-quad loads per trilinear sample, one
// 2-byte load per nearest-neighbour sample -- slab-major items) with the counters in global memory.  Fixed bins
// arrive RANKED by population: the rows of the a.rows_smem most populated fixed bins (48 rows at 1024 bins, 12 at 4096:
// the background and the most common tissue levels) are counted in shared memory and added to the global histogram
// once per item; every other update is a plain L2 reduction (round 1 ran __match_any_sync before every update,
// about 50 clocks per warp-wide update).
template <int INTERP, int U, bool MASK>
__global__ void __launch_bounds__(kHistThreads, 1) resample_wide_kernel(const __grid_constant__ WideArgs a) {
    extern __shared__ __align__(16) uint32_t sh_hist[];
    constexpr int NW = kHistThreads / 32;
    constexpr int TZ = NW / 8;
    const int nb = a.nb, pitch = a.pitch, rows_smem = a.rows_smem;
    for (int w = threadIdx.x; w < rows_smem * pitch; w += kHistThreads) sh_hist[w] = 0u;
    __syncthreads();
    unsigned sbase = (unsigned)__cvta_generic_to_shared(sh_hist);
    asm volatile("" : "+r"(sbase));
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wy = warp & 7, wz = warp >> 3;
    const int fnx = a.f.nx, fny = a.f.ny, fnz = a.f.nz;
    const int tiles_y = (fny + 7) >> 3;
    const int tiles_total = tiles_y * ((fnz + TZ - 1) / TZ);
    const unsigned pnx = (unsigned)a.m.nx + 2u, pny = (unsigned)a.m.ny + 2u;
    const unsigned mnx = (unsigned)a.m.nx, mny = (unsigned)a.m.ny;
    const unsigned fold_pad = (unsigned)(kFloorMagicBits - 1) * (pny * pnx + pnx + 1u);   // see MovingView::fold
    const unsigned fold_nn = (unsigned)kFloorMagicBits * (mny * mnx + mnx + 1u);
    const float fmx = (float)a.m.nx, fmy = (float)a.m.ny, fmz = (float)a.m.nz;
    const float hx = __fsub_rn(fmx, 0.5f), hy = __fsub_rn(fmy, 0.5f), hz = __fsub_rn(fmz, 0.5f);
    const float mlo = a.mlo, mscale = a.mscale;
    const int top = nb - 1;
    const float4* __restrict__ quad = a.moving_quad;
    const uint16_t* __restrict__ mbins = a.mbins;
    const float flane = (float)lane;

    const long long nitems = (long long)a.n_transforms * a.nslabs;
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        // slab-major: the SMs spread over the counters of ALL transforms of the call.  Grouping the transforms so
        // that one group's counters stay L2-resident (16 transforms at 1024 bins, one at 4096) measured 35 / 92 ms
        // against 24 / 45 ms on a 125-transform call at the C3 size: contention on the counters costs more than
        // their L2 misses.
        const int slab = (int)(item / a.n_transforms);
        const int t = (int)(item - (long long)slab * a.n_transforms);
        const int tile_lo = (int)((long long)tiles_total * slab / a.nslabs);
        const int tile_hi = (int)((long long)tiles_total * (slab + 1) / a.nslabs);
        float m[12];
#pragma unroll
        for (int i = 0; i < 12; ++i) m[i] = __ldg(a.M + (size_t)t * 12 + i);
        uint32_t* gh = a.hist + (size_t)t * nb * nb;

        int tz = tile_lo / tiles_y, ty = tile_lo - tz * tiles_y;
        for (int tile = tile_lo; tile < tile_hi; ++tile, ++ty) {
            if (ty == tiles_y) { ty = 0; ++tz; }
            const int iy = (ty << 3) + wy, iz = tz * TZ + wz;
            if (iy >= fny || iz >= fnz) continue;
            const unsigned row = (unsigned)(iz * fny + iy);
            const float fy = (float)iy, fz = (float)iz;
            // CANON-2: row terms, then one fma per voxel and axis
            const float rx = __fmaf_rn(m[1], fy, __fmaf_rn(m[2], fz, m[3]));
            const float ry = __fmaf_rn(m[5], fy, __fmaf_rn(m[6], fz, m[7]));
            const float rz = __fmaf_rn(m[9], fy, __fmaf_rn(m[10], fz, m[11]));
            const uint16_t* __restrict__ frow = a.fbins_ranked + (size_t)row * (unsigned)fnx;
            float fx0 = flane;
            for (unsigned ix0 = (unsigned)lane; ix0 < (unsigned)fnx; ix0 += 32u * U, fx0 += (float)(32 * U)) {
                unsigned idx[U];
                float wxs[U], wys[U], wzs[U];
                bool ok[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const float fx = fx0 + (float)(32 * u);
                    const float cx = __fmaf_rn(m[0], fx, rx), cy = __fmaf_rn(m[4], fx, ry), cz = __fmaf_rn(m[8], fx, rz);
                    bool v;
                    unsigned i;
                    if (INTERP == MI_INTERP_NEAREST) {
                        // CANON-3: r = floor(c + 0.5) (round half up), validity tested on r in float
                        const float tx = __fadd_rd(__fadd_rn(cx, 0.5f), kFloorMagic);
                        const float ty2 = __fadd_rd(__fadd_rn(cy, 0.5f), kFloorMagic);
                        const float tz2 = __fadd_rd(__fadd_rn(cz, 0.5f), kFloorMagic);
                        const float qx = __fsub_rn(tx, kFloorMagic), qy = __fsub_rn(ty2, kFloorMagic), qz = __fsub_rn(tz2, kFloorMagic);
                        v = qx >= 0.0f && qx < fmx && qy >= 0.0f && qy < fmy && qz >= 0.0f && qz < fmz;
                        i = (__float_as_uint(tz2) * mny + __float_as_uint(ty2)) * mnx + __float_as_uint(tx) - fold_nn;
                        wxs[u] = wys[u] = wzs[u] = 0.0f;
                    } else {
                        // CANON-4: region [-0.5, n-0.5), edge clamp (via the padded copy)
                        v = cx >= -0.5f && cx < hx && cy >= -0.5f && cy < hy && cz >= -0.5f && cz < hz;
                        const float tx = __fadd_rd(cx, kFloorMagic), ty2 = __fadd_rd(cy, kFloorMagic), tz2 = __fadd_rd(cz, kFloorMagic);
                        wxs[u] = __fsub_rn(cx, __fsub_rn(tx, kFloorMagic));
                        wys[u] = __fsub_rn(cy, __fsub_rn(ty2, kFloorMagic));
                        wzs[u] = __fsub_rn(cz, __fsub_rn(tz2, kFloorMagic));
                        i = (__float_as_uint(tz2) * pny + __float_as_uint(ty2)) * pnx + __float_as_uint(tx) - fold_pad;
                    }
                    v = v && (ix0 + 32u * u < (unsigned)fnx);
                    if (MASK) {
                        const unsigned vi = row * (unsigned)fnx + min(ix0 + 32u * u, (unsigned)fnx - 1u);
                        v = v && ((__ldg(a.mask_bits + (vi >> 5)) >> (vi & 31u)) & 1u);
                    }
                    idx[u] = v ? i : 0u;
                    ok[u] = v;
                }
                float4 q0[U], q1[U];
                unsigned mb[U], fa[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    if (INTERP == MI_INTERP_NEAREST) {
                        mb[u] = (unsigned)__ldg(mbins + idx[u]);
                    } else {
                        q0[u] = __ldg(quad + idx[u]);
                        q1[u] = __ldg(quad + idx[u] + 1);
                    }
                    fa[u] = ok[u] ? (unsigned)__ldg(frow + ix0 + 32u * u) : 0u;
                }
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    unsigned b;
                    if (INTERP == MI_INTERP_NEAREST) {
                        b = mb[u];
                    } else {
                        // x-, y-, z-lerps (CANON-4 order), binning (CANON-5)
                        const float v00 = lerp_rn(q0[u].x, q1[u].x, wxs[u]);
                        const float v10 = lerp_rn(q0[u].y, q1[u].y, wxs[u]);
                        const float v01 = lerp_rn(q0[u].z, q1[u].z, wxs[u]);
                        const float v11 = lerp_rn(q0[u].w, q1[u].w, wxs[u]);
                        const float w0 = lerp_rn(v00, v10, wys[u]);
                        const float w1 = lerp_rn(v01, v11, wys[u]);
                        const float v = lerp_rn(w0, w1, wzs[u]);
                        const float tt = __fmul_rn(__fsub_rn(v, mlo), mscale);
                        b = (unsigned)min(max(__float2int_rd(tt), 0), top);
                    }
                    const bool in_smem = (int)fa[u] < rows_smem;
                    if (ok[u] && in_smem) red_shared_inc32(sbase + (fa[u] * (unsigned)pitch + b) * 4u);
                    if (ok[u] && !in_smem) atomicAdd(&gh[(unsigned)__ldg(a.rank_inv + fa[u]) * (unsigned)nb + b], 1u);
                }
            }
        }
        __syncthreads();
        // the shared rows go to the transform's global histogram (un-ranking the fixed bin) and are zeroed again
        for (int r = warp; r < rows_smem; r += NW) {
            uint32_t* grow = gh + (size_t)__ldg(a.rank_inv + r) * nb;
            for (int b = lane; b < nb; b += 32) {
                const uint32_t v = sh_hist[r * pitch + b];
                if (v) {
                    sh_hist[r * pitch + b] = 0u;
                    atomicAdd(&grow[b], v);
                }
            }
        }
        __syncthreads();
    }
}

template <int INTERP>
static cudaError_t launch_wide2(const WideArgs& a, int unroll, int num_sms, cudaStream_t s) {
    const long long nitems = (long long)a.n_transforms * a.nslabs;
    long long grid = nitems < num_sms ? nitems : num_sms;
    if (grid < 1) return cudaSuccess;
    const bool mask = a.mask_bits != nullptr;
    const size_t smem = (size_t)a.rows_smem * a.pitch * sizeof(uint32_t);
    int carve = (int)((smem + 1024) * 100 / (228 * 1024));
    if (carve > 100) carve = 100;
#define MI_WIDE_K(KERN)                                                                                          \
    do {                                                                                                         \
        cudaError_t e = cudaFuncSetAttribute(KERN, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);      \
        if (e != cudaSuccess) return e;                                                                          \
        e = cudaFuncSetAttribute(KERN, cudaFuncAttributePreferredSharedMemoryCarveout, carve);                   \
        if (e != cudaSuccess) return e;                                                                          \
        KERN<<<(unsigned)grid, kHistThreads, smem, s>>>(a);                                                      \
        return cudaGetLastError();                                                                               \
    } while (0)
#define MI_WIDE(UU)                                                                                              \
    do {                                                                                                         \
        if (mask) MI_WIDE_K((resample_wide_kernel<INTERP, UU, true>));                                           \
        else MI_WIDE_K((resample_wide_kernel<INTERP, UU, false>));                                               \
    } while (0)
    if (unroll == 1) MI_WIDE(1);
    if (unroll == 2) MI_WIDE(2);
    if (unroll == 3) MI_WIDE(3);
    MI_WIDE(4);
#undef MI_WIDE
#undef MI_WIDE_K
}

cudaError_t launch_resample_hist_wide(const WideArgs& a, int interp, int num_sms, cudaStream_t s) {
    if (a.version == 2 && a.moving_quad != nullptr && a.fbins_ranked != nullptr && a.rows_smem >= 1) {
        // samples in flight per lane: as in launch_resample_hist (fewest idle chunks in the last trip of a row)
        int unroll = a.unroll;
        if (unroll < 1 || unroll > 4) {
            const int chunks = (a.f.nx + 31) / 32;
            int best_waste = 1 << 30;
            for (int u = 1; u <= 4; ++u) {
                const int waste = (chunks + u - 1) / u * u - chunks;
                if (waste <= best_waste) { best_waste = waste; unroll = u; }
            }
        }
        return interp == MI_INTERP_NEAREST ? launch_wide2<MI_INTERP_NEAREST>(a, unroll, num_sms, s)
                                           : launch_wide2<MI_INTERP_TRILINEAR>(a, unroll, num_sms, s);
    }
    const long long nitems = (long long)a.n_transforms * a.nslabs;
    long long grid = nitems < 4LL * num_sms ? nitems : 4LL * num_sms;
    if (grid < 1) return cudaSuccess;
    if (interp == MI_INTERP_NEAREST) resample_hist_wide_kernel<MI_INTERP_NEAREST><<<(unsigned)grid, 512, 0, s>>>(a);
    else resample_hist_wide_kernel<MI_INTERP_TRILINEAR><<<(unsigned)grid, 512, 0, s>>>(a);
    return cudaGetLastError();
}


}  // namespace mi
