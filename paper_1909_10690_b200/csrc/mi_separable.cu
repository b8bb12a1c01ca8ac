// mi_separable.cu -- the separable fast path of the exhaustive map (steps a3 + a4) for transform
// families whose matrix is diagonal: translation, scale, log-scale.
//
// With a diagonal index-space matrix the continuous moving index of fixed voxel (ix,iy,iz) is
//   c_x = fma(mx, ix, ox)   c_y = fma(my, iy, oy)   c_z = fma(mz, iz, oz)
// (the off-diagonal fmas of CANON-2 add exact zeros), where (mx,ox) depends on p0 only, (my,oy) on
// p1 only and (mz,oz) on p2 only.  CANON-4 interpolates x first, then y, then z, so the x-lerped
// rows are shared by every transform with the same p0 and the xy-lerped planes by every transform
// with the same (p0,p1) -- bit for bit the same fp32 values the generic kernel computes:
//   X_a  [z'][y'][ix]  = L(pad[z'][y'][jx+1], pad[z'][y'][jx+2], wx)          (x-pass, per p0)
//   XY_ab[z'][iy][ix]  = L(X_a[z'][jy+1][ix], X_a[z'][jy+2][ix], wy)          (y-pass, per (p0,p1))
//   v                  = L(XY_ab[jz+1][iy][ix], XY_ab[jz+2][iy][ix], wz)      (z-lerp, per transform)
// so one evaluation costs one z-lerp, one binning and one histogram update, with fully coalesced
// 16-byte loads and no gathers.  Nearest-neighbour mode uses the same three passes on moving BIN
// indices (uint8) with a plane select instead of the lerps.
#include <cuda_runtime.h>
#include <stdint.h>

#include "mi_internal.h"

namespace mi {

namespace {

constexpr float kMagic = 12582912.0f;  // 1.5 * 2^23: RD(c + kMagic) - kMagic == floor(c) for |c| < 2^22
constexpr int kMagicBits = 0x4B400000;

__device__ __forceinline__ float lerp_rn(float p, float q, float f) {
    return __fmaf_rn(f, __fsub_rn(q, p), p);
}

// One axis of CANON-3/4 for continuous index c on an axis of n voxels.
//   trilinear: ok = c in [-0.5, n-0.5); lower = floor(c)+1 (index into the replicate-padded axis);
//              w = c - floor(c)
//   nearest:   r = floor(c + 0.5); ok = r in [0, n); lower = r (unpadded); w unused
struct AxisSample {
    bool ok;
    int lower;
    float w;
};
template <bool NN>
__device__ __forceinline__ AxisSample axis_sample(float c, int n) {
    AxisSample s;
    if (NN) {
        const float t = __fadd_rd(__fadd_rn(c, 0.5f), kMagic);
        const float r = __fsub_rn(t, kMagic);
        s.ok = r >= 0.0f && r < (float)n;
        s.lower = __float_as_int(t) - kMagicBits;
        s.w = 0.0f;
    } else {
        const float t = __fadd_rd(c, kMagic);
        s.ok = c >= -0.5f && c < __fsub_rn((float)n, 0.5f);
        s.lower = __float_as_int(t) - kMagicBits + 1;
        s.w = __fsub_rn(c, __fsub_rn(t, kMagic));
    }
    return s;
}

// ---- x-pass -------------------------------------------------------------------------------------
// grid: (rows = planes*prows, ceil(fnx/128), na).  Trilinear: src = padded float volume, rows over
// padded (z', y').  Nearest: src = moving bins, rows over (z, y).
template <bool NN, typename VT>
__global__ void __launch_bounds__(128) xpass_kernel(const VT* __restrict__ src, int snx, int mnx,
                                                    const float2* __restrict__ ax, int a0, int fnx,
                                                    VT* __restrict__ X) {
    const int ix = blockIdx.y * 128 + threadIdx.x;
    if (ix >= fnx) return;
    const int row = blockIdx.x;          // up to 2^31-1 rows (gridDim.y/z stop at 65535)
    const int a = blockIdx.z;
    const float2 mo = ax[a0 + a];
    const AxisSample sx = axis_sample<NN>(__fmaf_rn(mo.x, (float)ix, mo.y), mnx);
    const VT* __restrict__ r = src + (size_t)row * snx;
    VT out = VT(0);
    if (sx.ok) {
        if (NN) out = r[sx.lower];
        else out = (VT)lerp_rn((float)r[sx.lower], (float)r[sx.lower + 1], sx.w);
    }
    X[((size_t)a * gridDim.x + row) * fnx + ix] = out;
}

// ---- y-pass -------------------------------------------------------------------------------------
// grid: (ceil(colpitch/4 / 128), npairs).  pair = a_local*n1 + b.  Every thread owns 4 adjacent
// columns of one pair, resolves their x/y samples once and then walks all planes (unrolled by 4 for
// memory-level parallelism), writing XY[pair][plane][col..col+3] as one 16-byte store per plane, and
// colvalid[pair][col..col+3].
template <bool NN, typename VT>
struct Quad;
template <>
struct Quad<false, float> {
    float4 q;
    __device__ __forceinline__ void set(int k, float v) { (&q.x)[k] = v; }
    __device__ __forceinline__ void store(float* p) const { *reinterpret_cast<float4*>(p) = q; }
};
template <>
struct Quad<true, uint8_t> {
    uint32_t q = 0u;
    __device__ __forceinline__ void set(int k, uint8_t v) { q |= (uint32_t)v << (8 * k); }
    __device__ __forceinline__ void store(uint8_t* p) const { *reinterpret_cast<uint32_t*>(p) = q; }
};

template <bool NN, typename VT>
__global__ void __launch_bounds__(128) ypass_kernel(const VT* __restrict__ X, int planes, int prows, int mnx,
                                                    int mny, const float2* __restrict__ ax,
                                                    const float2* __restrict__ ay, int a0, int n1, int fnx,
                                                    int cols, int colpitch, VT* __restrict__ XY,
                                                    uint8_t* __restrict__ colvalid) {
    const int col0 = (blockIdx.x * 128 + threadIdx.x) * 4;
    if (col0 >= colpitch) return;
    const int pair = blockIdx.y;
    const int a = pair / n1, b = pair - a * n1;
    const float2 mx = ax[a0 + a], my = ay[b];
    // per column: offset of X[a][plane 0][sy.lower][ix] (or -1 if the column is invalid) and the y weight
    long long off[4];
    float wy[4];
    uint32_t cv = 0u;
    int iy = col0 / fnx, ix = col0 - iy * fnx;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        off[k] = -1;
        wy[k] = 0.0f;
        if (col0 + k < cols) {
            const AxisSample sx = axis_sample<NN>(__fmaf_rn(mx.x, (float)ix, mx.y), mnx);
            const AxisSample sy = axis_sample<NN>(__fmaf_rn(my.x, (float)iy, my.y), mny);
            if (sx.ok && sy.ok) {
                off[k] = ((long long)a * planes * prows + sy.lower) * fnx + ix;
                wy[k] = sy.w;
                cv |= 1u << (8 * k);
            }
        }
        if (++ix == fnx) { ix = 0; ++iy; }
    }
    *reinterpret_cast<uint32_t*>(colvalid + (size_t)pair * colpitch + col0) = cv;
    const size_t pstride = (size_t)prows * fnx;
    VT* __restrict__ out = XY + (size_t)pair * planes * colpitch + col0;
#pragma unroll 4
    for (int plane = 0; plane < planes; ++plane) {
        Quad<NN, VT> q;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            VT v = VT(0);
            if (off[k] >= 0) {
                const VT* __restrict__ r = X + off[k] + plane * pstride;
                if (NN) v = __ldg(r);
                else v = (VT)lerp_rn((float)__ldg(r), (float)__ldg(r + fnx), wy[k]);
            }
            q.set(k, v);
        }
        q.store(out + (size_t)plane * colpitch);
    }
}

// ---- z-lerp + joint histogram ---------------------------------------------------------------------
__device__ __forceinline__ float4 ld4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ uint32_t ld_u32(const uint8_t* p) { return __ldg(reinterpret_cast<const uint32_t*>(p)); }

// Result-less shared-memory increment on a 32-bit shared address (SASS: ATOMS.POPC.INC, which
// counts the lanes of a warp that hit the same address in one pass).
__device__ __forceinline__ void red_shared_inc(unsigned addr) {
    asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory");
}

// Words of shared memory in front of the histogram: ws[fnz] + run_hi[planes], rounded up to a
// multiple of 4 words.
__host__ __device__ __forceinline__ int zhist_table_words(int fnz, int planes) {
    return (fnz + planes + 3) & ~3;
}

template <int COLS>
struct ColVec {                      // COLS adjacent columns of one plane / one fixed slice
    float v[COLS];
};
template <int COLS>
__device__ __forceinline__ void ld_cols(ColVec<COLS>& r, const float* p) {
#pragma unroll
    for (int j = 0; j < COLS / 4; ++j) {
        const float4 q = ld4(p + 4 * j);
        r.v[4 * j] = q.x; r.v[4 * j + 1] = q.y; r.v[4 * j + 2] = q.z; r.v[4 * j + 3] = q.w;
    }
}
template <int COLS>
struct BinVec {                      // COLS adjacent uint8 values
    uint32_t w[COLS / 4];
};
template <int COLS>
__device__ __forceinline__ void ld_bins(BinVec<COLS>& r, const uint8_t* p) {
    if (COLS == 8) {
        const uint2 q = __ldg(reinterpret_cast<const uint2*>(p));
        r.w[0] = q.x; r.w[COLS / 4 - 1] = q.y;
    } else {
        r.w[0] = ld_u32(p);
    }
}
__device__ __forceinline__ unsigned byte_of(uint32_t w, int k) { return __byte_perm(w, 0u, 0x4440u | (unsigned)k); }

// One CTA per (pair, p2) item at a time; every thread owns COLS adjacent columns (iy,ix) of the
// fixed volume and walks them along z.  The walk is organised by moving plane: for lower plane p the
// fixed slices iz with floor(c_z) = p form one contiguous run (c_z is non-decreasing in iz), during
// which the two xy-lerped plane values stay in registers; the next plane is prefetched one step
// ahead and the three register sets rotate by name (the plane loop is unrolled by 3), so a plane step
// costs one 16-byte load per 4 columns and a pointer increment.
//
// Histogram update, trilinear (CANON-4 z-lerp, CANON-5 binning, one RED):
//   v = fma(w, hi - lo, lo)              hi - lo is formed once per plane step
//   t = (v - mlo) * mscale               FAST: mlo == 0 and every moving voxel >= 0, so v - 0 == v
//   t = min(max(t, 0), nb - 1)           FAST: t >= 0 already; clamping before the floor == after it
//   r = RD(t + (1.5*2^23 + a*pitch))     the low mantissa bits of r are a*pitch + floor(t) EXACTLY
//                                        (ulp is 1 there and the second addend is an integer)
//   RED [4*bits(r) + const]              const folds the shared base and -4*bits(1.5*2^23)
// The shared histogram rows have a pitch of nb + pad words: bank = (a*pad + b) mod 32, so the rows
// of the (many) background fixed bins do not all start on bank 0.
//
// Shared memory: ws[fnz] z-weights | run_hi[planes] | histogram rows (pitch words each).
template <bool NN, int COLS, bool FAST>
__global__ void __launch_bounds__(kHistThreads, 1) zhist_kernel(const __grid_constant__ ZHistArgs a) {
    extern __shared__ __align__(16) uint32_t sh_raw[];
    float* ws = reinterpret_cast<float*>(sh_raw);
    int* run_hi = reinterpret_cast<int*>(sh_raw) + a.fnz;
    uint32_t* sh_hist = sh_raw + zhist_table_words(a.fnz, a.planes);
    __shared__ int s_lo, s_hi;
    const unsigned nb = (unsigned)a.nb;
    const unsigned pitch = (unsigned)a.pitch;
    const int rows_smem = a.rows_smem;   // includes the dump row
    const int words = rows_smem * a.pitch;
    for (int w = threadIdx.x; w < words; w += blockDim.x) sh_hist[w] = 0u;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int colpitch = a.colpitch;
    const float topf = (float)(a.nb - 1);
    const int ntiles = (colpitch + COLS * kHistThreads - 1) / (COLS * kHistThreads);
    const long long nitems = (long long)a.n_pairs * a.n2;
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(sh_hist);
    const unsigned cbase = sbase - 4u * (unsigned)kMagicBits;   // modulo 2^32
    const float mlo = a.mlo, mscale = a.mscale;

    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int pair = (int)(item / a.n2);
        const int c = (int)(item - (long long)pair * a.n2);
        const float2 mo = a.az[c];
        if (threadIdx.x == 0) { s_lo = 0x7FFFFFFF; s_hi = -1; }
        for (int p = threadIdx.x; p < a.planes; p += blockDim.x) run_hi[p] = 0;
        __syncthreads();
        for (int iz = threadIdx.x; iz < a.fnz; iz += blockDim.x) {
            const AxisSample sz = axis_sample<NN>(__fmaf_rn(mo.x, (float)iz, mo.y), a.mnz);
            ws[iz] = sz.w;
            if (sz.ok) {
                atomicMin(&s_lo, iz);
                atomicMax(&s_hi, iz);
                atomicMax(&run_hi[sz.lower], iz + 1);
            }
        }
        __syncthreads();
        const int iz_lo = s_lo, iz_hi = s_hi + 1;   // valid z is one interval (c_z is monotone in iz)
        uint32_t* gh = a.hist + (size_t)item * a.nb * a.nb;

        if (iz_lo < iz_hi) {
            // lower planes visited: p_lo .. p_hi (planes whose run is empty are stepped over)
            int p_lo = 0, p_hi = -1;
            {
                const AxisSample s0 = axis_sample<NN>(__fmaf_rn(mo.x, (float)iz_lo, mo.y), a.mnz);
                const AxisSample s1 = axis_sample<NN>(__fmaf_rn(mo.x, (float)(iz_hi - 1), mo.y), a.mnz);
                p_lo = s0.lower;
                p_hi = s1.lower;
            }
            for (int tile = 0; tile < ntiles; ++tile) {
                const int col0 = (tile * kHistThreads + threadIdx.x) * COLS;
                if (col0 >= colpitch) continue;
                // columns outside the moving volume count into the dump row: (fa & keep) | dump
                BinVec<COLS> cv, keep, dump;
                ld_bins<COLS>(cv, a.colvalid + (size_t)pair * colpitch + col0);
                uint32_t any = 0u;
#pragma unroll
                for (int j = 0; j < COLS / 4; ++j) {
                    any |= cv.w[j];
                    keep.w[j] = cv.w[j] * 0xFFu;                            // cv bytes are 0 or 1
                    dump.w[j] = (~keep.w[j]) & ((uint32_t)a.rows_real * 0x01010101u);
                }
                if (any == 0u) continue;
                const uint8_t* __restrict__ fbq = a.fb + (size_t)iz_lo * colpitch + col0;
                BinVec<COLS> fa_next;
                ld_bins<COLS>(fa_next, fbq);
                int iz = iz_lo;
                if (NN) {
                    const uint8_t* __restrict__ pp = static_cast<const uint8_t*>(a.xy) +
                                                     ((size_t)pair * a.planes + p_lo) * colpitch + col0;
                    for (int p = p_lo; p <= p_hi; ++p, pp += colpitch) {
                        const int hi = run_hi[p];
                        if (iz >= hi) continue;
                        BinVec<COLS> v;
                        ld_bins<COLS>(v, pp);
                        for (; iz < hi; ++iz) {
                            BinVec<COLS> fa;
#pragma unroll
                            for (int j = 0; j < COLS / 4; ++j) fa.w[j] = (fa_next.w[j] & keep.w[j]) | dump.w[j];
                            fbq += colpitch;
                            if (iz + 1 < iz_hi) ld_bins<COLS>(fa_next, fbq);
#pragma unroll
                            for (int k = 0; k < COLS; ++k)
                                red_shared_inc(sbase + (byte_of(fa.w[k / 4], k & 3) * pitch + byte_of(v.w[k / 4], k & 3)) * 4u);
                        }
                    }
                } else {
                    const float* __restrict__ pp = static_cast<const float*>(a.xy) +
                                                   ((size_t)pair * a.planes + p_lo) * colpitch + col0;
                    ColVec<COLS> r0, r1, r2;
                    ld_cols<COLS>(r0, pp);
                    ld_cols<COLS>(r1, pp + colpitch);
                    r2 = r1;
                    pp += 2 * (size_t)colpitch;   // next plane to prefetch: p + 2
                    int p = p_lo;
                    // one plane step: prefetch plane p+2 into `pre`, run the slices of plane p on (lo, hi)
                    auto step = [&](const ColVec<COLS>& lo, const ColVec<COLS>& hi, ColVec<COLS>& pre) {
                        if (p + 2 < a.planes) ld_cols<COLS>(pre, pp);
                        pp += colpitch;
                        const int end = run_hi[p];
                        if (iz < end) {
                            float d[COLS];
#pragma unroll
                            for (int k = 0; k < COLS; ++k) d[k] = __fsub_rn(hi.v[k], lo.v[k]);
                            for (; iz < end; ++iz) {
                                const float w = ws[iz];
                                BinVec<COLS> fa;
#pragma unroll
                                for (int j = 0; j < COLS / 4; ++j) fa.w[j] = (fa_next.w[j] & keep.w[j]) | dump.w[j];
                                fbq += colpitch;
                                if (iz + 1 < iz_hi) ld_bins<COLS>(fa_next, fbq);
#pragma unroll
                                for (int k = 0; k < COLS; ++k) {
                                    const float v = __fmaf_rn(w, d[k], lo.v[k]);
                                    float t = FAST ? __fmul_rn(v, mscale) : __fmul_rn(__fsub_rn(v, mlo), mscale);
                                    t = fminf(t, topf);
                                    if (!FAST) t = fmaxf(t, 0.0f);
                                    const unsigned mbits = byte_of(fa.w[k / 4], k & 3) * pitch + (unsigned)kMagicBits;
                                    const float r = __fadd_rd(t, __uint_as_float(mbits));
                                    red_shared_inc(__float_as_uint(r) * 4u + cbase);
                                }
                            }
                        }
                        ++p;
                    };
                    while (p <= p_hi) {
                        step(r0, r1, r2);
                        if (p > p_hi) break;
                        step(r1, r2, r0);
                        if (p > p_hi) break;
                        step(r2, r0, r1);
                    }
                }
            }
        }
        __syncthreads();
        // write the item's whole global histogram (un-ranking the fixed bin): counted rows from shared
        // memory (re-zeroed for the next item), rows of the rare ranks as zeros -- zrare_kernel adds
        // their voxels afterwards.  No other CTA touches this histogram, so plain stores suffice.
        for (int r = warp; r < (int)nb; r += nwarps) {
            uint32_t* grow = gh + (size_t)__ldg(a.rank_inv + r) * nb;
            const bool real = r < a.rows_real;
            for (unsigned b = lane; b < nb; b += 32) {
                uint32_t v = 0u;
                if (real) {
                    v = sh_hist[r * pitch + b];
                    if (v) sh_hist[r * pitch + b] = 0u;
                }
                grow[b] = v;
            }
        }
        if (a.rows_real < rows_smem)   // the dump row is only re-zeroed
            for (unsigned b = threadIdx.x; b < nb; b += blockDim.x) sh_hist[a.rows_real * pitch + b] = 0u;
        __syncthreads();
    }
}

// fixed ranked bins -> [fnz][colpitch] (plane pitch padded to a multiple of 4 so that four adjacent
// columns are one aligned 32-bit load); pad columns are 0.  Ranks >= rows_real are clamped to the
// dump row `rows_real` and the voxel is appended to the rare list as (col, iz | rank << 16).
__global__ void __launch_bounds__(256) pitch_bins_kernel(const uint8_t* __restrict__ in, int cols,
                                                         int colpitch, int rows_real,
                                                         uint8_t* __restrict__ out, uint2* __restrict__ rare,
                                                         unsigned* __restrict__ rare_count, unsigned rare_cap) {
    const int col = blockIdx.x * 256 + threadIdx.x;
    if (col >= colpitch) return;
    const int iz = blockIdx.y;
    int r = col < cols ? in[(size_t)iz * cols + col] : 0;
    if (r >= rows_real) {
        const unsigned slot = atomicAdd(rare_count, 1u);
        if (slot < rare_cap) rare[slot] = make_uint2((unsigned)col, (unsigned)iz | ((unsigned)r << 16));
        r = rows_real;
    }
    out[(size_t)iz * colpitch + col] = (uint8_t)r;
}

// CANON-5 on the integer side: PTX float->int conversions saturate to the destination range
// (NaN -> 0), so cvt.rmi.u8 is clamp(floor(t), 0, 255) in one instruction; bins < 256 need one min.
__device__ __forceinline__ unsigned bin_u8(float t, unsigned top) {
    unsigned b;
    asm("cvt.rmi.u8.f32 %0, %1;" : "=r"(b) : "f"(t));
    return min(b, top);
}

// Exact handling of the rare fixed-bin rows: for every item (pair, p2) and every rare voxel, the same
// z-lerp / plane select as the main kernel, added straight to the item's global histogram.
template <bool NN>
__global__ void __launch_bounds__(256) zrare_kernel(const __grid_constant__ ZHistArgs a) {
    const long long nitems = (long long)a.n_pairs * a.n2;
    const unsigned top = (unsigned)(a.nb - 1);
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int pair = (int)(item / a.n2);
        const int c = (int)(item - (long long)pair * a.n2);
        const float2 mo = a.az[c];
        uint32_t* gh = a.hist + (size_t)item * a.nb * a.nb;
        for (unsigned k = threadIdx.x; k < a.n_rare; k += blockDim.x) {
            const uint2 rv = a.rare[k];
            const unsigned col = rv.x, iz = rv.y & 0xFFFFu, rank = rv.y >> 16;
            if (!a.colvalid[(size_t)pair * a.colpitch + col]) continue;
            const AxisSample sz = axis_sample<NN>(__fmaf_rn(mo.x, (float)iz, mo.y), a.mnz);
            if (!sz.ok) continue;
            const size_t base = ((size_t)pair * a.planes + sz.lower) * a.colpitch + col;
            unsigned b;
            if (NN) {
                b = static_cast<const uint8_t*>(a.xy)[base];
            } else {
                const float* xy = static_cast<const float*>(a.xy);
                const float v = lerp_rn(xy[base], xy[base + a.colpitch], sz.w);
                b = bin_u8(__fmul_rn(__fsub_rn(v, a.mlo), a.mscale), top);
            }
            atomicAdd(&gh[(size_t)__ldg(a.rank_inv + rank) * a.nb + b], 1u);
        }
    }
}

}  // namespace

cudaError_t launch_pitch_bins(const uint8_t* in, int cols, int colpitch, int fnz, int rows_real, uint8_t* out,
                              uint2* rare, unsigned* rare_count, unsigned rare_cap, cudaStream_t s) {
    dim3 grid((colpitch + 255) / 256, fnz);
    pitch_bins_kernel<<<grid, 256, 0, s>>>(in, cols, colpitch, rows_real, out, rare, rare_count, rare_cap);
    return cudaGetLastError();
}

cudaError_t launch_xpass(bool nn, const void* src, int snx, int srows, int mnx, const float2* ax, int a0,
                         int na, int fnx, void* X, cudaStream_t s) {
    dim3 grid(srows, (fnx + 127) / 128, na);
    if (nn)
        xpass_kernel<true, uint8_t><<<grid, 128, 0, s>>>(static_cast<const uint8_t*>(src), snx, mnx, ax, a0, fnx,
                                                        static_cast<uint8_t*>(X));
    else
        xpass_kernel<false, float><<<grid, 128, 0, s>>>(static_cast<const float*>(src), snx, mnx, ax, a0, fnx,
                                                       static_cast<float*>(X));
    return cudaGetLastError();
}

cudaError_t launch_ypass(bool nn, const void* X, int planes, int prows, int mnx, int mny, const float2* ax,
                         const float2* ay, int a0, int n1, int npairs, int fnx, int cols, int colpitch,
                         void* XY, uint8_t* colvalid, cudaStream_t s) {
    dim3 grid((colpitch / 4 + 127) / 128, npairs);
    if (nn)
        ypass_kernel<true, uint8_t><<<grid, 128, 0, s>>>(static_cast<const uint8_t*>(X), planes, prows, mnx, mny, ax,
                                                        ay, a0, n1, fnx, cols, colpitch, static_cast<uint8_t*>(XY),
                                                        colvalid);
    else
        ypass_kernel<false, float><<<grid, 128, 0, s>>>(static_cast<const float*>(X), planes, prows, mnx, mny, ax, ay,
                                                       a0, n1, fnx, cols, colpitch, static_cast<float*>(XY), colvalid);
    return cudaGetLastError();
}

// Histogram rows (of `pitch` words) of the z kernel that fit in shared memory, the dump row included
// (at most nb + 1).
int zhist_rows_in_smem(int nb, int pitch, int fnz, int planes, size_t smem_optin) {
    const size_t reserve = 1024 + 4 * (size_t)zhist_table_words(fnz, planes);
    size_t rows = (smem_optin > reserve ? smem_optin - reserve : 0) / ((size_t)pitch * sizeof(uint32_t));
    if (rows > (size_t)nb + 1) rows = (size_t)nb + 1;
    return (int)rows;
}

template <bool NN, int COLS, bool FAST>
static cudaError_t launch_zhist_t(const ZHistArgs& a, unsigned grid, size_t smem, cudaStream_t s) {
    auto kern = zhist_kernel<NN, COLS, FAST>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kHistThreads, smem, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_zhist(bool nn, const ZHistArgs& a, int num_sms, cudaStream_t s) {
    if (a.rows_smem < 1 || a.pitch < a.nb || (a.colpitch % a.cols) != 0) return cudaErrorInvalidConfiguration;
    const size_t smem = 4 * (size_t)zhist_table_words(a.fnz, a.planes) + (size_t)a.rows_smem * a.pitch * sizeof(uint32_t);
    const long long nitems = (long long)a.n_pairs * a.n2;
    long long grid = nitems < num_sms ? nitems : num_sms;
    if (grid < 1) return cudaSuccess;
    cudaError_t e;
    const unsigned g = (unsigned)grid;
    if (nn) {
        e = a.cols == 8 ? launch_zhist_t<true, 8, false>(a, g, smem, s) : launch_zhist_t<true, 4, false>(a, g, smem, s);
    } else if (a.fast_bin) {
        e = a.cols == 8 ? launch_zhist_t<false, 8, true>(a, g, smem, s) : launch_zhist_t<false, 4, true>(a, g, smem, s);
    } else {
        e = a.cols == 8 ? launch_zhist_t<false, 8, false>(a, g, smem, s) : launch_zhist_t<false, 4, false>(a, g, smem, s);
    }
    if (e != cudaSuccess) return e;
    if (a.n_rare > 0) {
        long long g2 = nitems < 8LL * num_sms ? nitems : 8LL * num_sms;
        if (nn) zrare_kernel<true><<<(unsigned)g2, 256, 0, s>>>(a);
        else zrare_kernel<false><<<(unsigned)g2, 256, 0, s>>>(a);
    }
    return cudaGetLastError();
}

}  // namespace mi
