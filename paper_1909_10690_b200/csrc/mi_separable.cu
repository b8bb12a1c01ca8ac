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
// grid: (ceil(fnx/128), rows = planes*prows, na).  Trilinear: src = padded float volume, rows over
// padded (z', y').  Nearest: src = moving bins, rows over (z, y).
template <bool NN, typename VT>
__global__ void __launch_bounds__(128) xpass_kernel(const VT* __restrict__ src, int snx, int mnx,
                                                    const float2* __restrict__ ax, int a0, int fnx,
                                                    VT* __restrict__ X) {
    const int ix = blockIdx.x * 128 + threadIdx.x;
    if (ix >= fnx) return;
    const int row = blockIdx.y;
    const int a = blockIdx.z;
    const float2 mo = ax[a0 + a];
    const AxisSample sx = axis_sample<NN>(__fmaf_rn(mo.x, (float)ix, mo.y), mnx);
    const VT* __restrict__ r = src + (size_t)row * snx;
    VT out = VT(0);
    if (sx.ok) {
        if (NN) out = r[sx.lower];
        else out = (VT)lerp_rn((float)r[sx.lower], (float)r[sx.lower + 1], sx.w);
    }
    X[((size_t)a * gridDim.y + row) * fnx + ix] = out;
}

// ---- y-pass -------------------------------------------------------------------------------------
// grid: (ceil(colpitch/256), planes, npairs).  pair = a_local*n1 + b.  Writes XY[pair][plane][col]
// and (for plane 0) colvalid[pair][col].
template <bool NN, typename VT>
__global__ void __launch_bounds__(256) ypass_kernel(const VT* __restrict__ X, int prows, int mnx, int mny,
                                                    const float2* __restrict__ ax, const float2* __restrict__ ay,
                                                    int a0, int n1, int fnx, int cols, int colpitch,
                                                    VT* __restrict__ XY, uint8_t* __restrict__ colvalid) {
    const int col = blockIdx.x * 256 + threadIdx.x;
    if (col >= colpitch) return;
    const int plane = blockIdx.y, planes = gridDim.y;
    const int pair = blockIdx.z;
    const int a = pair / n1, b = pair - a * n1;
    const int iy = col / fnx, ix = col - iy * fnx;
    VT out = VT(0);
    bool ok = false;
    if (col < cols) {
        const float2 mx = ax[a0 + a], my = ay[b];
        const AxisSample sx = axis_sample<NN>(__fmaf_rn(mx.x, (float)ix, mx.y), mnx);
        const AxisSample sy = axis_sample<NN>(__fmaf_rn(my.x, (float)iy, my.y), mny);
        ok = sx.ok && sy.ok;
        if (ok) {
            const VT* __restrict__ r = X + (((size_t)a * planes + plane) * prows + sy.lower) * fnx + ix;
            if (NN) out = r[0];
            else out = (VT)lerp_rn((float)r[0], (float)r[fnx], sy.w);
        }
    }
    XY[((size_t)pair * planes + plane) * colpitch + col] = out;
    if (plane == 0) colvalid[(size_t)pair * colpitch + col] = ok ? 1 : 0;
}

// ---- z-lerp + joint histogram ---------------------------------------------------------------------
__device__ __forceinline__ float4 ld4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ uint32_t ld_u32(const uint8_t* p) { return __ldg(reinterpret_cast<const uint32_t*>(p)); }

// Result-less shared-memory increment on a 32-bit shared address (SASS: ATOMS.POPC.INC / ATOMS.ADD).
__device__ __forceinline__ void red_shared_inc(unsigned addr) {
    asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory");
}

// CANON-5 on the integer side: PTX float->int conversions saturate to the destination range
// (NaN -> 0), so cvt.rmi.u8 is clamp(floor(t), 0, 255) in one instruction; bins < 256 need one min.
__device__ __forceinline__ unsigned bin_u8(float t, unsigned top) {
    unsigned b;
    asm("cvt.rmi.u8.f32 %0, %1;" : "=r"(b) : "f"(t));
    return min(b, top);
}

// Words of shared memory in front of the histogram: ws[fnz] + run_lo[planes] + run_hi[planes],
// rounded up to a multiple of 4 words.
__host__ __device__ __forceinline__ int zhist_table_words(int fnz, int planes) {
    return (fnz + 2 * planes + 3) & ~3;
}

// One CTA per (pair, p2) item at a time; every thread owns 4 adjacent columns (iy,ix) of the fixed
// volume and walks them along z.  The walk is organised by moving plane: for lower plane p the fixed
// slices iz with floor(c_z) = p form one contiguous run (c_z is non-decreasing in iz), during which
// the two xy-lerped plane values stay in registers; the next plane is prefetched one step ahead and
// the three float4 registers rotate by name (the plane loop is unrolled by 3), so a plane step costs
// one 16-byte load and a pointer increment.
//
// Shared memory: ws[fnz] z-weights | run_lo[planes], run_hi[planes] | histogram rows.
template <bool NN>
__global__ void __launch_bounds__(kHistThreads, 1) zhist_kernel(const __grid_constant__ ZHistArgs a) {
    extern __shared__ __align__(16) uint32_t sh_raw[];
    float* ws = reinterpret_cast<float*>(sh_raw);
    int* run_lo = reinterpret_cast<int*>(sh_raw) + a.fnz;
    int* run_hi = run_lo + a.planes;
    uint32_t* sh_hist = sh_raw + zhist_table_words(a.fnz, a.planes);
    __shared__ int s_lo, s_hi;
    const unsigned nb = (unsigned)a.nb;
    const int rows_smem = a.rows_smem;   // includes the dump row
    const int words = rows_smem * a.nb;
    for (int w = threadIdx.x; w < words; w += blockDim.x) sh_hist[w] = 0u;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int colpitch = a.colpitch;
    const unsigned top = (unsigned)(a.nb - 1);
    const int ntiles = (colpitch + 4 * kHistThreads - 1) / (4 * kHistThreads);
    const long long nitems = (long long)a.n_pairs * a.n2;
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(sh_hist);

    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int pair = (int)(item / a.n2);
        const int c = (int)(item - (long long)pair * a.n2);
        const float2 mo = a.az[c];
        if (threadIdx.x == 0) { s_lo = 0x7FFFFFFF; s_hi = -1; }
        for (int p = threadIdx.x; p < a.planes; p += blockDim.x) { run_lo[p] = 0x7FFFFFFF; run_hi[p] = 0; }
        __syncthreads();
        for (int iz = threadIdx.x; iz < a.fnz; iz += blockDim.x) {
            const AxisSample sz = axis_sample<NN>(__fmaf_rn(mo.x, (float)iz, mo.y), a.mnz);
            ws[iz] = sz.w;
            if (sz.ok) {
                atomicMin(&s_lo, iz);
                atomicMax(&s_hi, iz);
                atomicMin(&run_lo[sz.lower], iz);
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
                const int col0 = (tile * kHistThreads + threadIdx.x) * 4;
                if (col0 >= colpitch) continue;
                const uint32_t cv = ld_u32(a.colvalid + (size_t)pair * colpitch + col0);
                if (cv == 0u) continue;
                // columns outside the moving volume count into the dump row: (fa & keep) | dump
                const uint32_t keep = cv * 0xFFu;                       // cv bytes are 0 or 1
                const uint32_t dump = (~keep) & ((uint32_t)a.rows_real * 0x01010101u);
                const uint8_t* __restrict__ fbq = a.fb + (size_t)iz_lo * colpitch + col0;
                uint32_t fa_next = ld_u32(fbq);
                int iz = iz_lo;
                if (NN) {
                    const uint8_t* __restrict__ pp = static_cast<const uint8_t*>(a.xy) +
                                                     ((size_t)pair * a.planes + p_lo) * colpitch + col0;
                    for (int p = p_lo; p <= p_hi; ++p, pp += colpitch) {
                        const int hi = run_hi[p];
                        if (iz >= hi) continue;
                        const uint32_t v = ld_u32(pp);
                        for (; iz < hi; ++iz) {
                            const uint32_t fa4 = (fa_next & keep) | dump;
                            fbq += colpitch;
                            if (iz + 1 < iz_hi) fa_next = ld_u32(fbq);
                            red_shared_inc(sbase + ((fa4 & 0xFF) * nb + (v & 0xFF)) * 4u);
                            red_shared_inc(sbase + (((fa4 >> 8) & 0xFF) * nb + ((v >> 8) & 0xFF)) * 4u);
                            red_shared_inc(sbase + (((fa4 >> 16) & 0xFF) * nb + ((v >> 16) & 0xFF)) * 4u);
                            red_shared_inc(sbase + ((fa4 >> 24) * nb + (v >> 24)) * 4u);
                        }
                    }
                } else {
                    const float* __restrict__ pp = static_cast<const float*>(a.xy) +
                                                   ((size_t)pair * a.planes + p_lo) * colpitch + col0;
                    float4 r0 = ld4(pp), r1 = ld4(pp + colpitch), r2 = r1;
                    pp += 2 * (size_t)colpitch;   // next plane to prefetch: p + 2
                    int p = p_lo;
                    // one plane step: prefetch plane p+2 into `pre`, run the slices of plane p on (lo, hi)
                    auto step = [&](const float4& lo, const float4& hi, float4& pre) {
                        if (p + 2 < a.planes) pre = ld4(pp);
                        pp += colpitch;
                        const int end = run_hi[p];
                        for (; iz < end; ++iz) {
                            const float w = ws[iz];
                            const uint32_t fa4 = (fa_next & keep) | dump;
                            fbq += colpitch;
                            if (iz + 1 < iz_hi) fa_next = ld_u32(fbq);
                            // CANON-4 z-lerp, CANON-5 binning (floor and clamp by the saturating convert)
                            const unsigned b0 = bin_u8(__fmul_rn(__fsub_rn(lerp_rn(lo.x, hi.x, w), a.mlo), a.mscale), top);
                            const unsigned b1 = bin_u8(__fmul_rn(__fsub_rn(lerp_rn(lo.y, hi.y, w), a.mlo), a.mscale), top);
                            const unsigned b2 = bin_u8(__fmul_rn(__fsub_rn(lerp_rn(lo.z, hi.z, w), a.mlo), a.mscale), top);
                            const unsigned b3 = bin_u8(__fmul_rn(__fsub_rn(lerp_rn(lo.w, hi.w, w), a.mlo), a.mscale), top);
                            red_shared_inc(sbase + ((fa4 & 0xFF) * nb + b0) * 4u);
                            red_shared_inc(sbase + (((fa4 >> 8) & 0xFF) * nb + b1) * 4u);
                            red_shared_inc(sbase + (((fa4 >> 16) & 0xFF) * nb + b2) * 4u);
                            red_shared_inc(sbase + ((fa4 >> 24) * nb + b3) * 4u);
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
        // merge the CTA-private rows into the item's global histogram (un-ranking the fixed bin);
        // the dump row (rare fixed ranks, handled exactly by zrare_kernel) is only re-zeroed
        for (int r = warp; r < rows_smem; r += nwarps) {
            uint32_t* grow = gh + (size_t)__ldg(a.rank_inv + r) * nb;
            const bool real = r < a.rows_real;
            for (unsigned b = lane; b < nb; b += 32) {
                const uint32_t v = sh_hist[r * nb + b];
                if (v) {
                    sh_hist[r * nb + b] = 0u;
                    if (real) atomicAdd(&grow[b], v);
                }
            }
        }
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
    dim3 grid((fnx + 127) / 128, srows, na);
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
    dim3 grid((colpitch + 255) / 256, planes, npairs);
    if (nn)
        ypass_kernel<true, uint8_t><<<grid, 256, 0, s>>>(static_cast<const uint8_t*>(X), prows, mnx, mny, ax, ay, a0,
                                                        n1, fnx, cols, colpitch, static_cast<uint8_t*>(XY), colvalid);
    else
        ypass_kernel<false, float><<<grid, 256, 0, s>>>(static_cast<const float*>(X), prows, mnx, mny, ax, ay, a0, n1,
                                                       fnx, cols, colpitch, static_cast<float*>(XY), colvalid);
    return cudaGetLastError();
}

// Histogram rows of the z kernel that fit in shared memory, the dump row included (at most nb + 1).
int zhist_rows_in_smem(int nb, int fnz, int planes, size_t smem_optin) {
    const size_t reserve = 1024 + 4 * (size_t)zhist_table_words(fnz, planes);
    size_t rows = (smem_optin > reserve ? smem_optin - reserve : 0) / ((size_t)nb * sizeof(uint32_t));
    if (rows > (size_t)nb + 1) rows = (size_t)nb + 1;
    return (int)rows;
}

cudaError_t launch_zhist(bool nn, const ZHistArgs& a, int num_sms, cudaStream_t s) {
    if (a.rows_smem < 1) return cudaErrorInvalidConfiguration;
    const size_t smem = 4 * (size_t)zhist_table_words(a.fnz, a.planes) + (size_t)a.rows_smem * a.nb * sizeof(uint32_t);
    const long long nitems = (long long)a.n_pairs * a.n2;
    long long grid = nitems < num_sms ? nitems : num_sms;
    if (grid < 1) return cudaSuccess;
    cudaError_t e;
    if (nn) {
        e = cudaFuncSetAttribute(zhist_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        zhist_kernel<true><<<(unsigned)grid, kHistThreads, smem, s>>>(a);
    } else {
        e = cudaFuncSetAttribute(zhist_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        zhist_kernel<false><<<(unsigned)grid, kHistThreads, smem, s>>>(a);
    }
    if (a.n_rare > 0) {
        long long g2 = nitems < 8LL * num_sms ? nitems : 8LL * num_sms;
        if (nn) zrare_kernel<true><<<(unsigned)g2, 256, 0, s>>>(a);
        else zrare_kernel<false><<<(unsigned)g2, 256, 0, s>>>(a);
    }
    return cudaGetLastError();
}

}  // namespace mi
