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
// grid: (ceil(colpitch/4 / 128), npairs).  pair = a_local*n1 + b_local (n1 = p1 values of the batch,
// the first one is b0).  Every thread owns 4 adjacent
// columns of one pair, resolves their x/y samples once and then walks all planes (unrolled by 4 for
// memory-level parallelism), writing XY[pair][plane][col..col+3] as one 16-byte store per plane, and
// colvalid[pair][col..col+3].  Trilinear values are stored times `prescale` (1, or the power-of-two
// bin scale in kBinFastPrescaled mode -- an exact multiplication).
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
                                                    const float2* __restrict__ ay, int a0, int b0, int n1, int fnx,
                                                    int cols, int colpitch, float prescale,
                                                    VT* __restrict__ XY, uint8_t* __restrict__ colvalid) {
    const int col0 = (blockIdx.x * 128 + threadIdx.x) * 4;
    if (col0 >= colpitch) return;
    const int pair = blockIdx.y;
    const int a = pair / n1, b = pair - a * n1;
    const float2 mx = ax[a0 + a], my = ay[b0 + b];
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
    // Common case (trilinear): the four columns are four adjacent, 16-byte aligned voxels of one moving
    // row pair -- two 16-byte loads per plane instead of eight 4-byte ones (same values, same lerps).
    bool vec = !NN && (fnx & 3) == 0 && off[0] >= 0;
#pragma unroll
    for (int k = 1; k < 4; ++k) vec = vec && off[k] == off[0] + k;
    if (vec) {
        const float w = wy[0];   // same iy for all four: same weight
        const float* __restrict__ r = reinterpret_cast<const float*>(X) + off[0];
#pragma unroll 4
        for (int plane = 0; plane < planes; ++plane) {
            const float4 lo = __ldg(reinterpret_cast<const float4*>(r + plane * pstride));
            const float4 hi = __ldg(reinterpret_cast<const float4*>(r + plane * pstride + fnx));
            float4 q;
            q.x = __fmul_rn(lerp_rn(lo.x, hi.x, w), prescale);
            q.y = __fmul_rn(lerp_rn(lo.y, hi.y, w), prescale);
            q.z = __fmul_rn(lerp_rn(lo.z, hi.z, w), prescale);
            q.w = __fmul_rn(lerp_rn(lo.w, hi.w, w), prescale);
            *reinterpret_cast<float4*>(reinterpret_cast<float*>(out) + (size_t)plane * colpitch) = q;
        }
        return;
    }
#pragma unroll 4
    for (int plane = 0; plane < planes; ++plane) {
        Quad<NN, VT> q;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            VT v = VT(0);
            if (off[k] >= 0) {
                const VT* __restrict__ r = X + off[k] + plane * pstride;
                if (NN) v = __ldg(r);
                else v = (VT)__fmul_rn(lerp_rn((float)__ldg(r), (float)__ldg(r + fnx), wy[k]), prescale);
            }
            q.set(k, v);
        }
        q.store(out + (size_t)plane * colpitch);
    }
}

// ---- z-lerp + joint histogram (+ fused entropy epilogue) --------------------------------------------
__device__ __forceinline__ float4 ld4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ uint32_t ld_u32(const uint8_t* p) { return __ldg(reinterpret_cast<const uint32_t*>(p)); }

// Result-less shared-memory increment on a 32-bit shared address (SASS: ATOMS.POPC.INC, which
// counts the lanes of a warp that hit the same address in one pass).
__device__ __forceinline__ void red_shared_inc(unsigned addr) {
    asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory");
}
// The alternative BASELINE.json's north_star names: software warp aggregation -- the lanes that hit the same
// counter are found with __match_any_sync and their leader adds the group's size.  Kept as an option
// (MI_OPT_ZHIST_MATCH_ANY) so that the choice of the plain RED stays a measured one (profiles/).
__device__ __forceinline__ void match_any_inc(unsigned addr) {
    const unsigned active = __activemask();
    const unsigned peers = __match_any_sync(active, addr);
    if ((unsigned)(threadIdx.x & 31) == (unsigned)(__ffs(peers) - 1))
        asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"((unsigned)__popc(peers)) : "memory");
}
template <bool AGG>
__device__ __forceinline__ void hist_inc(unsigned addr) {
    if (AGG) match_any_inc(addr); else red_shared_inc(addr);
}

__device__ __forceinline__ unsigned warp_sum_u(unsigned v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Shared-memory layout of the z kernel, in 32-bit words:
//   run_hi[planes] | (pad to 4) | pb[kEntropyPb] | red[kEntropyRed] | histogram rows
// pb / red are the fused entropy epilogue's scratch (moving marginal counts; per-warp partial sums).
constexpr int kEntropyAcc = 1 + kMaxQPerPass;                     // sum c ln c, sum c^q_k
constexpr int kEntropyPb = 272;                                   // 256 moving bins + 8 partial totals, multiple of 4
constexpr int kEntropyRed = 2 * kEntropyAcc * (kHistThreads / 32 + 16);  // doubles as word pairs
__host__ __device__ __forceinline__ int zhist_table_words(int planes) {
    return ((planes + 3) & ~3) + kEntropyPb + kEntropyRed;
}

struct Cols {                        // this thread's kZCols columns of one plane: 2 groups of 4
    float4 g[kZCols / 4];
};
__device__ __forceinline__ void ld_cols(Cols& r, const float* p) {
#pragma unroll
    for (int j = 0; j < kZCols / 4; ++j) r.g[j] = ld4(p + 128 * j);
}
__device__ __forceinline__ float col_of(const Cols& r, int k) { return (&r.g[k >> 2].x)[k & 3]; }
struct Bins {                        // the same columns of a uint8 plane / fixed slice
    uint32_t w[kZCols / 4];
};
__device__ __forceinline__ void ld_bins(Bins& r, const uint8_t* p) {
#pragma unroll
    for (int j = 0; j < kZCols / 4; ++j) r.w[j] = ld_u32(p + 128 * j);
}
__device__ __forceinline__ unsigned byte_of(uint32_t w, int k) { return __byte_perm(w, 0u, 0x4440u | (unsigned)k); }

// Accumulate the entropy terms of one count c > 0 (CANON-7 on integer counts):
//   acc[0] += c ln c,  acc[1+k] += c^q_k = exp(q_k ln c)
template <int NQ>
__device__ __forceinline__ void entropy_terms(double (&acc)[kEntropyAcc], unsigned c, const double (&qv)[kMaxQPerPass],
                                              int nq) {
    const double dv = (double)c;
    const double lc = log(dv);
    acc[0] += dv * lc;
#pragma unroll
    for (int k = 0; k < NQ; ++k)
        if (k < nq) acc[1 + k] += exp(qv[k] * lc);
}

// Step a5 from the finished shared histogram of one item (all kHistThreads threads call this; the
// CTA is synchronised on entry).  With c the integer counts and N their total (CANON-7):
//   H = ln N - (sum c ln c)/N,   sum p^q = exp(-q ln N) * sum c^q.
// Pass 1: every warp takes rows; each non-zero count adds its joint terms, is added to the moving
// marginal pb[b] and re-zeroed; the row sum (fixed marginal) is parked in the row's first word.
// Pass 2: threads 0..255 take the fixed marginal, threads 256..511 the moving marginal.
// Per-warp partial sums meet in sh_red (fixed summation order -> reproducible values).
__device__ __forceinline__ void zhist_entropy_epilogue(const ZHistArgs& a, long long item, uint32_t* sh_hist,
                                                       uint32_t* sh_pb, double* sh_red) {
    constexpr int nwarps = kHistThreads / 32;
    constexpr int kSlots = nwarps + 16;          // joint warps | 8 fixed-marginal warps | 8 moving-marginal warps
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned nb = (unsigned)a.nb, pitch = (unsigned)a.pitch;
    const int nq = a.nq;
    double qv[kMaxQPerPass];
#pragma unroll
    for (int k = 0; k < kMaxQPerPass; ++k) qv[k] = k < nq ? __ldg(a.q + k) : 1.0;

    double acc[kEntropyAcc];
#pragma unroll
    for (int i = 0; i < kEntropyAcc; ++i) acc[i] = 0.0;
    for (int r = warp; r < a.rows_real; r += nwarps) {
        uint32_t* row = sh_hist + r * pitch;
        unsigned rowsum = 0u;
        for (unsigned b = lane; b < nb; b += 32) {
            const unsigned v = row[b];
            if (v) {
                row[b] = 0u;
                rowsum += v;
                atomicAdd(&sh_pb[b], v);
                entropy_terms<kMaxQPerPass>(acc, v, qv, nq);
            }
        }
        rowsum = warp_sum_u(rowsum);
        if (lane == 0) row[0] = rowsum;
    }
#pragma unroll
    for (int i = 0; i < kEntropyAcc; ++i) {
        const double s = warp_sum_d(acc[i]);
        if (lane == 0) sh_red[i * kSlots + warp] = s;
        acc[i] = 0.0;
    }
    __syncthreads();

    if (warp < 16) {
        unsigned cnt = 0u;
        if (warp < 8) {
            const int r = threadIdx.x;
            if (r < a.rows_real) {
                cnt = sh_hist[r * pitch];
                sh_hist[r * pitch] = 0u;
            }
        } else {
            const unsigned b = threadIdx.x - 256u;
            if (b < nb) {
                cnt = sh_pb[b];
                sh_pb[b] = 0u;
            }
        }
        if (cnt) entropy_terms<kMaxQPerPass>(acc, cnt, qv, nq);
#pragma unroll
        for (int i = 0; i < kEntropyAcc; ++i) {
            const double s = warp_sum_d(acc[i]);
            if (lane == 0) sh_red[i * kSlots + nwarps + warp] = s;
        }
        const unsigned n = warp_sum_u(cnt);   // N_f < 2^31: the total fits
        if (lane == 0 && warp < 8) sh_pb[256 + warp] = n;
    }
    __syncthreads();

    if (threadIdx.x == 0) {
        unsigned long long n = 0;
        for (int w = 0; w < 8; ++w) n += sh_pb[256 + w];
        const size_t dst = a.om.dst(item);  // item order (p0, p1, p2 fastest) -> map order (p2, p1, p0 fastest)
        double* out = a.mi_out + dst * (size_t)(1 + a.nq_total);
        if (a.nvalid != nullptr) a.nvalid[dst] = (int64_t)n;
        if (n == 0) {
            out[0] = 0.0;
            for (int k = 0; k < nq; ++k) out[1 + k] = 0.0;
        } else {
            const double N = (double)n, lnN = log(N);
            double tA[kEntropyAcc], tB[kEntropyAcc], tAB[kEntropyAcc];
            for (int i = 0; i <= nq; ++i) {
                double sab = 0.0, sa = 0.0, sb = 0.0;
                for (int w = 0; w < nwarps; ++w) sab += sh_red[i * kSlots + w];
                for (int w = 0; w < 8; ++w) sa += sh_red[i * kSlots + nwarps + w];
                for (int w = 8; w < 16; ++w) sb += sh_red[i * kSlots + nwarps + w];
                tA[i] = sa; tB[i] = sb; tAB[i] = sab;
            }
            const double HA = lnN - tA[0] / N, HB = lnN - tB[0] / N, HAB = lnN - tAB[0] / N;
            const double I = HA + HB - HAB;  // eq. 2
            out[0] = I;
            for (int k = 0; k < nq; ++k) {
                const double qq = qv[k];
                double val;
                if (qq == 1.0) {
                    val = I;
                } else {
                    const double sc = exp(-qq * lnN);
                    const double SA = (1.0 - tA[1 + k] * sc) / (qq - 1.0);
                    const double SB = (1.0 - tB[1 + k] * sc) / (qq - 1.0);
                    const double SAB = (1.0 - tAB[1 + k] * sc) / (qq - 1.0);
                    val = SA + SB - SAB;
                    if (a.form == MI_TSALLIS_PSEUDO_ADDITIVE) val += (1.0 - qq) * SA * SB;
                }
                out[1 + k] = val;
            }
        }
    }
}

// One CTA per (pair, p2) item at a time; every thread owns kZCols columns (iy,ix) of the fixed volume
// -- two groups of 4 adjacent columns, the groups of a warp interleaved so that each 16-byte load
// instruction of a warp reads 512 contiguous bytes -- and walks them along z.  The walk is organised
// by moving plane: for lower plane p the fixed slices iz with floor(c_z) = p form one contiguous run
// (c_z is non-decreasing in iz), during which the two xy-lerped plane values stay in registers; the
// next plane is prefetched one step ahead and the three register sets rotate by name (the plane loop
// is unrolled by 3), so a plane step costs one 16-byte load per 4 columns and a pointer increment.
//
// Histogram update, trilinear (CANON-4 z-lerp, CANON-5 binning, one RED):
//   v = fma(w, hi - lo, lo)
//   t = (v - mlo) * mscale               kBinFast: t = v*mscale; kBinFastPrescaled: t = v
//   t = min(max(t, 0), nb - 1)           kBinFast*: not needed, t is in [0, nb] (mi_internal.h)
//   r = RD(t + (1.5*2^23 + a*pitch))     the low mantissa bits of r are a*pitch + floor(t) EXACTLY
//                                        (ulp is 1 there and the second addend is an integer)
//   RED [4*bits(r) + const]              const folds the shared base and -4*bits(1.5*2^23)
// The shared histogram rows have a pitch of nb + pad words: bank = (a*pad + b) mod 32, so the rows
// of the (many) background fixed bins do not all start on bank 0; pad column nb takes v == hi.
//
// Epilogue: either the histogram is written to global memory (un-ranking the fixed bin), or -- fused
// mode -- step a5 runs straight from shared memory: sum c ln c and sum c^q of the joint counts and
// of both marginals in double, then eq. 2 and its Tsallis forms, written to the
// item's position in the map.  Entropies do not depend on the order of the bins, so the ranked rows
// are used as they are.
template <bool NN, int MODE, bool AGG>
__global__ void __launch_bounds__(kHistThreads, 1) zhist_kernel(const __grid_constant__ ZHistArgs a) {
    extern __shared__ __align__(16) uint32_t sh_raw[];
    int* run_hi = reinterpret_cast<int*>(sh_raw);
    uint32_t* sh_pb = sh_raw + ((a.planes + 3) & ~3);
    double* sh_red = reinterpret_cast<double*>(sh_pb + kEntropyPb);
    uint32_t* sh_hist = sh_raw + zhist_table_words(a.planes);
    __shared__ int s_lo, s_hi;
    __shared__ unsigned long long s_issued;   // histogram updates this CTA issued (a.red_count)
    if (threadIdx.x == 0) s_issued = 0ull;
    const unsigned nb = (unsigned)a.nb;
    const unsigned pitch = (unsigned)a.pitch;
    const int rows_smem = a.rows_smem;   // includes the dump row
    const int words = rows_smem * a.pitch;
    for (int w = threadIdx.x; w < words; w += blockDim.x) sh_hist[w] = 0u;
    for (int w = threadIdx.x; w < kEntropyPb; w += blockDim.x) sh_pb[w] = 0u;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int nwarps = kHistThreads / 32;
    const int colpitch = a.colpitch;
    const float topf = (float)(a.nb - 1);
    const int ntiles = (colpitch + kZCols * kHistThreads - 1) / (kZCols * kHistThreads);
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
            if (sz.ok) {
                atomicMin(&s_lo, iz);
                atomicMax(&s_hi, iz);
                atomicMax(&run_hi[sz.lower], iz + 1);
            }
        }
        __syncthreads();
        const int iz_lo = s_lo, iz_hi = s_hi + 1;   // valid z is one interval (c_z is monotone in iz)

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
                const int wcol = (tile * kHistThreads + warp * 32) * kZCols;   // first column of the warp
                if (wcol >= colpitch) break;                                   // colpitch % kZColAlign == 0
                const int col0 = wcol + lane * 4;                              // groups at col0, col0 + 128
                // columns outside the moving volume count into the dump row: (fa & keep) | dump
                Bins cv, keep, dump;
                ld_bins(cv, a.colvalid + (size_t)pair * colpitch + col0);
                uint32_t any = 0u;
#pragma unroll
                for (int j = 0; j < kZCols / 4; ++j) {
                    any |= cv.w[j];
                    keep.w[j] = cv.w[j] * 0xFFu;                            // cv bytes are 0 or 1
                    dump.w[j] = (~keep.w[j]) & ((uint32_t)a.rows_real * 0x01010101u);
                }
                if (any == 0u) continue;
                const uint8_t* __restrict__ fbq = a.fb + (size_t)iz_lo * colpitch + col0;
                Bins fa_next;
                ld_bins(fa_next, fbq);
                int iz = iz_lo;
                if (NN) {
                    const uint8_t* __restrict__ pp = static_cast<const uint8_t*>(a.xy) +
                                                     ((size_t)pair * a.planes + p_lo) * colpitch + col0;
                    for (int p = p_lo; p <= p_hi; ++p, pp += colpitch) {
                        const int hi = run_hi[p];
                        if (iz >= hi) continue;
                        Bins v;
                        ld_bins(v, pp);
                        for (; iz < hi; ++iz) {
                            Bins fa;
#pragma unroll
                            for (int j = 0; j < kZCols / 4; ++j) fa.w[j] = (fa_next.w[j] & keep.w[j]) | dump.w[j];
                            fbq += colpitch;
                            if (iz + 1 < iz_hi) ld_bins(fa_next, fbq);
#pragma unroll
                            for (int k = 0; k < kZCols; ++k)
                                hist_inc<AGG>(sbase + (byte_of(fa.w[k / 4], k & 3) * pitch + byte_of(v.w[k / 4], k & 3)) * 4u);
                        }
                    }
                } else {
                    const float* __restrict__ pp = static_cast<const float*>(a.xy) +
                                                   ((size_t)pair * a.planes + p_lo) * colpitch + col0;
                    Cols r0, r1, r2;
                    ld_cols(r0, pp);
                    ld_cols(r1, pp + colpitch);
                    r2 = r1;
                    pp += 2 * (size_t)colpitch;   // next plane to prefetch: p + 2
                    int p = p_lo;
                    // one plane step: prefetch plane p+2 into `pre`, run the slices of plane p on (lo, hi)
                    auto step = [&](const Cols& lo, const Cols& hi, Cols& pre) {
                        if (p + 2 < a.planes) ld_cols(pre, pp);
                        pp += colpitch;
                        const int end = run_hi[p];
                        for (; iz < end; ++iz) {
                            // z weight c_z - floor(c_z) (CANON-4) recomputed per slice, 4 ALU instructions, rather
                            // than read from a shared table: the LSU data pipe is this kernel's bottleneck, the
                            // issue slots are not (658 -> 637 ms at C5; deriving the run ends the same way instead
                            // of reading run_hi measured no further gain)
                            const float czf = __fmaf_rn(mo.x, (float)iz, mo.y);
                            const float w = __fsub_rn(czf, __fsub_rn(__fadd_rd(czf, kMagic), kMagic));
                            Bins fa;
#pragma unroll
                            for (int j = 0; j < kZCols / 4; ++j) fa.w[j] = (fa_next.w[j] & keep.w[j]) | dump.w[j];
                            fbq += colpitch;
                            if (iz + 1 < iz_hi) ld_bins(fa_next, fbq);
#pragma unroll
                            for (int k = 0; k < kZCols; ++k) {
                                const float l = col_of(lo, k);
                                const float v = __fmaf_rn(w, __fsub_rn(col_of(hi, k), l), l);
                                float t;
                                if (MODE == kBinFastPrescaled) {
                                    t = v;
                                } else if (MODE == kBinFast) {
                                    t = __fmul_rn(v, mscale);
                                } else {
                                    t = __fmul_rn(__fsub_rn(v, mlo), mscale);
                                    t = fmaxf(fminf(t, topf), 0.0f);   // clamping before the floor == after it
                                }
                                const unsigned mbits = byte_of(fa.w[k / 4], k & 3) * pitch + (unsigned)kMagicBits;
                                const float r = __fadd_rd(t, __uint_as_float(mbits));
                                hist_inc<AGG>(__float_as_uint(r) * 4u + cbase);
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
        if (a.red_count != nullptr && iz_lo < iz_hi) {
            // updates issued for this item, recounted from the column flags outside the hot loop (a counter
            // carried through it costs registers the z kernel does not have: 1024 threads x 64)
            unsigned mine = 0u;
            for (int tile = 0; tile < ntiles; ++tile) {
                const int wcol = (tile * kHistThreads + warp * 32) * kZCols;
                if (wcol >= colpitch) break;
                Bins cv;
                ld_bins(cv, a.colvalid + (size_t)pair * colpitch + wcol + lane * 4);
                uint32_t any = 0u;
#pragma unroll
                for (int j = 0; j < kZCols / 4; ++j) any |= cv.w[j];
                mine += any != 0u;
            }
            mine = warp_sum_u(mine);
            if (lane == 0 && mine) atomicAdd(&s_issued, (unsigned long long)mine * (unsigned)(kZCols * (iz_hi - iz_lo)));
        }
        __syncthreads();
        if (!NN && MODE != kBinGeneral) {   // pad column nb (v == moving_hi) belongs to the last bin
            for (int r = threadIdx.x; r < rows_smem; r += blockDim.x) {
                const uint32_t v = sh_hist[r * pitch + nb];
                if (v) {
                    sh_hist[r * pitch + nb] = 0u;
                    sh_hist[r * pitch + nb - 1] += v;
                }
            }
            __syncthreads();
        }
        if (a.fused) {
            zhist_entropy_epilogue(a, item, sh_hist, sh_pb, sh_red);
        } else {
            // write the item's whole global histogram (un-ranking the fixed bin): counted rows from
            // shared memory (re-zeroed for the next item), rows of the rare ranks as zeros --
            // zrare_kernel adds their voxels afterwards.  No other CTA touches this histogram, so
            // plain stores suffice.
            uint32_t* gh = a.hist + (size_t)item * a.nb * a.nb;
            for (int r = warp; r < (int)nb; r += nwarps) {
                uint32_t* grow = gh + (size_t)__ldg(a.rank_inv + r) * nb;
                const bool real = r < a.rows_real;
                for (unsigned b = lane; b < nb; b += 32) {
                    uint32_t v = 0u;
                    if (real) {
                        v = sh_hist[r * pitch + b];
                        if (v) sh_hist[r * pitch + b] = 0u;
                    }
                    __stcs(grow + b, v);   // streaming: 256 KB per item must not push the xy planes out of L2
                }
            }
        }
        if (a.rows_real < rows_smem)   // the dump row is only re-zeroed
            for (unsigned b = threadIdx.x; b <= nb; b += blockDim.x) sh_hist[a.rows_real * pitch + b] = 0u;
        __syncthreads();
    }
    if (a.red_count != nullptr && threadIdx.x == 0 && s_issued) atomicAdd(a.red_count, s_issued);
}

// fixed ranked bins -> [fnz][colpitch] (plane pitch padded to a multiple of 4 so that four adjacent
// columns are one aligned 32-bit load); pad columns are 0.  Ranks >= rows_real are clamped to the
// dump row `rows_real` and the voxel is appended to the rare list as (col, iz | rank << 16).  Voxels
// outside the optional fixed-voxel mask (mi_set_fixed_mask) become the dump row as well: the z kernel
// then counts them where the entropy epilogue and the histogram write-out never look.
__global__ void __launch_bounds__(256) pitch_bins_kernel(const uint8_t* __restrict__ in,
                                                         const uint32_t* __restrict__ mask_bits, int cols,
                                                         int colpitch, int fnz, int rows_real,
                                                         uint8_t* __restrict__ out, uint2* __restrict__ rare,
                                                         unsigned* __restrict__ rare_count, unsigned rare_cap) {
    const int col = blockIdx.x * 256 + threadIdx.x;
    if (col >= colpitch) return;
    for (int iz = blockIdx.y; iz < fnz; iz += gridDim.y) {
        int r = col < cols ? in[(size_t)iz * cols + col] : 0;
        if (mask_bits != nullptr && col < cols) {
            const size_t vi = (size_t)iz * cols + col;
            if (((mask_bits[vi >> 5] >> (vi & 31u)) & 1u) == 0u) {
                out[(size_t)iz * colpitch + col] = (uint8_t)rows_real;   // masked-out voxel: counts into the dump row
                continue;
            }
        }
        if (r >= rows_real) {
            const unsigned slot = atomicAdd(rare_count, 1u);
            if (slot < rare_cap) rare[slot] = make_uint2((unsigned)col, (unsigned)iz | ((unsigned)r << 16));
            r = rows_real;
        }
        out[(size_t)iz * colpitch + col] = (uint8_t)r;
    }
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
                b = bin_u8(a.bin_mode == kBinFastPrescaled ? v : __fmul_rn(__fsub_rn(v, a.mlo), a.mscale), top);
            }
            atomicAdd(&gh[(size_t)__ldg(a.rank_inv + rank) * a.nb + b], 1u);
        }
    }
}

}  // namespace

cudaError_t launch_pitch_bins(const uint8_t* in, const uint32_t* mask_bits, int cols, int colpitch, int fnz, int rows_real, uint8_t* out,
                              uint2* rare, unsigned* rare_count, unsigned rare_cap, cudaStream_t s) {
    dim3 grid((colpitch + 255) / 256, fnz < 65535 ? fnz : 65535);
    pitch_bins_kernel<<<grid, 256, 0, s>>>(in, mask_bits, cols, colpitch, fnz, rows_real, out, rare, rare_count, rare_cap);
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
                         const float2* ay, int a0, int b0, int nb1, int npairs, int fnx, int cols, int colpitch,
                         float prescale, void* XY, uint8_t* colvalid, cudaStream_t s) {
    dim3 grid((colpitch / 4 + 127) / 128, npairs);
    if (nn)
        ypass_kernel<true, uint8_t><<<grid, 128, 0, s>>>(static_cast<const uint8_t*>(X), planes, prows, mnx, mny, ax,
                                                        ay, a0, b0, nb1, fnx, cols, colpitch, 1.0f,
                                                        static_cast<uint8_t*>(XY), colvalid);
    else
        ypass_kernel<false, float><<<grid, 128, 0, s>>>(static_cast<const float*>(X), planes, prows, mnx, mny, ax, ay,
                                                       a0, b0, nb1, fnx, cols, colpitch, prescale, static_cast<float*>(XY),
                                                       colvalid);
    return cudaGetLastError();
}

// Histogram rows (of `pitch` words) of the z kernel that fit in shared memory beside its tables,
// the dump row included (at most nb + 1).
int zhist_rows_in_smem(int nb, int pitch, int fnz, int planes, size_t smem_optin) {
    (void)fnz;
    const size_t reserve = 1024 + 4 * (size_t)zhist_table_words(planes);
    size_t rows = (smem_optin > reserve ? smem_optin - reserve : 0) / ((size_t)pitch * sizeof(uint32_t));
    if (rows > (size_t)nb + 1) rows = (size_t)nb + 1;
    return (int)rows;
}

template <bool NN, int MODE, bool AGG>
static cudaError_t launch_zhist_t(const ZHistArgs& a, unsigned grid, size_t smem, cudaStream_t s) {
    auto kern = zhist_kernel<NN, MODE, AGG>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kHistThreads, smem, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_zhist(bool nn, const ZHistArgs& a, int num_sms, cudaStream_t s) {
    if (a.rows_smem < 1 || a.pitch < a.nb + 1 || (a.colpitch % kZColAlign) != 0 || a.nb > 256)
        return cudaErrorInvalidConfiguration;
    if (a.fused && (a.n_rare > 0 || a.nq > kMaxQPerPass || a.mi_out == nullptr)) return cudaErrorInvalidConfiguration;
    const size_t smem = 4 * (size_t)zhist_table_words(a.planes) + (size_t)a.rows_smem * a.pitch * sizeof(uint32_t);
    const long long nitems = (long long)a.n_pairs * a.n2;
    long long grid = nitems < num_sms ? nitems : num_sms;
    if (grid < 1) return cudaSuccess;
    cudaError_t e;
    const unsigned g = (unsigned)grid;
    if (a.match_any) {
        if (nn) e = launch_zhist_t<true, kBinGeneral, true>(a, g, smem, s);
        else if (a.bin_mode == kBinFastPrescaled) e = launch_zhist_t<false, kBinFastPrescaled, true>(a, g, smem, s);
        else if (a.bin_mode == kBinFast) e = launch_zhist_t<false, kBinFast, true>(a, g, smem, s);
        else e = launch_zhist_t<false, kBinGeneral, true>(a, g, smem, s);
    } else if (nn) e = launch_zhist_t<true, kBinGeneral, false>(a, g, smem, s);
    else if (a.bin_mode == kBinFastPrescaled) e = launch_zhist_t<false, kBinFastPrescaled, false>(a, g, smem, s);
    else if (a.bin_mode == kBinFast) e = launch_zhist_t<false, kBinFast, false>(a, g, smem, s);
    else e = launch_zhist_t<false, kBinGeneral, false>(a, g, smem, s);
    if (e != cudaSuccess) return e;
    if (a.n_rare > 0) {
        long long g2 = nitems < 8LL * num_sms ? nitems : 8LL * num_sms;
        if (nn) zrare_kernel<true><<<(unsigned)g2, 256, 0, s>>>(a);
        else zrare_kernel<false><<<(unsigned)g2, 256, 0, s>>>(a);
    }
    return cudaGetLastError();
}

}  // namespace mi
