// mi_device.cuh -- small __device__ helpers shared by the kernel translation units (library-private;
// the library is built without relocatable device code, so shared device functions live in a header).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "mi_internal.h"

namespace mi {

// floor() of |c| < 2^22 without a conversion instruction: RD(c + 1.5*2^23) = 1.5*2^23 + floor(c)
// exactly (ulp is 1 there), so the low mantissa bits ARE floor(c) as a two's-complement offset.
constexpr float kFloorMagic = 12582912.0f;        // 1.5 * 2^23
constexpr int kFloorMagicBits = 0x4B400000;

__device__ __forceinline__ unsigned warp_sum(unsigned v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Last step of a5 for transform t from the three distributions' sums (tot[0..2] = sum c ln c of A, B, AB;
// tot[3 + 3k + {0,1,2}] = sum c^q_k) and the total count N (a double: voxels, or voxels as a multiple of
// 2^-15 for partial-volume histograms): eq. 1-2 and the Tsallis forms.
__device__ __forceinline__ void entropy_finish(const double* tot, double N, long long nvalid_count, int t,
                                               const double* qv, int nq_pass, int q_off, int nq_total, int form,
                                               double* __restrict__ mi_out, int64_t* __restrict__ nvalid,
                                               const OutMap& om) {
    const size_t dst = om.dst(t);  // item order (p0, p1, p2 fastest) -> map order (p2, p1, p0 fastest)
    double* out = mi_out + dst * (1 + nq_total);
    if (nvalid != nullptr) nvalid[dst] = (int64_t)nvalid_count;
    if (!(N > 0.0)) {
        out[0] = 0.0;
        for (int k = 0; k < nq_pass; ++k) out[1 + q_off + k] = 0.0;
        return;
    }
    const double lnN = log(N);
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

}  // namespace mi
