// mi_internal.h -- declarations shared by the translation units of libmi_b200.so (library-private).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "mi.h"

namespace mi {

constexpr int kMaxQPerPass = 8;      // Tsallis orders handled by one entropy-kernel pass
constexpr int kHistThreads = 1024;   // resample+histogram CTA size
constexpr int kEntropyThreads = 256;

// ---- host-side double math (mi_host.cpp; compiled with -ffp-contract=off) --------------------
int family_matrix(int family, const double p[3], double T[12]);
void index_affine(const double T[12], const int32_t fd[3], const double fs[3], const int32_t md[3],
                  const double ms[3], float out[12]);
float bin_scale(int nbins, float lo, float hi);

// ---- kernel launch wrappers (mi_kernels.cu) ---------------------------------------------------
struct VolumeDesc {
    int nx, ny, nz;
};

struct ResampleArgs {
    const uint8_t* fbins_ranked;  // fixed bins replaced by their population rank, [fz][fy][fx]
    const int* rank_inv;          // rank -> fixed bin
    const float* moving_pad;      // replicate-padded moving float32, dims (mx+2, my+2, mz+2)
    const uint8_t* mbins;         // moving bin indices (nearest neighbour), unpadded
    const float* M;               // n_transforms x 12 index-space affines (device)
    uint32_t* hist;               // n_transforms x nb x nb (row = fixed bin), zero on entry
    int rows_smem;                // ranked fixed-bin rows kept in shared memory
    VolumeDesc f, m;
    int nb;
    float mlo, mscale;       // moving binning (CANON-5)
    int n_transforms;
    int nslabs;              // CTAs cooperating on one transform (row slabs)
};

cudaError_t launch_prebin(const float* vol, uint8_t* bins, int64_t n, float lo, float scale, int nb,
                          cudaStream_t s);
cudaError_t launch_pad_replicate(const float* src, float* dst, int nx, int ny, int nz, cudaStream_t s);
cudaError_t launch_rank_fixed_bins(const uint8_t* bins, int64_t n, unsigned long long* counts_scratch,
                                   uint8_t* rank, int* inv, uint8_t* ranked_bins, cudaStream_t s);
int hist_rows_in_smem(int nb, size_t smem_optin);
cudaError_t launch_resample_hist(const ResampleArgs& a, int interp, int num_sms, cudaStream_t s);
cudaError_t launch_entropy(const uint32_t* hist, int nb, int n_transforms, const double* q_dev, int nq,
                           int q_off, int form, double* mi_out /* n x (1+nq) */, int64_t* nvalid,
                           cudaStream_t s);
cudaError_t launch_map_assemble(const double* mi /* n x nch */, int64_t n, int nch, double* map_out,
                                int64_t* argmax_out, cudaStream_t s);
cudaError_t run_shared_atomic_probe(int nbins, int pattern, int iters, int num_sms, size_t smem_optin,
                                    double* updates_per_s);

}  // namespace mi
