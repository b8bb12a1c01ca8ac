// mi_internal.h -- declarations shared by the translation units of libmi_b200.so (library-private).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "mi.h"

namespace mi {

// ---- shared host runtime pieces (mi_api.cu) -----------------------------------------------------
// stream-ordered allocation from the library's per-device pool / release back to it
cudaError_t dev_alloc(void** p, size_t bytes, int dev, cudaStream_t s);
void dev_free(void* p, cudaStream_t s);
void set_thread_error(const std::string& msg);   // text behind mi_last_error(NULL)
bool is_host_pointer(const void* p);
int sm_count();                                  // SMs of the current device (queried once per device)

constexpr int kMaxQPerPass = 8;      // Tsallis orders handled by one entropy-kernel pass
constexpr int kHistThreads = 1024;   // resample+histogram CTA size
constexpr int kEntropyThreads = 256;
constexpr int kMaxBinsWide = 4096;   // largest nbins (above 256: uint16 bins, global-memory histograms)

// ---- host-side double math (mi_host.cpp; compiled with -ffp-contract=off) --------------------
int family_matrix(int family, const double p[3], double T[12]);
void compose_matrix(const double p[9], double T[12]);
int seed_from_node(int family, const double p[3], double out[9]);
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
    const uint32_t* mask_bits;    // NULL, or one bit per fixed voxel (flat index): 0 = the voxel takes no part
    const float* moving_pad;      // replicate-padded moving float32, dims (mx+2, my+2, mz+2)
    const float4* moving_quad;    // yz-quads of the padded volume (same dims), or NULL
    int gather;                   // trilinear gather scheme: 0 eight 4-byte loads, 1 two 16-byte quad loads
    int threads;                  // CTA size of the quad kernel: 512, 768 or 1024
    int has_rare;                 // a populated fixed-bin rank >= rows_smem exists (its updates go to global memory)
    unsigned* sink;               // NULL; or (roofline probe) no histogram is built, bins are summed here
    const uint8_t* mbins;         // moving bin indices (nearest neighbour), unpadded
    const float* M;               // n_transforms x 12 index-space affines (device)
    uint32_t* hist;               // n_transforms x nb x nb (row = fixed bin), zero on entry
    int rows_smem;                // ranked fixed-bin rows kept in shared memory
    int pitch;                    // words per shared histogram row (>= nb)
    int ty_log2;                  // the CTA's 32 warps cover 2^ty_log2 (y) x 32/2^ty_log2 (z) fixed rows at a time
    VolumeDesc f, m;
    int nb;
    float mlo, mscale;       // moving binning (CANON-5)
    int n_transforms;
    int unroll;              // voxels per lane in flight (1..4); 0 = chosen from the row length
    int nslabs;              // CTAs cooperating on one transform (slabs of row tiles)
};

// flag (may be NULL): set to 1 if any voxel is negative, not finite or above the last bin edge
cudaError_t launch_prebin(const float* vol, uint8_t* bins, int64_t n, float lo, float scale, int nb,
                          unsigned* flag, cudaStream_t s);
cudaError_t launch_pad_replicate(const float* src, float* dst, int nx, int ny, int nz, cudaStream_t s);
cudaError_t launch_quad_build(const float* pad, float4* quad, int nx, int ny, int nz, cudaStream_t s);
cudaError_t launch_rank_fixed_bins(const uint8_t* bins, int64_t n, unsigned long long* counts_scratch,
                                   uint8_t* rank, int* inv, uint8_t* ranked_bins, cudaStream_t s);
int hist_rows_in_smem(int nb, int pitch, size_t smem_bytes);
// wide histograms (256 < nb <= kMaxBinsWide)
struct WideArgs {
    const uint16_t* fbins;        // fixed bins [fz][fy][fx]
    const uint16_t* mbins;        // moving bins (nearest neighbour)
    const uint32_t* mask_bits;    // NULL, or one bit per fixed voxel
    const float* moving_pad;      // replicate-padded moving float32
    const float* M;               // n_transforms x 12 (device)
    uint32_t* hist;               // n_transforms x nb x nb, zero on entry
    VolumeDesc f, m;
    int nb;
    float mlo, mscale;
    int n_transforms, nslabs;
    const float4* moving_quad;    // yz-quads of the padded moving volume (version 2, trilinear)
    const uint16_t* fbins_ranked; // version 2: fixed bins replaced by their population rank
    const int* rank_inv;          // version 2: rank -> fixed bin
    int rows_smem, pitch;         // version 2: ranked rows counted in shared memory, words per row
    int version, unroll;          // 2: resample_wide_kernel; 1: round 1's resample_hist_wide_kernel (MI_OPT_GENERIC_GATHER = 0)
};
cudaError_t launch_bin_count16(const uint16_t* bins, int64_t n, unsigned long long* counts, cudaStream_t s);
cudaError_t launch_remap16(const uint16_t* bins, uint16_t* ranked, int64_t n, const uint16_t* rank, cudaStream_t s);
cudaError_t launch_mask_bits(const uint8_t* mask, int64_t n, uint32_t* bits, cudaStream_t s);
cudaError_t launch_prebin16(const float* vol, uint16_t* bins, int64_t n, float lo, float scale, int nb, cudaStream_t s);
cudaError_t launch_resample_hist_wide(const WideArgs& a, int interp, int num_sms, cudaStream_t s);
cudaError_t launch_resample_hist(const ResampleArgs& a, int interp, int num_sms, cudaStream_t s);
// Where the entropy kernel writes the result of histogram `item`: transform-major position item
// (enabled == 0) or, for the separable path whose items are ordered (p0, p1, p2) with p2 fastest
// over a batch of nb1 p1 values starting at b0 and p0 values starting at a0, the map's transform
// index (p2*n1 + p1)*n0 + p0.
struct OutMap {
    int enabled;
    int n0, n1, n2, a0;
    int b0, nb1;
    __host__ __device__ size_t dst(long long item) const {
        if (!enabled) return (size_t)item;
        const long long c = item % n2, ab = item / n2;
        const long long b = ab % nb1, al = ab / nb1;
        return ((size_t)c * n1 + (size_t)(b0 + b)) * n0 + (size_t)(a0 + al);
    }
};
cudaError_t launch_entropy(const uint32_t* hist, int nb, int n_transforms, const double* q_dev, int nq,
                           int q_off, int form, double* mi_out /* n x (1+nq) */, int64_t* nvalid,
                           OutMap om, cudaStream_t s,
                           const uint8_t* row_used = nullptr /* nb > 256: flags of the populated fixed bins */);

// ---- partial-volume interpolation (mi_pv.cu) ---------------------------------------------------
struct PvArgs {
    const uint8_t* fbins_ranked;  // fixed bins replaced by their population rank, flat voxel order
    const int* rank_inv;          // rank -> fixed bin
    const uint32_t* mask_bits;    // NULL, or one bit per fixed voxel
    const uint32_t* mbins_quad;   // yz-quads of the replicate-padded moving BIN volume, dims (mx+2, my+2, mz+2)
    const float* M;               // n_transforms x 12 (device)
    unsigned long long* hist;     // n_transforms x nb x nb in units of 2^-15 voxel, zero on entry
    int rows_smem, pitch;         // shared histogram rows (ranked) and words per row
    VolumeDesc f, m;
    int nb, n_transforms;
    int nchunks, rows_per_chunk;  // set by the launcher: chunks of whole fixed rows per transform
    int hot_b;                    // most populated moving bin: cell (fixed rank 0, hot_b) is summed in registers
};
cudaError_t launch_bin_count(const uint8_t* bins, int64_t n, unsigned long long* counts, cudaStream_t s);
cudaError_t launch_bins_quad_build(const uint8_t* src, uint32_t* dst, int nx, int ny, int nz, cudaStream_t s);
cudaError_t launch_resample_hist_pv(PvArgs a, int num_sms, cudaStream_t s);
cudaError_t launch_entropy_pv(const unsigned long long* hist, int nb, int n_transforms, const double* q_dev, int nq,
                              int q_off, int form, double* mi_out, int64_t* nvalid, OutMap om, cudaStream_t s);

// ---- separable path (mi_separable.cu) ----------------------------------------------------------
struct ZHistArgs {
    const void* xy;            // [n_pairs][planes][colpitch] float (trilinear) or uint8 (nearest)
    const uint8_t* colvalid;   // [n_pairs][colpitch]: column (iy,ix) is inside the moving volume in x and y
    const uint8_t* fb;         // ranked fixed bins, [fnz][colpitch]
    const int* rank_inv;
    const float2* az;          // n2 z-axis (scale, offset) pairs
    uint32_t* hist;            // [n_pairs*n2][nb][nb], zero on entry
    int fnz, colpitch, planes, mnz;
    int nb, rows_smem;         // rows_smem: histogram rows in shared memory, dump row included
    int pitch;                 // words per shared histogram row (>= nb + 1; the pad spreads rows over banks)
    int bin_mode;              // kBinGeneral / kBinFast / kBinFastPrescaled (see below)
    int rows_real;             // ranks below rows_real are counted in shared memory; the rest are "rare"
    float mlo, mscale;
    int n_pairs, n2;
    const uint2* rare;         // rare voxels: (col, iz | rank << 16)
    unsigned n_rare;
    // fused entropy epilogue (step a5 straight from the shared histogram; needs n_rare == 0):
    // hist is not written, the (1 + nq_total) values of item go to mi_out at its map position
    int fused;
    const double* q;           // device, nq_total orders; the first nq (<= kMaxQPerPass) are computed
    int nq, nq_total, form;
    double* mi_out;
    int64_t* nvalid;
    OutMap om;
    int match_any;                  // 1: __match_any_sync aggregation instead of the plain RED (measurement option)
    unsigned long long* red_count;  // NULL, or device counter of the histogram updates issued
};
// Moving-side binning variants of the z kernel (CANON-5, t = (v - mlo) * mscale, clamp, floor):
//   kBinGeneral        the full sequence
//   kBinFast           mlo == 0 and every moving voxel v is finite with 0 <= v and v*mscale <= nb:
//                      every lerp result lies between its inputs, so t = v*mscale is in [0, nb]
//                      without clamps; floor(t) == nb (v == hi) is counted in pad column nb of the
//                      shared row and added to column nb-1 when the histogram is finished
//   kBinFastPrescaled  kBinFast and mscale is a power of two: the y-pass stores v*mscale (exact),
//                      and fma(w, s*hi - s*lo, s*lo) == s*fma(w, hi - lo, lo) bit for bit
enum { kBinGeneral = 0, kBinFast = 1, kBinFastPrescaled = 2 };
constexpr int kZCols = 8;            // columns per thread of the z kernel: 2 groups of 4
constexpr int kZColAlign = 32 * kZCols;  // colpitch is a multiple of this (one warp's columns)
cudaError_t launch_pitch_bins(const uint8_t* in, const uint32_t* mask_bits, int cols, int colpitch, int fnz, int rows_real, uint8_t* out,
                              uint2* rare, unsigned* rare_count, unsigned rare_cap, cudaStream_t s);
cudaError_t launch_xpass(bool nn, const void* src, int snx, int srows, int mnx, const float2* ax, int a0,
                         int na, int fnx, void* X, cudaStream_t s);
// pair = a_local*nb1 + b_local covers p0 index a0 + a_local and p1 index b0 + b_local
cudaError_t launch_ypass(bool nn, const void* X, int planes, int prows, int mnx, int mny, const float2* ax,
                         const float2* ay, int a0, int b0, int nb1, int npairs, int fnx, int cols, int colpitch,
                         float prescale, void* XY, uint8_t* colvalid, cudaStream_t s);
int zhist_rows_in_smem(int nb, int pitch, int fnz, int planes, size_t smem_optin);
cudaError_t launch_zhist(bool nn, const ZHistArgs& a, int num_sms, cudaStream_t s);
cudaError_t launch_map_assemble(const double* mi /* n x nch */, int64_t n, int nch, double* map_out,
                                int64_t* argmax_out, cudaStream_t s);
cudaError_t run_shared_atomic_probe(int nbins, int pattern, int iters, int num_sms, size_t smem_optin,
                                    double* updates_per_s);

}  // namespace mi
