/* mi.h -- C ABI of the B200-native exhaustive mutual-information map ("MICUDA" hot path of
 * Vianna & Murta 2019, arxiv 1909.10690).  Citations are PAPER.md line numbers.
 *
 * The library registers a moving volume v against a fixed volume u by EVALUATING (not optimising)
 * the metric F_m(u(x), v(T(x))) of eq. 3 for many transforms T at once:
 *   Transform block  v(T(x)): resample v at every fixed voxel x          (Fig. 1)
 *   Metric block     joint histogram over ALL voxels, "full histogram"
 *                    -> Shannon MI, eq. 1-2
 *                    -> Tsallis MI for a list of q from the SAME histogram
 *   Exhaustive map   one MI value per point of a 3-parameter grid of one transform family,
 *                    stored as a 3D image
 * Every step runs in hand-written CUDA kernels for sm_100a; there is NO CPU fallback: without a
 * CUDA device every compute entry point returns MI_ERR_CUDA.
 *
 * Conventions
 *   dims      (nx, ny, nz); x is fastest in memory: voxel (ix,iy,iz) is at [(iz*ny + iy)*nx + ix].
 *   frames    physical frames are volume-centred, axes = index axes, identity direction cosines:
 *             voxel i sits at spacing * (i - (n-1)/2) mm.
 *   transform T is a row-major 3x4 [A|t] of doubles mapping a FIXED physical point x (mm) to a
 *             MOVING physical point y = A x + t (mm) -- the direction of eq. 3.
 *   samples   falling outside the moving volume (continuous index outside [-0.5, n-0.5) on any
 *             axis) are skipped; probabilities are normalised by the number of valid samples.
 *   bins      uniform over [lo, hi]; b = clamp(floor((v - lo) * nbins/(hi-lo)), 0, nbins-1).
 *   pointers  BULK data -- the volumes and the mask given to mi_create / mi_set_fixed_mask, a map given
 *             to mi_map_gradient / mi_map_basins, and every OUTPUT array (mi_out, hist_out,
 *             nvalid_out, map_out, argmax_out, grad_out, label_out, steps_out, mi_get_bins' out) --
 *             may be HOST or DEVICE pointers (resolved with cudaPointerGetAttributes).  The small
 *             PARAMETER arrays -- dims, spacings, T, q, lo, hi, n, begin, end, p, delta, step0,
 *             step_min -- and the info/stats structs are read or written on the host and must be
 *             HOST pointers.  Inputs are only read.  Outputs are caller-owned and are written only
 *             when the call returns MI_OK.
 *   sync      a call returns after all HOST outputs are complete; DEVICE outputs are ordered on
 *             the context's stream (the cudaStream_t given to mi_create).
 *   threads   one context must not be used from two threads at once; distinct contexts are
 *             independent.
 *   errors    status codes only -- nothing throws or aborts across this ABI; mi_last_error gives
 *             the text of the last failure.
 */
#ifndef MI_B200_H
#define MI_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mi_ctx mi_ctx; /* opaque; owns all of its device memory until mi_destroy */

typedef enum {
    MI_OK = 0,
    MI_ERR_INVALID_ARG = 1,   /* NULL pointer, dim < 1, grid n < 1, spacing <= 0 or non-finite, lo >= hi,
                                 nbins < 2, N < 0, q <= 0, q > 32 or non-finite, non-finite matrix entry */
    MI_ERR_UNSUPPORTED = 2,   /* nbins > 4096; volume with more than 2^31-1 voxels */
    MI_ERR_OUT_OF_MEMORY = 3,
    MI_ERR_CUDA = 4,          /* any CUDA runtime failure, including "no device" */
    MI_ERR_INTERNAL = 5
} mi_status;

/* Interpolation of the Transform block v(T(x)) ("the effects of interpolation").
 * NEAREST and TRILINEAR interpolate the intensity and add one count per sample.  PARTIAL_VOLUME is the
 * method of Maes et al. (the paper's ref. [5]; reading A21): no intensity is
 * interpolated, the eight neighbours of the sample point each add their trilinear weight to the cell
 * (bin u(x), bin v(neighbour)).  Weights are products of per-axis fractions rounded to 1/32 voxel, so one
 * sample adds exactly 2^15 integer units and the histogram does not depend on the order of the updates.
 * nbins <= 256 only; every transform takes the generic path. */
typedef enum { MI_INTERP_NEAREST = 0, MI_INTERP_TRILINEAR = 1, MI_INTERP_PARTIAL_VOLUME = 2 } mi_interp;

/* Tsallis entropy S_q(X) = (1 - sum_{p>0} p^q)/(q - 1).  The paper prints no Tsallis formula
 * (reading A1); ADDITIVE puts S_q into the paper's own eq. 2 and is the default. */
typedef enum {
    MI_TSALLIS_ADDITIVE = 0,        /* I_q = S_q(A) + S_q(B) - S_q(A,B)                         */
    MI_TSALLIS_PSEUDO_ADDITIVE = 1  /* I_q = S_q(A) + S_q(B) + (1-q) S_q(A) S_q(B) - S_q(A,B)   */
} mi_tsallis_form;

/* Transform families of the maps (section 3.1-3.3). p = (p0,p1,p2). */
typedef enum {
    MI_FAMILY_TRANSLATION = 0,        /* A = I, t = p (mm)                                       */
    MI_FAMILY_ROTATION_EULER_DEG = 1, /* A = Rz(p2) Ry(p1) Rx(p0), degrees, about the centre     */
    MI_FAMILY_ROTATION_VERSOR = 2,    /* p = axis*sin(theta/2); |p| > 1 -> p/|p| */
    MI_FAMILY_SCALE = 3,              /* A = diag(p), 1 = identity                               */
    MI_FAMILY_SCALE_LOG = 4           /* A = diag(exp(p)), zero-centred           */
} mi_family;

/* mi_create -- take a fixed/moving pair and pre-bin it (step a1: fixed float -> uint8 bin
 * indices; the moving volume is kept as float32 for trilinear sampling and also pre-binned for
 * nearest-neighbour sampling).  "uses all the voxels and produces a full histogram" PAPER.md:212.
 *   out            receives the context; *out is NULL on failure.
 *   fixed, moving  float32 volumes (host or device), finite values; copied -- the caller may free
 *                  them on return.
 *   *_dims         (nx, ny, nz), each >= 1;  *_spacing  mm, each > 0 and finite.  At most 2^31-1 voxels
 *                  per volume.  A fixed volume with nz > 65535 is accepted but its maps take the generic
 *                  kernel (the separable kernels index z slices with 16 bits).
 *   nbins          2..4096 bins per axis of the joint histogram.  Up to 256 the histograms are built in
 *                  shared memory (and translation / scale maps take the separable kernels); above, the
 *                  "full histogram" of PAPER.md:212 for 12-bit data, they live in global memory
 *                  (nbins*nbins*4 bytes per transform) and every transform takes the generic kernel.
 *   *_lo, *_hi     intensity range of each volume, lo < hi, finite.
 *   device         CUDA device ordinal.   cuda_stream  a cudaStream_t (may be NULL = default).
 * Blocks until the context is ready.
 * Device memory of a context (nbins <= 256), from the library's pool, each buffer rounded up to 2 MB: per FIXED
 * voxel 3 B (bins, ranked bins, pitched ranked bins); per MOVING voxel 1 B (bins) + 4 B per padded voxel (the
 * replicate-padded float copy, dims + 2).  Built only by the first call that needs them (MI_INFO_QUADS_BUILT):
 * + 16 B per padded moving voxel for the generic trilinear kernels (any transform that is not a pure
 * translation / scale grid), + 4 B per padded voxel for partial volume.  Map calls add their scratch on
 * demand, bounded by the MI_OPT_*_BUDGET_MB options. */
mi_status mi_create(mi_ctx **out,
                    const float *fixed, const int32_t fixed_dims[3], const double fixed_spacing[3],
                    const float *moving, const int32_t moving_dims[3], const double moving_spacing[3],
                    int32_t nbins, float fixed_lo, float fixed_hi, float moving_lo, float moving_hi,
                    int32_t device, void *cuda_stream);

/* Select the Tsallis MI form used by later calls (default MI_TSALLIS_ADDITIVE). */
mi_status mi_set_tsallis_form(mi_ctx *ctx, mi_tsallis_form form);

/* mi_eval_batch -- F_m(u, v o T) for N transforms (eq. 3 without the arg max).
 *   T           N x 12 doubles, row-major [A|t] per transform (see "transform" above).  Singular
 *               matrices are legal; entries must be finite.
 *   q, nq       Tsallis orders, each in (0, 32]; q == 1 returns the Shannon value; nq may be 0
 *               (then q may be NULL).  The upper bound keeps sum c^q over integer counts c < 2^31
 *               inside the double range (32 ln 2^31 = 688 < 709); the paper uses q in [0.5, 2].
 *   mi_out      N x (1+nq) doubles: [Shannon I (nats), I_q0, I_q1, ...] per transform.  An empty
 *               overlap gives zeros.
 *   hist_out    NULL, or N x nbins x nbins uint32 joint histograms, row = fixed bin, column =
 *               moving bin.  Must be NULL with MI_INTERP_PARTIAL_VOLUME (see mi_eval_batch_pv).
 *   nvalid_out  NULL, or N int64: samples inside the moving volume per transform.
 * N == 0 is a no-op returning MI_OK.  Every transform takes the generic resample+histogram kernel (only
 * mi_map / mi_map_range recognise diagonal grids and take the separable kernels). */
mi_status mi_eval_batch(mi_ctx *ctx, const double *T, int64_t N, const double *q, int32_t nq,
                        mi_interp interp, double *mi_out, uint32_t *hist_out, int64_t *nvalid_out);

/* mi_eval_batch with MI_INTERP_PARTIAL_VOLUME and the histograms in their own unit: hist_out is NULL or
 * N x nbins x nbins uint64 weights in units of 2^-15 voxel (sum = 2^15 * nvalid).  Other arguments as
 * mi_eval_batch.  MI_ERR_UNSUPPORTED for nbins > 256. */
mi_status mi_eval_batch_pv(mi_ctx *ctx, const double *T, int64_t N, const double *q, int32_t nq,
                           double *mi_out, uint64_t *hist_out, int64_t *nvalid_out);

/* mi_eval_noalloc -- steps a3-a5 (resample, joint histogram, entropies: eq. 1-2
 * PAPER.md:25-32) for ONE transform, without a context and without allocating any device memory.
 *
 * Why it exists.  mi_create and the calls on a context take device memory from the library's pool.  A
 * caller whose process has given the whole GPU to another allocator (a tensor framework's caching
 * allocator, a renderer, a fixed MPS/MIG memory limit), or who sits in a latency-critical loop where the
 * device-wide synchronisation of cudaMalloc / cudaFree is not acceptable, cannot use them.  This call makes
 * no cudaMalloc, cudaFree or other allocating call: its only scratch, the nbins x nbins joint histogram
 * (plus the q list), lives in a static __device__ array inside the library.
 *
 * Cost and limits.  The array is 256 KB + 256 B; every GPU on which the library is loaded holds it until
 * the process exits.  nbins <= 256, nq <= 8, NEAREST or TRILINEAR, one transform per call; larger requests
 * return MI_ERR_UNSUPPORTED with a message in mi_last_error(NULL) -- nothing is truncated.
 *
 * Arguments.  fixed_dev, moving_dev: float32 volumes in DEVICE memory the caller owns (layout, dims,
 * spacing, ranges, nbins as in mi_create; read in place, not copied, so they must stay valid until the
 * work queued on cuda_stream has run).  T: one row-major 3x4 [A|t] (host); q, nq, interp as in
 * mi_eval_batch (host); form as in mi_set_tsallis_form.  Outputs are DEVICE pointers the caller owns:
 * mi_out_dev 1+nq doubles; hist_out_dev NULL or nbins x nbins uint32; nvalid_out_dev NULL or one int64.
 * A host pointer for a volume or an output is MI_ERR_INVALID_ARG (staging it would need a device buffer).
 * device, cuda_stream as in mi_create.  The call only queues work on cuda_stream and returns; the outputs
 * are complete when that stream has run, and a kernel fault shows up at the caller's next synchronisation.
 * Results are bit-identical to mi_eval_batch's for the same volumes and transform.
 *
 * One array, shared by every call:
 *   - it still holds the previous call's histogram; each call clears the cells it uses, on cuda_stream,
 *     before counting -- callers need not (and cannot) clear it themselves;
 *   - two calls whose GPU work overlaps in time on one device (different streams, threads or contexts)
 *     count into the same cells and spoil each other: serialise them on one stream or with events;
 *   - the FIRST call on each device looks up the array's device address (cudaGetSymbolAddress with that
 *     device current) and opts the kernel into large shared memory.  Make that first call during set-up,
 *     before any stream capture begins; later calls only launch kernels. */
mi_status mi_eval_noalloc(const float *fixed_dev, const int32_t fixed_dims[3], const double fixed_spacing[3],
                          const float *moving_dev, const int32_t moving_dims[3], const double moving_spacing[3],
                          int32_t nbins, float fixed_lo, float fixed_hi, float moving_lo, float moving_hi,
                          const double T[12], const double *q, int32_t nq, mi_interp interp, mi_tsallis_form form,
                          double *mi_out_dev, uint32_t *hist_out_dev, int64_t *nvalid_out_dev,
                          int32_t device, void *cuda_stream);

/* mi_map -- the exhaustive map of one family: "map with the MI function all
 * the space in a finite range and build a 3D image".
 *   lo, hi, n   inclusive grid per parameter axis: value k on axis d is
 *               lo[d] + k*(hi[d]-lo[d])/(n[d]-1) in double (n[d] == 1 -> lo[d]); n[d] >= 1.
 *   map_out     (1+nq) x n[2] x n[1] x n[0] doubles, channel-major, p0 fastest.
 *   argmax_out  NULL, or (1+nq) int64 linear indices into one channel: the largest value, ties to
 *               the lowest index (the arg max of eq. 3). */
mi_status mi_map(mi_ctx *ctx, mi_family family, const double lo[3], const double hi[3],
                 const int32_t n[3], const double *q, int32_t nq, mi_interp interp,
                 double *map_out, int64_t *argmax_out);

/* mi_map_range -- a sub-box of the same map: nodes begin[d] <= k_d < end[d] of the grid (lo, hi, n).
 * Node parameters are those of the WHOLE grid (lo[d] + k*(hi[d]-lo[d])/(n[d]-1)), so a slab computed
 * here equals the same nodes of mi_map bit for bit -- the unit of multi-GPU sharding (every map voxel
 * is a separate MI evaluation) and of spot checks of a large map.
 *   begin, end  NULL = the whole axis range (0 and n); else 0 <= begin[d] < end[d] <= n[d].
 *   map_out     (1+nq) x m[2] x m[1] x m[0] doubles with m[d] = end[d] - begin[d], p0 fastest.
 *   argmax_out  NULL, or (1+nq) linear indices into the SUB-BOX.
 *   hist_out    NULL, or m[2]*m[1]*m[0] joint histograms of nbins x nbins uint32 in sub-box node order
 *               (row = fixed bin).  Diagonal families then run the separable kernels with the
 *               histogram written out instead of the fused entropy epilogue.  Must be NULL with
 *               MI_INTERP_PARTIAL_VOLUME. */
mi_status mi_map_range(mi_ctx *ctx, mi_family family, const double lo[3], const double hi[3],
                       const int32_t n[3], const int32_t begin[3], const int32_t end[3],
                       const double *q, int32_t nq, mi_interp interp,
                       double *map_out, int64_t *argmax_out, uint32_t *hist_out);

/* Tuning and test options of a context -- the only way to change kernel selection (no environment
 * variable is read anywhere in the library).  Defaults are the measured optimum;
 * no option changes a result bit: they select between kernels that compute the same CANON sequence.
 * Values are validated (MI_ERR_INVALID_ARG).  MI_INFO_* keys are read-only (mi_get_option). */
typedef enum {
    MI_OPT_SEPARABLE = 0,          /* 1: translation / scale maps take the separable kernels; 0: generic kernel */
    MI_OPT_FUSE_ENTROPY = 1,       /* 1: step a5 as the z kernel's epilogue when possible                       */
    MI_OPT_BIN_MODE_MAX = 2,       /* cap on the z kernel's binning variant: 0 general, 1 clamp-free, 2 pre-scaled */
    MI_OPT_ZHIST_ROWS_MAX = 3,     /* cap on the z kernel's shared histogram rows (0 = all that fit), >= 2      */
    MI_OPT_ZHIST_PAD = 4,          /* pad words per shared row of the z kernel, 1..64 (default 9)               */
    MI_OPT_XY_BUDGET_MB = 5,       /* xy-plane scratch per separable batch (default 12288)                      */
    MI_OPT_SEP_HIST_BUDGET_MB = 6, /* histogram scratch per separable batch when not fused (default 3072)       */
    MI_OPT_HIST_BUDGET_MB = 7,     /* histogram scratch per chunk of the generic path (default 1024)            */
    MI_OPT_GENERIC_PAD = 8,        /* pad words per shared row of the generic kernel, 0..64 (default 5)         */
    MI_OPT_GENERIC_SMEM_KB = 9,    /* shared histogram of the generic kernel in KB (default 196; rest is L1)    */
    MI_OPT_GENERIC_TY_LOG2 = 10,   /* generic kernel row tile: 2^v rows in y x 32/2^v in z (default 3)          */
    MI_OPT_GENERIC_UNROLL = 11,    /* generic kernel voxels in flight per lane, 1..4 (0 = from the row length)  */
    MI_OPT_ZHIST_MATCH_ANY = 12,   /* 1: the z kernel aggregates equal addresses with __match_any_sync before the shared
                                      atomic (the scheme BASELINE.json's north_star names) instead of one plain RED per
                                      lane; slower on B200 (profiles/), kept so the choice stays a measured one  */
    MI_OPT_GENERIC_GATHER = 13,    /* generic kernel, trilinear: 1 (default) two 16-byte loads per sample from a yz-quad
                                      copy of the moving volume; 0 eight 4-byte loads from the padded volume        */
    MI_OPT_GENERIC_THREADS = 14,   /* CTA size of the quad-gather kernel: 512, 768 or 1024 (default)               */
    MI_OPT_GENERIC_SLAB_MB = 15,   /* quad-gather kernel: z slabs of the fixed volume sized so that a slab's share of
                                      the quad volume is at most this many MB (default 16; 0 = one slab)           */
    MI_INFO_NUM_SMS = 100,         /* multiprocessors of the context's device                                   */
    MI_INFO_BIN_MODE = 101,        /* binning variant in effect                                                 */
    MI_INFO_ZHIST_ROWS = 102,      /* fixed-bin ranks the z kernel counts in shared memory                      */
    MI_INFO_RARE_VOXELS = 103,     /* fixed voxels of the ranks that do not fit (0 = the epilogue can be fused) */
    MI_INFO_GENERIC_ROWS = 104,    /* fixed-bin ranks the generic kernel counts in shared memory                */
    MI_INFO_LAST_UPDATES_ISSUED = 106, /* shared-memory histogram updates the z kernel issued in the last call
                                      (-1 if the call did not take the separable path): evaluations minus the z
                                      slices that fall outside the moving volume                               */
    MI_INFO_QUADS_BUILT = 107,     /* bit 0: the float yz-quad copy of the moving volume exists (16 B per padded moving
                                      voxel; built by the first generic trilinear call with GENERIC_GATHER = 1, freed by
                                      GENERIC_GATHER = 0); bit 1: the bin-quad copy exists (4 B per padded voxel; first
                                      partial-volume call)                                                       */
    MI_INFO_LAST_PATH = 105        /* path of the last call: 0 generic, 1 separable, 2 wide-histogram, 3 partial-volume kernels */
} mi_option;
mi_status mi_set_option(mi_ctx *ctx, mi_option key, int64_t value);
mi_status mi_get_option(const mi_ctx *ctx, mi_option key, int64_t *value);

/* Restrict the metric to a subset of the fixed voxels (the random-sampling question of
 * "ITK Mattes uses a random sampling of the image ... while MICUDA uses all the voxels";
 * DESIGN.md A19).  mask: nx*ny*nz bytes in the fixed volume's layout, host or device, non-zero = the voxel
 * takes part; NULL restores all voxels.  The subset is an input (the caller draws it); it applies to every
 * later mi_eval_batch / mi_map / mi_multimetric_gradient of the context.  The mask is copied. */
mi_status mi_set_fixed_mask(mi_ctx *ctx, const uint8_t *mask);

/* Release the context.  Its device memory goes back to a library-level stream-ordered pool (one per
 * device) that keeps it cached for the next context -- the multi-GB scratch of a map is then not
 * mapped and unmapped by the driver on every create/destroy cycle.  NULL is a no-op. */
void mi_destroy(mi_ctx *ctx);

/* Return the memory cached by destroyed contexts on `device` to the driver.  Live contexts are not
 * affected.  MI_ERR_INVALID_ARG for a device that does not exist. */
mi_status mi_release_cached_memory(int32_t device);

/* Text of the last failure on this context (ctx != NULL) or of the last failed mi_create on this
 * thread (ctx == NULL).  The string is owned by the library and valid until the next call. */
const char *mi_last_error(const mi_ctx *ctx);

/* ---- multi-metric gradient ---------------------------------------------------
 * "we can use the same histogram to produce the Shannon and Tsallis results [so] the reasonable
 * strategy is to use multiple algorithms in the gradient descent ... the Tsallis in the translation
 * gradients and Shannon in the rotation and scale gradients".  The paper fixes
 * neither the parameterisation nor the difference rule; the reading (A18): nine parameters
 * p = (tx, ty, tz [mm], ax, ay, az [deg], sx, sy, sz [factors]), transform y = R(a) S(s) x + t with
 * R = Rz Ry Rx and S = diag(s) about the volume centre; component k is the central difference
 * (F_k(p + d_k e_k) - F_k(p - d_k e_k)) / (2 d_k), F_k = Tsallis MI of order q (the context's Tsallis
 * form) for k < 3 and Shannon MI for k >= 3.  All 2*9 + 1 transforms go through one mi_eval_batch,
 * one joint histogram each. */

/* Host side: physical 3x4 [A|t] of the nine parameters. */
mi_status mi_compose_matrix(const double p[9], double T_out[12]);

/* The hand-off "coarse exhaustive map -> gradient ascent" (an exhaustive search is the robust
 * way to start; then the multi-metric gradient): the nine parameters of the map node with
 * linear index `index` (an argmax_out of mi_map) on the grid (lo, hi, n) of `family`, identity in the other
 * parameter groups -- the p0 of mi_register.  Translation / Euler / scale nodes are copied, log-scale nodes
 * become factors exp(p), versor nodes the Euler angles of their rotation matrix.  Host pointers. */
mi_status mi_seed_from_map(mi_family family, const double lo[3], const double hi[3], const int32_t n[3],
                           int64_t index, double p_out[9]);

/* delta[k] <= 0 skips component k (grad_out[k] = 0).  grad_out: 9 doubles; value_out: NULL or 2
 * doubles (Shannon, Tsallis_q at p).  Host pointers; q > 0 and finite.
 * With MI_INTERP_PARTIAL_VOLUME the weights are quantised to 1/32 voxel per axis (A21), so MI is
 * piecewise constant in the transform and a finite difference needs a step the quantisation resolves:
 * every delta[k] > 0 must be at least mi_pv_min_delta's value for k, else MI_ERR_INVALID_ARG (the same
 * holds for mi_register).  NEAREST and TRILINEAR have no such bound. */
mi_status mi_multimetric_gradient(mi_ctx *ctx, const double p[9], const double delta[9], double q,
                                  mi_interp interp, double grad_out[9], double value_out[2]);

/* Smallest central-difference steps partial-volume interpolation resolves on this context's geometry, in the
 * units of p: [0..2] translation, moving spacing / 32 mm (one quantisation step of that moving axis);
 * [3..5] rotation in degrees and [6..8] scale factor, the change that moves a point at the reference radius
 * r = max(smallest fixed extent / 4, smallest fixed spacing) by one step of the coarsest moving axis, so that
 * every voxel farther than r from the centre moves at least one step.  Host pointer, 9 doubles. */
mi_status mi_pv_min_delta(const mi_ctx *ctx, double delta_min_out[9]);

/* The loop of the paper's Fig. 1 (Transform -> Metric -> Optimizer) around the
 * multi-metric gradient.  The paper names "gradient descent" and the strategy but prints no step rule;
 * the rule taken (A20) is regular-step gradient ascent per parameter group G (translation,
 * rotation, scale) with its own step length L_G (mm, degrees, factor):
 *     g = mi_multimetric_gradient(p);  d = g_G / |g_G|  (skipped when |g_G| == 0)
 *     if d . d_prev_G < 0: L_G = L_G / 2;   if L_G >= step_min[G]: p_G = p_G + L_G d
 * A group with step0[G] < step_min[G] (e.g. 0) never moves.  Stops when no group moved or after
 * max_iter iterations.  p_out: 9 doubles; trace_out: NULL or (max_iter + 1) x 9 doubles (the visited
 * p, row 0 = p0; rows beyond info.iterations are not written); info_out may be NULL.  Host pointers. */
typedef struct {
    int32_t iterations;       /* gradient evaluations made                                          */
    double steps[3];          /* final step lengths                                                 */
    double values[2];         /* (Shannon, Tsallis_q) at the last gradient evaluation               */
} mi_register_info;
mi_status mi_register(mi_ctx *ctx, const double p0[9], const double delta[9], const double step0[3],
                      const double step_min[3], int32_t max_iter, double q, mi_interp interp,
                      double p_out[9], double *trace_out, mi_register_info *info_out);

/* ---- capture-range analysis of a map ---------------------------------------
 * The paper reads its maps through "the paths the gradient descent algorithm will take" and the
 * regions "converging to the central point" or "to other points not related to our goal"
 * (Figs. 2-5).  It prints no algorithm for those paths (they were drawn by a
 * viewer), so the read-out is computed in its exact, parameter-free, discrete form (A17).
 * Both calls take ONE channel of a map: n[2] x n[1] x n[0] doubles, p0 fastest, host or device
 * memory, and work on `device` in `cuda_stream` (may be NULL); they return when their outputs are
 * complete.  n[0]*n[1]*n[2] must be < 2^31. */

/* Finite-difference gradient field in parameter units: grad_out is 3 x n[2] x n[1] x n[0] doubles
 * (component d = dM/dp_d), host or device.  Grid step h_d = (hi[d]-lo[d])/(n[d]-1); central
 * differences (M[k+1]-M[k-1])/(2 h_d) inside, one-sided (M[1]-M[0])/h_d and (M[n-1]-M[n-2])/h_d on
 * the faces; an axis with n[d] == 1 has gradient 0.  MI_ERR_INVALID_ARG if n[d] > 1 and
 * hi[d] == lo[d], or lo/hi are not finite. */
mi_status mi_map_gradient(const double *map, const int32_t n[3], const double lo[3], const double hi[3],
                          double *grad_out, int32_t device, void *cuda_stream);

typedef struct {
    int64_t n_extrema;        /* nodes that are their own best neighbour                            */
    int64_t target;           /* the node used as target (the argument, or the global extremum)     */
    int64_t target_label;     /* where the path from the target ends                                */
    int64_t captured;         /* nodes whose path ends at target_label                              */
    double capture_fraction;  /* captured / number of nodes                                         */
    int32_t max_steps;        /* longest path, in moves                                             */
    int32_t iterations;       /* pointer-doubling rounds the kernels took                           */
} mi_basin_stats;

/* Discrete steepest ascent (direction = +1, the arg max of eq. 3) or descent (direction = -1, "the
 * minimum value it can reach") on the parameter grid.  With v = direction * M, every
 * node steps to the neighbour (connectivity 6 or 26) with the largest v if that is strictly larger
 * than its own v -- ties between neighbours go to the lowest linear index -- until no neighbour is
 * better.  label_out (NULL or n[2] x n[1] x n[0] int64): linear index of the extremum reached;
 * steps_out (NULL or int32): moves taken.  target: linear index of the ground-truth node, or -1 for
 * the global extremum of v (lowest index on ties).  stats_out (host, may be NULL). */
mi_status mi_map_basins(const double *map, const int32_t n[3], int32_t direction, int32_t connectivity,
                        int64_t target, int64_t *label_out, int32_t *steps_out, mi_basin_stats *stats_out,
                        int32_t device, void *cuda_stream);

/* ---- host-side pieces of the path, exported so tests can check them without a GPU ------------ */

/* Step a2, family generator: parameter triple -> physical 3x4 [A|t] (double). */
mi_status mi_family_matrix(mi_family family, const double p[3], double T_out[12]);

/* Step a2, index-space composition (DESIGN.md CANON-1): physical [A|t] + the two geometries ->
 * fp32 3x4 [M|m0] with c = M i + m0 the continuous moving index of fixed voxel i. */
mi_status mi_index_affine(const double T[12], const int32_t fixed_dims[3], const double fixed_spacing[3],
                          const int32_t moving_dims[3], const double moving_spacing[3], float M_out[12]);

/* ---- introspection used by tests and the benchmark ------------------------------------------- */

/* Copy the pre-binned volumes out of the context (step a1 parity): which = 0 fixed, 1 moving;
 * out receives nx*ny*nz bin indices (host or device): uint8 for nbins <= 256, uint16 above. */
mi_status mi_get_bins(mi_ctx *ctx, int32_t which, void *out);

/* Device milliseconds (CUDA events on the context's stream) spent in the kernels of the last
 * mi_eval_batch / mi_map call: ms[0] transform upload + setup, ms[1] resample+histogram kernels,
 * ms[2] entropy kernels (0 when step a5 ran as the histogram kernel's epilogue), ms[3] map assembly +
 * arg max, ms[4] the dominant histogram kernel alone (z-lerp+histogram kernel of the separable path,
 * or the generic resample+histogram kernel; a part of ms[1]); launches[k] = kernels launched per
 * class (launches[4] is a subset of launches[1]). */
mi_status mi_last_timing(const mi_ctx *ctx, float ms[5], int64_t launches[5]);

/* Shared-memory atomic rate probe for the roofline: runs `iters` rounds of
 * atomicAdd(u32) into an nbins x nbins table in shared memory on every SM and reports
 * lane-updates per second.  pattern: 0 conflict-free (lane-distinct banks); 1 uniform random bins,
 * independent between the lanes of a warp (a hash of thread and update number) -- the roofline's
 * denominator; 2 all lanes on one address; 3 one linear congruential generator per thread seeded linearly in
 * the thread index (round 1's pattern: random in time, but the lanes of a warp form an arithmetic
 * progression, which spreads them over the banks more evenly than chance); 4 and 5 are patterns 2 and 1 with a
 * per-lane VALUE added instead of 1 (the weighted update of partial-volume interpolation); 6 is pattern 1's
 * statistics with the bins hashed once per thread BEFORE the timed loop (eight per thread, reused), so that no
 * integer arithmetic competes with the updates -- the probe that shows what the crossbar itself sustains
 * (pattern 1's hash costs about 5 % of it).  iters is rounded up to a multiple of 8.  Host pointers. */
mi_status mi_probe_shared_atomic_rate(int32_t device, int32_t nbins, int32_t pattern, int32_t iters,
                                      double *updates_per_s);

/* Gather-rate probe for the roofline of the generic (rotation) path: the resample+histogram kernel of
 * mi_eval_batch WITHOUT its histogram updates, run on the context's own volumes for the n physical
 * transforms T (n x 12 doubles, host) with the context's current options; reports fixed-voxel samples per
 * second (best of `reps` runs after one warm-up).  What it measures is the rate at which L1TEX delivers the
 * eight neighbours of every trilinear sample -- the term SURVEY.md 8(d) calls t_LSU -- for this data and these
 * angles; the full kernel adds one shared-memory update per sample on the same load/store pipe. */
mi_status mi_probe_gather_rate(mi_ctx *ctx, const double *T, int32_t n, int32_t reps, double *samples_per_s);

const char *mi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MI_B200_H */
