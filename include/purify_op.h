/* purify_op.h - C ABI of the B200-native measurement operator  Phi = W G F Z S  and its adjoint.
 *
 * What it computes (arXiv 1903.04502, /root/reference/PAPER.md):
 *   Eq. (2):  y = W G F Z S x  with S the gridding correction, Z zero padding
 *   (oversampling factor 2), F a 2-D FFT on the K x K oversampled grid (K = 2n), G the
 *   Kaiser-Bessel degridding onto M visibilities at continuous (u, v), W the noise weights;
 *   the adjoint Phi^dagger "consists of applying these operators in reverse"
 *   (S^dagger Z^dagger F^dagger G^dagger W^dagger).  Phi and Phi^dagger are applied once each per
 *   ADMM iteration (Algorithm 1 lines 3 and 6).  The interpolation matrix G is
 *   never stored (the thing PAPER.md:580-592 "Kernel Pre-Sampling" gets rid of): kernel weights are
 *   evaluated on the fly (ANALYTIC) or read from the paper's pre-sampled table (TABLE).
 *   Exact definitions, including every reading taken where the paper is silent: DESIGN.md.
 *
 * Conventions
 *   image   x[py*n + px], interleaved complex (re, im), px fastest; px <-> u, py <-> v; the pixel
 *           (n/2, n/2) is the phase centre.  n even.
 *   (u, v)  uv[k][0] = u_k, uv[k][1] = v_k in OVERSAMPLED-GRID CELLS, DC at 0, period K = 2n
 *           (paper's radians/pixel omega: u = omega K / 2 pi).  Any finite value with
 *           |u| < 2^30 is accepted and taken mod K.
 *   dtype   PURIFY_C64 : x, y complex64,  uv and w float32.   PURIFY_C128: complex128 / float64.
 *   order   "caller order" = the order of uv at create.  "native order" = the library's own order, a
 *           vector of M_native >= M entries (purify_op_info): native[i] = caller[perm[i]] with perm
 *           from purify_op_permutation(); perm[i] = 0xFFFFFFFF marks a PADDING entry (batched
 *           layout only): purify_degrid_native writes 0 there, purify_grid_native ignores it.
 *   memory  "_dev" pointers are CUDA device pointers on the current device, "_host" pointers are
 *           host pointers (pinned memory recommended).  The caller owns every buffer it passes; the
 *           handle owns its sorted copies, tables, grid workspace and cuFFT plan.
 *   stream  `cuda_stream` is a cudaStream_t cast to void* (NULL = legacy default stream).  All work
 *           is enqueued on it; only purify_op_create*, the *_host calls (they return after the
 *           result is in host memory) and purify_stage_times_ms synchronise.
 *   errors  every function returns a purify_status (0 = OK, < 0 = error); nothing throws, aborts or
 *           prints.  purify_last_error() gives a thread-local detail string for the last failure.
 *   thread  a handle is NOT re-entrant: it owns one grid workspace, one work queue and one set of lazily allocated
 *           vectors, so two calls on the same handle must not overlap - neither from two host threads nor on two
 *           streams (calls on ONE stream are ordered and fine).  Distinct handles are independent.
 *   determinism  degrid is bit-reproducible.  grid/normal flush partial tiles with floating-point
 *           atomics, so the last bits of the gridded image may vary from call to call.
 */
#ifndef PURIFY_OP_H
#define PURIFY_OP_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct purify_op purify_op; /* opaque */

typedef enum { PURIFY_C64 = 0, PURIFY_C128 = 1 } purify_dtype;
typedef enum { PURIFY_KERNEL_ANALYTIC = 0, PURIFY_KERNEL_TABLE = 1 } purify_kernel_mode;

typedef enum {
    PURIFY_OK = 0,
    PURIFY_ERR_INVALID_ARG = -1, /* NULL pointer, n odd or <= 0, M < 0 or >= 2^31, J not in {4,6,8} */
    PURIFY_ERR_UNSUPPORTED = -2, /* oversample != 2, unknown dtype / kernel mode                    */
    PURIFY_ERR_UV_NONFINITE = -3,/* a NaN / Inf / |u| >= 2^30 coordinate was found at create        */
    PURIFY_ERR_ALLOC = -4,       /* device or host allocation failed                                 */
    PURIFY_ERR_CUDA = -5,        /* a CUDA runtime / driver call failed (detail in last_error)       */
    PURIFY_ERR_CUFFT = -6,       /* a cuFFT call failed                                              */
    PURIFY_ERR_NO_DEVICE = -7    /* no CUDA device: there is NO CPU fallback                         */
} purify_status;

/* Options; pass NULL for defaults.  Zero in any field means "default". */
typedef struct {
    int kernel_mode;            /* purify_kernel_mode; default ANALYTIC                              */
    int table_samples_per_unit; /* TABLE mode: samples per grid cell R; default 4096
                                   (BASELINE.json configs[4]); paper used 2e5.
                                   T[i] = g(i/R), i = 0..R*J/2+1, lookup T[floor(|d| R + 1/2)].      */
    int chunk;                  /* complex128 (tile-sorted layout): visibilities per work item (CTA); default 4096.
                                   Ignored by the batched layout (items of 64 iterations x 32 lanes)        */
    int time_stages;            /* != 0: record CUDA events around each stage (also switchable later:
                                   purify_op_set_time_stages); while it is on, purify_normal is not replayed
                                   from its CUDA graph                                                        */
    int admm_unfused;           /* != 0: purify_admm_fidelity_step runs its unfused form (separate norm and update
                                   kernels) even where the fused kernels exist                                */
    int force_tile_sorted;      /* != 0: complex128 uses the tile-sorted kernels for every J (default: batched
                                   layout for J <= 6, tile-sorted for J = 8)                                   */
    int reserved[2];            /* must be 0                                                                   */
} purify_opts;

/* Facts about a handle (for tests, benches and roofline arithmetic). */
typedef struct {
    int n, K, J, dtype, kernel_mode, table_samples_per_unit;
    long long M;
    int tile;                   /* tile side T in grid cells                                         */
    int n_tiles;                /* tiles on the K x K grid                                           */
    int n_tiles_nonempty;
    int n_items;                /* work items (tile chunks) = CTAs per degrid / grid launch          */
    int poly_degree;            /* ANALYTIC: degree of the per-tap polynomial in the cell offset     */
    double poly_max_abs_err;    /* ANALYTIC: max |poly - g| over the support (fit check at create)   */
    long long device_bytes;     /* device memory owned by the handle                                 */
    long long max_tile_count;   /* visibilities in the fullest tile / band                           */
    long long M_native;         /* length of a native-order y vector (>= M: the batched layout pads)   */
    long long n_batches;        /* batched layout: batches of 32 cell-units                          */
    int layout;                 /* 0 = tile-sorted (complex128, J = 8), 1 = batched cell-stationary (complex64; complex128, J <= 6) */
    int tile_h;                 /* tile / band height in grid cells (tile = width)                   */
} purify_info;

/* Stage indices for purify_stage_times_ms (milliseconds of the LAST call that ran the stage). */
enum { PURIFY_STAGE_PAD = 0,   /* S + Z fused */
       PURIFY_STAGE_FFT = 1,   /* F, cuFFT                         (a2)                */
       PURIFY_STAGE_DEGRID = 2,/* W G                              (a3)                */
       PURIFY_STAGE_GRID = 3,  /* G^dagger W^dagger kernel         (a4)                */
       PURIFY_STAGE_IFFT = 4,  /* F^dagger, cuFFT                  (a5)                */
       PURIFY_STAGE_CROP = 5,  /* Z^dagger S^dagger fused          (a6)                */
       PURIFY_STAGE_PERMUTE = 6,
       PURIFY_STAGE_ZERO = 7,  /* zeroing of the grid before a4 (cudaMemsetAsync)      */
       PURIFY_STAGE_COUNT = 8 };

/* a0: build an operator for an n x n image, K = oversample*n, J-tap Kaiser-Bessel
 * kernel (beta = 2.34 J) and M visibilities.  uv_dev: [M][2] (u, v); w_dev: [M] real weights or NULL
 * (=> 1).  Copies uv and w (the caller may free them when this returns), bins the visibilities by
 * grid tile (device radix sort on tile/cell id, once), builds the correction vector, the kernel
 * polynomial or table and the cuFFT plan.  Synchronises the stream.  On error *out = NULL.         */
int purify_op_create(purify_op **out, int n, int oversample, int J, long long M,
                     const void *uv_dev, const void *w_dev, int dtype,
                     const purify_opts *opts, void *cuda_stream);
/* Same with uv / w in host memory. */
int purify_op_create_host(purify_op **out, int n, int oversample, int J, long long M,
                          const void *uv_host, const void *w_host, int dtype,
                          const purify_opts *opts, void *cuda_stream);
int purify_op_destroy(purify_op *op);
int purify_op_info(const purify_op *op, purify_info *info);
/* perm_dev[i] = caller index of the visibility at native position i, or 0xFFFFFFFF for padding
 * (device pointer, M_native entries). */
int purify_op_permutation(const purify_op *op, const unsigned **perm_dev);

/* Phi (a1-a3):  x_dev[n*n] -> y_dev[M], caller order. */
int purify_degrid(purify_op *op, const void *x_dev, void *y_dev, void *cuda_stream);
/* Phi^dagger (a4-a6):  y_dev[M] (caller order) -> x_dev[n*n]. */
int purify_grid(purify_op *op, const void *y_dev, void *x_dev, void *cuda_stream);
/* Phi^dagger Phi (a7): x_in_dev -> x_out_dev (may alias); y stays in the handle's workspace. */
int purify_normal(purify_op *op, const void *x_in_dev, void *x_out_dev, void *cuda_stream);

/* Same operators with y in NATIVE order (moves only the minimum bytes; an ADMM loop can keep all
 * its M-sized vectors in this order after one purify_permute_to_native of the data).  Native vectors have
 * M_native entries (purify_op_info); for PURIFY_C64 the y_native pointer given to purify_grid_native must be
 * 16-byte aligned (INVALID_ARG otherwise: the kernel streams it with bulk copies). */
int purify_degrid_native(purify_op *op, const void *x_dev, void *y_native_dev, void *cuda_stream);
int purify_grid_native(purify_op *op, const void *y_native_dev, void *x_dev, void *cuda_stream);
/* The permutation passes on their own (also what purify_degrid / purify_grid run after / before the native kernels).
 * Input and output must not overlap.  From 2^24 visibilities on the permutation is routed in three coalesced passes
 * (blocks permuted in shared memory, runs of consecutive elements written: native order -> grouped by ranges of the
 * caller index -> grouped by caller tiles of 4096 -> caller order; index arrays built at create) and the handle
 * lazily allocates M (from native) or 2 M (to native) complex entries of workspace; below, one gather. */
int purify_permute_to_native(purify_op *op, const void *y_caller_dev, void *y_native_dev, void *cuda_stream);
int purify_permute_from_native(purify_op *op, const void *y_native_dev, void *y_caller_dev, void *cuda_stream);

/* Host-buffer entry points (end-to-end path): copy in, run, copy out, synchronise. */
int purify_degrid_host(purify_op *op, const void *x_host, void *y_host, void *cuda_stream);
int purify_grid_host(purify_op *op, const void *y_host, void *x_host, void *cuda_stream);
int purify_normal_host(purify_op *op, const void *x_in_host, void *x_out_host, void *cuda_stream);

/* f3: the distributed-image operator - "each node has a replica of the image and its own section of
 * the visibilities": Phi_j needs no exchange (Eq. 37), x' = sum_j Phi_j^dagger y_j is an all-reduce
 * of the n x n image (Eq. 38; Algorithm 2 "AllSumAll").  The exchange is the CALLER's: these two
 * calls run Phi_j^dagger (resp. Phi_j^dagger Phi_j) and hand the image to `allreduce` in `bands` horizontal bands
 * (rows [n k / bands, n (k+1) / bands)) as each leaves the crop kernel, so that band k is reduced while band k + 1 is
 * cropped; when the call returns, work enqueued on cuda_stream afterwards sees the reduced image.
 *   allreduce(user, band_dev, count_reals, is_double, comm_stream) must ENQUEUE an in-place sum over the ranks of the
 *   count_reals floats (is_double = 0) or doubles at band_dev onto comm_stream (a stream owned by the handle, already
 *   ordered after the band's crop) and return 0; e.g. ncclAllReduce(band_dev, band_dev, count_reals, ncclFloat,
 *   ncclSum, comm, comm_stream).  allreduce = NULL: a single process, no exchange.  y in native order (M_native). */
typedef int (*purify_allreduce_fn)(void *user, void *band_dev, long long count_reals, int is_double, void *comm_stream);
int purify_grid_dist(purify_op *op, const void *y_native_dev, void *x_dev, int bands,
                     purify_allreduce_fn allreduce, void *user, void *cuda_stream);
int purify_normal_dist(purify_op *op, const void *x_in_dev, void *x_out_dev, int bands,
                       purify_allreduce_fn allreduce, void *user, void *cuda_stream);

/* f2: largest eigenvalue of Phi^dagger Phi = ||Phi||^2 by the power method ("We can normalize the
 * operator with the operator norm, by using the power method to estimate the largest eigenvalue").
 * x_1 = x0 / ||x0||; z_k = Phi^dagger Phi x_k; lambda_k = ||z_k||_2; x_{k+1} = z_k / lambda_k; stops after max_iter
 * iterations or when |lambda_k - lambda_{k-1}| <= rel_tol lambda_k (k >= 2; rel_tol = 0: run max_iter iterations).
 * x0_dev: n*n complex start vector on the device, or NULL for all ones.  Norms are accumulated in fp64.
 * lambda_out, iters_out: HOST pointers (iters_out may be NULL).  Synchronises the stream every iteration. */
int purify_op_norm(purify_op *op, const void *x0_dev, int max_iter, double rel_tol, double *lambda_out, int *iters_out,
                   void *cuda_stream);

/* f1: the data-fidelity half of one ADMM iteration around the operator - Algorithm 1 lines 3-6
 * with the l2-ball projection of Eq. (23):
 *     v = Phi x;   r = P_B(v + s), B = { z : ||z - y||_2 <= epsilon };   s <- s + varrho (v - r);
 *     g = Phi^dagger (v - r + s)          (the caller then forms x~ = x - rho g, line 6).
 * y_native_dev (measurements) and s_native_dev (dual variable, updated in place) are NATIVE-order vectors of M_native
 * entries (bring the data there once with purify_permute_to_native; padding entries are ignored and s is written as 0
 * there).  g_dev: n*n complex, device.  resid_norm_out: HOST pointer that receives ||v + s_old - y||_2 (may be NULL;
 * if given the call synchronises the stream).  epsilon >= 0.  PURIFY_C64 + ANALYTIC weights run fused: the norm is
 * accumulated inside the degridding kernel and r, s_new and v - r + s_new are formed inside the gridding kernel (the
 * vector handed to Phi^dagger is never stored); y_native and s_native must then be 16-byte aligned.  Other
 * configurations use separate norm / update kernels. */
int purify_admm_fidelity_step(purify_op *op, const void *x_dev, const void *y_native_dev, void *s_native_dev,
                              double epsilon, double varrho, void *g_dev, double *resid_norm_out, void *cuda_stream);

/* Stage access for tests (device pointers): the K x K Fourier grid workspace in the library's
 * internal layout is NOT exposed; these run single stages into caller buffers in the mathematical
 * layout B[ky*K + kx], ky, kx in [0, K) (DC at index 0), so they can be compared with the oracle. */
int purify_stage_fourier_grid(purify_op *op, const void *x_dev, void *B_dev /* K*K complex */, void *cuda_stream);
int purify_stage_gridded(purify_op *op, const void *y_dev /* caller order */, void *B_dev, void *cuda_stream);

/* Milliseconds per stage of the last call (needs stage timing switched on); synchronises. */
int purify_stage_times_ms(const purify_op *op, float out[PURIFY_STAGE_COUNT]);
/* Switch the per-stage CUDA events on (enable != 0) or off for the calls that follow. */
int purify_op_set_time_stages(purify_op *op, int enable);
/* Number of kernels of this library (cuFFT launches not counted) enqueued by the last call. */
int purify_last_launch_count(const purify_op *op);

/* Measurement aid: issue rate of the packed fp32 instruction forms the hot kernels consist of, on the
 * current device.  form 0: 2 x FFMA (3 registers); 1: FFMA2 broadcast scalar x pair + pair (degridding row pass);
 * 2: FFMA2 pair x pair + pair; 3: FFMA2 pair x pair + constant (Horner step); 4: FFMA2 varying scalar x shared pair +
 * pair (gridding).  warps_per_sm in {4, 8, ..., 32}.  *cycles_per_instr_out (HOST): SM cycles per warp instruction per
 * SM sub-partition, from clock64() inside the kernel; *sm_ghz_out (HOST, may be NULL): cycles / event time.
 * Allocates and frees its own scratch, uses the legacy default stream and synchronises. */
int purify_ubench_fma(int form, int warps_per_sm, double *cycles_per_instr_out, double *sm_ghz_out);

const char *purify_strerror(int status);
const char *purify_last_error(void);
int purify_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PURIFY_OP_H */
