/* purify_wavelet.h - C ABI of the sparsity side of one ADMM iteration (f4): the wavelet dictionary
 * Psi / Psi^dagger and the Dual Forward-Backward inner iteration (arXiv 1903.04502, /root/reference/PAPER.md).
 *
 * What it computes
 *   dictionary  "a collection of wavelet bases (Dirac and Daubechies 1-8)", 3 levels: n_w = 9
 *               bases; alpha = [alpha_1 .. alpha_9] (Eq. 40); Psi alpha = sum_b Psi_b alpha_b (Eq. 41, no normalisation:
 *               Psi Psi^dagger = 9 I); Psi^dagger x = [Psi_b^dagger x]_b (Eq. 43).
 *   Psi_b       b = 0: Dirac (identity); b = 1..8: the periodic orthonormal two-channel filter bank with the
 *               b-vanishing-moment extremal-phase Daubechies low-pass filter h (2b taps), g[m] = (-1)^m h[2b-1-m],
 *               lo[k] = sum_m h[m] x[(2k+m) mod len], hi[k] = sum_m g[m] x[(2k+m) mod len]; along x, then along y;
 *               Mallat layout (low-low block in the top-left corner), `levels` times (reading W1).
 *   S_gamma     soft threshold of Eq. (24)-(26) on the complex modulus; P_C the projection onto the
 *               real non-negative images.
 *   DUALFB      Algorithm 1 lines 12-13 (reading W3 for the garbled line 13):
 *                   d    <- (1/eta) (I - S_gamma)(eta d + Psi^dagger zbar_prev)
 *                   zbar <- P_C(z - Psi d)
 * Conventions: images n x n complex interleaved, row-major, n a multiple of 2^levels; coefficients [9][n][n] complex,
 * basis-major; dtype as in purify_op.h (PURIFY_C64 = 0, PURIFY_C128 = 1); "_dev" pointers are device pointers; every
 * call is enqueued on `cuda_stream` and returns without synchronising; status codes are purify_status (purify_op.h),
 * detail in purify_last_error().  A handle owns its filters and scratch and is not re-entrant. */
#ifndef PURIFY_WAVELET_H
#define PURIFY_WAVELET_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct purify_wavelet purify_wavelet; /* opaque */

/* n even multiple of 2^levels, 1 <= levels <= 8; builds the eight Daubechies filters (spectral factorisation of
 * Daubechies' polynomial, long double, at create) and allocates 25 n^2 complex of scratch.  Synchronises. */
int purify_wavelet_create(purify_wavelet **out, int n, int levels, int dtype, void *cuda_stream);
int purify_wavelet_destroy(purify_wavelet *w);
/* filter of basis b = 1..8: writes its 2b low-pass taps to h_host (HOST, double); returns the number of taps or < 0 */
int purify_wavelet_filter(const purify_wavelet *w, int basis, double *h_host);
/* alpha = Psi^dagger x:  x_dev[n*n] -> alpha_dev[9*n*n]  (analysis) */
int purify_wavelet_adjoint(purify_wavelet *w, const void *x_dev, void *alpha_dev, void *cuda_stream);
/* x = Psi alpha:  alpha_dev[9*n*n] -> x_dev[n*n]  (synthesis and sum over the bases); alpha is not modified */
int purify_wavelet_forward(purify_wavelet *w, const void *alpha_dev, void *x_dev, void *cuda_stream);
/* one DUALFB pass (lines 12-13): z_dev, zbar_prev_dev: n*n (inputs); d_dev: 9*n*n, updated in place;
 * zbar_out_dev: n*n (may alias zbar_prev_dev).  gamma >= 0, eta > 0. */
int purify_dualfb_step(purify_wavelet *w, const void *z_dev, const void *zbar_prev_dev, void *d_dev, void *zbar_out_dev,
                       double gamma, double eta, void *cuda_stream);
/* zbar = P_C(z) (line 10) */
int purify_project_positive(purify_wavelet *w, const void *z_dev, void *zbar_dev, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* PURIFY_WAVELET_H */
