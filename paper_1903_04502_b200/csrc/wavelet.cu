// f4: the wavelet dictionary Psi / Psi^dagger (Dirac + Daubechies 1-8, periodic, Mallat layout) and
// one Dual Forward-Backward pass (Algorithm 1 lines 12-13) - C ABI of include/purify_wavelet.h, sm_100a.
// HBM-bound stencils: every pass streams its arrays once with coalesced accesses along x; the eight wavelet bases
// are batched in one launch (blockIdx.z); the last synthesis pass sums the nine bases and applies the epilogue
// (plain store, or P_C(z - .)) so that Psi d is never stored.  Filters: own spectral factorisation (Durand-Kerner +
// Newton in long double) - shares nothing with oracle/.
#include "../../include/purify_op.h"
#include "../../include/purify_wavelet.h"

#include <cuda_runtime.h>

#include <cmath>
#include <complex>
#include <cstdarg>
#include <cstdio>
#include <new>
#include <vector>

extern "C" const char* purify_last_error(void);
namespace pkerr { int set(int status, const char* fmt, ...); }      // purify_op.cu: the thread-local detail string

namespace {

constexpr int NB = 8;           // wavelet bases proper (Daubechies 1..8); basis 0 of the dictionary is the Dirac basis
constexpr int LMAX = 16;        // longest filter

template <typename R> struct C2T;
template <> struct C2T<float> { typedef float2 type; };
template <> struct C2T<double> { typedef double2 type; };

struct Filters { int len[NB]; };                          // taps live in device memory: filt[(b * 2 + {0: h, 1: g}) * LMAX + m]

// periodic index: i is at most a filter length outside [0, m) (no integer division in the tap loops)
__device__ __forceinline__ int wrap_nonneg(int i, int m) { while (i >= m) i -= m; return i; }
__device__ __forceinline__ int wrap_any(int i, int m) { while (i < 0) i += m; while (i >= m) i -= m; return i; }

// The per-level kernels below are templated on the filter length L (a switch on the basis picks the instantiation),
// so that the tap loops unroll and every thread produces several outputs from one sliding window of inputs:
// KPT low / high pairs (analysis) or 2 KPT samples (synthesis) per thread - about (2 KPT + L) loads instead of KPT L.
constexpr int KPT = 4;

#define WL_SWITCH_L(b, CALL)                    \
    switch (b) {                                \
        case 0: { constexpr int L = 2; CALL; } break;   \
        case 1: { constexpr int L = 4; CALL; } break;   \
        case 2: { constexpr int L = 6; CALL; } break;   \
        case 3: { constexpr int L = 8; CALL; } break;   \
        case 4: { constexpr int L = 10; CALL; } break;  \
        case 5: { constexpr int L = 12; CALL; } break;  \
        case 6: { constexpr int L = 14; CALL; } break;  \
        default: { constexpr int L = 16; CALL; } break; \
    }

// ---- the analysis pass along x goes through shared memory: a CTA of 128 threads takes ROW_SPAN outputs of one row,
// stages the inputs they need with coalesced loads, split into even and odd samples so that the stride-2 reads of
// neighbouring outputs become unit-stride, and every thread then produces outputs 128 apart: coalesced stores.
constexpr int ROW_SPAN = 512;           // low / high pairs per CTA

template <typename R, int L>
__device__ __forceinline__ void row_fwd_body(const typename C2T<R>::type* __restrict__ s, typename C2T<R>::type* __restrict__ t,
                                             int m, int kb, const R* __restrict__ h, const R* __restrict__ g,
                                             typename C2T<R>::type* ev, typename C2T<R>::type* od) {
    typedef typename C2T<R>::type C;
    const int mh = m >> 1, cnt = min(ROW_SPAN, mh - kb), span = 2 * cnt + L - 2;
    for (int e = threadIdx.x; e < span; e += 128) {
        const C v = s[wrap_nonneg(2 * kb + e, m)];
        if (e & 1) od[e >> 1] = v; else ev[e >> 1] = v;
    }
    __syncthreads();
    for (int q = threadIdx.x; q < cnt; q += 128) {
        R lx = 0, ly = 0, hx = 0, hy = 0;
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const C v = (i & 1) ? od[q + (i >> 1)] : ev[q + (i >> 1)];
            lx += h[i] * v.x; ly += h[i] * v.y; hx += g[i] * v.x; hy += g[i] * v.y;
        }
        C lo; lo.x = lx; lo.y = ly;
        C hi; hi.x = hx; hi.y = hy;
        t[kb + q] = lo;
        t[mh + kb + q] = hi;
    }
}

template <typename R>
__global__ void __launch_bounds__(128) wl_row_fwd(const typename C2T<R>::type* __restrict__ src, long long src_stride, int pitch,
                                                  typename C2T<R>::type* __restrict__ tmp, long long tmp_stride, int n, int m,
                                                  const R* __restrict__ filt) {
    typedef typename C2T<R>::type C;
    __shared__ C ev[ROW_SPAN + LMAX / 2], od[ROW_SPAN + LMAX / 2];
    const int kb = blockIdx.x * ROW_SPAN, r = blockIdx.y, b = blockIdx.z;
    const C* s = src + (long long)b * src_stride + (long long)r * pitch;
    C* t = tmp + (long long)b * tmp_stride + (long long)r * n;
    const R* h = filt + (b * 2) * LMAX;
    const R* g = h + LMAX;
    WL_SWITCH_L(b, (row_fwd_body<R, L>(s, t, m, kb, h, g, ev, od)))
}

// ---- analysis along y: tmp[b] (m x m block) -> dst[b] top-left m x m block (rows [0, m/2) low, [m/2, m) high).
// Thread = one column, KPT consecutive output rows; loads coalesced across the columns.
template <typename R, int L>
__device__ __forceinline__ void col_fwd_body(const typename C2T<R>::type* __restrict__ t, typename C2T<R>::type* __restrict__ d,
                                             int n, int m, int k0, const R* __restrict__ h, const R* __restrict__ g) {
    typedef typename C2T<R>::type C;
    const int mh = m >> 1;
    R lx[KPT], ly[KPT], hx[KPT], hy[KPT];
#pragma unroll
    for (int q = 0; q < KPT; ++q) lx[q] = ly[q] = hx[q] = hy[q] = (R)0;
    int idx = wrap_nonneg(2 * k0, m);
#pragma unroll
    for (int r = 0; r < 2 * KPT + L - 2; ++r) {
        const C v = t[(long long)idx * n];
        if (++idx == m) idx = 0;
#pragma unroll
        for (int q = 0; q < KPT; ++q) {
            const int i = r - 2 * q;
            if (i >= 0 && i < L) { lx[q] += h[i] * v.x; ly[q] += h[i] * v.y; hx[q] += g[i] * v.x; hy[q] += g[i] * v.y; }
        }
    }
#pragma unroll
    for (int q = 0; q < KPT; ++q)
        if (k0 + q < mh) {
            C lo; lo.x = lx[q]; lo.y = ly[q];
            C hi; hi.x = hx[q]; hi.y = hy[q];
            d[(long long)(k0 + q) * n] = lo;
            d[(long long)(mh + k0 + q) * n] = hi;
        }
}

template <typename R>
__global__ void __launch_bounds__(128) wl_col_fwd(const typename C2T<R>::type* __restrict__ tmp, long long tmp_stride,
                                                  typename C2T<R>::type* __restrict__ dst, long long dst_stride, int n, int m,
                                                  const R* __restrict__ filt) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x, k0 = blockIdx.y * KPT, b = blockIdx.z;
    if (c >= m) return;
    const auto* t = tmp + (long long)b * tmp_stride + c;
    auto* d = dst + (long long)b * dst_stride + c;
    const R* h = filt + (b * 2) * LMAX;
    const R* g = h + LMAX;
    WL_SWITCH_L(b, (col_fwd_body<R, L>(t, d, n, m, k0, h, g)))
}

// ---- synthesis, one axis: 2 KPT consecutive samples j0 .. j0 + 2 KPT - 1 (j0 even) from the low / high coefficients
// kk = kmin .. kmin + KPT + L/2 - 2, kmin = (j0 - (L - 2)) / 2:  out[j0 + jj] = sum h[i] lo[kk] + g[i] hi[kk], i = jj - 2 kr + L - 2
template <typename R, int L, typename LoadLo, typename LoadHi, typename Store>
__device__ __forceinline__ void inv_body(int mh, int j0, const R* __restrict__ h, const R* __restrict__ g, LoadLo load_lo, LoadHi load_hi,
                                         Store store) {
    typedef typename C2T<R>::type C;
    R ax[2 * KPT], ay[2 * KPT];
#pragma unroll
    for (int jj = 0; jj < 2 * KPT; ++jj) ax[jj] = ay[jj] = (R)0;
    int kk = wrap_any((j0 - (L - 2)) / 2, mh);                 // (j0 - L + 2 is even; C division of a negative even number is exact)
#pragma unroll
    for (int kr = 0; kr < KPT + L / 2 - 1; ++kr) {
        const C lo = load_lo(kk), hi = load_hi(kk);
        if (++kk == mh) kk = 0;
#pragma unroll
        for (int jj = 0; jj < 2 * KPT; ++jj) {
            const int i = jj - 2 * kr + (L - 2);
            if (i >= 0 && i < L) { ax[jj] += h[i] * lo.x + g[i] * hi.x; ay[jj] += h[i] * lo.y + g[i] * hi.y; }
        }
    }
#pragma unroll
    for (int jj = 0; jj < 2 * KPT; ++jj) { C o; o.x = ax[jj]; o.y = ay[jj]; store(jj, o); }
}

// ---- synthesis along y: the m x m block whose low-low quadrant comes from `ll` (the level below, already synthesised)
// and whose other three quadrants come from `det` (the coefficients) -> tmp[b] rows j < m.  Thread = one column.
template <typename R>
__global__ void __launch_bounds__(128) wl_col_inv(const typename C2T<R>::type* __restrict__ ll, long long ll_stride,
                                                  const typename C2T<R>::type* __restrict__ det, long long det_stride,
                                                  typename C2T<R>::type* __restrict__ tmp, long long tmp_stride, int n, int m,
                                                  const R* __restrict__ filt) {
    typedef typename C2T<R>::type C;
    const int c = blockIdx.x * blockDim.x + threadIdx.x, j0 = blockIdx.y * 2 * KPT, b = blockIdx.z, mh = m >> 1;
    if (c >= m) return;
    const C* lo_src = (c < mh ? ll + (long long)b * ll_stride : det + (long long)b * det_stride) + c;     // rows [0, m/2)
    const C* hi_src = det + (long long)b * det_stride + (long long)mh * n + c;                          // rows [m/2, m)
    C* out = tmp + (long long)b * tmp_stride + c;
    const R* h = filt + (b * 2) * LMAX;
    const R* g = h + LMAX;
    auto load_lo = [&](int kk) { return lo_src[(long long)kk * n]; };
    auto load_hi = [&](int kk) { return hi_src[(long long)kk * n]; };
    auto store = [&](int jj, C o) { if (j0 + jj < m) out[(long long)(j0 + jj) * n] = o; };
    WL_SWITCH_L(b, (inv_body<R, L>(mh, j0, h, g, load_lo, load_hi, store)))
}

// ---- synthesis along x: tmp[b] (m x m block) -> out[b] (m x m block).  Thread = 2 KPT consecutive samples of one row
// (the shared-memory staging that pays for the analysis was measured slower here: 0.58 vs 0.31 ms for Psi at n = 2048).
template <typename R>
__global__ void __launch_bounds__(128) wl_row_inv(const typename C2T<R>::type* __restrict__ tmp, long long tmp_stride,
                                                  typename C2T<R>::type* __restrict__ out, long long out_stride, int n, int m,
                                                  const R* __restrict__ filt) {
    typedef typename C2T<R>::type C;
    const int j0 = (blockIdx.x * blockDim.x + threadIdx.x) * 2 * KPT, r = blockIdx.y, b = blockIdx.z, mh = m >> 1;
    if (j0 >= m) return;
    const C* t = tmp + (long long)b * tmp_stride + (long long)r * n;
    C* o_ = out + (long long)b * out_stride + (long long)r * n;
    const R* h = filt + (b * 2) * LMAX;
    const R* g = h + LMAX;
    auto load_lo = [&](int kk) { return t[kk]; };
    auto load_hi = [&](int kk) { return t[mh + kk]; };
    auto store = [&](int jj, C o) { if (j0 + jj < m) o_[j0 + jj] = o; };
    WL_SWITCH_L(b, (inv_body<R, L>(mh, j0, h, g, load_lo, load_hi, store)))
}

// ---- last synthesis pass (level 0, along x) of all eight bases + the Dirac coefficients, summed (Eq. 41), with the
// epilogue: MODE 0: x = sum; MODE 1: zbar = P_C(z - sum) (Algorithm 1 line 13).  Thread = 2 KPT consecutive samples.
template <typename R, int MODE>
__global__ void __launch_bounds__(128) wl_row_inv_sum(const typename C2T<R>::type* __restrict__ tmp, long long tmp_stride,
                                                      const typename C2T<R>::type* __restrict__ dirac,
                                                      const typename C2T<R>::type* __restrict__ z,
                                                      typename C2T<R>::type* __restrict__ out, int n,
                                                      const R* __restrict__ filt) {
    typedef typename C2T<R>::type C;
    const int j0 = (blockIdx.x * blockDim.x + threadIdx.x) * 2 * KPT, r = blockIdx.y, mh = n >> 1;
    if (j0 >= n) return;
    R sx[2 * KPT], sy[2 * KPT];
#pragma unroll
    for (int jj = 0; jj < 2 * KPT; ++jj) {
        sx[jj] = sy[jj] = (R)0;
        if (j0 + jj < n) { const C d0 = dirac[(long long)r * n + j0 + jj]; sx[jj] = d0.x; sy[jj] = d0.y; }
    }
    auto store = [&](int jj, C o) { sx[jj] += o.x; sy[jj] += o.y; };
#pragma unroll 1
    for (int b = 0; b < NB; ++b) {
        const C* t = tmp + (long long)b * tmp_stride + (long long)r * n;
        const R* h = filt + (b * 2) * LMAX;
        const R* g = h + LMAX;
        auto load_lo = [&](int kk) { return t[kk]; };
        auto load_hi = [&](int kk) { return t[mh + kk]; };
        WL_SWITCH_L(b, (inv_body<R, L>(mh, j0, h, g, load_lo, load_hi, store)))
    }
#pragma unroll
    for (int jj = 0; jj < 2 * KPT; ++jj)
        if (j0 + jj < n) {
            C o;
            if (MODE == 0) { o.x = sx[jj]; o.y = sy[jj]; }
            else { const C zz = z[(long long)r * n + j0 + jj]; const R v = zz.x - sx[jj]; o.x = v > (R)0 ? v : (R)0; o.y = (R)0; }
            out[(long long)r * n + j0 + jj] = o;
        }
}

// ---- d <- (1/eta) (I - S_gamma)(eta d + a)   (Algorithm 1 line 12; Eq. 26 on the complex modulus)
template <typename R>
__global__ void __launch_bounds__(256) dual_update_kernel(typename C2T<R>::type* __restrict__ d, const typename C2T<R>::type* __restrict__ a,
                                                          long long count, R gamma, R eta) {
    typedef typename C2T<R>::type C;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        const C dv = d[i], av = a[i];
        const R ux = eta * dv.x + av.x, uy = eta * dv.y + av.y;
        const R mod = sqrt(ux * ux + uy * uy);
        // u - S_gamma(u) = u where |u| <= gamma, u gamma / |u| elsewhere
        const R f = mod > gamma ? gamma / mod : (R)1;
        C o; o.x = ux * f / eta; o.y = uy * f / eta;
        d[i] = o;
    }
}

template <typename R>
__global__ void __launch_bounds__(256) project_positive_kernel(const typename C2T<R>::type* __restrict__ z,
                                                               typename C2T<R>::type* __restrict__ o, long long count) {
    typedef typename C2T<R>::type C;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        C v; v.x = z[i].x > (R)0 ? z[i].x : (R)0; v.y = (R)0;
        o[i] = v;
    }
}

// ---------------------------------------------------------------- host: Daubechies filters (reading W1)
typedef long double ld;
typedef std::complex<ld> cld;

// low-pass filter with N vanishing moments, extremal phase: H(q) = sqrt2 ((1+q)/2)^N L(q), L(q) L(1/q) = P((2-q-1/q)/4),
// P(y) = sum_{k<N} C(N-1+k, k) y^k; L collects, for every root y_k of P, the zero of z^2 - (2 - 4 y_k) z + 1 inside the circle.
void daubechies(int N, std::vector<double>& h) {
    h.assign(2 * N, 0.0);
    if (N == 1) { h[0] = h[1] = (double)(1 / sqrtl(2.0L)); return; }
    std::vector<ld> P(N);
    P[0] = 1;
    for (int k = 1; k < N; ++k) P[k] = P[k - 1] * (ld)(N - 1 + k) / (ld)k;
    auto eval = [&](cld y) { cld v = 0; for (int k = N - 1; k >= 0; --k) v = v * y + P[k]; return v; };
    auto deriv = [&](cld y) { cld v = 0; for (int k = N - 1; k >= 1; --k) v = v * y + P[k] * (ld)k; return v; };
    const int D = N - 1;
    std::vector<cld> y(D);
    for (int j = 0; j < D; ++j) y[j] = std::pow(cld(0.4L, 0.9L), (ld)j) * (ld)0.7;       // Durand-Kerner start values
    for (int it = 0; it < 2000; ++it) {
        ld move = 0;
        for (int j = 0; j < D; ++j) {
            cld den = P[D];
            for (int i = 0; i < D; ++i) if (i != j) den *= (y[j] - y[i]);
            const cld step = eval(y[j]) / den;
            y[j] -= step;
            move = fmaxl(move, std::abs(step));
        }
        if (move < 1e-19L) break;
    }
    for (int it = 0; it < 6; ++it)                                                        // Newton polish
        for (int j = 0; j < D; ++j) y[j] -= eval(y[j]) / deriv(y[j]);
    std::vector<cld> L(1, cld(1, 0));
    for (int j = 0; j < D; ++j) {
        const cld b = (ld)2 - (ld)4 * y[j], disc = std::sqrt(b * b - (ld)4);
        const cld z1 = (b + disc) / (ld)2, z2 = (b - disc) / (ld)2;
        const cld zk = std::abs(z1) < 1 ? z1 : z2;
        std::vector<cld> Ln(L.size() + 1, cld(0, 0));
        for (size_t i = 0; i < L.size(); ++i) { Ln[i] += L[i] / ((ld)1 - zk); Ln[i + 1] -= L[i] * zk / ((ld)1 - zk); }
        L.swap(Ln);
    }
    std::vector<cld> H(1, cld(1, 0));
    for (int k = 0; k < N; ++k) {
        std::vector<cld> Hn(H.size() + 1, cld(0, 0));
        for (size_t i = 0; i < H.size(); ++i) { Hn[i] += H[i] * (ld)0.5; Hn[i + 1] += H[i] * (ld)0.5; }
        H.swap(Hn);
    }
    for (size_t i = 0; i < H.size(); ++i)
        for (size_t j = 0; j < L.size(); ++j) h[i + j] += (double)((H[i] * L[j]).real() * sqrtl(2.0L));
}

#define WCK(call)                                                                                           \
    do {                                                                                                    \
        cudaError_t e_ = (call);                                                                            \
        if (e_ != cudaSuccess)                                                                              \
            return pkerr::set(e_ == cudaErrorMemoryAllocation ? PURIFY_ERR_ALLOC : PURIFY_ERR_CUDA,          \
                              "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__);   \
    } while (0)

}  // namespace

struct purify_wavelet {
    int n = 0, levels = 0, dtype = 0;
    Filters F;
    std::vector<double> taps[NB];
    void* filt = nullptr;       // device: [NB][2][LMAX] reals
    void* tmp = nullptr;        // NB n^2 complex: between the two passes of a level
    void* work = nullptr;       // NB n^2 complex: the synthesis' evolving low-low blocks
    void* coef = nullptr;       // 9 n^2 complex: Psi^dagger zbar of the DUALFB pass
    int launches = 0;
};

namespace {

size_t csz(const purify_wavelet* w) { return w->dtype == PURIFY_C64 ? 8 : 16; }

template <typename R>
int adjoint_t(purify_wavelet* w, const void* x, void* alpha, cudaStream_t st) {
    typedef typename C2T<R>::type C;
    const int n = w->n;
    const long long nn = (long long)n * n;
    WCK(cudaMemcpyAsync(alpha, x, csz(w) * (size_t)nn, cudaMemcpyDeviceToDevice, st));               // Dirac basis: identity
    C* a = (C*)alpha + nn;                                                                          // bases 1..8
    for (int lev = 0; lev < w->levels; ++lev) {
        const int m = n >> lev, mh = m >> 1;
        const C* src = lev == 0 ? (const C*)x : a;
        wl_row_fwd<R><<<dim3((mh + ROW_SPAN - 1) / ROW_SPAN, m, NB), 128, 0, st>>>(src, lev == 0 ? 0 : nn, n, (C*)w->tmp, nn, n, m, (const R*)w->filt);
        wl_col_fwd<R><<<dim3((m + 127) / 128, (mh + KPT - 1) / KPT, NB), 128, 0, st>>>((const C*)w->tmp, nn, a, nn, n, m, (const R*)w->filt);
        w->launches += 2;
    }
    WCK(cudaGetLastError());
    return PURIFY_OK;
}

// MODE 0: x = Psi alpha; MODE 1: out = P_C(z - Psi alpha)
template <typename R, int MODE>
int forward_t(purify_wavelet* w, const void* alpha, const void* z, void* out, cudaStream_t st) {
    typedef typename C2T<R>::type C;
    const int n = w->n;
    const long long nn = (long long)n * n;
    const C* a = (const C*)alpha + nn;
    C* wk = (C*)w->work;
    for (int lev = w->levels - 1; lev >= 0; --lev) {
        const int m = n >> lev;
        const C* ll = lev == w->levels - 1 ? a : wk;          // the deepest level takes its low-low block from the coefficients
        const int blk = (m + 2 * KPT - 1) / (2 * KPT);            // 2 KPT samples per thread along the blocked axis
        wl_col_inv<R><<<dim3((m + 127) / 128, blk, NB), 128, 0, st>>>(ll, nn, a, nn, (C*)w->tmp, nn, n, m, (const R*)w->filt);
        if (lev > 0)
            wl_row_inv<R><<<dim3((blk + 127) / 128, m, NB), 128, 0, st>>>((const C*)w->tmp, nn, wk, nn, n, m, (const R*)w->filt);
        else
            wl_row_inv_sum<R, MODE><<<dim3((blk + 127) / 128, n), 128, 0, st>>>((const C*)w->tmp, nn, (const C*)alpha, (const C*)z, (C*)out, n,
                                                                              (const R*)w->filt);
        w->launches += 2;
    }
    WCK(cudaGetLastError());
    return PURIFY_OK;
}

}  // namespace

extern "C" {

int purify_wavelet_create(purify_wavelet** out, int n, int levels, int dtype, void* cuda_stream) {
    if (!out) return pkerr::set(PURIFY_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (levels < 1 || levels > 8) return pkerr::set(PURIFY_ERR_INVALID_ARG, "levels must be in [1, 8] (got %d)", levels);
    if (n <= 0 || n > 16384 || (n % (1 << levels))) return pkerr::set(PURIFY_ERR_INVALID_ARG, "n must be a positive multiple of 2^levels (got %d)", n);
    if (dtype != PURIFY_C64 && dtype != PURIFY_C128) return pkerr::set(PURIFY_ERR_UNSUPPORTED, "unknown dtype %d", dtype);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) {
        cudaGetLastError();
        return pkerr::set(PURIFY_ERR_NO_DEVICE, "no CUDA device available; this library has no CPU fallback");
    }
    purify_wavelet* w = new (std::nothrow) purify_wavelet();
    if (!w) return pkerr::set(PURIFY_ERR_ALLOC, "host allocation failed");
    w->n = n; w->levels = levels; w->dtype = dtype;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t rs = dtype == PURIFY_C64 ? 4 : 8, nn = (size_t)n * n;
    std::vector<double> host((size_t)NB * 2 * LMAX, 0.0);
    for (int b = 0; b < NB; ++b) {
        daubechies(b + 1, w->taps[b]);
        const int L = 2 * (b + 1);
        w->F.len[b] = L;
        for (int m = 0; m < L; ++m) {
            host[(size_t)(b * 2) * LMAX + m] = w->taps[b][m];
            host[(size_t)(b * 2 + 1) * LMAX + m] = ((m & 1) ? -1.0 : 1.0) * w->taps[b][L - 1 - m];
        }
    }
    auto bail = [&](int code) { purify_wavelet_destroy(w); return code; };
    if (cudaMalloc(&w->filt, rs * host.size()) != cudaSuccess || cudaMalloc(&w->tmp, csz(w) * nn * NB) != cudaSuccess ||
        cudaMalloc(&w->work, csz(w) * nn * NB) != cudaSuccess || cudaMalloc(&w->coef, csz(w) * nn * (NB + 1)) != cudaSuccess) {
        cudaGetLastError();
        return bail(pkerr::set(PURIFY_ERR_ALLOC, "cudaMalloc of the wavelet scratch (25 n^2 complex) failed"));
    }
    cudaError_t e;
    if (dtype == PURIFY_C64) {
        std::vector<float> hf(host.begin(), host.end());
        e = cudaMemcpyAsync(w->filt, hf.data(), rs * host.size(), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    } else {
        e = cudaMemcpyAsync(w->filt, host.data(), rs * host.size(), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    }
    if (e != cudaSuccess) { cudaGetLastError(); return bail(pkerr::set(PURIFY_ERR_CUDA, "filter upload failed: %s", cudaGetErrorString(e))); }
    *out = w;
    return PURIFY_OK;
}

int purify_wavelet_destroy(purify_wavelet* w) {
    if (!w) return PURIFY_OK;
    cudaFree(w->filt); cudaFree(w->tmp); cudaFree(w->work); cudaFree(w->coef);
    cudaGetLastError();
    delete w;
    return PURIFY_OK;
}

int purify_wavelet_filter(const purify_wavelet* w, int basis, double* h_host) {
    if (!w || !h_host) return pkerr::set(PURIFY_ERR_INVALID_ARG, "NULL argument");
    if (basis < 1 || basis > NB) return pkerr::set(PURIFY_ERR_INVALID_ARG, "basis must be in [1, 8] (got %d)", basis);
    for (int m = 0; m < 2 * basis; ++m) h_host[m] = w->taps[basis - 1][m];
    return 2 * basis;
}

int purify_wavelet_adjoint(purify_wavelet* w, const void* x_dev, void* alpha_dev, void* cuda_stream) {
    if (!w || !x_dev || !alpha_dev) return pkerr::set(PURIFY_ERR_INVALID_ARG, "NULL argument");
    w->launches = 0;
    return w->dtype == PURIFY_C64 ? adjoint_t<float>(w, x_dev, alpha_dev, (cudaStream_t)cuda_stream)
                                  : adjoint_t<double>(w, x_dev, alpha_dev, (cudaStream_t)cuda_stream);
}

int purify_wavelet_forward(purify_wavelet* w, const void* alpha_dev, void* x_dev, void* cuda_stream) {
    if (!w || !x_dev || !alpha_dev) return pkerr::set(PURIFY_ERR_INVALID_ARG, "NULL argument");
    w->launches = 0;
    return w->dtype == PURIFY_C64 ? forward_t<float, 0>(w, alpha_dev, nullptr, x_dev, (cudaStream_t)cuda_stream)
                                  : forward_t<double, 0>(w, alpha_dev, nullptr, x_dev, (cudaStream_t)cuda_stream);
}

int purify_dualfb_step(purify_wavelet* w, const void* z_dev, const void* zbar_prev_dev, void* d_dev, void* zbar_out_dev,
                       double gamma, double eta, void* cuda_stream) {
    if (!w || !z_dev || !zbar_prev_dev || !d_dev || !zbar_out_dev) return pkerr::set(PURIFY_ERR_INVALID_ARG, "NULL argument");
    if (!(gamma >= 0.0) || !(eta > 0.0)) return pkerr::set(PURIFY_ERR_INVALID_ARG, "need gamma >= 0 and eta > 0");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    w->launches = 0;
    const long long cnt = (long long)w->n * w->n * (NB + 1);
    const int blocks = (int)((cnt + 255) / 256 < 148 * 32 ? (cnt + 255) / 256 : 148 * 32);
    int rc;
    if (w->dtype == PURIFY_C64) {
        if ((rc = adjoint_t<float>(w, zbar_prev_dev, w->coef, st))) return rc;
        dual_update_kernel<float><<<blocks, 256, 0, st>>>((float2*)d_dev, (const float2*)w->coef, cnt, (float)gamma, (float)eta);
        w->launches++;
        return forward_t<float, 1>(w, d_dev, z_dev, zbar_out_dev, st);
    }
    if ((rc = adjoint_t<double>(w, zbar_prev_dev, w->coef, st))) return rc;
    dual_update_kernel<double><<<blocks, 256, 0, st>>>((double2*)d_dev, (const double2*)w->coef, cnt, gamma, eta);
    w->launches++;
    return forward_t<double, 1>(w, d_dev, z_dev, zbar_out_dev, st);
}

int purify_project_positive(purify_wavelet* w, const void* z_dev, void* zbar_dev, void* cuda_stream) {
    if (!w || !z_dev || !zbar_dev) return pkerr::set(PURIFY_ERR_INVALID_ARG, "NULL argument");
    const long long cnt = (long long)w->n * w->n;
    const int blocks = (int)((cnt + 255) / 256 < 148 * 32 ? (cnt + 255) / 256 : 148 * 32);
    if (w->dtype == PURIFY_C64) project_positive_kernel<float><<<blocks, 256, 0, (cudaStream_t)cuda_stream>>>((const float2*)z_dev, (float2*)zbar_dev, cnt);
    else project_positive_kernel<double><<<blocks, 256, 0, (cudaStream_t)cuda_stream>>>((const double2*)z_dev, (double2*)zbar_dev, cnt);
    WCK(cudaGetLastError());
    return PURIFY_OK;
}

}  // extern "C"
