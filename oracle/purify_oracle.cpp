// CPU ORACLE for the measurement operator Phi = W G F Z S and its adjoint.
//
// *** TEST INFRASTRUCTURE, NOT PRODUCT. ***  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may call this.  It shares no
// code with the CUDA path (paper_1903_04502_b200/csrc) and neither imports the other.
//
// Plain, slow, step-by-step restatement of the algorithm in the paper's order
// (Eq. (2): y = W G F Z S x; adjoint = "these operators in reverse"),
// always in fp64.  Phi is an approximation (a NUFFT) of Eq. (1), so the
// oracle follows the algorithm; the plain definition (brute-force NUDFT) is what the
// tests check it against.  Where the paper is silent the readings R1..R13 of
// SURVEY.md 8(c) / DESIGN.md "Readings" are taken; each function names the one it uses.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): I0 vs scipy + printed constants,
// sum_c g(delta-c) closed form, g-hat vs numerical quadrature, FFT vs direct DFT and
// numpy, Phi vs brute-force NUDFT (Eq. 1), adjoint identity, centred / off-centre point
// sources, single-visibility adjoint, periodic wrap, table accuracy.
// The tap set of W G at integer / half-integer (u, v) (R7) is pinned on a one-hot Fourier grid and through the adjoint
// identity at such coordinates; the fp32 branch of the table index (R11) against exact integer arithmetic.
// Parity unpinned by the paper: WHICH of the two equally valid tie-breaks at integer u is taken (R7) - convention only.
//
// Conventions: image x[py*n+px] complex interleaved (re,im), px fastest, px<->u, py<->v;
// centred pixel coordinate p^ = p - n/2; grid side K = 2n; (u,v) in grid cells, period K.
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
static const double PI = 3.14159265358979323846264338327950288;
static const int MAXJ = 32;   // largest kernel support the C entry points accept

// ---------------------------------------------------------------- O1: kernel
// Modified Bessel function of the first kind, order 0, by its power series
// I0(z) = sum_k ((z/2)^2)^k / (k!)^2  (all terms positive: no cancellation).
static double i0_series(double z) {
    const double q = 0.25 * z * z;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 500; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < 1e-18 * sum) break;
    }
    return sum;
}

// R1: Kaiser-Bessel g(d) = I0(beta sqrt(1-(2d/J)^2)) / I0(beta), |d| <= J/2, else 0;
// beta = 2.34 J (the alpha = 2 choice of the NUFFT paper [34] cited at PAPER.md:51).
static double kb_beta(int J) { return 2.34 * (double)J; }

static double kb_g(double d, int J) {
    const double h = 0.5 * (double)J;
    if (std::fabs(d) > h) return 0.0;
    const double r = d / h;
    double a = 1.0 - r * r;
    if (a < 0.0) a = 0.0;
    return i0_series(kb_beta(J) * std::sqrt(a)) / i0_series(kb_beta(J));
}

// O2 / R2: continuous Fourier transform of g,
// g^(xi) = (J / I0(beta)) sinh(sqrt(beta^2 - (pi J xi)^2)) / sqrt(beta^2 - (pi J xi)^2)
// (real for |xi| <= 1/4 because pi J / 4 < 2.34 J).
static double kb_ghat(double xi, int J) {
    const double beta = kb_beta(J);
    const double t = PI * (double)J * xi;
    const double a2 = beta * beta - t * t;
    double val;
    if (a2 > 0.0) {
        const double a = std::sqrt(a2);
        val = std::sinh(a) / a;
    } else if (a2 < 0.0) {
        const double a = std::sqrt(-a2);
        val = std::sin(a) / a;
    } else {
        val = 1.0;
    }
    return (double)J / i0_series(beta) * val;
}

// O5 / R11: pre-sampled kernel table: T[i] = g(i/R), i = 0..R*J/2+1
// (guard entry; g = 0 beyond J/2), zeroth-order (nearest-sample) lookup, even symmetry,
// same table for G and G^dagger.
static void build_table(int J, int R, std::vector<double>& T) {
    const long len = (long)R * J / 2 + 2;
    T.resize(len);
    for (long i = 0; i < len; ++i) T[i] = kb_g((double)i / (double)R, J);
}

// Kernel weight of tap c for coordinate u.  mode 0: analytic g(u - c) in double.
// mode 1: table lookup T[floor(|d| R + 1/2)].  idx_prec 64: d and the index are
// evaluated in double; idx_prec 32: in float (the CUDA C64 path's precision - task
// rule 3: "where floating point decides an integer, both sides take that decision in
// the same precision").  u arrives already rounded to the storage precision.
// R11: index of the nearest table sample for the distance |u - c|: floor(|d| R + 1/2), each step ONE IEEE operation
// in the storage precision of the problem (idx_prec 32: float, 64: double).
static long table_index(double u, long c, int R, int idx_prec) {
    if (idx_prec == 32) {
        volatile float df = (float)u - (float)c;          // one IEEE fp32 subtraction
        volatile float a = std::fabs(df) * (float)R;      // one fp32 multiply
        volatile float b = a + 0.5f;                      // one fp32 add
        return (long)std::floor((double)b);
    }
    volatile double d = u - (double)c;
    volatile double a = std::fabs(d) * (double)R;
    volatile double b = a + 0.5;
    return (long)std::floor(b);
}

struct KernelEval {
    int J, mode, R, idx_prec;
    std::vector<double> T;
    KernelEval(int J_, int mode_, int R_, int idx_prec_) : J(J_), mode(mode_), R(R_), idx_prec(idx_prec_) {
        if (mode == 1) build_table(J, R, T);
    }
    double operator()(double u, long c) const {
        if (mode == 0) return kb_g(u - (double)c, J);
        const long idx = table_index(u, c, R, idx_prec);
        if (idx >= (long)T.size()) return 0.0;
        return T[idx];
    }
};

static inline long mod_pos(long a, long K) {
    long r = a % K;
    return r < 0 ? r + K : r;
}

// ---------------------------------------------------------------- O3(2): FFT
// Unnormalised DFT, B[k] = sum_j b[j] exp(sign * 2 pi i j k / K)  (R5: forward sign = -1,
// F^dagger = +1 with NO 1/K^2).  Radix-2 decimation-in-time for powers of two,
// directly computed twiddles; direct O(K^2) DFT otherwise (R13).
static bool is_pow2(long K) { return K > 0 && (K & (K - 1)) == 0; }

static void dft1_direct(const cplx* in, cplx* out, long K, long stride_in, int sign) {
    for (long k = 0; k < K; ++k) {
        cplx acc(0.0, 0.0);
        for (long j = 0; j < K; ++j) {
            const long jk = (j * k) % K;   // exact phase reduction
            const double ang = (double)sign * 2.0 * PI * (double)jk / (double)K;
            acc += in[j * stride_in] * cplx(std::cos(ang), std::sin(ang));
        }
        out[k] = acc;
    }
}

static void fft1_radix2(cplx* a, long K, int sign, const std::vector<cplx>& tw) {
    // bit reversal
    for (long i = 1, j = 0; i < K; ++i) {
        long bit = K >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(a[i], a[j]);
    }
    for (long len = 2; len <= K; len <<= 1) {
        const long half = len >> 1, step = K / len;
        for (long i = 0; i < K; i += len)
            for (long k = 0; k < half; ++k) {
                cplx w = tw[k * step];
                if (sign > 0) w = std::conj(w);
                const cplx t = a[i + k + half] * w;
                a[i + k + half] = a[i + k] - t;
                a[i + k] += t;
            }
    }
}

static void fft2(cplx* data, long K, int sign) {
    const bool p2 = is_pow2(K);
    std::vector<cplx> tw;
    if (p2) {
        tw.resize(K / 2 > 0 ? K / 2 : 1);
        for (long k = 0; k < K / 2; ++k) {
            const double ang = -2.0 * PI * (double)k / (double)K;   // forward twiddle
            tw[k] = cplx(std::cos(ang), std::sin(ang));
        }
    }
    // rows
#pragma omp parallel
    {
        std::vector<cplx> tmp(K), out(K);
#pragma omp for schedule(static)
        for (long r = 0; r < K; ++r) {
            cplx* row = data + r * K;
            if (p2) fft1_radix2(row, K, sign, tw);
            else { dft1_direct(row, out.data(), K, 1, sign); std::memcpy((void*)row, out.data(), sizeof(cplx) * K); }
        }
        // columns
#pragma omp for schedule(static)
        for (long c = 0; c < K; ++c) {
            for (long r = 0; r < K; ++r) tmp[r] = data[r * K + c];
            if (p2) { fft1_radix2(tmp.data(), K, sign, tw); for (long r = 0; r < K; ++r) data[r * K + c] = tmp[r]; }
            else { dft1_direct(tmp.data(), out.data(), K, 1, sign); for (long r = 0; r < K; ++r) data[r * K + c] = out[r]; }
        }
    }
}

// ---------------------------------------------------------------- O2: correction vector
// s[p] = 1 / g^(p^/K), p^ = p - n/2  (R2, R3: a == 1, pure kernel correction, exact scale).
static void correction(int n, int K, int J, std::vector<double>& s) {
    s.resize(n);
    for (int p = 0; p < n; ++p) s[p] = 1.0 / kb_ghat((double)(p - n / 2) / (double)K, J);
}

// O3(1): S then Z.  b = 0; b[p^y mod K, p^x mod K] = s[py] s[px] x[py,px]   (R6)
static void pad_correct(int n, int K, const std::vector<double>& s, const cplx* x, cplx* b) {
    for (long i = 0; i < (long)K * K; ++i) b[i] = cplx(0.0, 0.0);
    for (int py = 0; py < n; ++py)
        for (int px = 0; px < n; ++px) {
            const long gy = mod_pos(py - n / 2, K), gx = mod_pos(px - n / 2, K);
            b[gy * K + gx] = s[py] * s[px] * x[(long)py * n + px];
        }
}

// O4(3): Z^dagger then S^dagger.  x'[py,px] = s[py] s[px] b'[p^y mod K, p^x mod K]
static void crop_correct(int n, int K, const std::vector<double>& s, const cplx* b, cplx* x) {
    for (int py = 0; py < n; ++py)
        for (int px = 0; px < n; ++px) {
            const long gy = mod_pos(py - n / 2, K), gx = mod_pos(px - n / 2, K);
            x[(long)py * n + px] = s[py] * s[px] * b[gy * K + gx];
        }
}

// O3(3): W G.  For each k: cell = floor(u_k); taps c = cell - J/2 + b, b = 1..J, i.e. the
// integers in (u - J/2, u + J/2] (R7); y_k = w_k sum_a sum_b g(v_k - cy_a) g(u_k - cx_b)
// B[cy_a mod K, cx_b mod K]  (R8: periodic wrap).
static void degrid_core(int K, int J, long M, const cplx* B, const double* uv, const double* w,
                        const KernelEval& ker, cplx* y) {
#pragma omp parallel for schedule(static)
    for (long k = 0; k < M; ++k) {
        const double u = uv[2 * k], v = uv[2 * k + 1];
        const long cx0 = (long)std::floor(u) - J / 2, cy0 = (long)std::floor(v) - J / 2;
        double gxs[MAXJ + 1], gys[MAXJ + 1];
        for (int t = 1; t <= J; ++t) { gxs[t] = ker(u, cx0 + t); gys[t] = ker(v, cy0 + t); }
        cplx acc(0.0, 0.0);
        for (int a = 1; a <= J; ++a) {
            const long row = mod_pos(cy0 + a, K);
            for (int b = 1; b <= J; ++b)
                acc += (gys[a] * gxs[b]) * B[row * K + mod_pos(cx0 + b, K)];
        }
        y[k] = (w ? w[k] : 1.0) * acc;
    }
}

// O4(1): G^dagger W^dagger.  B' = 0; B'[cy_a mod K, cx_b mod K] += g g conj(w_k) y_k (R9: w real).
// Threads own private grids that are summed in thread order (deterministic).
static void grid_core(int K, int J, long M, const cplx* y, const double* uv, const double* w,
                      const KernelEval& ker, cplx* Bp) {
    const long KK = (long)K * K;
    int nt = 1;
#ifdef _OPENMP
    nt = omp_get_max_threads();
    // bound the private-grid memory to ~8 GB
    const long cap = (long)(8.0e9 / (16.0 * (double)KK));
    if (nt > cap) nt = (int)(cap < 1 ? 1 : cap);
#endif
    std::vector<std::vector<cplx> > priv(nt);
#pragma omp parallel num_threads(nt)
    {
        int t = 0;
#ifdef _OPENMP
        t = omp_get_thread_num();
#endif
        std::vector<cplx>& g = priv[t];
        g.assign(KK, cplx(0.0, 0.0));
        const long k0 = M * t / nt, k1 = M * (t + 1) / nt;
        for (long k = k0; k < k1; ++k) {
            const double u = uv[2 * k], v = uv[2 * k + 1];
            const long cx0 = (long)std::floor(u) - J / 2, cy0 = (long)std::floor(v) - J / 2;
            const cplx z = (w ? w[k] : 1.0) * y[k];
            double gxs[MAXJ + 1], gys[MAXJ + 1];
            for (int t2 = 1; t2 <= J; ++t2) { gxs[t2] = ker(u, cx0 + t2); gys[t2] = ker(v, cy0 + t2); }
            for (int a = 1; a <= J; ++a) {
                const long row = mod_pos(cy0 + a, K);
                for (int b = 1; b <= J; ++b)
                    g[row * K + mod_pos(cx0 + b, K)] += (gys[a] * gxs[b]) * z;
            }
        }
    }
    for (long i = 0; i < KK; ++i) Bp[i] = cplx(0.0, 0.0);
    for (int t = 0; t < nt; ++t) {
#pragma omp parallel for schedule(static)
        for (long i = 0; i < KK; ++i) Bp[i] += priv[t][i];
        std::vector<cplx>().swap(priv[t]);
    }
}

// ---------------------------------------------------------------- C ABI (ctypes)
extern "C" {

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void oracle_set_num_threads(int t) {
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

double oracle_i0(double z) { return i0_series(z); }
double oracle_kb(double d, int J) { return kb_g(d, J); }
double oracle_kb_ghat(double xi, int J) { return kb_ghat(xi, J); }

void oracle_correction(int n, int J, double* s_out) {
    std::vector<double> s;
    correction(n, 2 * n, J, s);
    for (int p = 0; p < n; ++p) s_out[p] = s[p];
}

long oracle_table_len(int J, int R) { return (long)R * J / 2 + 2; }
void oracle_table(int J, int R, double* T_out) {
    std::vector<double> T;
    build_table(J, R, T);
    for (size_t i = 0; i < T.size(); ++i) T_out[i] = T[i];
}
// kernel weight exactly as the operator evaluates it (for the table-accuracy pin)
double oracle_kernel_weight(double u, long c, int J, int mode, int R, int idx_prec) {
    KernelEval ker(J, mode, R, idx_prec);
    return ker(u, c);
}

// the table index rule on its own, for n (u, c) pairs (pin of the idx_prec = 32 branch)
void oracle_table_index(long n, const double* u, const long* c, int R, int idx_prec, long* out) {
    for (long i = 0; i < n; ++i) out[i] = table_index(u[i], c[i], R, idx_prec);
}

// in-place unnormalised 2-D DFT of a K x K complex array, sign = -1 forward, +1 adjoint
void oracle_fft2(double* data, int K, int sign) { fft2((cplx*)data, K, sign); }
// direct separable O(K^3) DFT (cross-check of the radix-2 code on small K)
void oracle_dft2_direct(const double* in, double* out, int K, int sign) {
    const cplx* a = (const cplx*)in;
    cplx* o = (cplx*)out;
    std::vector<cplx> tmp((size_t)K * K), col(K), res(K);
    for (long r = 0; r < K; ++r) dft1_direct(a + r * K, tmp.data() + r * K, K, 1, sign);
    for (long c = 0; c < K; ++c) {
        for (long r = 0; r < K; ++r) col[r] = tmp[r * K + c];
        dft1_direct(col.data(), res.data(), K, 1, sign);
        for (long r = 0; r < K; ++r) o[r * K + c] = res[r];
    }
}

// S + Z only: x[n*n] -> b[K*K]
void oracle_pad(int n, int J, const double* x, double* b) {
    std::vector<double> s;
    correction(n, 2 * n, J, s);
    pad_correct(n, 2 * n, s, (const cplx*)x, (cplx*)b);
}
// Z^dagger S^dagger only
void oracle_crop(int n, int J, const double* b, double* x) {
    std::vector<double> s;
    correction(n, 2 * n, J, s);
    crop_correct(n, 2 * n, s, (const cplx*)b, (cplx*)x);
}
// W G only, from a given Fourier grid B[K*K]
void oracle_degrid_from_grid(int K, int J, long M, const double* B, const double* uv, const double* w,
                             int mode, int R, int idx_prec, double* y) {
    KernelEval ker(J, mode, R, idx_prec);
    degrid_core(K, J, M, (const cplx*)B, uv, w, ker, (cplx*)y);
}
// G^dagger W^dagger only, to a Fourier grid B'[K*K]
void oracle_grid_to_grid(int K, int J, long M, const double* y, const double* uv, const double* w,
                         int mode, int R, int idx_prec, double* Bp) {
    KernelEval ker(J, mode, R, idx_prec);
    grid_core(K, J, M, (const cplx*)y, uv, w, ker, (cplx*)Bp);
}

// Phi: y = W G F Z S x   (O3)
void oracle_degrid(int n, int J, long M, const double* x, const double* uv, const double* w,
                   int mode, int R, int idx_prec, double* y) {
    const int K = 2 * n;
    std::vector<double> s;
    correction(n, K, J, s);
    std::vector<cplx> b((size_t)K * K);
    pad_correct(n, K, s, (const cplx*)x, b.data());
    fft2(b.data(), K, -1);
    KernelEval ker(J, mode, R, idx_prec);
    degrid_core(K, J, M, b.data(), uv, w, ker, (cplx*)y);
}

// Phi^dagger: x' = S^dagger Z^dagger F^dagger G^dagger W^dagger y   (O4)
void oracle_grid(int n, int J, long M, const double* y, const double* uv, const double* w,
                 int mode, int R, int idx_prec, double* x) {
    const int K = 2 * n;
    std::vector<double> s;
    correction(n, K, J, s);
    std::vector<cplx> b((size_t)K * K);
    KernelEval ker(J, mode, R, idx_prec);
    grid_core(K, J, M, (const cplx*)y, uv, w, ker, b.data());
    fft2(b.data(), K, +1);
    crop_correct(n, K, s, b.data(), (cplx*)x);
}

}  // extern "C"
