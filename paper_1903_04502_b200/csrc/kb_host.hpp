// Host-side (create-time) mathematics of the CUDA path: Kaiser-Bessel kernel, its Fourier
// transform (gridding correction), the per-tap polynomial fit and the pre-sampled table.
// Written in long double from the definitions in DESIGN.md "Readings" (R1, R2, R11); shares no
// code with oracle/ (the oracle has its own, in double).
#pragma once
#include <cmath>
#include <vector>

namespace kbhost {

typedef long double ld;
static const ld PI_L = 3.141592653589793238462643383279502884L;

// I0 by its everywhere-convergent, all-positive power series.
inline ld bessel_i0(ld z) {
    const ld q = z * z / 4;
    ld term = 1, sum = 1;
    for (int k = 1; k < 1000; ++k) {
        term *= q / ((ld)k * (ld)k);
        sum += term;
        if (term < sum * 1e-22L) break;
    }
    return sum;
}

inline ld beta_of(int J) { return 2.34L * (ld)J; }   // R1: beta = 2.34 J (alpha = 2)

// R1: g(d) = I0(beta sqrt(1 - (2d/J)^2)) / I0(beta) on |d| <= J/2, 0 outside.
inline ld kb(ld d, int J) {
    const ld h = (ld)J / 2;
    if (fabsl(d) > h) return 0;
    ld a = 1 - (d / h) * (d / h);
    if (a < 0) a = 0;
    return bessel_i0(beta_of(J) * sqrtl(a)) / bessel_i0(beta_of(J));
}

// Analytic continuation of g just past the support edge (the same entire function of
// a = 1 - (2d/J)^2, I0(beta sqrt(a)) = J0(beta sqrt(-a)) for a < 0) - used only so that the
// polynomial fit of the outermost tap sees a smooth function on its whole unit interval.
inline ld kb_smooth(ld d, int J) {
    const ld h = (ld)J / 2;
    const ld a = 1 - (d / h) * (d / h);
    const ld q = beta_of(J) * beta_of(J) * a / 4;     // series in q is entire, valid for q < 0
    ld term = 1, sum = 1;
    for (int k = 1; k < 1000; ++k) {
        term *= q / ((ld)k * (ld)k);
        sum += term;
        if (fabsl(term) < 1e-24L) break;
    }
    return sum / bessel_i0(beta_of(J));
}

// R2: g^(xi) = (J / I0(beta)) sinh(sqrt(beta^2 - (pi J xi)^2)) / sqrt(beta^2 - (pi J xi)^2).
inline ld kb_ghat(ld xi, int J) {
    const ld b = beta_of(J), t = PI_L * (ld)J * xi;
    const ld a2 = b * b - t * t;
    ld v;
    if (a2 > 0) { const ld a = sqrtl(a2); v = sinhl(a) / a; }
    else if (a2 < 0) { const ld a = sqrtl(-a2); v = sinl(a) / a; }
    else v = 1;
    return (ld)J / bessel_i0(b) * v;
}

// Gridding-correction vector s[p] = 1 / g^((p - n/2)/K), K = 2n.
inline void correction(int n, int J, std::vector<double>& s) {
    s.resize(n);
    for (int p = 0; p < n; ++p) s[p] = (double)(1 / kb_ghat((ld)(p - n / 2) / (ld)(2 * n), J));
}

// Pre-sampled table T[i] = g(i/R), i = 0 .. R*J/2 + 1.
inline void table(int J, int R, std::vector<double>& T) {
    const long len = (long)R * J / 2 + 2;
    T.resize(len);
    for (long i = 0; i < len; ++i) T[i] = (double)kb((ld)i / (ld)R, J);
}

// Per-tap polynomial.  For a coordinate u with cell = floor(u), f = u - cell in [0,1), the J taps
// are c_j = cell - J/2 + 1 + j, j = 0..J-1, at distance d_j = f + (J/2 - 1 - j).  With
// t = f - 1/2 in [-1/2, 1/2):  g(d_j) = P_j(t) and, by evenness of g, g(d_{J-1-j}) = P_j(-t).
// Split P_j(t) = E_j(t^2) + t O_j(t^2): one pair of taps costs one even and one odd Horner chain.
// Coefficients: Chebyshev interpolation (64 nodes) of P_j on [-1/2, 1/2], truncated at `degree`,
// converted to monomials in t in long double.  e[j][m] multiplies t^(2m), o[j][m] t^(2m+1).
struct PolyFit {
    int J, degree, ne, no;
    double e[4][12], o[4][12];
    double max_abs_err;
};

inline void fit_poly(int J, int degree, PolyFit& out) {
    const int NN = 64;
    out.J = J; out.degree = degree;
    out.ne = degree / 2 + 1;
    out.no = (degree + 1) / 2;
    out.max_abs_err = 0;
    for (int j = 0; j < 4; ++j) for (int m = 0; m < 12; ++m) { out.e[j][m] = 0; out.o[j][m] = 0; }
    for (int j = 0; j < J / 2; ++j) {
        const ld shift = 0.5L + (ld)(J / 2 - 1 - j);
        // Chebyshev coefficients in s = 2t
        std::vector<ld> c(degree + 1, 0);
        for (int m = 0; m <= degree; ++m) {
            ld acc = 0;
            for (int i = 0; i < NN; ++i) {
                const ld th = PI_L * ((ld)i + 0.5L) / NN;
                const ld t = 0.5L * cosl(th);
                acc += kb_smooth(t + shift, J) * cosl((ld)m * th);
            }
            c[m] = acc * 2 / NN;
        }
        c[0] /= 2;
        // monomial coefficients of sum_m c_m T_m(s)
        std::vector<ld> mono(degree + 1, 0), Tm2(degree + 1, 0), Tm1(degree + 1, 0), Tm(degree + 1, 0);
        Tm2[0] = 1;                                   // T_0
        mono[0] += c[0];
        if (degree >= 1) { Tm1[1] = 1; mono[1] += c[1]; }   // T_1 = s
        for (int m = 2; m <= degree; ++m) {
            for (int i = 0; i <= degree; ++i) Tm[i] = -Tm2[i] + (i > 0 ? 2 * Tm1[i - 1] : 0);
            for (int i = 0; i <= degree; ++i) mono[i] += c[m] * Tm[i];
            Tm2 = Tm1; Tm1 = Tm;
        }
        ld p2 = 1;
        for (int i = 0; i <= degree; ++i) {           // s = 2t
            const ld a = mono[i] * p2;
            if (i % 2 == 0) out.e[j][i / 2] = (double)a; else out.o[j][i / 2] = (double)a;
            p2 *= 2;
        }
        // fit check against the true (truncated) kernel, Horner in double as on the device
        for (int i = 0; i <= 2000; ++i) {
            const double t = -0.5 + (double)i / 2000.0 * (1.0 - 1e-12);
            const double t2 = t * t;
            double E = out.e[j][out.ne - 1], O = out.no > 0 ? out.o[j][out.no - 1] : 0.0;
            for (int m = out.ne - 2; m >= 0; --m) E = E * t2 + out.e[j][m];
            for (int m = out.no - 2; m >= 0; --m) O = O * t2 + out.o[j][m];
            const double hi = E + t * O, lo = E - t * O;
            const double e1 = fabs(hi - (double)kb((ld)t + shift, J));
            const double e2 = fabs(lo - (double)kb(-(ld)t + shift, J));
            if (e1 > out.max_abs_err) out.max_abs_err = e1;
            if (e2 > out.max_abs_err) out.max_abs_err = e2;
        }
    }
}

}  // namespace kbhost
