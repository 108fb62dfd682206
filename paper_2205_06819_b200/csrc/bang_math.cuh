// bang_math.cuh -- scalar device functions of the path: Hernquist projections, Jeans l.o.s. quadrature, modified Bessel
// functions and the Freeman-disc function, NFW enclosed mass, and the pseudo-logarithmic table index.
//
// Everything here is written from the formulas cited (PAPER.md:<line>, DLMF section numbers for the special functions);
// nothing is shared with oracle/.  Functions are BANG_HD so that the same source can be exercised on the host by
// development probes; the library only ever calls them from kernels.
#pragma once
#include <math.h>
#include <stdint.h>

#if defined(__CUDACC__)
#define BANG_HD __host__ __device__ __forceinline__
#define BANG_D __device__ __forceinline__
#else
#define BANG_HD inline
#define BANG_D inline
#endif

namespace bang {

constexpr double kG = 4.30091727004e-6;              // kpc km^2 s^-2 Msun^-1
constexpr double kKpcPerArcsecPerMpc = 4.84813681109536e-3;
constexpr double kH0 = 0.07;                         // km/s/kpc = 70 km/s/Mpc (reading H)
constexpr double kPi = 3.14159265358979323846;
constexpr double kEulerGamma = 0.57721566490153286061;
constexpr int kRFloorLog2 = -16;                     // radii are floored at 2^-16 kpc (reading V)

// ---------------------------------------------------------------------------------------------------------------
// T5(u) = -ln(1-u) - u - u^2/2 - u^3/3 - u^4/4 = sum_{n>=5} u^n/n, 0 <= u < 1.
// rho_b v_r^2 = G M_b^2/(2 pi R_b^4) T5(R_b/(r+R_b)) is eq. 1 x eq. 3 with the Jeans integral done by
// partial fractions (reading C): the printed eq. 3 cancels catastrophically for r >> R_b, this form does not.
BANG_HD double T5(double u) {
    if (u <= 0.0) return 0.0;
    if (u < 0.75) {
        double p = u * u * u * u * u, sum = 0.0;
        for (int n = 5; n < 200; ++n) {
            double term = p / n;
            sum += term;
            if (term < 2e-18 * sum) break;
            p *= u;
        }
        return sum;
    }
    double u2 = u * u;
    return -log1p(-u) - u - 0.5 * u2 - u2 * u * (1.0 / 3.0) - 0.25 * u2 * u2;
}

// Scale-free Jeans l.o.s. integral (eq. 6 first form):
//   Sigma_b sigma_b^2 (R) = 2 int_0^inf rho_b v_r^2 dz = G M_b^2/(2 pi R_b^3) * 2 * J(s),   s = R/R_b,
//   J(s) = int_0^inf T5(1/(1 + sqrt(s^2 + z^2))) dz          (z in units of R_b).
// Rule (reading B): Gauss-Legendre on t in (0,1), z = L t^2/(1-t), dz/dt = L t (2-t)/(1-t)^2, L = sqrt(s^2+1).
// glx, glw: the N_J nodes and weights on (-1,1).
BANG_HD double jeans_J(double s, int NJ, const double* glx, const double* glw) {
    const double L = sqrt(s * s + 1.0);
    double sum = 0.0;
    for (int k = 0; k < NJ; ++k) {
        const double t = 0.5 * (glx[k] + 1.0), w = 0.5 * glw[k];
        const double omt = 1.0 - t;
        const double z = L * t * t / omt;
        const double dzdt = L * t * (2.0 - t) / (omt * omt);
        const double r = sqrt(s * s + z * z);
        sum += w * dzdt * T5(1.0 / (1.0 + r));
    }
    return sum;
}

// Hernquist projected profile (eq. 4-5): Sigma_b = M_b/(2 pi R_b^2) SigmaTilde(s),
//   SigmaTilde = [(2+s^2) X(s) - 3]/(1-s^2)^2.
// With w = 1 - s^2, X = atanh(sqrt w)/sqrt w (w>0) = atan(sqrt -w)/sqrt -w (w<0) = sum_n w^n/(2n+1), which turns the
// removable singularity at s = 1 into the power series  SigmaTilde = sum_{n>=2} 4(n-1)/(4n^2-1) w^(n-2)  (|w| < 1).
BANG_HD double sigma_tilde(double s) {
    const double w = 1.0 - s * s;
    if (fabs(w) < 0.25) {
        double p = 1.0, sum = 0.0;
        for (int n = 2; n < 80; ++n) {
            double term = 4.0 * (n - 1) / (4.0 * n * n - 1.0) * p;
            sum += term;
            if (fabs(term) < 1e-18 * fabs(sum)) break;
            p *= w;
        }
        return sum;
    }
    double X;
    if (w > 0.0) {
        double q = sqrt(w);
        X = log((1.0 + q) / s) / q;
    } else {
        double q = sqrt(-w);
        X = acos(1.0 / s) / q;
    }
    return ((2.0 + s * s) * X - 3.0) / (w * w);
}

// ---------------------------------------------------------------------------------------------------------------
// Jaffe bulge (Appendix B; reading J).
// eq. B4: Sigma_b = M_b/R_b^2 SigmaTildeJ(s),  SigmaTildeJ = 1/(4s) + [1 - (2 - s^2) X(s)]/(2 pi (1 - s^2)).
//   |1 - s^2| < 1/4: with w = 1 - s^2 and X = sum_n w^n/(2n+1),  [1 - (1+w) X]/w = -sum_{n>=1} 4n/(4n^2-1) w^(n-1);
//   s >= 8: the two terms cancel to ~1/(8 s^3); use the projection of the large-r expansion of eq. B1 term by term,
//           rho = (1/4 pi) sum_k (-1)^k (k+1) r^-(k+4),  2 int_0^inf (s^2+z^2)^(-m/2) dz = c_m s^(1-m),
//           c_4 = pi/2, c_5 = 4/3, c_(m+2) = c_m (m-1)/m.
BANG_HD double jaffe_sigma_tilde(double s) {
    const double w = 1.0 - s * s;
    if (fabs(w) < 0.25) {
        double p = 1.0, sum = 0.0;
        for (int n = 1; n < 80; ++n) {
            double term = 4.0 * n / (4.0 * n * n - 1.0) * p;
            sum += term;
            if (fabs(term) < 1e-18 * fabs(sum)) break;
            p *= w;
        }
        return 0.25 / s - sum / (2.0 * kPi);
    }
    if (s >= 8.0) {
        const double is = 1.0 / s;
        double ce = 0.5 * kPi, co = 4.0 / 3.0;           // c_m for even / odd m, starting at m = 4, 5
        double p = is * is * is, sum = 0.0;
        for (int k = 0; k < 60; ++k) {
            const int m = k + 4;
            const double c = (m & 1) ? co : ce;
            const double term = ((k & 1) ? -1.0 : 1.0) * (k + 1) * c * p;
            sum += term;
            if (fabs(term) < 1e-18 * fabs(sum)) break;
            if (m & 1) co *= (double)(m - 1) / m; else ce *= (double)(m - 1) / m;
            p *= is;
        }
        return sum / (4.0 * kPi);
    }
    double X;
    if (w > 0.0) { const double q = sqrt(w); X = log((1.0 + q) / s) / q; }
    else { const double q = sqrt(-w); X = acos(1.0 / s) / q; }
    return 0.25 / s + (1.0 - (2.0 - s * s) * X) / (2.0 * kPi * w);
}

// rho_b v_r^2 = G M_b^2/(4 pi R_b^4) J3(t), t = r/R_b: the isotropic Jeans integral of eqs. B1-B2,
//   J3 = int_t^inf dt'/(t'^3 (1+t')^3) = sum_{n>=5} (n-3)(n-4)/2 u^n/n  (u = 1/(1+t); equals rho_b x eq. B3 as corrected
//   by reading J; the closed form cancels like t^-5 for large t, hence the series for t > 1).
BANG_HD double jaffe_J3(double t) {                      // argument t = r/R_b (u would lose t for t << 1)
    if (t > 1.0) {
        const double u = 1.0 / (1.0 + t);
        double p = u * u * u * u * u, sum = 0.0;
        for (int n = 5; n < 400; ++n) {
            double term = 0.5 * (n - 3) * (n - 4) * p / n;
            sum += term;
            if (term < 2e-18 * sum) break;
            p *= u;
        }
        return sum;
    }
    return 1.0 / (2.0 * t * t) - 3.0 / t - 3.0 / (1.0 + t) - 1.0 / (2.0 * (1.0 + t) * (1.0 + t)) + 6.0 * log1p(1.0 / t);
}

// Scale-free l.o.s. integral for the Jaffe bulge with the same N_J-node rule as jeans_J (reading B):
//   Sigma_b sigma_b^2 (R) = G M_b^2/(4 pi R_b^3) * 2 * JJ(s),  JJ(s) = int_0^inf J3(sqrt(s^2+z^2)) dz.
BANG_HD double jaffe_jeans_J(double s, int NJ, const double* glx, const double* glw) {
    const double L = sqrt(s * s + 1.0);
    double sum = 0.0;
    for (int k = 0; k < NJ; ++k) {
        const double t = 0.5 * (glx[k] + 1.0), w = 0.5 * glw[k];
        const double omt = 1.0 - t;
        const double z = L * t * t / omt;
        const double dzdt = L * t * (2.0 - t) / (omt * omt);
        const double r = sqrt(s * s + z * z);
        sum += w * dzdt * jaffe_J3(r);
    }
    return sum;
}

// ---------------------------------------------------------------------------------------------------------------
// Modified Bessel functions I0, I1, K0, K1, exponentially scaled: I_nu(y) e^-y and K_nu(y) e^y.
//   y <= 2 : ascending series, DLMF 10.25.2 (I_nu) and 10.31.1-2 (K_0, K_1)
//   y  > 2 : integral representations DLMF 10.32.3  I_n(y) = (1/pi) int_0^pi e^{y cos t} cos(n t) dt  and
//            10.32.9  K_nu(y) = int_0^inf e^{-y cosh t} cosh(nu t) dt, by the trapezoid rule (geometric convergence
//            for these analytic integrands).
struct Bessel4 { double i0e, i1e, k0e, k1e; };

BANG_HD Bessel4 bessel_series(double y) {
    const double q = 0.25 * y * y;                       // (y/2)^2
    double term0 = 1.0, term1 = 1.0;                     // q^k/(k!)^2 and q^k/(k!(k+1)!)
    double i0 = 1.0, i1 = 1.0;
    double H = 0.0;                                      // harmonic number H_k
    double k0s = 0.0;                                    // sum_k H_k q^k/(k!)^2
    double k1s = (1.0 - 2.0 * kEulerGamma);              // sum_k [psi(k+1)+psi(k+2)] q^k/(k!(k+1)!), k = 0 term: -2 gamma + 1
    for (int k = 1; k < 40; ++k) {
        term0 *= q / ((double)k * k);
        term1 *= q / ((double)k * (k + 1));
        H += 1.0 / k;
        i0 += term0;
        i1 += term1;
        k0s += H * term0;
        k1s += (2.0 * H + 1.0 / (k + 1) - 2.0 * kEulerGamma) * term1;
        if (term0 < 1e-19 * i0) break;
    }
    i1 *= 0.5 * y;
    const double lh = log(0.5 * y);
    const double k0 = -(lh + kEulerGamma) * i0 + k0s;
    const double k1 = 1.0 / y + lh * i1 - 0.25 * y * k1s;
    const double e = exp(y), em = 1.0 / e;
    Bessel4 b;
    b.i0e = i0 * em; b.i1e = i1 * em; b.k0e = k0 * e; b.k1e = k1 * e;
    return b;
}

BANG_HD Bessel4 bessel_quadrature(double y) {
    Bessel4 b;
    {   // I_n: trapezoid on [0, pi] with N intervals (error ~ I_{2N}(y) e^-y, negligible for 2N >> y)
        const int N = 256;
        const double h = kPi / N;
        double s0 = 0.5 * (1.0 + exp(-2.0 * y)), s1 = 0.5 * (1.0 - exp(-2.0 * y));
        for (int j = 1; j < N; ++j) {
            const double c = cos(j * h);
            const double e = exp(y * (c - 1.0));
            s0 += e;
            s1 += e * c;
        }
        b.i0e = s0 / N;
        b.i1e = s1 / N;
    }
    {   // K_nu: trapezoid on [0, inf) with step h; integrand e^{-y (cosh t - 1)} cosh(nu t)
        const double h = 0.0625;
        double s0 = 0.5, s1 = 0.5;
        for (int j = 1; j < 4000; ++j) {
            const double t = j * h;
            const double ch = cosh(t);
            const double a = y * (ch - 1.0);
            if (a > 745.0) break;
            const double e = exp(-a);
            s0 += e;
            s1 += e * ch;
        }
        b.k0e = s0 * h;
        b.k1e = s1 * h;
    }
    return b;
}

// Freeman (1970) disc, eq. 9 in its dimensionally consistent form (reading D):
//   v_c^2(r) = (2 G M_d / R_d) F(y),  y = r/(2 R_d),  F(y) = y^2 [I0(y) K0(y) - I1(y) K1(y)].
// y > 32: large-argument expansion of the products, DLMF 10.40.6:
//   I_nu K_nu ~ 1/(2y) sum_k (-1)^k [(2k-1)!!/(2k)!!] (mu-1)(mu-9)...(mu-(2k-1)^2) / (2y)^(2k),  mu = 4 nu^2.
BANG_HD double freeman_F(double y) {
    if (y <= 0.0) return 0.0;
    if (y <= 2.0) {
        Bessel4 b = bessel_series(y);
        return y * y * (b.i0e * b.k0e - b.i1e * b.k1e);
    }
    if (y <= 32.0) {
        Bessel4 b = bessel_quadrature(y);
        return y * y * (b.i0e * b.k0e - b.i1e * b.k1e);
    }
    const double iz2 = 1.0 / (4.0 * y * y);
    double a0 = 1.0, a1 = 1.0, sum = 0.0, prev = 1e300;   // k-th terms of the nu = 0 and nu = 1 series
    for (int k = 1; k < 40; ++k) {
        const double odd = 2.0 * k - 1.0;
        const double f = -(odd / (2.0 * k)) * iz2;
        a0 *= f * (0.0 - odd * odd);
        a1 *= f * (4.0 - odd * odd);
        const double term = a0 - a1;
        if (fabs(term) >= prev) break;
        prev = fabs(term);
        sum += term;
        if (prev < 1e-18 * fabs(sum)) break;
    }
    return 0.5 * y * sum;
}

// NFW enclosed-mass shape mu(x) = ln(1+x) - x/(1+x) (reading H); series sum_{n>=2} (-1)^n (n-1)/n x^n for small x.
template <typename T>
BANG_HD T nfw_mu(T x) {
    if (x < T(0.03125)) {
        // alternating series; 10 terms give x^12 ~ 1e-18 at x = 1/32
        T sum = T(0), p = x * x, sgn = T(1);
        for (int n = 2; n < 13; ++n) {
            sum += sgn * (T(n - 1) / T(n)) * p;
            p *= x;
            sgn = -sgn;
        }
        return sum;
    }
    return (T)log1p((double)x) - x / (T(1) + x);
}
template <>
BANG_HD float nfw_mu<float>(float x) {
    if (x < 0.25f) {                                  // 15 terms: x^17 < 6e-11; beyond, ln(1+x) - x/(1+x) cancels < 10x
        float sum = 0.f, p = x * x, sgn = 1.f;
#pragma unroll
        for (int n = 2; n < 17; ++n) {
            sum += sgn * ((float)(n - 1) / (float)n) * p;
            p *= x;
            sgn = -sgn;
        }
        return sum;
    }
    return log1pf(x) - x / (1.f + x);
}

// r200 of an NFW halo of mass M200: mean density 200 rho_c inside, rho_c = 3 H0^2/(8 pi G) (reading H).
BANG_HD double nfw_r200(double M200) {
    const double rho_c = 3.0 * kH0 * kH0 / (8.0 * kPi * kG);
    return cbrt(3.0 * M200 / (4.0 * kPi * 200.0 * rho_c));
}

// ---------------------------------------------------------------------------------------------------------------
// Pseudo-logarithmic table index.  A positive floating-point number u = 2^e (1 + f) is its own table address: the
// table has 2^M equal sub-intervals per octave of u, the interval number is the top bits (exponent and M mantissa bits)
// and the position inside the interval, mapped to t in [-1, 1), is the remaining mantissa bits.  No logarithm is taken.
// Every table stores, per interval, the D+1 coefficients of a polynomial in t (Chebyshev-node interpolant, monomial
// form): D = 3, M = 3 in fp32 mode (8 cubics per octave: relative error 4e-6 for SigmaTilde, 8e-6 for J, 6e-7 for F,
// 2e-7 for v_c -- measured against direct evaluation; the mode's tolerance is 1e-4), D = 7, M = 3 in fp64 mode (~1e-11).
// Round 1 used M = 4 in fp32 mode (3e-7): halving the tables is what lets the theta's slice of the bulge table live in
// shared memory next to its v_c table.
template <typename T> struct TabCfg;
template <> struct TabCfg<float>  { static constexpr int D = 3, M = 3; };
template <> struct TabCfg<double> { static constexpr int D = 7, M = 3; };

// global interval number of u (before subtracting the table's first interval): (biased exponent << M) | top mantissa bits
BANG_HD int tab_cell(float u, float& t) {
    constexpr int M = TabCfg<float>::M, LOW = 23 - M;
#if defined(__CUDA_ARCH__)
    const int bits = __float_as_int(u);
    // tau = 1 + (low 23-M mantissa bits) 2^-23 in [1, 1 + 2^-M);  t = 2^(M+1) tau - (2^(M+1) + 1), exact: one LOP3 and one
    // FFMA (both masks as register operands, or ptxas splits (bits & m) | c into two LOP3 with one immediate each)
    int tau;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(tau) : "r"(bits), "r"((1 << LOW) - 1), "r"(0x3F800000));
    t = fmaf(__int_as_float(tau), (float)(2 << M), -(float)((2 << M) + 1));
#else
    union { float f; int i; } c; c.f = u;
    const int bits = c.i;
    union { int i; float f; } d; d.i = ((bits & ((1 << LOW) - 1)) << M) | 0x40000000;
    t = d.f - 3.0f;
#endif
    return bits >> LOW;
}
BANG_HD int tab_cell(double u, double& t) {
#if defined(__CUDA_ARCH__)
    const long long bits = __double_as_longlong(u);
    t = __longlong_as_double(((bits & 0x1FFFFFFFFFFFFLL) << 3) | 0x4000000000000000LL) - 3.0;
#else
    union { double f; long long i; } c; c.f = u;
    const long long bits = c.i;
    union { long long i; double f; } d; d.i = ((bits & 0x1FFFFFFFFFFFFLL) << 3) | 0x4000000000000000LL;
    t = d.f - 3.0;
#endif
    return (int)(bits >> 49);                            // 52 - M, M = 3
}
// first global interval number of the octave 2^e
template <typename T> BANG_HD int tab_first_cell(int e);
template <> BANG_HD int tab_first_cell<float>(int e) { return (e + 127) << TabCfg<float>::M; }
template <> BANG_HD int tab_first_cell<double>(int e) { return (e + 1023) << 3; }

// lower edge and width of interval `cell` (global number), as doubles
template <typename T>
BANG_HD void tab_interval(int cell, double& lo, double& width) {
    constexpr int M = TabCfg<T>::M;
    constexpr int bias = sizeof(T) == 4 ? 127 : 1023;
    const int e = (cell >> M) - bias;
    const int j = cell & ((1 << M) - 1);
    const double p = ldexp(1.0, e);
    width = p / (1 << M);
    lo = p + j * width;
}

}  // namespace bang
