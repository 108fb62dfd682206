// bang_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, fp64 CPU restatement of the batched likelihood of Rigamonti et al. 2022
// (arXiv 2205.06819, "BANG"), written from /root/reference/PAPER.md and the readings listed in
// DESIGN.md ("Readings of the paper").  It exists so that the CUDA library can be checked against
// something that can be compared with the paper by eye.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header, table or
// constant generator with paper_2205_06819_b200/ (the CUDA path) and neither includes the other.
//
// Every quantity is evaluated DIRECTLY at every fine cell: no radial tables, no interpolation, no
// tiling, no fusion.  The only "library primitives" are libm, libquadmath and the C++17 special
// functions std::cyl_bessel_i / std::cyl_bessel_k.
//
// Pins (tests/test_oracle_*.py, `-m "not gpu"`): every function below is pinned to something other
// than itself -- mpmath closed forms / direct numerical integration, textbook limits, invariants,
// brute-force 2-D PSF sums, and the survey-time cross-check values in tests/golden/.  One choice is
// a definition rather than a derivable fact and is therefore "parity unpinned" beyond its
// invariants: WHICH fields are PSF-convolved and that they are convolved unweighted (reading G).
//
// Notation follows the paper: R = sky-plane radius, r = radius in the disc plane, s = R/R_b,
// Sigma = surface density, B = surface brightness, k_j = Satoh parameter, i = inclination.
//
// Build: g++ -O2 -std=c++17 -fopenmp -shared -fPIC bang_oracle.cpp -o libbang_oracle.so -lquadmath

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <vector>
#include <quadmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---- constants -------------------------------------------
const double kG = 4.30091727004e-6;            // kpc km^2 s^-2 Msun^-1
const double kArcsecKpcPerMpc = 4.84813681109536e-3;   // kpc per arcsec per Mpc of distance
const double kH0 = 0.07;                        // km s^-1 kpc^-1  (70 km/s/Mpc; reading H)
const double kPi = 3.14159265358979323846;
const double kRFloor = 1.52587890625e-05;       // 2^-16 kpc: floor on R and r (reading V)

const unsigned C_BULGE = 1u, C_DISC1 = 2u, C_DISC2 = 4u, C_HALO = 8u;

int g_threads = 0;   // 0 = OpenMP default

// ---- eq. 5: X(s) -----------------------------------------------------------------------------
template <typename T> T sqrtT(T x);
template <> double sqrtT(double x) { return std::sqrt(x); }
template <> __float128 sqrtT(__float128 x) { return sqrtq(x); }
template <typename T> T logT(T x);
template <> double logT(double x) { return std::log(x); }
template <> __float128 logT(__float128 x) { return logq(x); }
template <typename T> T acosT(T x);
template <> double acosT(double x) { return std::acos(x); }
template <> __float128 acosT(__float128 x) { return acosq(x); }

// PAPER.md:100 (eq. 5).  s > 0, s != 1.
template <typename T> T hernquist_X(T s) {
    const T one = 1;
    if (s < one) {
        T q = sqrtT<T>(one - s * s);
        return logT<T>((one + q) / s) / q;
    }
    T q = sqrtT<T>(s * s - one);
    return acosT<T>(one / s) / q;
}

// PAPER.md:96 (eq. 4): Sigma_b(R) = M_b/(2 pi R_b^2) * SigmaTilde(s),
// SigmaTilde(s) = [(2+s^2) X(s) - 3] / (1-s^2)^2.
template <typename T> T sigma_tilde_T(T s) {
    const T one = 1;
    T d = one - s * s;
    return ((T(2) + s * s) * hernquist_X<T>(s) - T(3)) / (d * d);
}

// Removable singularity at s = 1 (reading I): the printed form is evaluated in binary128 for
// 0.5 < s < 2 (cancellation ~1/eps^2), and by its Taylor series 4/15 - (16/35)e + (8/15)e^2 for
// |e| = |s-1| < 1e-7 (pinned against mpmath in tests/test_oracle_pins.py).
double sigma_tilde(double s) {
    double e = s - 1.0;
    if (std::fabs(e) < 1e-7) return 4.0 / 15.0 - (16.0 / 35.0) * e + (8.0 / 15.0) * e * e;
    if (s > 0.5 && s < 2.0) return (double)sigma_tilde_T<__float128>((__float128)s);
    return sigma_tilde_T<double>(s);
}

// PAPER.md:105 (eq. 6, second form; reading A for the broken line):
// Sigma_b sigma_b^2 = G M_b^2/(12 pi R_b^3) * ITilde(s),
// ITilde = [ -3 s^2 X (8 s^6 - 28 s^4 + 35 s^2 - 20) - 24 s^6 + 68 s^4 - 65 s^2 + 6 ] / (2 (1-s^2)^3) - 6 pi s.
// Cancels catastrophically near s = 1 and for s >> 1, so it is evaluated in binary128 throughout.
// NOT on the model path (the N_J-node quadrature is): it is the pin for that quadrature.
double I_tilde_closed(double sd) {
    double e = sd - 1.0;
    if (std::fabs(e) < 1e-5)
        return (664.0 / 35.0 - 6.0 * kPi) - 0.259079731063 * e + (80.0 / 231.0) * e * e;
    __float128 s = sd, s2 = s * s, s4 = s2 * s2, s6 = s4 * s2;
    __float128 X = hernquist_X<__float128>(s);
    __float128 d = 1 - s2;
    __float128 num = -3 * s2 * X * (8 * s6 - 28 * s4 + 35 * s2 - 20) - 24 * s6 + 68 * s4 - 65 * s2 + 6;
    __float128 v = num / (2 * d * d * d) - 6 * (4 * atanq((__float128)1)) * s;
    return (double)v;
}

// PAPER.md:89 (eq. 3) as printed, in binary128 (pin only; reading C explains why it is not used).
double vr2_printed(double r, double Mb, double Rb) {
    __float128 x = (__float128)r / Rb;
    __float128 t = 12 * x * (1 + x) * (1 + x) * (1 + x) * logq((1 + x) / x)
                 - x / (1 + x) * (25 + 52 * x + 42 * x * x + 12 * x * x * x);
    return (double)((__float128)(kG * Mb / (12.0 * Rb)) * t);
}

// ---- reading C: rho_b * v_r^2 = G M_b^2/(2 pi R_b^4) * T5(u), u = R_b/(r + R_b) ---------------
// T5(u) = -ln(1-u) - u - u^2/2 - u^3/3 - u^4/4 = sum_{n>=5} u^n/n  (the isotropic Jeans integral
// int_r^inf rho G M(<x)/x^2 dx of eqs. 1-2 by partial fractions; identical to eq. 1 x eq. 3).
double T5(double u) {
    if (u <= 0.0) return 0.0;
    if (u < 0.5) {
        double un = u * u * u * u * u, sum = 0.0;
        for (int n = 5; n < 400; ++n) {
            double term = un / n;
            sum += term;
            if (term < 1e-18 * sum) break;
            un *= u;
        }
        return sum;
    }
    return -std::log1p(-u) - u - u * u / 2 - u * u * u / 3 - u * u * u * u / 4;
}

double rho_vr2(double r, double Mb, double Rb) {
    return kG * Mb * Mb / (2 * kPi * Rb * Rb * Rb * Rb) * T5(Rb / (r + Rb));
}

// ---- Appendix B: Jaffe bulge (reading J) -----------------------------
// eq. B1: rho_b = M_b R_b / (4 pi r^2 (r + R_b)^2);  M(<r) = M_b r/(r + R_b);  eq. B2: v_c^2 = G M_b/(r + R_b).
double vc2_jaffe(double r, double M, double a) { return kG * M / (r + a); }

// eq. B4: Sigma_b(R) = M_b/R_b^2 * SigmaTildeJ(s),
// SigmaTildeJ(s) = 1/(4 s) + [1 - (2 - s^2) X(s)] / (2 pi (1 - s^2)),  X(s) of eq. 5.
template <typename T> T jaffe_sigma_tilde_T(T s) {
    const T one = 1, pi = T(4) * (sizeof(T) == 8 ? T(std::atan(1.0)) : T(atanq((__float128)1)));
    return one / (T(4) * s) + (one - (T(2) - s * s) * hernquist_X<T>(s)) / (T(2) * pi * (one - s * s));
}
// Removable singularity at s = 1 (value 1/4 - 2/(3 pi)): Taylor series for |s-1| < 1e-7.  For s >> 1 the two terms
// cancel to Sigma ~ 1/(8 s^3) (relative loss ~ eps s^2), so binary128 is used for every s > 0.5.
double jaffe_sigma_tilde(double s) {
    double e = s - 1.0;
    if (std::fabs(e) < 1e-7) return (0.25 - 2.0 / (3.0 * kPi)) - 0.0802347273686449752 * e + 0.116613000075362963 * e * e;
    if (s > 0.5) return (double)jaffe_sigma_tilde_T<__float128>((__float128)s);
    return jaffe_sigma_tilde_T<double>(s);
}

// Isotropic Jeans integral of eqs. B1-B2: rho_b v_r^2 = int_r^inf rho_b G M(<x)/x^2 dx
//   = G M_b^2/(4 pi R_b^4) * J3(t),  t = r/R_b,  u = R_b/(r + R_b) = 1/(1+t),
//   J3 = int_t^inf dt'/(t'^3 (1+t')^3) = 1/(2t^2) - 3/t - 3/(1+t) - 1/(2(1+t)^2) + 6 ln(1 + 1/t),  t = r/R_b
//      = int_0^u u'^4/(1-u')^3 du' = sum_{n>=5} (n-3)(n-4)/2 u^n/n      (the closed form cancels like t^-5 for t >> 1).
// Equals rho_b x eq. B3 with the sign of B3's braces reversed and a = R_b (reading J; pinned in tests).
double J3(double t) {                          // argument: t = r/R_b (not u, which loses t for t << 1)
    if (!(t < INFINITY)) return 0.0;
    if (t > 1.0) {
        double u = 1.0 / (1.0 + t);
        double un = u * u * u * u * u, sum = 0.0;
        for (int n = 5; n < 400; ++n) {
            double term = 0.5 * (n - 3) * (n - 4) * un / n;
            sum += term;
            if (term < 1e-18 * sum) break;
            un *= u;
        }
        return sum;
    }
    return 1.0 / (2 * t * t) - 3.0 / t - 3.0 / (1 + t) - 1.0 / (2 * (1 + t) * (1 + t)) + 6.0 * std::log1p(1.0 / t);
}
double rho_vr2_jaffe(double r, double Mb, double Rb) {
    return kG * Mb * Mb / (4 * kPi * Rb * Rb * Rb * Rb) * J3(r / Rb);
}
// eq. B3 with reading J's corrections (a = R_b, sign), in binary128: pin only.
double vr2_jaffe_corrected(double r, double Mb, double Rb) {
    __float128 x = (__float128)r / Rb;
    __float128 br = 6 * logq(1 + 1 / x) - 3 / x - (6 * x + 7) / (2 * (x + 1) * (x + 1)) + 1 / (2 * x * x);
    return (double)((__float128)(kG * Mb / Rb) * x * x * (1 + x) * (1 + x) * br);
}
// eq. B5 times Sigma_b: Sigma_b sigma_b^2 = G M_b^2/(4 pi R_b^3) * ITildeJ(s),
// ITildeJ = [pi/(2s) + 11 - (13/2) pi s - 12 s^2 + 6 pi s^3 - X(s)(6 - 19 s^2 + 12 s^4)] / (1 - s^2); binary128.
// NOT on the model path: the pin for the N_J-node quadrature below.
double jaffe_I_tilde_closed(double sd) {
    double e = sd - 1.0;
    if (std::fabs(e) < 1e-5) return 0.0545737385894705218 - 0.153685581666989383 * e + 0.2755582315567978 * e * e;
    __float128 s = sd, s2 = s * s, pi = 4 * atanq((__float128)1);
    __float128 X = hernquist_X<__float128>(s);
    __float128 num = pi / (2 * s) + 11 - (__float128)13 / 2 * pi * s - 12 * s2 + 6 * pi * s2 * s - X * (6 - 19 * s2 + 12 * s2 * s2);
    return (double)(num / (1 - s2));
}

// ---- Gauss-Legendre nodes on (-1,1) ----------------------------------------------------------
void gauss_legendre(int n, double *x, double *w) {
    for (int i = 0; i < (n + 1) / 2; ++i) {
        double z = std::cos(kPi * (i + 0.75) / (n + 0.5)), pp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) {
                double p3 = p2;
                p2 = p1;
                p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
            }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (std::fabs(dz) < 1e-16) break;
        }
        x[i] = -z;
        x[n - 1 - i] = z;
        w[i] = w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

// ---- eq. 6, FIRST form, by the N_J-node rule of reading B --------------------------------------
// I_b(R) = Sigma_b sigma_b^2 = 2 int_0^inf rho_b v_r^2 dz,  r = sqrt(R^2 + z^2)
// Rule: Gauss-Legendre on t in (0,1), z = L t^2/(1-t), dz/dt = L t (2-t)/(1-t)^2, L = sqrt(R^2+R_b^2).
double Ib_quadrature(double R, double Mb, double Rb, int NJ, const double *glx, const double *glw) {
    double L = std::sqrt(R * R + Rb * Rb), sum = 0.0;
    for (int k = 0; k < NJ; ++k) {
        double t = 0.5 * (glx[k] + 1.0), wt = 0.5 * glw[k];
        double z = L * t * t / (1.0 - t);
        double dzdt = L * t * (2.0 - t) / ((1.0 - t) * (1.0 - t));
        double r = std::sqrt(R * R + z * z);
        sum += wt * dzdt * T5(Rb / (Rb + r));
    }
    return kG * Mb * Mb / (2 * kPi * Rb * Rb * Rb * Rb) * 2.0 * sum;
}

// The same N_J-node rule for the Jaffe bulge: I_b(R) = 2 int_0^inf rho_b v_r^2 dz with rho_b v_r^2 of rho_vr2_jaffe.
double Ib_quadrature_jaffe(double R, double Mb, double Rb, int NJ, const double *glx, const double *glw) {
    double L = std::sqrt(R * R + Rb * Rb), sum = 0.0;
    for (int k = 0; k < NJ; ++k) {
        double t = 0.5 * (glx[k] + 1.0), wt = 0.5 * glw[k];
        double z = L * t * t / (1.0 - t);
        double dzdt = L * t * (2.0 - t) / ((1.0 - t) * (1.0 - t));
        double r = std::sqrt(R * R + z * z);
        sum += wt * dzdt * J3(r / Rb);
    }
    return kG * Mb * Mb / (4 * kPi * Rb * Rb * Rb * Rb) * 2.0 * sum;
}

// ---- eq. 9 (reading D): v_c^2 = (2 G M_d / R_d) F(r / 2R_d), F(y) = y^2 [I0 K0 - I1 K1](y) ------
double freeman_F(double y) {
    if (y <= 0.0) return 0.0;
    if (y < 30.0) {   // extended precision: the bracket cancels like 2 y^2 (8e-13 in binary64 at y = 20)
        long double z = y;
        return (double)(z * z * (std::cyl_bessel_i(0.0L, z) * std::cyl_bessel_k(0.0L, z) -
                                 std::cyl_bessel_i(1.0L, z) * std::cyl_bessel_k(1.0L, z)));
    }
    // y >= 30: large-argument expansion (asymptotic; smallest term ~ e^{-2y}, summed until it stops shrinking)
    // I_nu K_nu ~ 1/(2y) sum_k (-1)^k [(2k-1)!!/(2k)!!] prod_{j<=k}(mu-(2j-1)^2) / (2y)^{2k}, mu = 4 nu^2.
    double z2 = 4.0 * y * y, sum = 0.0, c0 = 1.0, c1 = 1.0, prev = 1e300;   // c_nu = k-th term of each series
    for (int k = 1; k < 60; ++k) {
        double odd = (2.0 * k - 1.0), f = -(odd / (2.0 * k)) / z2;
        c0 *= f * (0.0 - odd * odd);
        c1 *= f * (4.0 - odd * odd);
        double term = c0 - c1;
        if (std::fabs(term) >= prev) break;
        prev = std::fabs(term);
        sum += term;
        if (prev < 1e-18 * std::fabs(sum)) break;
    }
    return y * y * sum / (2.0 * y);
}

// eq. 2: Hernquist circular speed squared.
double vc2_hernquist(double r, double M, double a) { return kG * M * r / ((r + a) * (r + a)); }

double vc2_expdisc(double r, double Md, double Rd) { return 2.0 * kG * Md / Rd * freeman_F(r / (2.0 * Rd)); }

// reading H: NFW halo, (M200, c); rho_c from H0 = 70 km/s/Mpc.
double nfw_mu(double x) {
    if (x < 1e-2) {   // mu = sum_{n>=2} (-1)^n (n-1)/n x^n
        double xn = x * x, sum = 0.0, sgn = 1.0;
        for (int n = 2; n < 40; ++n) {
            sum += sgn * (n - 1.0) / n * xn;
            xn *= x;
            sgn = -sgn;
        }
        return sum;
    }
    return std::log1p(x) - x / (1.0 + x);
}
double nfw_r200(double M200) {
    double rho_c = 3.0 * kH0 * kH0 / (8.0 * kPi * kG);
    return std::cbrt(3.0 * M200 / (4.0 * kPi * 200.0 * rho_c));
}
double vc2_nfw(double r, double M200, double c) {
    if (r <= 0.0) return 0.0;
    double rs = nfw_r200(M200) / c;
    return kG * M200 * nfw_mu(r / rs) / (r * nfw_mu(c));
}

// ---- decoded parameter vector (Table 1; layout in DESIGN.md) ----------------
struct Theta {
    double x0, y0, pa, inc;            // arcsec, arcsec, rad, rad
    double Mb, Rb, Md[2], Rd[2], Mh, Rh;   // Msun, kpc  (Rh = concentration c when halo is NFW)
    double MLb, MLd[2], k[2];
    bool valid;
};

Theta decode(const double *th, unsigned comps) {
    Theta t;
    t.x0 = th[0]; t.y0 = th[1];
    t.pa = th[2] * kPi / 180.0; t.inc = th[3] * kPi / 180.0;
    t.Mb = std::pow(10.0, th[4]); t.Rb = th[5];
    t.Md[0] = std::pow(10.0, th[6]); t.Rd[0] = th[7];
    t.Md[1] = std::pow(10.0, th[8]); t.Rd[1] = th[9];
    t.Mh = std::pow(10.0, th[10]); t.Rh = th[11];
    t.MLb = th[12]; t.MLd[0] = th[13]; t.MLd[1] = th[14];
    t.k[0] = th[15]; t.k[1] = th[16];
    bool ok = std::isfinite(th[0]) && std::isfinite(th[1]) && std::isfinite(th[2]) && std::isfinite(th[3]);
    ok = ok && std::fabs(th[3]) < 90.0;   // cos i > 0, decided on the angle in degrees
    if (comps & C_BULGE) ok = ok && std::isfinite(th[4]) && th[5] > 0 && std::isfinite(th[5]) && th[12] > 0 && std::isfinite(th[12]);
    for (int j = 0; j < 2; ++j)
        if (comps & (j ? C_DISC2 : C_DISC1))
            ok = ok && std::isfinite(th[6 + 2 * j]) && th[7 + 2 * j] > 0 && std::isfinite(th[7 + 2 * j]) &&
                 th[13 + j] > 0 && std::isfinite(th[13 + j]) && std::fabs(th[15 + j]) <= 1.0;
    if (comps & C_HALO) ok = ok && std::isfinite(th[10]) && th[11] > 0 && std::isfinite(th[11]);
    t.valid = ok;
    return t;
}

// circular speed squared of everything but the bulge at radius x (eq. 9 per disc, halo): the "external" potential of
// reading U'
double vc2_ext(double x, const Theta &t, unsigned comps, int halo_profile) {
    double v2 = 0.0;
    for (int j = 0; j < 2; ++j)
        if (comps & (j ? C_DISC2 : C_DISC1)) v2 += vc2_expdisc(x, t.Md[j], t.Rd[j]);
    if (comps & C_HALO) v2 += (halo_profile == 1) ? vc2_nfw(x, t.Mh, t.Rh) : vc2_hernquist(x, t.Mh, t.Rh);
    return v2;
}

struct Setup {
    int nx, ny, s, rk, nfx, nfy, NJ;
    double pix, kappa;
    unsigned comps;
    int halo_profile;                  // 0 Hernquist (paper), 1 NFW (reading H)
    int bulge_profile;                 // 0 Hernquist (paper default), 1 Jaffe (App. B)
    int psf_weighting;                 // 0: the paper's eq. 21 on B, v, sigma, <L/M> (reading G); 1: flux-weighted moments (reading G')
    int bulge_potential;               // 0: the bulge's dispersion in its own potential (the paper); 1: in the
                                       //    total potential of eq. 10 (reading U')
    std::vector<double> taps, glx, glw;
};

int psf_halfwidth(double sigma_pix, int s, double trunc) {
    return (int)std::ceil(trunc * sigma_pix * s - 1e-9);
}

// eq. 21 on the fine grid, separable reading F: taps exp(-m^2/(2 sigma_f^2)),
// m = -r_k..r_k, normalised to sum 1 (the denominator of eq. 21).
void psf_taps(double sigma_pix, int s, double trunc, std::vector<double> &g) {
    int rk = psf_halfwidth(sigma_pix, s, trunc);
    double sf = sigma_pix * s, sum = 0.0;
    g.assign(2 * rk + 1, 0.0);
    for (int m = -rk; m <= rk; ++m) {
        g[m + rk] = (sf > 0.0) ? std::exp(-0.5 * m * m / (sf * sf)) : (m == 0 ? 1.0 : 0.0);
        sum += g[m + rk];
    }
    for (double &v : g) v /= sum;
}

// profiles: bits 0-7 halo profile, bits 8-15 bulge profile, bits 16-23 PSF weighting, bits 24-31 bulge potential
bool make_setup(Setup &S, int nx, int ny, double pix, int s, double dist_mpc, double sigma_pix,
                double trunc, unsigned comps, int profiles, int NJ) {
    const int halo_profile = profiles & 0xff, bulge_profile = (profiles >> 8) & 0xff;
    const int psf_weighting = (profiles >> 16) & 0xff, bulge_potential = (profiles >> 24) & 0xff;
    if (halo_profile > 1 || bulge_profile > 1 || psf_weighting > 1 || bulge_potential > 1) return false;
    if (nx < 1 || ny < 1 || s < 1 || !(pix > 0) || !(dist_mpc > 0) || sigma_pix < 0 || NJ < 1) return false;
    if (!(comps & (C_BULGE | C_DISC1 | C_DISC2))) return false;
    S.nx = nx; S.ny = ny; S.s = s; S.pix = pix; S.kappa = dist_mpc * kArcsecKpcPerMpc;
    S.comps = comps; S.halo_profile = halo_profile; S.bulge_profile = bulge_profile; S.psf_weighting = psf_weighting; S.bulge_potential = bulge_potential; S.NJ = NJ;
    psf_taps(sigma_pix, s, trunc, S.taps);
    S.rk = (int(S.taps.size()) - 1) / 2;
    S.nfx = nx * s + 2 * S.rk; S.nfy = ny * s + 2 * S.rk;
    S.glx.resize(NJ); S.glw.resize(NJ);
    gauss_legendre(NJ, S.glx.data(), S.glw.data());
    return true;
}

// ---- reading U' (variant; PAPER.md:107 and :417-419 name it as the model's first limitation): the bulge's dispersion in
// the TOTAL potential.  Isotropic spherical Jeans equation with the enclosed mass read off the total circular speed of
// eq. 10, G M(<x) = x v_c,tot^2(x):   rho_b v_r^2 (r) = int_r^inf rho_b(x) v_c,tot^2(x) / x dx,
// and its l.o.s. integral with the order of integration exchanged (z <= sqrt(x^2 - R^2)), an exact identity:
//     I_b(R) = Sigma_b sigma_b^2 = 2 int_0^inf rho_b v_r^2 (sqrt(R^2+z^2)) dz = 2 int_R^inf rho_b(x) v_c,tot^2(x) sqrt(x^2 - R^2) / x dx.
// v_c,tot^2 = v_c,b^2 + v_ext^2: the bulge's own part is eq. 6 exactly as in the paper's path (Ib_quadrature above), so
// the variant reduces to it identically when discs and halo vanish; the part of the other components is
//     I_ext(R) = 2 int_R^inf rho_b(x) v_ext^2(x) sqrt(x^2 - R^2) / x dx,   v_ext^2 = sum_j eq. 9 + halo,
// by the N_J-node Gauss-Legendre rule on t in (0,1) with x = R + L t^2/(1-t), L = sqrt(R^2 + R_b^2) (the map of reading B:
// sqrt(x^2 - R^2) = t sqrt(L (2R + d)/(1-t)), d = x - R, is smooth in t).  rho_b: eq. 1 (Hernquist) or eq. B1 (Jaffe).
double rho_bulge(double x, double Mb, double Rb, int bulge_profile) {
    if (bulge_profile == 1) return Mb * Rb / (4 * kPi * x * x * (x + Rb) * (x + Rb));        // eq. B1
    return Mb * Rb / (2 * kPi * x * (x + Rb) * (x + Rb) * (x + Rb));                          // eq. 1
}
double Ib_ext_quadrature(double R, const Theta &t, unsigned comps, int halo_profile, int bulge_profile, double Mb, double Rb,
                         int NJ, const double *glx, const double *glw) {
    double L = std::sqrt(R * R + Rb * Rb), sum = 0.0;
    for (int k = 0; k < NJ; ++k) {
        double tt = 0.5 * (glx[k] + 1.0), wt = 0.5 * glw[k];
        double d = L * tt * tt / (1.0 - tt);                      // x - R
        double dxdt = L * tt * (2.0 - tt) / ((1.0 - tt) * (1.0 - tt));
        double x = R + d;
        double root = std::sqrt(d * (2.0 * R + d));               // sqrt(x^2 - R^2) without cancellation
        sum += wt * dxdt * rho_bulge(x, Mb, Rb, bulge_profile) * vc2_ext(x, t, comps, halo_profile) * root / x;
    }
    return 2.0 * sum;
}

// ---- one fine cell: steps 1-8 of the definition (PAPER.md secs 2.1-2.4) -------------
// Jx, Jy: fine-cell indices in [-r_k, N s + r_k).  out = {B_tot, v_los, sigma_los, <L/M>}.
void fine_cell(const Setup &S, const Theta &t, int Jx, int Jy, double out[4]) {
    // 1. sky position of the cell centre [arcsec], then offset from the galaxy centre [kpc]
    double xs = ((Jx + 0.5) / S.s - 0.5 * S.nx) * S.pix;
    double ys = ((Jy + 0.5) / S.s - 0.5 * S.ny) * S.pix;
    double X = (xs - t.x0) * S.kappa, Y = (ys - t.y0) * S.kappa;
    // 2. rotate so that the major axis lies along x' (fn 2)
    double cp = std::cos(t.pa), sp = std::sin(t.pa);
    double xp = X * cp + Y * sp, yp = -X * sp + Y * cp;
    // 3. radii
    double ci = std::cos(t.inc), si = std::sin(t.inc);
    double R = std::max(std::hypot(xp, yp), kRFloor);
    double r = std::max(std::hypot(xp, yp / ci), kRFloor);
    double cosphi = xp / r;
    // 4. bulge: eq. 4 and eq. 6 (first form, N_J nodes)
    double Sb = 0.0, Ib = 0.0, vc2 = 0.0;
    if ((S.comps & C_BULGE) && S.bulge_profile == 0) {
        Sb = t.Mb / (2 * kPi * t.Rb * t.Rb) * sigma_tilde(R / t.Rb);
        Ib = Ib_quadrature(R, t.Mb, t.Rb, S.NJ, S.glx.data(), S.glw.data());
        vc2 += vc2_hernquist(r, t.Mb, t.Rb);
    } else if (S.comps & C_BULGE) {            // Jaffe: eq. B4, B2 and the l.o.s. integral of rho_b v_r^2 (B1, B3)
        Sb = t.Mb / (t.Rb * t.Rb) * jaffe_sigma_tilde(R / t.Rb);
        Ib = Ib_quadrature_jaffe(R, t.Mb, t.Rb, S.NJ, S.glx.data(), S.glw.data());
        vc2 += vc2_jaffe(r, t.Mb, t.Rb);
    }
    if ((S.comps & C_BULGE) && S.bulge_potential == 1)          // reading U': + the discs' and the halo's pull on the bulge
        Ib += Ib_ext_quadrature(R, t, S.comps, S.halo_profile, S.bulge_profile, t.Mb, t.Rb, S.NJ, S.glx.data(), S.glw.data());
    // 5. discs: eq. 7-8;  6. circular speed: eq. 2, 9, 10
    double Sd[2] = {0.0, 0.0};
    for (int j = 0; j < 2; ++j)
        if (S.comps & (j ? C_DISC2 : C_DISC1)) {
            Sd[j] = t.Md[j] / (2 * kPi * t.Rd[j] * t.Rd[j] * ci) * std::exp(-r / t.Rd[j]);
            vc2 += vc2_expdisc(r, t.Md[j], t.Rd[j]);
        }
    if (S.comps & C_HALO)
        vc2 += (S.halo_profile == 1) ? vc2_nfw(r, t.Mh, t.Rh) : vc2_hernquist(r, t.Mh, t.Rh);
    // 7. Satoh decomposition: eq. 11-12
    double vint = std::sqrt(vc2);
    double vd[2], sd2[2];
    for (int j = 0; j < 2; ++j) {
        vd[j] = -t.k[j] * si * cosphi * vint;
        sd2[j] = (1.0 - t.k[j] * t.k[j]) * vc2 / 3.0;
    }
    // 8. light-weighted observables: eq. 13, 14, 15, 19   (B in Lsun/pc^2: 1e-6 kpc^-2 -> pc^-2)
    double Bb = (S.comps & C_BULGE) ? Sb / t.MLb * 1e-6 : 0.0;
    double Bd[2];
    for (int j = 0; j < 2; ++j) Bd[j] = (S.comps & (j ? C_DISC2 : C_DISC1)) ? Sd[j] / t.MLd[j] * 1e-6 : 0.0;
    double Btot = Bb + Bd[0] + Bd[1];
    double IbL = (S.comps & C_BULGE) ? Ib / t.MLb * 1e-6 : 0.0;      // B_b sigma_b^2
    out[0] = Btot;
    out[1] = (Bd[0] * vd[0] + Bd[1] * vd[1]) / Btot;
    out[2] = std::sqrt((IbL + Bd[0] * sd2[0] + Bd[1] * sd2[1]) / Btot);
    out[3] = Btot / ((Sb + Sd[0] + Sd[1]) * 1e-6);
    if (S.psf_weighting == 1) {
        // reading G': what the beam averages is light, not velocity -- the fields handed to
        // the PSF are the zeroth, first and second velocity moments of the light and the mass surface density:
        // B, B v_los, B (sigma_los^2 + v_los^2), Sigma_tot [x 1e-6], with v_los, sigma_los of eqs. 14-15 above
        const double v = out[1], sg = out[2];
        out[1] = Btot * v;
        out[2] = Btot * (sg * sg + v * v);
        out[3] = (Sb + Sd[0] + Sd[1]) * 1e-6;
    }
}

// fine maps [4][nfy][nfx], un-convolved
void fine_maps(const Setup &S, const Theta &t, double *fine) {
    const size_t plane = (size_t)S.nfx * S.nfy;
#pragma omp parallel for schedule(dynamic, 1) num_threads(g_threads > 0 ? g_threads : omp_get_max_threads())
    for (int jy = 0; jy < S.nfy; ++jy)
        for (int jx = 0; jx < S.nfx; ++jx) {
            double o[4];
            fine_cell(S, t, jx - S.rk, jy - S.rk, o);
            for (int q = 0; q < 4; ++q) fine[q * plane + (size_t)jy * S.nfx + jx] = o[q];
        }
}

// steps 9-10: separable PSF ("valid" region), mean over s x s, then M/L = 1/<L/M>
void convolve_rebin(const Setup &S, const double *fine, double *maps) {
    const int nfx = S.nfx, nfy = S.nfy, rk = S.rk, nix = S.nx * S.s, niy = S.ny * S.s;
    const size_t plane = (size_t)nfx * nfy;
    std::vector<double> tx((size_t)nfy * nix), txy((size_t)niy * nix);
    for (int q = 0; q < 4; ++q) {
        const double *f = fine + q * plane;
        for (int jy = 0; jy < nfy; ++jy)            // along x
            for (int ix = 0; ix < nix; ++ix) {
                double a = 0.0;
                for (int m = -rk; m <= rk; ++m) a += S.taps[m + rk] * f[(size_t)jy * nfx + (ix + rk + m)];
                tx[(size_t)jy * nix + ix] = a;
            }
        for (int iy = 0; iy < niy; ++iy)            // along y
            for (int ix = 0; ix < nix; ++ix) {
                double a = 0.0;
                for (int m = -rk; m <= rk; ++m) a += S.taps[m + rk] * tx[(size_t)(iy + rk + m) * nix + ix];
                txy[(size_t)iy * nix + ix] = a;
            }
        for (int py = 0; py < S.ny; ++py)           // rebin
            for (int px = 0; px < S.nx; ++px) {
                double a = 0.0;
                for (int by = 0; by < S.s; ++by)
                    for (int bx = 0; bx < S.s; ++bx) a += txy[(size_t)(py * S.s + by) * nix + (px * S.s + bx)];
                a /= (double)(S.s * S.s);
                maps[((size_t)q * S.ny + py) * S.nx + px] = (q == 3 && S.psf_weighting == 0) ? 1.0 / a : a;
            }
    }
    if (S.psf_weighting == 1) {
        // reading G': observables from the beam-averaged moments M0..M3 of a pixel:
        // B = M0, v = M1/M0, sigma = sqrt(M2/M0 - v^2) (never negative analytically; floored at 0), M/L = M3/M0
        const size_t np = (size_t)S.nx * S.ny;
        for (size_t i = 0; i < np; ++i) {
            const double M0 = maps[i], v = maps[np + i] / M0;
            maps[np + i] = v;
            maps[2 * np + i] = std::sqrt(std::max(maps[2 * np + i] / M0 - v * v, 0.0));
            maps[3 * np + i] = maps[3 * np + i] / M0;
        }
    }
}

void model_one(const Setup &S, const double *theta, double *maps, std::vector<double> &fine) {
    Theta t = decode(theta, S.comps);
    const size_t npix = (size_t)S.nx * S.ny;
    if (!t.valid) {
        for (size_t p = 0; p < 4 * npix; ++p) maps[p] = std::numeric_limits<double>::quiet_NaN();
        return;
    }
    fine.resize((size_t)4 * S.nfx * S.nfy);
    fine_maps(S, t, fine.data());
    convolve_rebin(S, fine.data(), maps);
}

}  // namespace

extern "C" {

void bo_set_threads(int n) { g_threads = n; }
int bo_get_threads() {
#ifdef _OPENMP
    return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
    return 1;
#endif
}

// ---- scalar entry points (pins) ----
double bo_hernquist_X(double s) { return hernquist_X<double>(s); }
double bo_sigma_tilde(double s) { return sigma_tilde(s); }
double bo_I_tilde_closed(double s) { return I_tilde_closed(s); }
double bo_vr2_printed(double r, double Mb, double Rb) { return vr2_printed(r, Mb, Rb); }
double bo_T5(double u) { return T5(u); }
double bo_rho_vr2(double r, double Mb, double Rb) { return rho_vr2(r, Mb, Rb); }
double bo_Ib_quadrature(double R, double Mb, double Rb, int NJ) {
    std::vector<double> x(NJ), w(NJ);
    gauss_legendre(NJ, x.data(), w.data());
    return Ib_quadrature(R, Mb, Rb, NJ, x.data(), w.data());
}
void bo_gauss_legendre(int n, double *x, double *w) { gauss_legendre(n, x, w); }
double bo_freeman_F(double y) { return freeman_F(y); }
double bo_vc2_hernquist(double r, double M, double a) { return vc2_hernquist(r, M, a); }
double bo_vc2_expdisc(double r, double Md, double Rd) { return vc2_expdisc(r, Md, Rd); }
double bo_nfw_mu(double x) { return nfw_mu(x); }
double bo_nfw_r200(double M200) { return nfw_r200(M200); }
double bo_vc2_nfw(double r, double M200, double c) { return vc2_nfw(r, M200, c); }
double bo_hernquist_Sigma(double R, double Mb, double Rb) { return Mb / (2 * kPi * Rb * Rb) * sigma_tilde(R / Rb); }
double bo_jaffe_sigma_tilde(double s) { return jaffe_sigma_tilde(s); }
double bo_jaffe_I_tilde_closed(double s) { return jaffe_I_tilde_closed(s); }
double bo_J3(double t) { return J3(t); }
double bo_rho_vr2_jaffe(double r, double Mb, double Rb) { return rho_vr2_jaffe(r, Mb, Rb); }
double bo_vr2_jaffe_corrected(double r, double Mb, double Rb) { return vr2_jaffe_corrected(r, Mb, Rb); }
double bo_vc2_jaffe(double r, double M, double a) { return vc2_jaffe(r, M, a); }
double bo_Ib_quadrature_jaffe(double R, double Mb, double Rb, int NJ) {
    std::vector<double> x(NJ), w(NJ);
    gauss_legendre(NJ, x.data(), w.data());
    return Ib_quadrature_jaffe(R, Mb, Rb, NJ, x.data(), w.data());
}
// reading U': I_ext(R) for a bulge (Mb, Rb, profile) in the field of up to two discs and a halo (pins)
double bo_Ib_ext_quadrature(double R, double Mb, double Rb, int bulge_profile, double Md1, double Rd1, double Md2, double Rd2,
                            double Mh, double Rh, int halo_profile, unsigned comps, int NJ) {
    Theta t{};
    t.Mb = Mb; t.Rb = Rb; t.Md[0] = Md1; t.Rd[0] = Rd1; t.Md[1] = Md2; t.Rd[1] = Rd2; t.Mh = Mh; t.Rh = Rh;
    std::vector<double> x(NJ), w(NJ);
    gauss_legendre(NJ, x.data(), w.data());
    return Ib_ext_quadrature(R, t, comps, halo_profile, bulge_profile, Mb, Rb, NJ, x.data(), w.data());
}
double bo_rho_bulge(double x, double Mb, double Rb, int bulge_profile) { return rho_bulge(x, Mb, Rb, bulge_profile); }
double bo_G() { return kG; }
double bo_kappa(double dist_mpc) { return dist_mpc * kArcsecKpcPerMpc; }

int bo_psf_halfwidth(double sigma_pix, int s, double trunc) { return psf_halfwidth(sigma_pix, s, trunc); }
int bo_psf_taps(double sigma_pix, int s, double trunc, double *g /*[2 r_k + 1]*/) {
    std::vector<double> t;
    psf_taps(sigma_pix, s, trunc, t);
    std::memcpy(g, t.data(), t.size() * sizeof(double));
    return (int(t.size()) - 1) / 2;
}

// ---- maps ----
// fine: [4][N_y s + 2 r_k][N_x s + 2 r_k], un-convolved B_tot, v_los, sigma_los, <L/M>. Returns 0, or -1 (bad setup), -2 (theta out of domain).
int bo_model_fine(const double *theta, int nx, int ny, double pix, int s, double dist_mpc, double sigma_pix,
                  double trunc, unsigned comps, int profiles, int NJ, double *fine) {
    Setup S;
    if (!make_setup(S, nx, ny, pix, s, dist_mpc, sigma_pix, trunc, comps, profiles, NJ)) return -1;
    Theta t = decode(theta, comps);
    if (!t.valid) return -2;
    fine_maps(S, t, fine);
    return 0;
}

// steps 9-10 alone on caller-supplied fine maps (pin: brute-force 2-D sums, flux conservation)
int bo_convolve_rebin(const double *fine, int nx, int ny, int s, double sigma_pix, double trunc, int psf_weighting,
                      double *maps) {
    Setup S;
    if (!make_setup(S, nx, ny, 1.0, s, 1.0, sigma_pix, trunc, C_DISC1, psf_weighting << 16, 1)) return -1;
    convolve_rebin(S, fine, maps);
    return 0;
}

// maps: [B][4][ny][nx] = B [Lsun/pc^2], v_los [km/s], sigma_los [km/s], M/L.  Out-of-domain theta -> NaN.
int bo_model_maps(const double *theta, int B, int nx, int ny, double pix, int s, double dist_mpc,
                  double sigma_pix, double trunc, unsigned comps, int profiles, int NJ, double *maps) {
    Setup S;
    if (!make_setup(S, nx, ny, pix, s, dist_mpc, sigma_pix, trunc, comps, profiles, NJ)) return -1;
    std::vector<double> fine;
    for (int b = 0; b < B; ++b) model_one(S, theta + 17 * (size_t)b, maps + (size_t)b * 4 * nx * ny, fine);
    return 0;
}

// eq. 20 with the error model of App. C: log10 (M/L)_alpha = a + b (m_beta - m_gamma);
// its uncertainty propagates the magnitude errors and adds the scatter sigma_alpha of the relation in quadrature:
// d log10(M/L) = sqrt(b^2 (dm_beta^2 + dm_gamma^2) + sigma_alpha^2);  to first order d(M/L) = ln 10 (M/L) d log10(M/L).
void bo_ml_from_colour(const double *m_beta, const double *m_gamma, const double *dm_beta, const double *dm_gamma,
                       long n, double a, double b, double sigma_alpha, double *ml, double *ml_err) {
    for (long i = 0; i < n; ++i) {
        double logml = a + b * (m_beta[i] - m_gamma[i]);
        double dlog = std::sqrt(b * b * (dm_beta[i] * dm_beta[i] + dm_gamma[i] * dm_gamma[i]) + sigma_alpha * sigma_alpha);
        ml[i] = std::pow(10.0, logml);
        ml_err[i] = std::log(10.0) * ml[i] * dlog;
    }
}

// step 11, eq. 18 (reading L): Gaussian log-likelihood of given model maps.
double bo_loglike_of_maps(const double *maps, const double *data, const double *err, const unsigned char *mask,
                          int nx, int ny) {
    double sum = 0.0;
    for (size_t p = 0; p < (size_t)4 * nx * ny; ++p)
        if (mask[p]) {
            double z = (data[p] - maps[p]) / err[p];
            sum += -0.5 * (z * z + std::log(2 * kPi * err[p] * err[p]));
        }
    return sum;
}

// logL[B]; out-of-domain theta -> -inf.  maps_out may be NULL, else receives [B][4][ny][nx].
int bo_loglike(const double *theta, int B, int nx, int ny, double pix, int s, double dist_mpc, double sigma_pix,
               double trunc, unsigned comps, int profiles, int NJ, const double *data, const double *err,
               const unsigned char *mask, double *logL, double *maps_out) {
    Setup S;
    if (!make_setup(S, nx, ny, pix, s, dist_mpc, sigma_pix, trunc, comps, profiles, NJ)) return -1;
    std::vector<double> fine, maps((size_t)4 * nx * ny);
    for (int b = 0; b < B; ++b) {
        Theta t = decode(theta + 17 * (size_t)b, comps);
        double *m = maps_out ? maps_out + (size_t)b * 4 * nx * ny : maps.data();
        model_one(S, theta + 17 * (size_t)b, m, fine);
        logL[b] = t.valid ? bo_loglike_of_maps(m, data, err, mask, nx, ny)
                          : -std::numeric_limits<double>::infinity();
    }
    return 0;
}

}  // extern "C"
