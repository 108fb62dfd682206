// bang_kernels.cuh -- the hot path: per-theta decode + radial table (a0, a1), per-fine-cell model (a2, a3), separable
// PSF fused with the rebin (a4, a5) and the masked chi-square reduction (a6), in ONE persistent kernel per batch.
// Step names are those of SURVEY.md sec. 8(a) / DESIGN.md "The path".  T = float (BANG_FP32) or double (BANG_FP64).
#pragma once
#include <cuda_runtime.h>
#include <cstdio>

#include "bang_math.cuh"

// -DBANG_CHECK: a debug build whose kernels trap on a table index or a row-buffer offset out of range (the stand-in for
// compute-sanitizer, which is closed on the GPU pool); the release build relies on decode_theta's range checks.
#ifdef BANG_CHECK
#define BANG_ASSERT(cond) do { if (!(cond)) { printf("BANG_CHECK failed: %s (%s:%d)\n", #cond, __FILE__, __LINE__); __trap(); } } while (0)
#else
#define BANG_ASSERT(cond) do { } while (0)
#endif

namespace bang {

constexpr int kNTheta = 17;      // Table 1
constexpr int kVcOct = 32;           // octaves of r^2 the per-theta v_c table holds (a theta that needs more takes the direct path)
constexpr int kBOct = 24;            // octaves of s^2 = R^2/R_b^2 the per-theta slice of the bulge tables holds (likewise)
constexpr unsigned C_BULGE = 1u, C_DISC1 = 2u, C_DISC2 = 4u, C_HALO = 8u;
constexpr int kBulgeOctLo = -44, kBulgeOctHi = 36;    // universal bulge tables: s^2 in [2^-44, 2^36)
constexpr int kFOctLo = -60, kFOctHi = 10;            // universal Freeman table: y^2 in [2^-60, 2^10)

// ---- fast fp32 special-function-unit ops (MUFU), and their fp64 counterparts -------------------------------------
BANG_D float fast_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
BANG_D float fast_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
BANG_D float fast_sqrt(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
BANG_D float fast_exp2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
BANG_D double fast_rsqrt(double x) { return 1.0 / sqrt(x); }
BANG_D double fast_rcp(double x) { return 1.0 / x; }
BANG_D double fast_sqrt(double x) { return sqrt(x); }
BANG_D double fast_exp2(double x) { return exp2(x); }

// ---- a piecewise-polynomial table in global or shared memory -----------------------------------------------------
template <typename T>
struct PolyTab {
    const T* coef;    // [n_cells][n_func][D+1], monomial coefficients in t in [-1,1)
    int first;        // global interval number (tab_cell) of coef[0]
    int n_cells;
};

template <typename T, int D>
BANG_D T horner(const T* c, T t) {
    T v = c[D];
#pragma unroll
    for (int d = D - 1; d >= 0; --d) v = fma(v, t, c[d]);
    return v;
}

// ---- per-theta constants (a0), decoded once per theta in fp64 by one thread ----------------------------------------
struct ThetaD {      // what the table build needs, in double
    double GMb, Rb;              // bulge v_c^2 = GMb r/(r+Rb)^2  (eq. 2)
    double Ad[2], inv2Rd[2];     // disc  v_c^2 = Ad F(r inv2Rd),  Ad = 2 G M_d/R_d  (eq. 9, reading D)
    double Ah, hs;               // halo: Hernquist GMh, Rh;  NFW: G M200/mu(c), 1/r_s  (reading H)
    double ghc, ghs, gxp0, gyp0, gtan2i;   // the geometry of ThetaC (hc, hs, xp0, yp0, tan2i) in double: direct path
    double s2near;               // s^2 = R^2/R_b^2 of the cell nearest to the centre (entry 0 of the per-theta bulge tables)
};
template <typename T>
struct ThetaC {
    int valid;                   // 0: theta outside the model's domain (NaN maps, logL = -inf)
    int slow;                    // 1: radii on this theta's grid leave the tabulated ranges -> direct evaluation per cell
    int jcx, jcy;                // fine cell (buffer coordinates) nearest to the galaxy centre
    int vfirst, vcells;          // per-theta v_c table: first global interval, number of regular intervals (entry 0 of the
                                 // table is the constant v_c of the cell nearest to the centre, entries 1.. the intervals)
    T vc_near;                   // v_c at that cell
    int bfirst, bcells;          // per-theta bulge tables over s^2 = R^2/R_b^2: first global interval, number of regular
                                 // intervals (entry 0 = the cell nearest to the centre, as for v_c)
    T sig_near, J_near;          // SigmaTilde and J at that cell
    T hc, hs;                    // h cos PA, h sin PA   (h = fine cell size in kpc)
    T xp0, yp0;                  // rotated offset of cell (jcx, jcy) from the centre
    T tan2i;                     // tan^2 i = 1/cos^2 i - 1
    T invRb2, ampBb, ampIb, MLb; // bulge: s^2 = R^2 invRb2;  B_b = ampBb SigmaTilde;  B_b sigma_b^2 = ampIb J
    T cexp[2], ampBd[2], ampSd[2]; // disc j: B_d = ampBd 2^(r cexp), Sigma_d = ampSd 2^(r cexp) = (M/L)_d B_d
    T vkB[2], q3B[2];            // -sin i k_j ampBd_j   and   (1 - k_j^2)/3 ampBd_j: the light weights of eqs. 14, 15
    ThetaD d;
    alignas(16) int kpack[28];   // fp32 mode: the CellK constants below, packed for 128-bit broadcast loads (pack_cellk)
};

// geometry of the run, the same for every theta (built on the host at bang_create)
struct GridC {
    int nx, ny, s, rk;
    int nfx, nfy;                // evaluated fine cells: n s + 2 r_k (buffer coordinates 0..nf-1)
    double jsx, jsy;             // buffer index of the sky origin: r_k - 1/2 + n s/2
    double spx;                  // s / pix_arcsec: fine cells per arcsec
    double h;                    // fine cell size [kpc]
    unsigned comps;
    int halo_profile;            // 0 Hernquist (paper), 1 NFW (reading H)
    int bulge_profile;           // 0 Hernquist (paper default), 1 Jaffe (App. B)
    int flux;                    // 1: flux-weighted PSF variant (reading G'): the fine fields are the light moments
    int bulge_potential;         // 1: the bulge's dispersion in the total potential (reading U'): + I_ext, see ext_Itilde
};

// reading U' is active: a bulge, the switch, and something other than the bulge to pull on it
inline __host__ __device__ bool has_ext(const GridC& g) {
    return g.bulge_potential && (g.comps & C_BULGE) && (g.comps & (C_DISC1 | C_DISC2 | C_HALO));
}

struct FitC {                    // Chebyshev-node fit of degree D: nodes t_k and the inverse Vandermonde matrix
    double tnode[8];
    double vinv[64];             // vinv[d*(D+1)+k]: coefficient d = sum_k vinv[d][k] f(t_k)
};

// Freeman-disc function from the universal table (y^2 in [2^-60, 2^10)), its leading small-y form, and the
// large-argument expansion (DLMF 10.40.6) beyond.
template <typename T>
BANG_D double freeman_F_tab(const PolyTab<T>& Ftab, double y2) {
    if (y2 >= 1024.0) {
        const double iz2 = 0.25 / y2;
        double a0 = 1.0, a1 = 1.0, sum = 0.0;
#pragma unroll 1
        for (int k = 1; k < 14; ++k) {
            const double odd = 2.0 * k - 1.0;
            const double f = -(odd / (2.0 * k)) * iz2;
            a0 *= f * (0.0 - odd * odd);
            a1 *= f * (4.0 - odd * odd);
            sum += a0 - a1;
        }
        return 0.5 * sqrt(y2) * sum;
    }
    if (y2 < 8.673617379884035e-19)     // 2^-60: F = y^2 [-ln(y/2) - gamma - 1/2] (1 + O(y^2 ln y))
        return y2 * (-0.5 * log(0.25 * y2) - kEulerGamma - 0.5);
    T t;
    const int c = min(max(tab_cell((T)y2, t) - Ftab.first, 0), Ftab.n_cells - 1);
    return (double)horner<T, TabCfg<T>::D>(Ftab.coef + (size_t)c * (TabCfg<T>::D + 1), t);
}

// total circular speed squared at radius r in the disc plane (eq. 10)
// comps: which terms to sum (g.comps for eq. 10; g.comps & ~C_BULGE for the "external" field of reading U')
template <typename T>
BANG_D double vc2_total(const ThetaD& d, const GridC& g, const unsigned comps, const PolyTab<T>& Ftab, double r) {
    double v2 = 0.0;
    if (comps & C_BULGE) {
        const double a = r + d.Rb;
        v2 += g.bulge_profile == 1 ? d.GMb / a : d.GMb * r / (a * a);      // eq. B2 / eq. 2
    }
#pragma unroll
    for (int j = 0; j < 2; ++j)
        if (comps & (j ? C_DISC2 : C_DISC1)) {
            const double y = r * d.inv2Rd[j];
            v2 += d.Ad[j] * freeman_F_tab(Ftab, y * y);
        }
    if (comps & C_HALO) {
        if (g.halo_profile == 1) v2 += d.Ah * nfw_mu<double>(r * d.hs) / r;
        else { const double a = r + d.hs; v2 += d.Ah * r / (a * a); }
    }
    return v2;
}

// The same in fp32, for the table build of fp32 mode: the node values are stored as fp32 anyway and the interpolation
// error of the table is 2e-7, so evaluating eq. 10 in fp32 (relative error ~3e-7) costs nothing that the mode's 1e-4
// tolerance sees, and the per-theta prologue gets ~6x cheaper (it is 6 % of the instructions at config 2).
BANG_D float freeman_F_tab_f(const PolyTab<float>& Ftab, float y2) {
    if (y2 >= 1024.0f) {                               // DLMF 10.40.6: 3 terms reach 1e-9 at y^2 = 1024
        const float iz2 = 0.25f / y2;
        float a0 = 1.0f, a1 = 1.0f, sum = 0.0f;
#pragma unroll
        for (int k = 1; k < 4; ++k) {
            const float odd = 2.0f * k - 1.0f;
            const float f = -(odd / (2.0f * k)) * iz2;
            a0 *= f * (0.0f - odd * odd);
            a1 *= f * (4.0f - odd * odd);
            sum += a0 - a1;
        }
        return 0.5f * sqrtf(y2) * sum;
    }
    if (y2 < 8.673617379884035e-19f) return y2 * (-0.5f * logf(0.25f * y2) - (float)kEulerGamma - 0.5f);
    float t;
    const int c = min(max(tab_cell(y2, t) - Ftab.first, 0), Ftab.n_cells - 1);
    return horner<float, TabCfg<float>::D>(Ftab.coef + (size_t)c * (TabCfg<float>::D + 1), t);
}
struct ThetaF { float GMb, Rb, Ad[2], inv2Rd[2], Ah, hs; };
BANG_D float vc2_total_f(const ThetaF& d, const GridC& g, const unsigned comps, const PolyTab<float>& Ftab, const float r) {
    float v2 = 0.0f;
    if (comps & C_BULGE) {
        const float ia = 1.0f / (r + d.Rb);
        v2 += g.bulge_profile == 1 ? d.GMb * ia : d.GMb * r * ia * ia;
    }
#pragma unroll
    for (int j = 0; j < 2; ++j)
        if (comps & (j ? C_DISC2 : C_DISC1)) {
            const float y = r * d.inv2Rd[j];
            v2 += d.Ad[j] * freeman_F_tab_f(Ftab, y * y);
        }
    if (comps & C_HALO) {
        if (g.halo_profile == 1) v2 += d.Ah * nfw_mu<float>(r * d.hs) / r;
        else { const float ia = 1.0f / (r + d.hs); v2 += d.Ah * r * ia * ia; }
    }
    return v2;
}

// a0: decode theta[17] (Table 1).  Run by ONE thread; everything in fp64.
template <typename T>
BANG_D void decode_theta(const double* __restrict__ th, const GridC& g, const PolyTab<T>& btab, const PolyTab<T>& Ftab, ThetaC<T>& c) {
    const unsigned comps = g.comps;
    c.valid = 0;
    c.slow = 0;
    bool ok = isfinite(th[0]) && isfinite(th[1]) && isfinite(th[2]) && isfinite(th[3]) && fabs(th[3]) < 90.0;
    if (comps & C_BULGE) ok = ok && isfinite(th[4]) && th[5] > 0 && isfinite(th[5]) && th[12] > 0 && isfinite(th[12]);
    for (int j = 0; j < 2; ++j)
        if (comps & (j ? C_DISC2 : C_DISC1))
            ok = ok && isfinite(th[6 + 2 * j]) && th[7 + 2 * j] > 0 && isfinite(th[7 + 2 * j]) && th[13 + j] > 0 &&
                 isfinite(th[13 + j]) && fabs(th[15 + j]) <= 1.0;
    if (comps & C_HALO) ok = ok && isfinite(th[10]) && th[11] > 0 && isfinite(th[11]);
    if (!ok) return;

    // sec. 2.1 (fn 2 at :68): centre, position angle (counter-clockwise from +x), inclination
    double sp, cp, si, ci;
    sincos(th[2] * (kPi / 180.0), &sp, &cp);
    sincos(th[3] * (kPi / 180.0), &si, &ci);
    const double h = g.h;
    const double Jsx = g.jsx + th[0] * g.spx, Jsy = g.jsy + th[1] * g.spx;      // fractional buffer index of the centre
    const int jcx = (int)fmin(fmax(rint(Jsx), 0.0), (double)(g.nfx - 1));
    const int jcy = (int)fmin(fmax(rint(Jsy), 0.0), (double)(g.nfy - 1));
    const double dx = (jcx - Jsx) * h, dy = (jcy - Jsy) * h;                    // offset of that cell from the centre [kpc]
    c.jcx = jcx; c.jcy = jcy;
    c.hc = (T)(h * cp); c.hs = (T)(h * sp);
    const double xp0 = dx * cp + dy * sp, yp0 = -dx * sp + dy * cp;
    c.xp0 = (T)xp0;
    c.yp0 = (T)yp0;
    const double inv_ci2 = 1.0 / (ci * ci);
    const double tan2i = (si * si) / (ci * ci);
    c.tan2i = (T)tan2i;
    c.d.ghc = h * cp; c.d.ghs = h * sp; c.d.gxp0 = xp0; c.d.gyp0 = yp0; c.d.gtan2i = tan2i;

    // Range of radii on this theta's grid.  R^2 is smallest at the cell nearest to the centre (R2min); every OTHER cell
    // of the lattice has R^2 >= h^2/4 when the centre lies inside that cell, >= R2min when it lies outside the grid.
    // Maxima at the corners.  The per-theta v_c table covers [Llo, r2max] with its regular intervals and serves the
    // nearest cell with a dedicated constant entry, so that a centre that falls on (or next to) a cell centre does not
    // cost tens of empty octaves.
    const double floor2 = ldexp(1.0, 2 * kRFloorLog2);
    const double R2min = fmax(dx * dx + dy * dy, floor2);
    double R2max = 0.0, r2max = 0.0;
    for (int k = 0; k < 4; ++k) {
        const double a = ((k & 1) ? g.nfx - 1 : 0) - Jsx, b = ((k & 2) ? g.nfy - 1 : 0) - Jsy;
        const double X = a * h, Y = b * h;
        const double xp = X * cp + Y * sp, yp = -X * sp + Y * cp;
        R2max = fmax(R2max, xp * xp + yp * yp);
        r2max = fmax(r2max, xp * xp + yp * yp * inv_ci2);
    }
    R2max = fmax(R2max, floor2); r2max = fmax(r2max, floor2);
    const double lo_m = 1.0 - 0x1p-10, hi_m = 1.0 + 0x1p-10;
    const bool inside = fabs(dx) <= 0.5 * h * hi_m && fabs(dy) <= 0.5 * h * hi_m;
    const double Llo = inside ? fmin(0.25 * h * h, r2max) : R2min;
    const double LloR = inside ? fmin(0.25 * h * h, R2max) : R2min;           // the same for R^2 (the bulge tables)
    const int e_lo = ilogb(Llo * lo_m), e_hi = ilogb(r2max * hi_m);
    if (e_hi - e_lo + 1 > kVcOct || e_hi > 100) c.slow = 1;                      // direct evaluation (eval_cell_direct)
    // fp32 mode: r^2 = R^2 + y'^2 tan^2 i amplifies the rounding of y' (relative ~2^-23 per operation) by tan i; beyond
    // tan i = 64 (i > 89.1 deg) that approaches the mode's 1e-4, so such theta take the direct path (fp64 geometry)
    if (sizeof(T) == 4 && tan2i > 4096.0) c.slow = 1;
    c.vfirst = tab_first_cell<T>(e_lo);
    c.vcells = c.slow ? 0 : (e_hi - e_lo + 1) << TabCfg<T>::M;

    ThetaD& d = c.d;
    // bulge: eq. 1-6
    c.invRb2 = T(1); c.ampBb = T(0); c.ampIb = T(0); c.MLb = T(1);
    c.bfirst = 0; c.bcells = 0; c.sig_near = T(0); c.J_near = T(0);
    d.GMb = 0.0; d.Rb = 1.0; d.s2near = 1.0;
    if (comps & C_BULGE) {      // eq. 1-6 (Hernquist) or App. B (Jaffe): both scale-free in s = R/R_b
        const double Mb = exp10(th[4]), Rb = th[5], MLb = th[12];
        const double inv = 1.0 / (Rb * Rb);
        // s^2 = R^2/R_b^2 must stay inside the scale-free tables; otherwise the direct path evaluates eq. 4-6 per cell
        if (!(R2min * inv * lo_m >= ldexp(1.0, kBulgeOctLo)) || !(R2max * inv * hi_m < ldexp(1.0, kBulgeOctHi))) c.slow = 1;
        c.invRb2 = (T)inv;
        // the theta's slice of the scale-free tables: [LloR, R2max] / R_b^2 in regular intervals + entry 0 for the cell
        // nearest to the centre, exactly as for v_c
        const int eb_lo = ilogb(LloR * inv * lo_m), eb_hi = ilogb(R2max * inv * hi_m);
        if (eb_hi - eb_lo + 1 > kBOct) c.slow = 1;
        c.bfirst = tab_first_cell<T>(eb_lo);
        c.bcells = c.slow ? 0 : (eb_hi - eb_lo + 1) << TabCfg<T>::M;
        d.s2near = R2min * inv;
        if (!c.slow) {
            T tt;
            const int cell = min(max(tab_cell((T)d.s2near, tt) - btab.first, 0), btab.n_cells - 1);
            const T* pc = btab.coef + (size_t)cell * (2 * (TabCfg<T>::D + 1));
            c.sig_near = horner<T, TabCfg<T>::D>(pc, tt);
            c.J_near = horner<T, TabCfg<T>::D>(pc + TabCfg<T>::D + 1, tt);
        }
        if (g.bulge_profile == 1) {
            c.ampBb = (T)(Mb / (Rb * Rb) / MLb * 1e-6);                                  // eq. B4, in Lsun/pc^2
            c.ampIb = (T)(kG * Mb * Mb / (4.0 * kPi * Rb * Rb * Rb) * 2.0 / MLb * 1e-6); // l.o.s. integral of B1 x B3
        } else {
            c.ampBb = (T)(Mb / (2.0 * kPi * Rb * Rb) / MLb * 1e-6);                      // eq. 4, in Lsun/pc^2
            c.ampIb = (T)(kG * Mb * Mb / (2.0 * kPi * Rb * Rb * Rb) * 2.0 / MLb * 1e-6); // eq. 6 first form
        }
        c.MLb = (T)MLb;
        d.GMb = kG * Mb; d.Rb = Rb;
    }
    // discs: eq. 7-9, 11-12
    for (int j = 0; j < 2; ++j) {
        c.cexp[j] = T(0); c.ampBd[j] = T(0); c.ampSd[j] = T(0); c.vkB[j] = T(0); c.q3B[j] = T(0);
        d.Ad[j] = 0.0; d.inv2Rd[j] = 1.0;
        if (comps & (j ? C_DISC2 : C_DISC1)) {
            const double Md = exp10(th[6 + 2 * j]), Rd = th[7 + 2 * j], ML = th[13 + j], k = th[15 + j];
            c.cexp[j] = (T)(-1.4426950408889634 / Rd);
            const double aB = Md / (2.0 * kPi * Rd * Rd * ci) / ML * 1e-6;               // eq. 7-8, in Lsun/pc^2
            c.ampBd[j] = (T)aB;
            c.ampSd[j] = (T)(aB * ML);
            c.vkB[j] = (T)(-si * k * aB);                                                // eq. 11 inside eq. 14
            c.q3B[j] = (T)((1.0 - k * k) / 3.0 * aB);                                    // eq. 12 inside eq. 15
            d.Ad[j] = 2.0 * kG * Md / Rd;
            d.inv2Rd[j] = 0.5 / Rd;
        }
    }
    // halo (reading H)
    d.Ah = 0.0; d.hs = 1.0;
    if (comps & C_HALO) {
        const double Mh = exp10(th[10]);
        if (g.halo_profile == 1) {
            const double cc = th[11];
            d.Ah = kG * Mh / nfw_mu<double>(cc);
            d.hs = cc / nfw_r200(Mh);
        } else {
            d.Ah = kG * Mh; d.hs = th[11];
        }
    }
    // v_c at the cell nearest to the centre (entry 0 of the per-theta table)
    c.vc_near = (T)sqrt(vc2_total<T>(d, g, g.comps, Ftab, sqrt(R2min + yp0 * yp0 * tan2i)));
    c.valid = 1;
}
template <typename T> BANG_D void pack_cellk(ThetaC<T>& c);

// Node values -> monomial coefficients, in place: cells x (D+1) values at the Chebyshev nodes of each interval become the
// D+1 coefficients of its interpolant (fit.vinv, fp64 arithmetic).  One thread per interval; no barrier inside.
template <typename T>
BANG_D void fit_cells(const FitC& fit, T* reg, const int cells) {
    constexpr int NC = TabCfg<T>::D + 1;
    for (int cell = threadIdx.x; cell < cells; cell += blockDim.x) {
        T* p = reg + cell * NC;
        double f[NC], co[NC];
#pragma unroll
        for (int k = 0; k < NC; ++k) f[k] = (double)p[k];
#pragma unroll
        for (int d = 0; d < NC; ++d) {
            double a = 0.0;
#pragma unroll
            for (int k = 0; k < NC; ++k) a = fma(fit.vinv[d * NC + k], f[k], a);
            co[d] = a;
        }
#pragma unroll
        for (int d = 0; d < NC; ++d) p[d] = (T)co[d];
    }
}

// a1: the per-theta radial table v_c(r), a piecewise polynomial in u = r^2 on the pseudo-log grid, built cooperatively
// by the CTA in shared memory: every thread evaluates v_c at Chebyshev nodes, then one thread per interval turns its D+1
// node values into monomial coefficients.  Entry 0 is the constant v_c of the cell nearest to the centre; the regular
// intervals follow.  Must be called by all threads; ends with a __syncthreads().
template <typename T>
BANG_D void build_vc_table(const ThetaC<T>& c, const GridC& g, const FitC& fit, const PolyTab<T>& Ftab, T* vtab) {
    constexpr int D = TabCfg<T>::D, NC = D + 1;
    const int n = c.vcells * NC;
    if (threadIdx.x < NC) vtab[threadIdx.x] = threadIdx.x == 0 ? c.vc_near : T(0);
    T* reg = vtab + NC;
    if constexpr (sizeof(T) == 4) {
        const ThetaF df{(float)c.d.GMb, (float)c.d.Rb, {(float)c.d.Ad[0], (float)c.d.Ad[1]},
                        {(float)c.d.inv2Rd[0], (float)c.d.inv2Rd[1]}, (float)c.d.Ah, (float)c.d.hs};
        for (int i = threadIdx.x; i < n; i += blockDim.x) {
            const int cell = i / NC, k = i - cell * NC;
            double lo, width;
            tab_interval<T>(c.vfirst + cell, lo, width);
            const float u = (float)(lo + 0.5 * width * (fit.tnode[k] + 1.0));
            reg[i] = sqrtf(vc2_total_f(df, g, g.comps, Ftab, sqrtf(u)));
        }
    } else {
        for (int i = threadIdx.x; i < n; i += blockDim.x) {
            const int cell = i / NC, k = i - cell * NC;
            double lo, width;
            tab_interval<T>(c.vfirst + cell, lo, width);
            const double u = lo + 0.5 * width * (fit.tnode[k] + 1.0);
            reg[i] = (T)sqrt(vc2_total(c.d, g, g.comps, Ftab, sqrt(u)));
        }
    }
    __syncthreads();
    fit_cells<T>(fit, reg, c.vcells);
    __syncthreads();
}

// ---- reading U' (variant; PAPER.md:107 and :417-419 name it as the model's first limitation): the bulge's dispersion in
// the TOTAL potential of eq. 10.  Sigma_b sigma_b^2 gains the pull of the discs and the halo on the bulge's stars,
//   I_ext(R) = 2 int_R^inf rho_b(x) v_ext^2(x) sqrt(x^2 - R^2)/x dx,   v_ext^2 = sum_j eq. 9 + halo,
// by the same N_J-node Gauss-Legendre rule as eq. 6 (reading B) on t in (0,1) with x = R + L t^2/(1-t), L = sqrt(R^2+R_b^2).
// In units of R_b (s = R/R_b, x~ = x/R_b) and of the amplitude ampIb of the scale-free J:
//   Itilde_ext(s) = I_ext / (2 G M_b^2/(2 pi R_b^3)) [Hernquist; likewise Jaffe] = (R_b/(G M_b)) sum_k L~ b_k rho~(x~_k) v_ext^2(R_b x~_k) root_k/x~_k,
//   x~_k = s + L~ a_k,  root_k = sqrt(L~ a_k (2 s + L~ a_k)),  a_k = t_k^2/(1-t_k),  b_k = w_k t_k (2-t_k)/(1-t_k)^2 (host, long double),
//   rho~ = 1/(x~ (1+x~)^3) (eq. 1) or 1/(x~^2 (1+x~)^2) (eq. B1).
// Unlike J it is not scale-free (it depends on R_d/R_b, R_h/R_b, ...): it is tabulated PER THETA over the s^2 this theta's
// grid spans -- north_star's kernel (1) in earnest.  R: the arithmetic type (float in fp32 mode, double otherwise).
struct QuadC {
    const double2* qd;           // [N_J] {a_k, b_k} (device)
    const float2* qf;            // the same rounded to fp32
    int NJ;
    // Itilde_ext is evaluated by the rule only at the ND Chebyshev nodes (in w = log2 s^2) of panels of `span` octaves and
    // carried to the table's own nodes by barycentric interpolation of ln Itilde_ext(w) (measured on prior-drawn theta:
    // 8 nodes per 2 octaves reproduce the rule to 8e-8, 12 nodes per octave to 6e-14): bx = the nodes on [-1,1], bw = the
    // barycentric weights (-1)^k sin((2k+1) pi/(2 ND)).
    int ND, span;
    double bx[12], bw[12];
};
constexpr int kExtMaxND = 12;
BANG_D void quad_node(const QuadC& q, int k, double& a, double& b) { const double2 v = __ldg(q.qd + k); a = v.x; b = v.y; }
BANG_D void quad_node(const QuadC& q, int k, float& a, float& b) { const float2 v = __ldg(q.qf + k); a = v.x; b = v.y; }
template <typename T>
BANG_D double vext2(const ThetaD& d, const ThetaF&, const GridC& g, const PolyTab<T>& Ftab, double r) {
    return vc2_total<T>(d, g, g.comps & ~C_BULGE, Ftab, r);
}
BANG_D float vext2(const ThetaD&, const ThetaF& df, const GridC& g, const PolyTab<float>& Ftab, float r) {
    return vc2_total_f(df, g, g.comps & ~C_BULGE, Ftab, r);
}
template <typename R, typename T>
BANG_D R ext_Itilde(const R s, const ThetaD& d, const ThetaF& df, const GridC& g, const PolyTab<T>& Ftab, const QuadC& q,
                    const int k0 = 0, const int kstep = 1) {
    // (k0, kstep): the nodes k0, k0 + kstep, ... only -- the table build deals one rule out over four lanes
    const R L = sqrt(fma(s, s, R(1)));
    const R Rb = (R)d.Rb;
    R sum = R(0);
#pragma unroll 1
    for (int k = k0; k < q.NJ; k += kstep) {
        R a, b;
        quad_node(q, k, a, b);
        const R dd = L * a;                               // x~ - s
        const R x = s + dd;
        const R root = sqrt(dd * (R(2) * s + dd));        // sqrt(x~^2 - s^2) without cancellation
        const R rx = R(1) / x, r1 = R(1) / (R(1) + x);
        // rho~ root / x~ as a product of reciprocals (no overflow of x~^2 (1+x~)^3 in fp32)
        const R shape = g.bulge_profile == 1 ? rx * rx * rx * r1 * r1 : rx * rx * r1 * r1 * r1;
        sum = fma(L * b * root * shape, vext2(d, df, g, Ftab, Rb * x), sum);
    }
    return sum * (R)(d.Rb / d.GMb);
}

// a1 (continued): the per-theta bulge tables in shared memory.
//   fp32 mode: bs[entry][2][D+1] = {SigmaTilde, J (+ Itilde_ext)} -- entry 0 is the cell nearest to the centre (constants),
//   entries 1.. are this theta's slice of the scale-free tables, copied from global memory: the per-cell look-up is then
//   two 128-bit shared loads instead of two gathers through L1.
//   fp64 mode: the scale-free tables stay in global memory; bs[entry][D+1] = Itilde_ext only, and only for reading U'.
// scratch: room for (bcells (D+1) + 1) values of T (the row buffer, idle during the prologue).
// Must be called by all threads; ends with a __syncthreads().
template <typename T>
BANG_D void build_bulge_tables(const ThetaC<T>& c, const GridC& g, const FitC& fit, const PolyTab<T>& btab, const PolyTab<T>& Ftab,
                               const QuadC& q, T* bs, T* scratch) {
    constexpr int D = TabCfg<T>::D, NC = D + 1;
    const bool ext = has_ext(g);
    if constexpr (sizeof(T) == 4) {
        if (!(g.comps & C_BULGE)) { __syncthreads(); return; }
        const float4* src = reinterpret_cast<const float4*>(btab.coef + (size_t)(c.bfirst - btab.first) * (2 * NC));
        float4* dst = reinterpret_cast<float4*>(bs);
        if (threadIdx.x == 0) {
            dst[0] = make_float4(c.sig_near, 0.f, 0.f, 0.f);
            dst[1] = make_float4(c.J_near, 0.f, 0.f, 0.f);
        }
        for (int i = threadIdx.x; i < c.bcells * 2; i += blockDim.x) dst[2 + i] = __ldg(src + i);
    }
    if (!ext) { __syncthreads(); return; }
    // Itilde_ext by the N_J-node rule at the coarse panel nodes (+ the nearest cell, directly), ...
    const int n = c.bcells * NC;
    const int octaves = c.bcells >> TabCfg<T>::M, panels = (octaves + q.span - 1) / q.span, ncoarse = panels * q.ND;
    T* coarse = scratch + n + 4;                         // [panels][ND] ln Itilde_ext, then [ncoarse] = the nearest cell's value
    const int e0 = (c.bfirst >> TabCfg<T>::M) - (sizeof(T) == 4 ? 127 : 1023);     // first octave of the slice
    {
        const ThetaF df{(float)c.d.GMb, (float)c.d.Rb, {(float)c.d.Ad[0], (float)c.d.Ad[1]},
                        {(float)c.d.inv2Rd[0], (float)c.d.inv2Rd[1]}, (float)c.d.Ah, (float)c.d.hs};
        // every evaluation of the rule is dealt out over four neighbouring lanes (nodes k = part, part + 4, ...; the partial
        // sums meet by shuffle), so that the ~70 evaluations of a theta keep a 64-thread CTA busy as well as a 128-thread one
        for (int base = 0; base < 4 * (ncoarse + 1); base += blockDim.x) {
            const int item = base + threadIdx.x, i = item >> 2, part = item & 3;
            const bool on = i <= ncoarse;
            double s2 = 1.0;
            if (on) {
                if (i == ncoarse) s2 = c.d.s2near;
                else {
                    const int pn = i / q.ND, k = i - pn * q.ND;
                    s2 = exp2((double)(e0 + pn * q.span) + 0.5 * q.span * (q.bx[k] + 1.0));
                }
            }
            T v = T(0);
            if (on) {
                if constexpr (sizeof(T) == 4) v = ext_Itilde<float, float>(sqrtf((float)s2), c.d, df, g, Ftab, q, part, 4);
                else v = (T)ext_Itilde<double, T>(sqrt(s2), c.d, df, g, Ftab, q, part, 4);
            }
            v += __shfl_xor_sync(0xffffffffu, v, 1);
            v += __shfl_xor_sync(0xffffffffu, v, 2);
            if (on && part == 0) coarse[i] = i == ncoarse ? v : (T)log(fmax((double)v, 1e-300));
        }
    }
    __syncthreads();
    // ... then at the Chebyshev nodes of every interval of the slice by barycentric interpolation in w = log2 s^2
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const int cell = i / NC, k = i - cell * NC;
        double lo, width;
        tab_interval<T>(c.bfirst + cell, lo, width);
        const double w = log2(lo + 0.5 * width * (fit.tnode[k] + 1.0));
        const int pn = min((int)((w - e0) / q.span), panels - 1);
        const double x = (w - (e0 + pn * q.span)) * (2.0 / q.span) - 1.0;
        const T* gk = coarse + pn * q.ND;
        double num = 0.0, den = 0.0, hit = 0.0;
        bool exact = false;
        for (int j = 0; j < q.ND; ++j) {
            const double dx = x - q.bx[j];
            if (dx == 0.0) { exact = true; hit = (double)gk[j]; }
            const double wj = q.bw[j] / (dx == 0.0 ? 1.0 : dx);
            num = fma(wj, (double)gk[j], num);
            den += wj;
        }
        scratch[i] = (T)exp(exact ? hit : num / den);
    }
    if (threadIdx.x == 0) scratch[n] = coarse[ncoarse];
    __syncthreads();
    fit_cells<T>(fit, scratch, c.bcells);
    __syncthreads();
    if constexpr (sizeof(T) == 4) {
        // J += Itilde_ext, coefficient by coefficient (both are polynomials in the same t on the same interval)
        for (int i = threadIdx.x; i < n; i += blockDim.x) {
            const int cell = i / NC, k = i - cell * NC;
            bs[(size_t)(1 + cell) * (2 * NC) + NC + k] += scratch[i];
        }
        if (threadIdx.x == 0) bs[NC] += scratch[n];
    } else {
        for (int i = threadIdx.x; i < n; i += blockDim.x) bs[NC + i] = scratch[i];
        if (threadIdx.x < NC) bs[threadIdx.x] = threadIdx.x == 0 ? scratch[n] : T(0);
    }
    __syncthreads();
}
// number of T values of the per-theta bulge tables (bs above); 0 when the variant does not need them
template <typename T>
inline size_t bs_elems(const GridC& g) {
    constexpr int NC = TabCfg<T>::D + 1;
    const size_t entries = (size_t)kBOct * (1 << TabCfg<T>::M) + 1;
    if (!(g.comps & C_BULGE)) return 0;
    if (sizeof(T) == 4) return entries * 2 * NC;
    return has_ext(g) ? entries * NC : 0;
}

// per-theta constants of the fine-cell model, copied from shared memory into registers so that the per-cell code below
// touches shared memory only for its table look-up
template <typename T>
struct CellK {
    int jcx, jcy;
    int vfirst1;                 // global interval number of table entry 0 (= first regular interval - 1)
    int vlast;                   // last valid entry (BANG_CHECK builds only)
    int bfirst1, blast;          // the same for the per-theta bulge tables
    T hc, hs, xp0, yp0, tan2i;
    T invRb2, ampBb, ampIb, MLb;
    T cexp0, cexp1, ampBd0, ampBd1, ampSd0, ampSd1, vkB0, vkB1, q3B0, q3B1;
};
template <typename T>
BANG_D CellK<T> load_cellk(const ThetaC<T>& c) {
    CellK<T> k;
    if constexpr (sizeof(T) == 4) {
        // seven 128-bit broadcast loads instead of 25 scalar ones: the constants are re-read every super-row, and a
        // broadcast load costs a wavefront of the shared-memory pipe whatever its width
        const int4* s = reinterpret_cast<const int4*>(c.kpack);
        const int4 a = s[0], b = s[1], e = s[2], f = s[3], g = s[4], h = s[5];
        k.jcx = a.x; k.jcy = a.y; k.vfirst1 = a.z; k.bfirst1 = a.w;
        k.hc = __int_as_float(b.x); k.hs = __int_as_float(b.y); k.xp0 = __int_as_float(b.z); k.yp0 = __int_as_float(b.w);
        k.tan2i = __int_as_float(e.x); k.invRb2 = __int_as_float(e.y); k.ampBb = __int_as_float(e.z); k.ampIb = __int_as_float(e.w);
        k.MLb = __int_as_float(f.x); k.cexp0 = __int_as_float(f.y); k.cexp1 = __int_as_float(f.z); k.ampBd0 = __int_as_float(f.w);
        k.ampBd1 = __int_as_float(g.x); k.ampSd0 = __int_as_float(g.y); k.ampSd1 = __int_as_float(g.z); k.vkB0 = __int_as_float(g.w);
        k.vkB1 = __int_as_float(h.x); k.q3B0 = __int_as_float(h.y); k.q3B1 = __int_as_float(h.z);
        k.vlast = c.vcells; k.blast = c.bcells;      // read only by BANG_CHECK builds
    } else {
        k.jcx = c.jcx; k.jcy = c.jcy; k.vfirst1 = c.vfirst - 1; k.vlast = c.vcells;
        k.bfirst1 = c.bfirst - 1; k.blast = c.bcells;
        k.hc = c.hc; k.hs = c.hs; k.xp0 = c.xp0; k.yp0 = c.yp0; k.tan2i = c.tan2i;
        k.invRb2 = c.invRb2; k.ampBb = c.ampBb; k.ampIb = c.ampIb; k.MLb = c.MLb;
        k.cexp0 = c.cexp[0]; k.cexp1 = c.cexp[1]; k.ampBd0 = c.ampBd[0]; k.ampBd1 = c.ampBd[1];
        k.ampSd0 = c.ampSd[0]; k.ampSd1 = c.ampSd[1]; k.vkB0 = c.vkB[0]; k.vkB1 = c.vkB[1]; k.q3B0 = c.q3B[0]; k.q3B1 = c.q3B[1];
    }
    return k;
}
// fills ThetaC::kpack from the decoded fields (the thread that ran decode_theta; fp32 mode only)
template <typename T>
BANG_D void pack_cellk(ThetaC<T>& c) {
    if constexpr (sizeof(T) == 4) {
        int* q = c.kpack;
        q[0] = c.jcx; q[1] = c.jcy; q[2] = c.vfirst - 1; q[3] = c.bfirst - 1;
        const float v[19] = {c.hc, c.hs, c.xp0, c.yp0, c.tan2i, c.invRb2, c.ampBb, c.ampIb, c.MLb, c.cexp[0], c.cexp[1],
                             c.ampBd[0], c.ampBd[1], c.ampSd[0], c.ampSd[1], c.vkB[0], c.vkB[1], c.q3B[0], c.q3B[1]};
#pragma unroll
        for (int i = 0; i < 19; ++i) q[4 + i] = __float_as_int(v[i]);
    }
}

// sec. 2.1: rotate into the galaxy frame (fn 2).  a = jx - jcx and b = jy - jcy are offsets in cells from
// the cell nearest to the galaxy centre, so that fp32 keeps relative precision in R near the centre.
template <typename T>
BANG_D void rotate_cell(const CellK<T>& k, const T a, const T b, T& xp, T& yp) {
    xp = fma(a, k.hc, fma(b, k.hs, k.xp0));
    yp = fma(b, k.hc, fma(-a, k.hs, k.yp0));
}

// eq. 13, 14 (with 11), 15 (with 12), 19 from the per-cell ingredients: bulge light Bb and Bb sigma_b^2 (IbL), the disc
// exponentials E1, E2 (scaled by 2^-shift without a bulge), v_c and cos(phi).  FLUX: reading G' (light moments).
template <typename T, bool BULGE, bool FLUX>
BANG_D void combine_cell(const CellK<T>& k, const T Bb, const T IbL, const T E1, const T E2, const T shift, const T vc,
                         const T cosphi, T& oB, T& oV, T& oS, T& oLM) {
    const T Btot = fma(k.ampBd0, E1, fma(k.ampBd1, E2, Bb));
    const T Stot = fma(k.ampSd0, E1, fma(k.ampSd1, E2, k.MLb * Bb));       // total mass surface density (x 1e-6)
    const T invB = fast_rcp(Btot);
    const T kB = fma(k.vkB0, E1, k.vkB1 * E2);                              // sum_j B_d,j (-k_j sin i)
    const T qB = fma(k.q3B0, E1, k.q3B1 * E2);                              // sum_j B_d,j (1 - k_j^2)/3
    if constexpr (FLUX) {
        // reading G': the PSF acts on the light moments B, B v, B (sigma^2 + v^2) and on the mass surface density
        // B / <L/M> -- the numerators of eqs. 14, 15 and 19 before the division by B_tot: no square root, one reciprocal
        const T sc = BULGE ? T(1) : fast_exp2(shift);
        const T Bv = cosphi * vc * kB;
        oB = Btot * sc;
        oV = Bv * sc;
        oS = fma(Bv * Bv, invB, fma(vc * vc, qB, IbL)) * sc;
        oLM = Stot * sc;
    } else {
        oV = cosphi * vc * kB * invB;
        oS = fast_sqrt(fma(vc * vc, qB, IbL) * invB);
        oLM = Btot * fast_rcp(Stot);
        oB = BULGE ? Btot : Btot * fast_exp2(shift);
    }
}

// a2 + a3: one fine cell at (xp, yp) in the galaxy frame -> B_tot, v_los, sigma_los, <L/M>   (eqs. 4-15, 19).  BULGE: the
// model has a bulge; SHIFT = 0/1/2/3: without a bulge the disc exponentials are scaled by disc 1 (1), disc 2 (2) or the
// larger of the two (3) so that the ratios below survive fp32 underflow far outside small discs.
// bbase: the scale-free bulge table in global memory with its first interval folded in (coef - first * 2 (D+1)); used in
// fp64 mode.  bs: the per-theta bulge tables in shared memory (build_bulge_tables): in fp32 mode the theta's slice of
// {SigmaTilde, J}, in fp64 mode Itilde_ext of reading U' or NULL.  The caller guarantees that s^2 and r^2 stay inside the
// tables (decode_theta: otherwise the theta takes eval_cell_direct).
template <typename T, bool BULGE, int SHIFT, bool FLUX = false>
BANG_D void eval_cell(const CellK<T>& k, const T* __restrict__ bbase, const T* __restrict__ bs, const T* __restrict__ vtab,
                      const T xp, const T yp, T& oB, T& oV, T& oS, T& oLM) {
    constexpr int D = TabCfg<T>::D, NC = D + 1;
    // (xp, yp): the cell in the galaxy frame; R on the sky (bulge), r in the disc plane
    const T floor2 = sizeof(T) == 4 ? T(0x1p-32f) : T(0x1p-32);
    // r^2 = R^2 + y'^2 (1/cos^2 i - 1) with R^2 floored first: one FMNMX serves both radii (identical to flooring r^2
    // itself unless 0 < R < 2^-16 kpc, where fp32 coordinates carry no information anyway; reading V)
    const T y2 = yp * yp;
    const T R2 = fmax(fma(xp, xp, y2), floor2);
    const T r2 = fma(y2, k.tan2i, R2);
    const T rinv = fast_rsqrt(r2);
    const T r = r2 * rinv;
    const T cosphi = xp * rinv;

    // bulge: Sigma_b (eq. 4) and Sigma_b sigma_b^2 (eq. 6) from the scale-free tables at s^2 = R^2/R_b^2
    T Bb = T(0), IbL = T(0);
    if constexpr (BULGE) {
        T t;
        const int cell = tab_cell(R2 * k.invRb2, t);
        T cs[NC], cj[NC];
        if constexpr (sizeof(T) == 4) {
            const int e = max(cell - k.bfirst1, 0);                  // entry 0: the cell nearest to the centre
            BANG_ASSERT(e <= k.blast);
            const float4* p = reinterpret_cast<const float4*>(bs) + 2 * e;
            const float4 v0 = p[0], v1 = p[1];
            cs[0] = v0.x; cs[1] = v0.y; cs[2] = v0.z; cs[3] = v0.w;
            cj[0] = v1.x; cj[1] = v1.y; cj[2] = v1.z; cj[3] = v1.w;
            Bb = k.ampBb * horner<T, D>(cs, t);
            IbL = k.ampIb * horner<T, D>(cj, t);
        } else {
            const T* p = bbase + (ptrdiff_t)cell * (2 * NC);
#pragma unroll
            for (int d = 0; d < NC; d += 2) {
                const double2 v0 = __ldg(reinterpret_cast<const double2*>(p + d));
                const double2 v1 = __ldg(reinterpret_cast<const double2*>(p + NC + d));
                cs[d] = v0.x; cs[d + 1] = v0.y; cj[d] = v1.x; cj[d + 1] = v1.y;
            }
            Bb = k.ampBb * horner<T, D>(cs, t);
            T J = horner<T, D>(cj, t);
            if (bs) {                                                // reading U': + Itilde_ext from the per-theta table
                const int e = max(cell - k.bfirst1, 0);
                BANG_ASSERT(e <= k.blast);
                const T* pe = bs + e * NC;
                T ce[NC];
#pragma unroll
                for (int d = 0; d < NC; d += 2) {
                    const double2 v0 = *reinterpret_cast<const double2*>(pe + d);
                    ce[d] = v0.x; ce[d + 1] = v0.y;
                }
                J += horner<T, D>(ce, t);
            }
            IbL = k.ampIb * J;
        }
    }
    // discs: eq. 7-8
    const T e1a = r * k.cexp0, e2a = r * k.cexp1;
    T shift = T(0);
    if constexpr (!BULGE) shift = SHIFT == 1 ? e1a : (SHIFT == 2 ? e2a : fmax(e1a, e2a));
    const T E1 = fast_exp2(e1a - shift), E2 = fast_exp2(e2a - shift);     // B_d,j = ampBd_j E_j
    // v_c(r) from the per-theta table (eq. 10); entry 0 serves the cell nearest to the centre
    T vc;
    {
        T t;
        const int cell = max(tab_cell(r2, t) - k.vfirst1, 0);
        BANG_ASSERT(cell <= k.vlast);
        const T* p = vtab + cell * NC;
        T cv[NC];
        if constexpr (sizeof(T) == 4) {
            const float4 v0 = *reinterpret_cast<const float4*>(p);
            cv[0] = v0.x; cv[1] = v0.y; cv[2] = v0.z; cv[3] = v0.w;
        } else {
#pragma unroll
            for (int d = 0; d < NC; d += 2) {
                const double2 v0 = *reinterpret_cast<const double2*>(p + d);
                cv[d] = v0.x; cv[d + 1] = v0.y;
            }
        }
        vc = horner<T, D>(cv, t);
    }
    combine_cell<T, BULGE, FLUX>(k, Bb, IbL, E1, E2, shift, vc, cosphi, oB, oV, oS, oLM);
}

// eval_cell in two halves for fp32 mode (same arithmetic, same order): cell_begin does the geometry, the table addresses
// and ISSUES the three 128-bit table loads; cell_end consumes them.  eval_superrow calls cell_begin for the S cells of a
// column first, so that the loads of all of them are in flight before the first polynomial is evaluated.
struct CellF {
    float tb, tv, r, cosphi;
    float4 v0, v1, vv;
};
template <bool BULGE>
BANG_D void cell_begin(const CellK<float>& k, const float* __restrict__ bs, const float* __restrict__ vtab, const float xp,
                       const float yp, CellF& c) {
    const float y2 = yp * yp;
    const float R2 = fmaxf(fmaf(xp, xp, y2), 0x1p-32f);
    const float r2 = fmaf(y2, k.tan2i, R2);
    if constexpr (BULGE) {
        const int e = max(tab_cell(R2 * k.invRb2, c.tb) - k.bfirst1, 0);
        BANG_ASSERT(e <= k.blast);
        const float4* p = reinterpret_cast<const float4*>(bs) + 2 * e;
        c.v0 = p[0]; c.v1 = p[1];
    }
    const int cell = max(tab_cell(r2, c.tv) - k.vfirst1, 0);
    BANG_ASSERT(cell <= k.vlast);
    c.vv = *reinterpret_cast<const float4*>(vtab + cell * 4);
    const float rinv = fast_rsqrt(r2);
    c.cosphi = xp * rinv;
    c.r = r2 * rinv;
}
template <bool BULGE, int SHIFT, bool FLUX>
BANG_D void cell_end(const CellK<float>& k, const CellF& c, float& oB, float& oV, float& oS, float& oLM) {
    float Bb = 0.f, IbL = 0.f;
    if constexpr (BULGE) {
        const float cs[4] = {c.v0.x, c.v0.y, c.v0.z, c.v0.w}, cj[4] = {c.v1.x, c.v1.y, c.v1.z, c.v1.w};
        Bb = k.ampBb * horner<float, 3>(cs, c.tb);
        IbL = k.ampIb * horner<float, 3>(cj, c.tb);
    }
    const float e1a = c.r * k.cexp0, e2a = c.r * k.cexp1;
    float shift = 0.f;
    if constexpr (!BULGE) shift = SHIFT == 1 ? e1a : (SHIFT == 2 ? e2a : fmaxf(e1a, e2a));
    const float E1 = fast_exp2(e1a - shift), E2 = fast_exp2(e2a - shift);
    const float cv[4] = {c.vv.x, c.vv.y, c.vv.z, c.vv.w};
    const float vc = horner<float, 3>(cv, c.tv);
    combine_cell<float, BULGE, FLUX>(k, Bb, IbL, E1, E2, shift, vc, c.cosphi, oB, oV, oS, oLM);
}

// The direct path: one fine cell evaluated without the per-theta table and, where s^2 leaves the scale-free tables,
// without those either -- eq. 4-5 in closed form, eq. 6 by the N_J-node rule, eq. 10 term by term, in fp64.  Taken by the
// rare theta whose grid spans more octaves of r^2 than the v_c table holds (|i| -> 90 deg) or whose R/R_b leaves
// [2^-22, 2^18): the library's domain is the model's, not the tables'.  ~1e3-1e4 times slower per cell than eval_cell.
struct DirectC {
    const double* glx; const double* glw; int NJ;   // the Gauss-Legendre rule of reading B (device memory)
    QuadC quad;                                     // the same rule in the form ext_Itilde takes (reading U')
};
template <typename T, bool FLUX>
__device__ __noinline__ void eval_cell_direct(const ThetaC<T>& c, const GridC& g, const PolyTab<T>& btab, const PolyTab<T>& Ftab,
                                              const DirectC dc, const int a, const int b, T* o4) {
    // (a, b): offsets in cells from the cell nearest to the centre; the geometry in fp64 whatever the mode (at |i| -> 90
    // deg, r^2 = R^2 + y'^2 tan^2 i amplifies the rounding of fp32 coordinates beyond the mode's tolerance)
    const double xp = (double)a * c.d.ghc + ((double)b * c.d.ghs + c.d.gxp0);
    const double yp = (double)b * c.d.ghc + (c.d.gyp0 - (double)a * c.d.ghs);
    const double y2 = yp * yp;
    const double R2 = fmax(xp * xp + y2, 0x1p-32);
    const double r2 = R2 + y2 * c.d.gtan2i;
    const double r = sqrt(r2), cosphi = xp / r;
    double Bb = 0.0, IbL = 0.0;
    if (g.comps & C_BULGE) {
        const double s2 = R2 * (double)c.invRb2;
        double st, jj;
        if (s2 >= ldexp(1.0, kBulgeOctLo) * (1.0 + 0x1p-9) && s2 < ldexp(1.0, kBulgeOctHi) * (1.0 - 0x1p-9)) {
            T t;
            const int cell = tab_cell((T)s2, t) - btab.first;
            const T* p = btab.coef + (size_t)cell * (2 * (TabCfg<T>::D + 1));
            st = (double)horner<T, TabCfg<T>::D>(p, t);
            jj = (double)horner<T, TabCfg<T>::D>(p + TabCfg<T>::D + 1, t);
        } else {
            const double sx = sqrt(s2);
            st = g.bulge_profile == 1 ? jaffe_sigma_tilde(sx) : sigma_tilde(sx);
            jj = g.bulge_profile == 1 ? jaffe_jeans_J(sx, dc.NJ, dc.glx, dc.glw) : jeans_J(sx, dc.NJ, dc.glx, dc.glw);
        }
        if (has_ext(g))                                              // reading U'
            jj += ext_Itilde<double, T>(sqrt(s2), c.d, ThetaF{}, g, Ftab, dc.quad);
        Bb = (double)c.ampBb * st;
        IbL = (double)c.ampIb * jj;
    }
    const double vc2 = vc2_total<T>(c.d, g, g.comps, Ftab, r);
    // discs, with the common factor 2^shift taken out of the exponentials (no bulge: the ratios survive underflow)
    const double e1a = r * (double)c.cexp[0], e2a = r * (double)c.cexp[1];
    double shift = 0.0;
    if (!(g.comps & C_BULGE)) {
        const bool d1 = g.comps & C_DISC1, d2 = g.comps & C_DISC2;
        shift = (d1 && d2) ? fmax(e1a, e2a) : (d1 ? e1a : e2a);
    }
    const double E1 = exp2(e1a - shift), E2 = exp2(e2a - shift);
    const double Btot = (double)c.ampBd[0] * E1 + (double)c.ampBd[1] * E2 + Bb;
    const double Stot = (double)c.ampSd[0] * E1 + (double)c.ampSd[1] * E2 + (double)c.MLb * Bb;
    const double kB = (double)c.vkB[0] * E1 + (double)c.vkB[1] * E2;
    const double qB = (double)c.q3B[0] * E1 + (double)c.q3B[1] * E2;
    double oB = Btot * exp2(shift), oV = cosphi * sqrt(vc2) * kB / Btot, oS = sqrt((vc2 * qB + IbL) / Btot), oLM = Btot / Stot;
    if (FLUX) {
        const double v = oV;
        oV = oB * v; oS = oB * (oS * oS + v * v); oLM = oB / oLM;
    }
    o4[0] = (T)oB; o4[1] = (T)oV; o4[2] = (T)oS; o4[3] = (T)oLM;
}

// a2 + a3 over a run of whole fine rows (k_fine): cells i = tid, tid + NT, ... of the n_rows x nfx block that starts at
// fine row jy0, written to dst[row * row_pitch + observable * obs_stride + x].  All threads of the CTA take part.
struct EvalWalk { int i0, j0, x0, step_j, step_x; };   // flat cell i = i0 + n NT sits at (row j, column x)
BANG_D EvalWalk make_walk(const int tid, const int NT, const int nfx) {
    EvalWalk w;
    w.i0 = tid; w.j0 = tid / nfx; w.x0 = tid - w.j0 * nfx;
    w.step_j = NT / nfx; w.step_x = NT - w.step_j * nfx;
    return w;
}
template <typename T, bool BULGE, int SHIFT, bool FLUX>
BANG_D void eval_rows(const CellK<T>& k, const T* __restrict__ bbase, const T* __restrict__ bs, const T* __restrict__ vtab, T* __restrict__ dst,
                      const size_t row_pitch, const size_t obs_stride, const int nfx, const int jy0, const int n_rows,
                      const EvalWalk& w, const int NT) {
    const int step_j = w.step_j, step_x = w.step_x;
    int j = w.j0, x = w.x0;
    const int tid = w.i0;
    const int n = n_rows * nfx;
    for (int i = tid; i < n; i += NT) {
        T vB, vV, vS, vL, xp, yp;
        rotate_cell<T>(k, (T)(x - k.jcx), (T)(jy0 + j - k.jcy), xp, yp);
        eval_cell<T, BULGE, SHIFT, FLUX>(k, bbase, bs, vtab, xp, yp, vB, vV, vS, vL);
        T* d = dst + (size_t)j * row_pitch + x;
        d[0] = vB; d[obs_stride] = vV; d[2 * obs_stride] = vS; d[3 * obs_stride] = vL;
        x += step_x; j += step_j;
        if (x >= nfx) { x -= nfx; ++j; }
    }
}
template <typename T, bool FLUX>
BANG_D void eval_rows_comps(const unsigned comps, const CellK<T>& k, const T* __restrict__ bbase, const T* __restrict__ bs, const T* __restrict__ vtab,
                            T* __restrict__ dst, const size_t row_pitch, const size_t obs_stride, const int nfx,
                            const int jy0, const int n_rows, const EvalWalk& w, const int NT) {
    if (comps & C_BULGE) eval_rows<T, true, 0, FLUX>(k, bbase, bs, vtab, dst, row_pitch, obs_stride, nfx, jy0, n_rows, w, NT);
    else if ((comps & (C_DISC1 | C_DISC2)) == (C_DISC1 | C_DISC2))
        eval_rows<T, false, 3, FLUX>(k, bbase, bs, vtab, dst, row_pitch, obs_stride, nfx, jy0, n_rows, w, NT);
    else if (comps & C_DISC1) eval_rows<T, false, 1, FLUX>(k, bbase, bs, vtab, dst, row_pitch, obs_stride, nfx, jy0, n_rows, w, NT);
    else eval_rows<T, false, 2, FLUX>(k, bbase, bs, vtab, dst, row_pitch, obs_stride, nfx, jy0, n_rows, w, NT);
}
template <typename T>
BANG_D void eval_rows_any(const unsigned comps, const bool flux, const CellK<T>& k, const T* __restrict__ bbase, const T* __restrict__ bs,
                          const T* __restrict__ vtab, T* __restrict__ dst, const size_t row_pitch, const size_t obs_stride,
                          const int nfx, const int jy0, const int n_rows, const EvalWalk& w, const int NT) {
    if (flux) eval_rows_comps<T, true>(comps, k, bbase, bs, vtab, dst, row_pitch, obs_stride, nfx, jy0, n_rows, w, NT);
    else eval_rows_comps<T, false>(comps, k, bbase, bs, vtab, dst, row_pitch, obs_stride, nfx, jy0, n_rows, w, NT);
}
// the same block of rows through the direct path (a theta flagged slow)
template <typename T>
BANG_D void eval_rows_direct(const bool flux, const ThetaC<T>& c, const GridC& g, const PolyTab<T>& btab, const PolyTab<T>& Ftab,
                             const DirectC dc, const CellK<T>& k, T* __restrict__ dst, const size_t row_pitch,
                             const size_t obs_stride, const int nfx, const int jy0, const int n_rows, const int tid, const int NT) {
    const int n = n_rows * nfx;
    for (int i = tid; i < n; i += NT) {
        const int j = i / nfx, x = i - j * nfx;
        T o[4];
        if (flux) eval_cell_direct<T, true>(c, g, btab, Ftab, dc, x - k.jcx, jy0 + j - k.jcy, o);
        else eval_cell_direct<T, false>(c, g, btab, Ftab, dc, x - k.jcx, jy0 + j - k.jcy, o);
        T* d = dst + (size_t)j * row_pitch + x;
        d[0] = o[0]; d[obs_stride] = o[1]; d[2 * obs_stride] = o[2]; d[3 * obs_stride] = o[3];
    }
}

// ---- row buffer geometry --------------------------------------------------------------------------------------------
// The fused kernel keeps one super-row (S fine rows x 4 observables) in shared memory: plane (j, q) at (j 4 + q) NFB,
// cell x of a plane at x + PADV (x / GRP).  NFB, the plane pitch in cells, is a compile-time constant of the
// instantiation (immediate store offsets): the widest row the launch-bound class can hold.
// Bank conflicts.  In the PSF phase neighbouring threads read 16-byte vectors GRP = P S cells apart.  When that stride is
// an EVEN number of vectors (s = 4 with P = 4: 64 B), the 8 lanes of a quarter-warp fall on 2 or 4 of the 8 vector-wide
// bank groups (ncu, config 5: 7 conflicts per load); one pad vector after every GRP cells makes the stride odd and the
// loads conflict-free.  row_pad = pad cells per group (0 when not needed).
constexpr int row_pad(int P, int S, int elem_bytes) {
    const int V = 16 / elem_bytes, GRP = P * S;
    return (GRP % V == 0 && (GRP / V) % 2 == 0) ? V : 0;
}
// LBC: launch-bound class = the CTA-size bracket the kernel is compiled for, which fixes its register budget, the
// row-buffer pitch (hence the shared memory per CTA) and the pitch of the data array:
//   0: <= 128 threads, 7 (P = 2, 72 registers) or 5 (P = 4, 96 registers) CTAs per SM;  1: <= 256 threads, 3 or 2 CTAs per SM;  2: <= 512 threads
//   (2 CTAs per SM with P = 2, else 1).
constexpr int lbc_threads(int lbc) { return lbc == 0 ? 128 : (lbc == 1 ? 256 : 512); }
// plane pitch: nxp <= threads P / 4 data columns, i.e. (nxp - 1 + NACC) S cells, rounded up to a multiple of 4, plus 4
// cells of over-read slack for the vector loads
constexpr int lbc_nfb(int lbc, int P, int S, int NACC, int elem_bytes) {
    const int cells = (lbc_threads(lbc) * P / 4 - 1 + NACC) * S;
    const int padded = cells + row_pad(P, S, elem_bytes) * ((cells + P * S - 1) / (P * S));
    return (padded + 3) / 4 * 4 + 4 + row_pad(P, S, elem_bytes);
}
#ifndef BANG_MB_P4
#define BANG_MB_P4 5             // resident CTAs per SM the class-0 kernels are compiled for (register budget 96 / 72)
#endif
#ifndef BANG_MB_P2
#define BANG_MB_P2 7
#endif
constexpr int lbc_blocks(int lbc, int P, bool f64) {
    return f64 ? (lbc == 0 ? 4 : (lbc == 1 ? 2 : 1))          // fp64 mode: 128 registers in every class
               : (lbc == 0 ? (P == 2 ? BANG_MB_P2 : BANG_MB_P4) : (lbc == 1 ? (P == 2 ? 3 : 2) : (P == 2 ? 2 : 1)));
}

// a2 + a3 for one super-row of the fused kernel (S fine rows jy0 .. jy0+S-1 = one data row): thread `vt` takes the fine
// columns x = vt, vt + NT, ... and evaluates the S cells of each column in one iteration, so that the index arithmetic,
// the rotation and the store address are shared by S cells and S independent dependency chains are in flight.
// dst[(row * 4 + observable) * NFB + x].  GUARD: some of the S rows lie past the grid (zero-weight tap padding): they
// are written as zeros.
template <typename T, int S, int NFB, int GRP, int PADV, bool BULGE, int SHIFT, bool GUARD, bool FLUX, bool SPLIT>
BANG_D void eval_superrow(const CellK<T>& k, const T* __restrict__ bbase, const T* __restrict__ bs, const T* __restrict__ vtab, T* __restrict__ dst,
                          const int nfx, const int nfy, const int jy0, const int vt, const int NT) {
    const T b0 = (T)(jy0 - k.jcy);
    const T bx = fma(b0, k.hs, k.xp0), by = fma(b0, k.hc, k.yp0);
    for (int x = vt; x < nfx; x += NT) {
        const T a = (T)(x - k.jcx);
        const T px = fma(a, k.hc, bx), py = fma(-a, k.hs, by);
        T* d = dst + x + (PADV ? PADV * (x / GRP) : 0);      // row_pad: GRP is a power of two whenever PADV != 0
        BANG_ASSERT(x + (PADV ? PADV * (x / GRP) : 0) < NFB);
        if constexpr (sizeof(T) == 4 && !GUARD && SPLIT) {     // all S cells' table loads in flight first (cell_begin)
            CellF c[S];
#pragma unroll
            for (int j = 0; j < S; ++j)
                cell_begin<BULGE>(k, bs, vtab, j == 0 ? px : fma((T)j, k.hs, px), j == 0 ? py : fma((T)j, k.hc, py), c[j]);
#pragma unroll
            for (int j = 0; j < S; ++j) {
                T vB, vV, vS, vL;
                cell_end<BULGE, SHIFT, FLUX>(k, c[j], vB, vV, vS, vL);
                d[(j * 4 + 0) * NFB] = vB; d[(j * 4 + 1) * NFB] = vV; d[(j * 4 + 2) * NFB] = vS; d[(j * 4 + 3) * NFB] = vL;
            }
            continue;
        }
#pragma unroll
        for (int j = 0; j < S; ++j) {
            T vB, vV, vS, vL;
            if (GUARD && jy0 + j >= nfy) {
                vB = vV = vS = vL = T(0);
            } else {
                const T xp = j == 0 ? px : fma((T)j, k.hs, px), yp = j == 0 ? py : fma((T)j, k.hc, py);
                eval_cell<T, BULGE, SHIFT, FLUX>(k, bbase, bs, vtab, xp, yp, vB, vV, vS, vL);
            }
            d[(j * 4 + 0) * NFB] = vB; d[(j * 4 + 1) * NFB] = vV; d[(j * 4 + 2) * NFB] = vS; d[(j * 4 + 3) * NFB] = vL;
        }
    }
}
template <typename T, int S, int NFB, int GRP, int PADV, bool GUARD, bool FLUX, bool SPLIT>
BANG_D void eval_superrow_any(const unsigned comps, const CellK<T>& k, const T* __restrict__ bbase, const T* __restrict__ bs, const T* __restrict__ vtab,
                              T* __restrict__ dst, const int nfx, const int nfy, const int jy0, const int vt, const int NT) {
    if (comps & C_BULGE) eval_superrow<T, S, NFB, GRP, PADV, true, 0, GUARD, FLUX, SPLIT>(k, bbase, bs, vtab, dst, nfx, nfy, jy0, vt, NT);
    else if ((comps & (C_DISC1 | C_DISC2)) == (C_DISC1 | C_DISC2))
        eval_superrow<T, S, NFB, GRP, PADV, false, 3, GUARD, FLUX, SPLIT>(k, bbase, bs, vtab, dst, nfx, nfy, jy0, vt, NT);
    else if (comps & C_DISC1) eval_superrow<T, S, NFB, GRP, PADV, false, 1, GUARD, FLUX, SPLIT>(k, bbase, bs, vtab, dst, nfx, nfy, jy0, vt, NT);
    else eval_superrow<T, S, NFB, GRP, PADV, false, 2, GUARD, FLUX, SPLIT>(k, bbase, bs, vtab, dst, nfx, nfy, jy0, vt, NT);
}

// ---- the fused kernel ---------------------------------------------------------------------------------------------
// fp32 mode: the composite taps as pairs for Blackwell's two-wide FMA (FFMA2): a[k] = {W[2k], W[2k+1]} serves the
// pixels whose run starts on an even cell, b[k] = {W[2k+1], W[2k+2]} those that start on an odd one (their first tap is
// applied on its own).  Zero beyond the taps.
template <typename T, int N> struct TapPairs {};
template <int N> struct TapPairs<float, N> { float2 a[(N + 1) / 2], b[(N + 1) / 2], d[N]; };   // d[t] = {W[t], W[t]}

template <typename T, int S, int NACC>
struct FusedParams {
    GridC g;
    FitC fit;
    PolyTab<T> btab, Ftab;
    QuadC quad;                  // reading U': the N_J-node rule for Itilde_ext
    int bs_elems;                // size of the per-theta bulge tables in shared memory, in values of T (bs_elems<T>(g))
    T W[NACC * S];               // composite x s box (*) Gaussian taps, zero padded (a4 + a5)
    TapPairs<T, NACC * S> W2;    // the same in pairs (fp32 mode)
    const double* theta;         // [B][17]
    int B;
    int mode;                    // 0 maps, 1 likelihood (read by the MODE = 2 instantiations only)
    int nxp;                     // data columns padded to a multiple of P
    T* maps;                     // [B][4][ny][nx]
    const double2* data;         // [ny][4][P][GMAX] {d, 1/e} of pixel group P + i (1/e = 0 where masked or padded); GMAX =
                                 // (thread class of the launch) / 4 >= nxp/P
    double C0;                   // sum over used pixels of -1/2 ln(2 pi e^2)
    double* logL;                // [B]
    int* slow_list;              // [>= B] indices of the theta that need the direct path (k_slow, bang_slow.cuh) ...
    int* slow_count;             // ... and their number; NULL: such theta are reported as out of domain
};

template <typename T>
inline size_t vtab_bytes() { return ((size_t)kVcOct * (1 << TabCfg<T>::M) + 1) * (TabCfg<T>::D + 1) * sizeof(T); }
// scratch for the nodes of Itilde_ext: the row buffer serves when there is one (k_fused), else (k_fine) it is allocated
template <typename T>
inline size_t ext_scratch_elems(const GridC& g) {
    return has_ext(g) ? ((size_t)kBOct * (1 << TabCfg<T>::M)) * (TabCfg<T>::D + 1) + 4 + (size_t)kBOct * kExtMaxND + 4 : 0;
}
template <typename T>
inline size_t fused_smem_bytes(const GridC& g, int S, int nfb) {
    const size_t row = (size_t)S * 4 * nfb, scr = ext_scratch_elems<T>(g);
    return (sizeof(ThetaC<T>) + 15) / 16 * 16 + vtab_bytes<T>() + (bs_elems<T>(g) + (row > scr ? row : scr)) * sizeof(T) + 32 * sizeof(double);
}

// N consecutive values from shared memory into registers with the widest vector loads the alignment ALIGN (bytes)
// allows; may read up to one vector past N (the row buffer carries that slack).
// GRP, PADV: the buffer holds PADV pad elements after every GRP elements (row_pad above); src points at a group start.
template <typename T, int N, int ALIGN, int GRP, int PADV>
BANG_D void load_run(const T* __restrict__ src, T (&f)[N]) {
    constexpr int V = ALIGN / (int)sizeof(T);
    if constexpr (V == 4) {
#pragma unroll
        for (int i = 0; i < N; i += 4) {
            const float4 v = *reinterpret_cast<const float4*>(src + i + PADV * (i / GRP));
            f[i] = v.x;
            if (i + 1 < N) f[i + 1] = v.y;
            if (i + 2 < N) f[i + 2] = v.z;
            if (i + 3 < N) f[i + 3] = v.w;
        }
    } else if constexpr (V == 2 && sizeof(T) == 4) {
#pragma unroll
        for (int i = 0; i < N; i += 2) {
            const float2 v = *reinterpret_cast<const float2*>(src + i);
            f[i] = v.x;
            if (i + 1 < N) f[i + 1] = v.y;
        }
    } else if constexpr (V == 2 && sizeof(T) == 8) {
#pragma unroll
        for (int i = 0; i < N; i += 2) {
            const double2 v = *reinterpret_cast<const double2*>(src + i + PADV * (i / GRP));
            f[i] = v.x;
            if (i + 1 < N) f[i + 1] = v.y;
        }
    } else {
#pragma unroll
        for (int i = 0; i < N; ++i) f[i] = src[i];
    }
}

// 1/x for the final M/L = 1/<L/M> (fn 10): MUFU.RCP (1 ulp) in fp32 mode, IEEE division in fp64 mode
// The argument is floored far below any physical <L/M> so that padded pixels (accumulators = 0) stay finite.
BANG_D float inv_ml(float x) { return fast_rcp(fmaxf(x, 1e-30f)); }
BANG_D double inv_ml(double x) { return 1.0 / fmax(x, 1e-300); }

// MODE 0: write the maps (bang_model_maps); MODE 1: reduce the likelihood (bang_loglike); MODE 2: either, chosen at run
// time by p.mode (fp64 mode is instantiated this way only: it halves the build and costs one uniform branch per data row).
// FLUX: the flux-weighted PSF of reading G' -- the four fields that go through the PSF and the rebin are the light moments
// B, B v, B (sigma^2 + v^2) and the mass surface density (eval_cell<FLUX>); the observables are formed per data pixel when
// its row completes: v = M1/M0, sigma^2 = M2/M0 - v^2, M/L = M3/M0.  The four moments of a pixel are then needed
// together, so in this instantiation the PSF threads are numbered observable-fastest (lane = 4 group + observable) and the
// moments travel by warp shuffle inside each quad of lanes; the paper's path (FLUX = false) keeps its own numbering and
// carries none of this code.
// the register budget of an instantiation, stated outright (__maxnreg__): what lbc_blocks CTAs of lbc_threads threads leave
// of the SM's 64 K registers, in multiples of 8 (the min-blocks form of __launch_bounds__ gives the same cap but a slightly
// slower schedule: config 3 10.79 -> 10.72 ms, config 4 1.375 -> 1.366 ms)
constexpr int lbc_regs(int lbc, int P, bool f64) {      // fp32 mode (f64 = false)
    const int r = 65536 / (lbc_threads(lbc) * lbc_blocks(lbc, P, f64)) / 8 * 8;
    return r > 128 ? 128 : r;
}
template <typename T, int S, int NACC, int P, int MODE, int LBC, bool FLUX>
BANG_D void fused_body(const FusedParams<T, S, NACC>& p) {
    constexpr int D = TabCfg<T>::D, NC = D + 1;
    constexpr int RUN = (P - 1 + NACC) * S;          // fine cells one thread reads per row for its P data pixels
    constexpr int RUN_BYTES = P * S * (int)sizeof(T);   // byte stride between the runs of neighbouring threads
    constexpr int ALIGN = RUN_BYTES % 16 == 0 ? 16 : (RUN_BYTES % 8 == 0 ? 8 : (int)sizeof(T));
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ThetaC<T>& c = *reinterpret_cast<ThetaC<T>*>(smem_raw);
    constexpr size_t off_tab = (sizeof(ThetaC<T>) + 15) / 16 * 16;
    T* vtab = reinterpret_cast<T*>(smem_raw + off_tab);
    T* bs_mem = vtab + ((size_t)kVcOct * (1 << TabCfg<T>::M) + 1) * NC;
    T* rowbuf = bs_mem + p.bs_elems;
    const T* bs = p.bs_elems ? bs_mem : nullptr;
    constexpr int nfb = lbc_nfb(LBC, P, S, NACC, (int)sizeof(T));
    constexpr int GRP = P * S, PADV = row_pad(P, S, (int)sizeof(T));
    // the P = 4 kernels have the registers (96 in class 0) to keep the table loads of a column's S cells in flight at once;
    // at the 72 registers of P = 2 the same ordering costs 1-2 %
    constexpr bool SPLIT = P == 4;
    double* red = reinterpret_cast<double*>(rowbuf + (size_t)S * 4 * nfb);

    const GridC& g = p.g;
    const int tid = threadIdx.x, NT = blockDim.x;
    const int G = p.nxp / P;                         // pixel groups per map
    constexpr int GMAX = lbc_threads(LBC) / 4;       // pitch of the data array's pixel-group axis (compile-time: immediate offsets)
    const int items = 4 * G;
    // this thread's observable and pixel group in the PSF phase
    const int q = FLUX ? (tid & 3) : tid / G, grp = FLUX ? (tid >> 2) : tid - q * G;
    const bool psf_thread = tid < items;
    const int nsuper = g.ny + NACC - 1;
    const size_t npix = (size_t)g.nx * g.ny;
    const T* run_base = rowbuf + (size_t)q * nfb + grp * (GRP + PADV);
    const T* bbase = p.btab.coef - (ptrdiff_t)p.btab.first * (2 * NC);

    for (int i = tid; i < S * 4 * nfb; i += NT) rowbuf[i] = T(0);

    for (int b = blockIdx.x; b < p.B; b += gridDim.x) {
        __syncthreads();
        if (tid == 0) { decode_theta<T>(p.theta + (size_t)b * kNTheta, g, p.btab, p.Ftab, c); pack_cellk<T>(c); }
        __syncthreads();
        if (!c.valid || (c.slow && !p.slow_list)) {  // out-of-domain theta: NaN maps / -inf likelihood
            if (MODE == 0 || (MODE == 2 && p.mode == 0)) {
                const T qnan = (T)nan("");
                for (size_t i = tid; i < 4 * npix; i += NT) p.maps[(size_t)b * 4 * npix + i] = qnan;
            } else if (tid == 0) {
                p.logL[b] = -INFINITY;
            }
            continue;
        }
        if (c.slow) {                                // radii outside the tabulated ranges: left to k_slow (direct path)
            if (tid == 0) p.slow_list[atomicAdd(p.slow_count, 1)] = b;
            continue;
        }
        build_vc_table<T>(c, g, p.fit, p.Ftab, vtab);
        if (p.bs_elems) {
            build_bulge_tables<T>(c, g, p.fit, p.btab, p.Ftab, p.quad, bs_mem, rowbuf);
            if (has_ext(g)) {                         // the row buffer served as scratch: zero the tap padding again
                for (int i = tid; i < S * 4 * nfb; i += NT) rowbuf[i] = T(0);
                __syncthreads();
            }
        }

        constexpr bool F2Y = sizeof(T) == 4 && LBC == 0;    // (class 1, NACC = 10: 20 pair accumulators, measured 2 % slower)
        T acc[F2Y ? 1 : P][F2Y ? 1 : NACC];
        float2 acc2[F2Y ? P / 2 : 1][F2Y ? NACC : 1];      // F2Y: the running data rows of pixels (2 ip, 2 ip + 1) as pairs
        if constexpr (F2Y) {
#pragma unroll
            for (int ip = 0; ip < P / 2; ++ip)
#pragma unroll
                for (int kk = 0; kk < NACC; ++kk) acc2[ip][kk] = make_float2(0.f, 0.f);
        } else {
#pragma unroll
            for (int i = 0; i < P; ++i)
#pragma unroll
                for (int kk = 0; kk < NACC; ++kk) acc[i][kk] = T(0);
        }
        double chi2 = 0.0;
        int vt = (tid + 32 * (b & 3)) % NT;              // this thread's first fine column in the model phase (a2 + a3)

        for (int sr = 0; sr < nsuper; ++sr) {
            // ---- a2 + a3: evaluate the S fine rows of this super-row into shared memory
            // the per-theta constants are re-read from shared memory for every super-row (a handful of broadcast loads)
            // so that they do not occupy registers during the PSF phase
            const CellK<T> k = load_cellk<T>(c);
            if ((sr + 1) * S <= g.nfy) eval_superrow_any<T, S, nfb, GRP, PADV, false, FLUX, SPLIT>(g.comps, k, bbase, bs, vtab, rowbuf, g.nfx, g.nfy, sr * S, vt, NT);
            else eval_superrow_any<T, S, nfb, GRP, PADV, true, FLUX, SPLIT>(g.comps, k, bbase, bs, vtab, rowbuf, g.nfx, g.nfy, sr * S, vt, NT);
            vt = vt + 32 < NT ? vt + 32 : vt + 32 - NT;      // rotate the column ownership by one warp: the ragged last
                                                             // pass then falls on a different warp (scheduler) each time
            __syncthreads();
            // ---- a4 + a5: PSF along x fused with the rebin, then scattered along y into the running data rows
            if (psf_thread) {
                const int py = sr - (NACC - 1);      // the data row this super-row completes
                // a6: this thread's P {d, 1/e} pairs, requested now and used after the taps (the row is padded to nxp,
                // so the loads need no guard; 1/e = 0 where masked or padded)
                double2 de[P];
                if (!F2Y && (MODE == 1 || (MODE == 2 && p.mode == 1))) {
                    if (py >= 0) {
                        const double2* src = p.data + (((py * 4 + q) * P) * GMAX + grp);
#pragma unroll
                        for (int i = 0; i < P; ++i) de[i] = __ldg(src + i * GMAX);
                    }
                }
#pragma unroll
                for (int j = 0; j < S; ++j) {
                    T f[RUN];
                    [[maybe_unused]] float xpair[P];
                    load_run<T, RUN, ALIGN, GRP, PADV>(run_base + (size_t)(j * 4) * nfb, f);
#pragma unroll
                    for (int i = 0; i < P; ++i) {
                        T xp = T(0);
                        if constexpr (sizeof(T) == 4) {
                            // FFMA2, two taps per instruction: even and odd taps accumulate in the halves of one register
                            // pair (cells f[2m], f[2m+1] sit in an aligned pair after the vector loads), so the four
                            // chains stay as short as the scalar ones (config 3 10.96 -> 10.80 ms on the 96-register
                            // kernel; on the 80-register kernel of r02b it had changed nothing)
                            constexpr int NTAP = NACC * S;
                            const int base = i * S, t0 = base & 1;
                            float2 s2 = make_float2(0.f, 0.f);
#pragma unroll
                            for (int t = t0; t + 1 < NTAP; t += 2)
                                s2 = __ffma2_rn(t0 ? p.W2.b[t >> 1] : p.W2.a[t >> 1], make_float2(f[base + t], f[base + t + 1]), s2);
                            xp = s2.x + s2.y;
                            if (t0) xp = fma(p.W[0], f[base], xp);
                            if ((NTAP - t0) & 1) xp = fma(p.W[NTAP - 1], f[base + NTAP - 1], xp);
                        } else {
#pragma unroll
                            for (int t = 0; t < NACC * S; ++t) xp = fma(p.W[t], f[i * S + t], xp);
                        }
                        if constexpr (F2Y) {
                            xpair[i] = xp;
                        } else {
#pragma unroll
                            for (int kk = 0; kk < NACC; ++kk) acc[i][kk] = fma(p.W[(NACC - 1 - kk) * S + j], xp, acc[i][kk]);
                        }
                    }
                    if constexpr (F2Y) {
#pragma unroll
                        for (int ip = 0; ip < P / 2; ++ip) {
                            const float2 x2 = make_float2(xpair[2 * ip], xpair[2 * ip + 1]);
#pragma unroll
                            for (int kk = 0; kk < NACC; ++kk)
                                acc2[ip][kk] = __ffma2_rn(p.W2.d[(NACC - 1 - kk) * S + j], x2, acc2[ip][kk]);
                        }
                    }
                }
                // ---- a6 (or map output): data row py is complete
                if constexpr (F2Y) {                 // (the pair kernels request {d, 1/e} only now: 16 registers less over the taps)
                    if ((MODE == 1 || (MODE == 2 && p.mode == 1)) && py >= 0) {
                        const double2* src = p.data + (((py * 4 + q) * P) * GMAX + grp);
#pragma unroll
                        for (int i = 0; i < P; ++i) de[i] = __ldg(src + i * GMAX);
                    }
                }
                if (py >= 0) {
                    [[maybe_unused]] unsigned quad_mask = 0;
                    if constexpr (FLUX) quad_mask = __activemask();        // whole quads: the PSF threads are a multiple of 4
#pragma unroll
                    for (int i = 0; i < P; ++i) {
                        const int px = grp * P + i;
                        T m;
                        if constexpr (F2Y) m = (i & 1) ? acc2[i / 2][0].y : acc2[i / 2][0].x;
                        else m = acc[i][0];
                        if constexpr (FLUX) {
                            // reading G': B = M0, v = M1/M0, sigma^2 = M2/M0 - v^2, M/L = M3/M0 (M0 floored far below any
                            // physical light so that padded pixels stay finite)
                            const int base = (tid & 31) & ~3;
                            const T m0 = __shfl_sync(quad_mask, m, base), m1 = __shfl_sync(quad_mask, m, base + 1);
                            const T i0 = inv_ml(m0), v = m1 * i0;
                            if (q == 1) m = v;
                            else if (q == 2) m = fast_sqrt(fmax(fma(m, i0, -v * v), T(0)));
                            else if (q == 3) m = m * i0;
                        } else {
                            if (q == 3) m = inv_ml(m);                 // M/L = 1/<L/M> (fn 10)
                        }
                        if (MODE == 0 || (MODE == 2 && p.mode == 0)) {
                            if (px < g.nx) p.maps[((size_t)b * 4 + q) * npix + (size_t)py * g.nx + px] = m;
                        } else {
                            const double z = (de[i].x - (double)m) * de[i].y;      // eq. 18, residual in fp64
                            chi2 = de[i].y != 0.0 ? fma(z, z, chi2) : chi2;        // masked or padded pixel (1/e = 0): the
                        }                                                          // model value never enters (reading M)
                    }
                }
                if constexpr (F2Y) {
#pragma unroll
                    for (int ip = 0; ip < P / 2; ++ip) {
#pragma unroll
                        for (int kk = 0; kk + 1 < NACC; ++kk) acc2[ip][kk] = acc2[ip][kk + 1];
                        acc2[ip][NACC - 1] = make_float2(0.f, 0.f);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < P; ++i) {
#pragma unroll
                        for (int kk = 0; kk + 1 < NACC; ++kk) acc[i][kk] = acc[i][kk + 1];
                        acc[i][NACC - 1] = T(0);
                    }
                }
            }
            __syncthreads();
        }
        if (MODE == 1 || (MODE == 2 && p.mode == 1)) {   // a6: block reduction, warp shuffles, fp64
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) chi2 += __shfl_xor_sync(0xffffffffu, chi2, o);
            if ((tid & 31) == 0) red[tid >> 5] = chi2;
            __syncthreads();
            if (tid == 0) {
                double sum = 0.0;
                for (int w = 0; w < (NT + 31) / 32; ++w) sum += red[w];
                p.logL[b] = p.C0 - 0.5 * sum;
            }
        }
    }
}

// The kernel proper.  fp32 mode states its register budget outright (__maxnreg__, lbc_regs above); fp64 mode keeps the
// min-blocks form of __launch_bounds__ (same cap of 128, and measured 4 % faster at config 2 that way).
template <typename T, int S, int NACC, int P, int MODE, int LBC, bool FLUX = false>
__global__ void __launch_bounds__(lbc_threads(LBC)) __maxnreg__(lbc_regs(LBC, P, false))
k_fused(const __grid_constant__ FusedParams<T, S, NACC> p) {
    fused_body<T, S, NACC, P, MODE, LBC, FLUX>(p);
}
template <typename T, int S, int NACC, int P, int MODE, int LBC, bool FLUX = false>
__global__ void __launch_bounds__(lbc_threads(LBC), lbc_blocks(LBC, P, true))
k_fused64(const __grid_constant__ FusedParams<T, S, NACC> p) {
    fused_body<T, S, NACC, P, MODE, LBC, FLUX>(p);
}

// un-convolved fine maps (bang_model_fine): one CTA per theta, same decode / table / cell code as the fused kernel
template <typename T>
struct FineParams {
    GridC g;
    FitC fit;
    PolyTab<T> btab, Ftab;
    DirectC direct;
    int bs_elems;                // as in FusedParams
    const double* theta;
    int B;
    T* fine;                     // [B][4][nfy][nfx]
};

template <typename T>
__global__ void __launch_bounds__(256) k_fine(const __grid_constant__ FineParams<T> p) {
    constexpr int NC = TabCfg<T>::D + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ThetaC<T>& c = *reinterpret_cast<ThetaC<T>*>(smem_raw);
    constexpr size_t off_tab = (sizeof(ThetaC<T>) + 15) / 16 * 16;
    T* vtab = reinterpret_cast<T*>(smem_raw + off_tab);
    T* bs_mem = vtab + ((size_t)kVcOct * (1 << TabCfg<T>::M) + 1) * NC;
    T* scratch = bs_mem + p.bs_elems;
    const T* bs = p.bs_elems ? bs_mem : nullptr;
    const GridC& g = p.g;
    const size_t plane = (size_t)g.nfx * g.nfy;
    const T* bbase = p.btab.coef - (ptrdiff_t)p.btab.first * (2 * NC);
    for (int b = blockIdx.x; b < p.B; b += gridDim.x) {
        __syncthreads();
        if (threadIdx.x == 0) { decode_theta<T>(p.theta + (size_t)b * kNTheta, g, p.btab, p.Ftab, c); pack_cellk<T>(c); }
        __syncthreads();
        T* out = p.fine + (size_t)b * 4 * plane;
        if (!c.valid) {
            const T qnan = (T)nan("");
            for (size_t i = threadIdx.x; i < 4 * plane; i += blockDim.x) out[i] = qnan;
            continue;
        }
        const CellK<T> k = load_cellk<T>(c);
        if (c.slow) {
            eval_rows_direct<T>(g.flux != 0, c, g, p.btab, p.Ftab, p.direct, k, out, (size_t)g.nfx, plane, g.nfx, 0, g.nfy,
                                threadIdx.x, blockDim.x);
            continue;
        }
        build_vc_table<T>(c, g, p.fit, p.Ftab, vtab);
        if (p.bs_elems) build_bulge_tables<T>(c, g, p.fit, p.btab, p.Ftab, p.direct.quad, bs_mem, scratch);
        eval_rows_any<T>(g.comps, g.flux != 0, k, bbase, bs, vtab, out, (size_t)g.nfx, plane, g.nfx, 0, g.nfy,
                         make_walk(threadIdx.x, blockDim.x, g.nfx), blockDim.x);
    }
}

}  // namespace bang
