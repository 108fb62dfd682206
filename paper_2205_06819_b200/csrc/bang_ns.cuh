// bang_ns.cuh -- the replacement step of nested sampling on the device ("the worst
// live point is replaced by a point of higher likelihood found by MCMC"): K constrained random walks advance in lock-step,
// proposal -> batched likelihood (k_fused) -> accept/reject, with the walkers, their likelihoods and the parameter vectors
// resident in device memory for all `steps` MCMC steps -- no host round trip inside a call (bang_ns_walk).
//
// The walkers live in the unit cube u in [0,1]^d under a uniform prior; theta = theta0 with theta[free[j]] = lo[j] +
// (hi[j] - lo[j]) u[j] (a box prior).  Walker k belongs to group g = group[k] (one group per independent run / retire
// batch): groups have their own proposal covariance (Cholesky factor) and step scale, walkers their own likelihood bound.
// Random numbers: Philox4x32-10 (Salmon et al. 2011), counter = (walker, step, draw), key = seed -- each side of a test can
// reproduce any draw without state.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bang {

constexpr int kNsMaxDim = 17;

struct Philox4 { uint32_t x, y, z, w; };
__host__ __device__ inline Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return Philox4{c0, c1, c2, c3};
}
// two standard normals from two 32-bit words (Box-Muller on u1 in (0,1], u2 in [0,1))
__host__ __device__ inline void normal_pair(uint32_t a, uint32_t b, double& n0, double& n1) {
    const double u1 = ((double)a + 1.0) * (1.0 / 4294967296.0), u2 = (double)b * (1.0 / 4294967296.0);
    const double r = sqrt(-2.0 * log(u1));
    double s, c;
    sincos(6.283185307179586476925 * u2, &s, &c);
    n0 = r * c; n1 = r * s;
}

struct NsParams {
    int K, d, step;
    uint64_t seed;
    int free_idx[kNsMaxDim];
    double lo[kNsMaxDim], hi[kNsMaxDim];
    double theta0[17];
    const double* u;             // [K][d] current positions
    const double* logL;          // [K] their likelihoods
    const double* Lstar;         // [K] likelihood bounds
    const int* group;            // [K]
    const double* chol;          // [G][d][d] lower-triangular Cholesky factors of the proposal covariances, row-major
    const double* scale;         // [G] step scales (already times 2.38/sqrt(d))
    double* prop;                // [K][d] proposals
    double* theta;               // [K][17] proposals as parameter vectors (NaN when outside the cube: logL = -inf)
};

__global__ void k_ns_propose(const NsParams p) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= p.K) return;
    const int d = p.d, g = p.group[k];
    double z[kNsMaxDim + 3];
    for (int j = 0; j < d; j += 4) {
        const Philox4 r = philox4x32_10((uint32_t)k, (uint32_t)p.step, (uint32_t)(j >> 2), 0u, (uint32_t)p.seed, (uint32_t)(p.seed >> 32));
        normal_pair(r.x, r.y, z[j], z[j + 1]);
        normal_pair(r.z, r.w, z[j + 2], z[j + 3]);
    }
    const double* L = p.chol + (size_t)g * d * d;
    const double sc = p.scale[g];
    bool inside = true;
    double th[17];
    for (int i = 0; i < 17; ++i) th[i] = p.theta0[i];
    for (int i = 0; i < d; ++i) {
        double a = 0.0;
        for (int j = 0; j <= i; ++j) a = fma(L[i * d + j], z[j], a);
        const double v = p.u[(size_t)k * d + i] + sc * a;
        p.prop[(size_t)k * d + i] = v;
        inside = inside && v >= 0.0 && v <= 1.0;
        th[p.free_idx[i]] = fma(p.hi[i] - p.lo[i], v, p.lo[i]);
    }
    const double qnan = nan("");
    for (int i = 0; i < 17; ++i) p.theta[(size_t)k * 17 + i] = inside ? th[i] : qnan;
}

// accept the proposals whose likelihood beats the walker's bound; counts per group
__global__ void k_ns_accept(int K, int d, const double* __restrict__ prop, const double* __restrict__ pl,
                            const double* __restrict__ Lstar, const int* __restrict__ group, double* __restrict__ u,
                            double* __restrict__ logL, int* __restrict__ n_acc) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= K) return;
    const double l = pl[k];
    if (l > Lstar[k]) {                              // false for NaN and -inf
        for (int i = 0; i < d; ++i) u[(size_t)k * d + i] = prop[(size_t)k * d + i];
        logL[k] = l;
        atomicAdd(n_acc + group[k], 1);
    }
}

}  // namespace bang
