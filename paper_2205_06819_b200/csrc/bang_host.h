// bang_host.h -- host-side glue shared by bang_api.cu and the per-(T,S) instantiation units.  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>

#include "bang_kernels.cuh"

namespace bang {

// everything a fused launch needs, precision-agnostic (the instantiation unit converts to T)
struct FusedLaunch {
    GridC g;
    FitC fit;
    const void* btab; int btab_first, btab_cells;
    const void* Ftab; int Ftab_first, Ftab_cells;
    QuadC quad;                  // reading U': N_J-node rule as {a_k, b_k} pairs (device)
    const double* W; int nacc;   // composite taps, nacc * s of them
    const double* theta; int B;
    int P, nxp, mode;
    void* maps;
    const double2* data;
    double C0;
    double* logL;
    int* slow_list; int* slow_count;   // theta left to the direct path (k_slow), see FusedParams
    int threads, ctas;           // launch shape (ctas = 0: let the launcher size a persistent grid)
    int n_sm;
    int smem_optin;              // the device's opt-in maximum of dynamic shared memory per CTA
    int* cache;                  // [2] resident CTAs per SM of the mode's kernel once configured (0 = not yet), or NULL
    cudaStream_t stream;
};

// One per (T, S) translation unit (bang_fused_inst.cu compiled with -DBANG_INST_T / -DBANG_INST_S).
// Returns cudaErrorInvalidValue when (nacc, P) is not instantiated.  query_only: just report occupancy/resources.
struct FusedInfo { int regs; int max_ctas_per_sm; size_t smem; int ctas; };
#define BANG_DECL_FUSED(TN, S) cudaError_t launch_fused_##TN##_##S(const FusedLaunch& L, FusedInfo* info, bool query_only);
BANG_DECL_FUSED(float, 1) BANG_DECL_FUSED(float, 2) BANG_DECL_FUSED(float, 3) BANG_DECL_FUSED(float, 4)
BANG_DECL_FUSED(double, 1) BANG_DECL_FUSED(double, 2) BANG_DECL_FUSED(double, 3) BANG_DECL_FUSED(double, 4)
#undef BANG_DECL_FUSED

// accumulator depths instantiated: NACC = ceil((2 r_k + s)/s) is rounded up to one of these (taps zero padded)
constexpr int kNaccList[] = {1, 4, 7, 10, 13};
inline int round_nacc(int need) {
    for (int v : kNaccList) if (v >= need) return v;
    return -1;
}

}  // namespace bang
