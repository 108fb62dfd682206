// bang_fused_inst.cu -- instantiations of the fused kernel for one (T, S); compiled once per pair with
//   -DBANG_INST_T=float|double -DBANG_INST_TN=float|double -DBANG_INST_S=1..4
// so that the heavy, fully unrolled PSF code builds in parallel translation units.
#include <cstdio>
#include <cstdlib>

#include "bang_host.h"

#ifndef BANG_INST_T
#error "compile with -DBANG_INST_T=<type> -DBANG_INST_TN=<name> -DBANG_INST_S=<s>"
#endif

namespace bang {
namespace {

template <typename T, int S, int NACC, int P, int MODE, int LBC, bool FLUX>
cudaError_t launch_mode(const FusedLaunch& L, FusedInfo* info, bool query_only) {
    auto kern = []() {
        if constexpr (sizeof(T) == 8) return k_fused64<T, S, NACC, P, MODE, LBC, FLUX>;
        else return k_fused<T, S, NACC, P, MODE, LBC, FLUX>;
    }();
    if (L.threads > lbc_threads(LBC)) return cudaErrorInvalidValue;
    const size_t smem = fused_smem_bytes<T>(L.g, S, lbc_nfb(LBC, P, S, NACC, (int)sizeof(T)));
    // the shared-memory opt-in and the occupancy query are done once per context and mode (L.cache, owned by the
    // context): repeating them on every call costs ~10 us of host time, which a small batch notices
    int per_sm = L.cache ? L.cache[L.mode] : 0;
    cudaError_t e;
    if (per_sm < 1) {
        if (smem > (size_t)L.smem_optin) return cudaErrorLaunchOutOfResources;
        // opted in to the device maximum, not to this launch's size: the attribute is per function, and another context
        // of the same instantiation (reading U' in fp64 mode) may need more
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, L.smem_optin);
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, L.threads, smem);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) return cudaErrorLaunchOutOfResources;
        if (L.cache && !query_only) L.cache[L.mode] = per_sm;
    }
    int ctas = L.ctas > 0 ? L.ctas : per_sm * L.n_sm;
    if (ctas > L.B) ctas = L.B;
    if (info) {
        cudaFuncAttributes fa;
        cudaFuncGetAttributes(&fa, kern);
        info->regs = fa.numRegs; info->max_ctas_per_sm = per_sm; info->smem = smem; info->ctas = ctas;
    }
    if (query_only || L.B <= 0) return cudaSuccess;
#ifdef BANG_TUNING
    if (getenv("BANG_VERBOSE")) {
        cudaFuncAttributes fa;
        cudaFuncGetAttributes(&fa, kern);
        fprintf(stderr, "[bang] k_fused<%s,S=%d,NACC=%d,P=%d,MODE=%d,LBC=%d,FLUX=%d> regs=%d smem=%zu threads=%d ctas/SM=%d grid=%d B=%d\n",
                sizeof(T) == 4 ? "f32" : "f64", S, NACC, P, MODE, LBC, (int)FLUX, fa.numRegs, smem, L.threads, per_sm, ctas, L.B);
    }
#endif

    FusedParams<T, S, NACC> p;
    p.g = L.g; p.fit = L.fit;
    p.btab = PolyTab<T>{static_cast<const T*>(L.btab), L.btab_first, L.btab_cells};
    p.Ftab = PolyTab<T>{static_cast<const T*>(L.Ftab), L.Ftab_first, L.Ftab_cells};
    p.quad = L.quad; p.bs_elems = (int)bs_elems<T>(L.g);
    for (int t = 0; t < NACC * S; ++t) p.W[t] = (T)L.W[t];
    if constexpr (sizeof(T) == 4) {
        constexpr int N = NACC * S;
        auto w = [&](int t) { return t < N ? (float)L.W[t] : 0.f; };
        for (int k = 0; k < (N + 1) / 2; ++k) {
            p.W2.a[k] = make_float2(w(2 * k), w(2 * k + 1));
            p.W2.b[k] = make_float2(w(2 * k + 1), w(2 * k + 2));
        }
        for (int t = 0; t < N; ++t) p.W2.d[t] = make_float2(w(t), w(t));
    }
    p.theta = L.theta; p.B = L.B; p.mode = L.mode; p.nxp = L.nxp;
    p.maps = static_cast<T*>(L.maps); p.data = L.data; p.C0 = L.C0; p.logL = L.logL;
    p.slow_list = L.slow_list; p.slow_count = L.slow_count;
    kern<<<ctas, L.threads, smem, L.stream>>>(p);
    return cudaGetLastError();
}

template <typename T, int S, int NACC, int P, int LBC>
cudaError_t launch_lbc(const FusedLaunch& L, FusedInfo* info, bool query_only) {
    if constexpr (sizeof(T) == 8) {
        // fp64 mode: one instantiation serves both calls (MODE 2: p.mode read at run time), which halves its build
        return L.g.flux ? launch_mode<T, S, NACC, P, 2, LBC, true>(L, info, query_only)
                        : launch_mode<T, S, NACC, P, 2, LBC, false>(L, info, query_only);
    } else {
        if (L.g.flux)      // reading G': a separate instantiation, so that the paper's path keeps its registers
            return L.mode == 0 ? launch_mode<T, S, NACC, P, 0, LBC, true>(L, info, query_only)
                               : launch_mode<T, S, NACC, P, 1, LBC, true>(L, info, query_only);
        return L.mode == 0 ? launch_mode<T, S, NACC, P, 0, LBC, false>(L, info, query_only)
                           : launch_mode<T, S, NACC, P, 1, LBC, false>(L, info, query_only);
    }
}
template <typename T, int S, int NACC, int P>
cudaError_t launch_one(const FusedLaunch& L, FusedInfo* info, bool query_only) {
    if (L.threads <= 128) return launch_lbc<T, S, NACC, P, 0>(L, info, query_only);
#ifndef BANG_TUNING
    // fp32 mode takes P = 2 only for maps of up to 64 columns, i.e. 128 threads: the wider classes would be dead code
    if constexpr (sizeof(T) == 4 && P == 2) return cudaErrorInvalidValue;
    else
#endif
    {
        if (L.threads <= 256) return launch_lbc<T, S, NACC, P, 1>(L, info, query_only);
        return launch_lbc<T, S, NACC, P, 2>(L, info, query_only);
    }
}

template <typename T, int S, int P>
cudaError_t launch_nacc(const FusedLaunch& L, FusedInfo* info, bool q) {
#ifdef BANG_ONLY_NACC      // development builds: instantiate one accumulator depth only (seconds instead of minutes)
    if (L.nacc == BANG_ONLY_NACC) return launch_one<T, S, BANG_ONLY_NACC, P>(L, info, q);
    return cudaErrorInvalidValue;
#else
    switch (L.nacc) {
        case 1: return launch_one<T, S, 1, P>(L, info, q);
        case 4: return launch_one<T, S, 4, P>(L, info, q);
        case 7: return launch_one<T, S, 7, P>(L, info, q);
        case 10: return launch_one<T, S, 10, P>(L, info, q);
        case 13: return launch_one<T, S, 13, P>(L, info, q);
        default: return cudaErrorInvalidValue;
    }
#endif
}

}  // namespace

#define BANG_CAT3(a, b, c) a##b##_##c
#define BANG_NAME(tn, s) BANG_CAT3(launch_fused_, tn, s)

cudaError_t BANG_NAME(BANG_INST_TN, BANG_INST_S)(const FusedLaunch& L, FusedInfo* info, bool query_only) {
    using T = BANG_INST_T;
    constexpr int S = BANG_INST_S;
    if (L.g.s != S) return cudaErrorInvalidValue;
    if constexpr (sizeof(T) == 8) {
        if (L.P == 2) return launch_nacc<T, S, 2>(L, info, query_only);
    } else {
        if (L.P == 4) return launch_nacc<T, S, 4>(L, info, query_only);
#ifdef BANG_TUNING      // fp32 mode always takes P = 4; the P = 2 kernels exist in development builds only
        if (L.P == 2) return launch_nacc<T, S, 2>(L, info, query_only);
#endif
    }
    return cudaErrorInvalidValue;
}

}  // namespace bang
