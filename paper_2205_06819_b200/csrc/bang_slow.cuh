// bang_slow.cuh -- the direct path of the fused call: the rare theta whose radii leave the tabulated ranges of the fast
// kernel (more octaves of r^2 on the grid than the per-theta v_c table holds, |i| -> 90 deg; or R/R_b outside the
// scale-free bulge tables) are recorded by k_fused in a list and evaluated here, cell by cell, by eval_cell_direct:
// eq. 4-5 in closed form, eq. 6 by the N_J-node rule, eq. 10 term by term, in fp64.  Same dataflow as k_fused (fine row ->
// composite taps along x at stride s -> scatter along y into NACC running data rows -> chi-square), written generically
// (run-time s, NACC, P) with the accumulators in shared memory: it is 1e3-1e4 times slower per cell and is launched
// after every fused launch; with an empty list it returns at once.
#pragma once
#include "bang_kernels.cuh"

namespace bang {

template <typename T>
struct SlowParams {
    GridC g;
    PolyTab<T> btab, Ftab;
    DirectC direct;
    const double* W;             // composite taps (device), nacc * s of them, zero padded
    int nacc;
    const double* theta;         // [B][17]
    const int* slow_list;        // indices into theta
    int* slow_count;             // number of entries; reset to 0 by the last CTA to finish
    int* done;                   // CTAs finished (reset likewise)
    T* maps;                     // MODE 0: [B][4][ny][nx]
    const double2* data;         // MODE 1: [ny][4][P][gmax] {d, 1/e}
    int P, gmax;
    double C0;
    double* logL;                // MODE 1: [B]
};

template <typename T>
inline size_t slow_smem_bytes(const GridC& g, int nacc) {
    return (sizeof(ThetaC<T>) + 15) / 16 * 16 + ((size_t)4 * g.nfx + (size_t)nacc * 4 * g.nx) * sizeof(T) + 32 * sizeof(double);
}

template <typename T, int MODE>
__global__ void __launch_bounds__(256) k_slow(const __grid_constant__ SlowParams<T> p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ThetaC<T>& c = *reinterpret_cast<ThetaC<T>*>(smem_raw);
    constexpr size_t off = (sizeof(ThetaC<T>) + 15) / 16 * 16;
    const GridC& g = p.g;
    const int S = g.s, NACC = p.nacc, nx = g.nx, nfx = g.nfx;
    T* fine = reinterpret_cast<T*>(smem_raw + off);                  // [4][nfx]: the current fine row
    T* acc = fine + (size_t)4 * nfx;                                 // [NACC][4][nx]: running data rows (ring)
    double* red = reinterpret_cast<double*>(acc + (size_t)NACC * 4 * nx);
    const int tid = threadIdx.x, NT = blockDim.x;
    const int n = *p.slow_count;
    const size_t npix = (size_t)nx * g.ny;
    const int ntap = 2 * g.rk + S;

    for (int li = blockIdx.x; li < n; li += gridDim.x) {
        const int b = p.slow_list[li];
        __syncthreads();
        if (tid == 0) { decode_theta<T>(p.theta + (size_t)b * kNTheta, g, p.btab, p.Ftab, c); pack_cellk<T>(c); }
        for (int i = tid; i < NACC * 4 * nx; i += NT) acc[i] = T(0);
        __syncthreads();
        const CellK<T> k = load_cellk<T>(c);
        double chi2 = 0.0;
        const int nrows = (g.ny + NACC - 1) * S;
        for (int jy = 0; jy < nrows; ++jy) {
            const int sr = jy / S, j = jy - sr * S;
            // a2 + a3: one fine row, directly (reading G': the light moments)
            for (int x = tid; x < nfx; x += NT) {
                T o[4] = {T(0), T(0), T(0), T(0)};
                if (jy < g.nfy) {
                    if (g.flux) eval_cell_direct<T, true>(c, g, p.btab, p.Ftab, p.direct, x - k.jcx, jy - k.jcy, o);
                    else eval_cell_direct<T, false>(c, g, p.btab, p.Ftab, p.direct, x - k.jcx, jy - k.jcy, o);
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) fine[q * nfx + x] = o[q];
            }
            __syncthreads();
            // a4 + a5: composite taps along x at stride s, then the same taps along y into the running data rows
            for (int item = tid; item < 4 * nx; item += NT) {
                const int q = item / nx, px = item - q * nx;
                T xs = T(0);
                for (int t = 0; t < ntap; ++t) xs = fma((T)p.W[t], fine[q * nfx + px * S + t], xs);
                for (int kk = 0; kk < NACC; ++kk) {
                    const int py = sr - (NACC - 1) + kk;             // data row that accumulator kk of this super-row feeds
                    if (py >= 0 && py < g.ny) {
                        T& a = acc[((py % NACC) * 4 + q) * nx + px];
                        a = fma((T)p.W[(NACC - 1 - kk) * S + j], xs, a);
                    }
                }
            }
            __syncthreads();
            const int py0 = sr - (NACC - 1);
            if (j == S - 1 && py0 >= 0) {                            // a6 (or map output): data row py0 is complete
                T* row = acc + (size_t)(py0 % NACC) * 4 * nx;
                for (int item = tid; item < 4 * nx; item += NT) {
                    const int q = item / nx, px = item - q * nx;
                    T m = row[q * nx + px];
                    if (g.flux) {                                    // reading G': v = M1/M0, sigma^2 = M2/M0 - v^2, M/L = M3/M0
                        const T i0 = inv_ml(row[px]), v = row[nx + px] * i0;
                        if (q == 1) m = v;
                        else if (q == 2) m = fast_sqrt(fmax(fma(m, i0, -v * v), T(0)));
                        else if (q == 3) m = m * i0;
                    } else if (q == 3) {
                        m = inv_ml(m);
                    }
                    if constexpr (MODE == 0) {
                        p.maps[((size_t)b * 4 + q) * npix + (size_t)py0 * nx + px] = m;
                    } else {
                        const int grp = px / p.P, i = px - grp * p.P;
                        const double2 de = p.data[((size_t)(py0 * 4 + q) * p.P + i) * p.gmax + grp];
                        const double z = (de.x - (double)m) * de.y;
                        chi2 = de.y != 0.0 ? fma(z, z, chi2) : chi2;
                    }
                }
                __syncthreads();
                for (int item = tid; item < 4 * nx; item += NT) row[item] = T(0);
                __syncthreads();
            }
        }
        if constexpr (MODE == 1) {
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
    // the last CTA to finish empties the list for the next call on this stream
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(p.done, 1) == (int)gridDim.x - 1) { *p.slow_count = 0; *p.done = 0; }
    }
}

}  // namespace bang
