// grad_hybrid.cuh -- analytic gradient on MIPWA_PATH_HYBRID (some shapes float, some are fixed): the passes of grad.cuh
// with north_star (d) applied term by term, as in k_nll_hybrid.  `m` holds the spline tables of the call and ONLY the
// floating resonances (device slots d < F: spin 1 first, then spin 2); the symmetrised values of the RC fixed-shape
// resonances come from the per-point caches of the hybrid path (column 1 + k of the tile layout of cached.cuh, built in
// the cell-sorted point order this kernel walks), enter A with the coefficients cc.c[k] and need no Breit-Wigner,
// barrier or Zemach arithmetic at all: 26-52 FP64 instructions per point and cached term less than k_grad_recompute.
//
// result / partial layout (doubles), Rt = F + RC: [0] sum ln|A|^2, [1] sum w|A|^2, [2 + 2d + {0,1}] F_ev of slot d
// (d < F floating: f conj(T_d) without sqrt(n_R n_D); d >= F cached: f conj(b_k), fold factor included in the column),
// [2 + 2Rt + 2d + {0,1}] F_nm, then bins_ev[4][N-1][2], bins_nm[4][N-1][2];  NV = 2 + 4 Rt + 16 (N-1).
#pragma once
#include "grad.cuh"
#include "hybrid.cuh"

// dynamic shared memory of k_grad_hybrid beyond the segment moments: MIPWA_GRAD_RING_STAGES x (1 + RC) columns x block
__host__ __device__ constexpr size_t mipwa_grad_ring_bytes(int rct)
{
    return (size_t)MIPWA_GRAD_RING_STAGES * (1 + rct) * MIPWA_GRAD_BLOCK * sizeof(double2);
}

template <int R1, int R2, int RCT, int FL>
__global__ void __launch_bounds__(MIPWA_GRAD_BLOCK, MIPWA_GRAD_MINBLOCKS)
k_grad_hybrid(const __grid_constant__ DevModel m, const __grid_constant__ HybCoef cc,
              const double* __restrict__ e12, const double* __restrict__ e13, const unsigned short* __restrict__ eseg,
              const double2* __restrict__ ev_cache, long long n_ev,
              const double* __restrict__ g12, const double* __restrict__ g13, const double* __restrict__ gw,
              const unsigned short* __restrict__ gseg, const double2* __restrict__ nm_cache, long long n_norm,
              double* __restrict__ partials, double2* __restrict__ f_ev, double2* __restrict__ f_nm)
{
    constexpr int RR = GradDims<R1, R2>::RR, F = R1 + R2, RT = F + RCT;
    extern __shared__ double grad_bins[];                  // [2][4][N-1][2], then the cp.async ring of grad_pass
    __shared__ SplineCoefSmem sm;
    const int NS = m.N - 1, nb = 8 * NS, NV = 2 + 4 * RT + 2 * nb;
    double2* const ring = reinterpret_cast<double2*>(grad_bins + 2 * nb) + threadIdx.x;   // 16 NS doubles: 16-byte aligned
    for (int k = threadIdx.x; k < 2 * nb; k += blockDim.x) grad_bins[k] = 0.0;
    load_spline_coef_smem(sm, m);                          // ends with __syncthreads()

    double* mine = partials + (size_t)blockIdx.x * NV;
    __shared__ double wpart[2][MIPWA_GRAD_BLOCK / 32][1 + 2 * RT];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        double Sc = 0.0, Fr[RR], Fi[RR], Cr[RCT], Ci[RCT];
#pragma unroll
        for (int r = 0; r < RR; ++r) Fr[r] = Fi[r] = 0.0;
#pragma unroll
        for (int k = 0; k < RCT; ++k) Cr[k] = Ci[k] = 0.0;
        double qsum = 0.0;
        if (pass == 0)
            grad_pass<R1, R2, FL, true, false, RCT>(sm, m, e12, e13, nullptr, eseg, n_ev, f_ev, 0.0, qsum, grad_bins, Sc, Fr, Fi,
                                                    ev_cache, cc.c, Cr, Ci, ring);
        else
            grad_pass<R1, R2, FL, false, false, RCT>(sm, m, g12, g13, gw, gseg, n_norm, f_nm, 0.0, qsum, grad_bins + nb, Sc, Fr,
                                                     Fi, nm_cache, cc.c, Cr, Ci, ring);
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) Sc += __shfl_down_sync(0xffffffffu, Sc, off);
        if (lane == 0) wpart[pass][warp][0] = Sc;
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            double a = r < F ? Fr[r < F ? r : 0] : Cr[r >= F ? r - F : 0];
            double bq = r < F ? Fi[r < F ? r : 0] : Ci[r >= F ? r - F : 0];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                a += __shfl_down_sync(0xffffffffu, a, off);
                bq += __shfl_down_sync(0xffffffffu, bq, off);
            }
            if (lane == 0) { wpart[pass][warp][1 + 2 * r] = a; wpart[pass][warp][2 + 2 * r] = bq; }
        }
    }
    __syncthreads();                                       // every warp has left both sets of sums
    for (int t = threadIdx.x; t < 2 * (1 + 2 * RT); t += blockDim.x) {
        const int pass = t / (1 + 2 * RT), k = t - pass * (1 + 2 * RT);
        double v = 0.0;
        for (int w = 0; w < nwarp; ++w) v += wpart[pass][w][k];            // fixed order
        mine[k == 0 ? pass : 2 + 2 * RT * pass + (k - 1)] = v;
    }
    __syncthreads();                                       // all flushes into grad_bins are done
    for (int k = threadIdx.x; k < 2 * nb; k += blockDim.x) mine[2 + 4 * RT + k] = grad_bins[k];
}
