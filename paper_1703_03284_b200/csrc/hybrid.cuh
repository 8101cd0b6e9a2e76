// hybrid.cuh -- MIPWA_PATH_HYBRID: some resonance shapes float, others are fixed (BASELINE configs[3]: only the
// rho(770) mass and width float).  North_star (d) applied term by term: the fixed-shape resonances are linear
// basis functions whose symmetrised values are cached once per point (compact layout of cached.cuh: col 0 =
// (s12, s13), col 1+k = B of the k-th FIXED resonance, for events AND for normalisation points), the floating ones and
// the spline are re-evaluated every call.  The normalisation integral stays a sum over the points (the floating terms
// rule out a Gram matrix).  Per point: 16 + 16 RC bytes streamed + the arithmetic of R - RC resonances.
//
// `m` holds the spline tables of the call and ONLY the floating resonances (device slots: spin 1 first, then spin 2);
// cc.c[k] = coefficient of the k-th fixed resonance (its cache column carries sqrt(n_R n_D)).
#pragma once
#include "cached.cuh"

struct HybCoef {
    int32_t RC, pad;
    double2 c[MIPWA_DEV_MAX_RES];
};

template <int R1, int R2, int RCT, int FL>
__device__ __forceinline__ double hybrid_abs2(const SplineCoefSmem& sm, const DevModel& m, const HybCoef& cc, double2 s,
                                              unsigned int sg, const double2 (&b)[RCT])
{
    double re, im;
    amplitude_seg<R1, R2, FL>(sm, m, s.x, s.y, sg, re, im);   // spline + floating resonances
#pragma unroll
    for (int k = 0; k < RCT; ++k) {
        const double2 c = cc.c[k];
        re = fma(c.x, b[k].x, fma(-c.y, b[k].y, re));
        im = fma(c.x, b[k].y, fma(c.y, b[k].x, im));
    }
    return fma(re, re, im * im);
}

// One launch over [events | normalisation points]; one point per thread and tile, the next tile's columns are
// loaded before the current tile is evaluated.  result[0] = sum ln|A|^2, result[1] = sum w |A|^2 (w == NULL: weight 1).
// eseg / gseg: the stored segment pairs of the same (cell-sorted or caller's) point order the caches were built in.
template <int R1, int R2, int RCT, int FL>
__global__ void __launch_bounds__(MIPWA_TILE, 2)
k_nll_hybrid(const __grid_constant__ DevModel m, const __grid_constant__ HybCoef cc,
             const double2* __restrict__ ev_cache, const unsigned short* __restrict__ eseg, long long n_ev,
             const double2* __restrict__ nm_cache, const double* __restrict__ gw,
             const unsigned short* __restrict__ gseg, long long n_norm,
             double2* __restrict__ partials, unsigned int* __restrict__ ticket, double* __restrict__ result)
{
    __shared__ SplineCoefSmem sm;
    __shared__ double red[2 * 32];
    __shared__ bool is_last;
    load_spline_coef_smem(sm, m);
    constexpr int C = 1 + RCT;
    LogProd lp;
    double integ = 0.0;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        const double2* cache = pass == 0 ? ev_cache : nm_cache;
        const unsigned short* segs = pass == 0 ? eseg : gseg;
        const long long n = pass == 0 ? n_ev : n_norm;
        const long long n_tiles = (n + MIPWA_TILE - 1) / MIPWA_TILE;
        double2 s = make_double2(1.0, 1.0), b[RCT];
        double w = 0.0;
        unsigned int sg = 0u;
#pragma unroll
        for (int k = 0; k < RCT; ++k) b[k] = make_double2(0.0, 0.0);
        long long tile = blockIdx.x;
        if (tile < n_tiles) {
            const double2* p = cache + (size_t)tile * C * MIPWA_TILE + threadIdx.x;
            s = ld_stream(p);
#pragma unroll
            for (int k = 0; k < RCT; ++k) b[k] = ld_stream(p + (size_t)(1 + k) * MIPWA_TILE);
            const long long i = tile * MIPWA_TILE + threadIdx.x;
            if (pass == 1) w = i < n ? (gw ? gw[i] : 1.0) : 0.0;
            if (i < n) sg = segs[i];
        }
        for (; tile < n_tiles; tile += gridDim.x) {
            double2 ns = make_double2(1.0, 1.0), nb[RCT];
            double nw = 0.0;
            unsigned int nsg = 0u;
#pragma unroll
            for (int k = 0; k < RCT; ++k) nb[k] = make_double2(0.0, 0.0);
            const long long nt = tile + gridDim.x;
            if (nt < n_tiles) {
                const double2* p = cache + (size_t)nt * C * MIPWA_TILE + threadIdx.x;
                ns = ld_stream(p);
#pragma unroll
                for (int k = 0; k < RCT; ++k) nb[k] = ld_stream(p + (size_t)(1 + k) * MIPWA_TILE);
                const long long i = nt * MIPWA_TILE + threadIdx.x;
                if (pass == 1) nw = i < n ? (gw ? gw[i] : 1.0) : 0.0;
                if (i < n) nsg = segs[i];
            }
            const bool live = tile * MIPWA_TILE + threadIdx.x < n;
            // padding slots of the last tile hold (0, 0): evaluate a harmless point instead
            const double v = hybrid_abs2<R1, R2, RCT, FL>(sm, m, cc, live ? s : make_double2(1.0, 1.0), live ? sg : 0u, b);
            if (pass == 0) lp.add(live ? v : 1.0);
            else integ = fma(w, v, integ);
            s = ns; w = nw; sg = nsg;
#pragma unroll
            for (int k = 0; k < RCT; ++k) b[k] = nb[k];
        }
    }
    double v[2] = { lp.value(), integ };
    block_reduce<2>(v, red);
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = make_double2(v[0], v[1]);
        __threadfence();
        is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        double f[2] = { 0.0, 0.0 };
        for (int k = threadIdx.x; k < gridDim.x; k += blockDim.x) {
            const double2 q = __ldcg(&partials[k]);
            f[0] += q.x; f[1] += q.y;
        }
        block_reduce<2>(f, red);
        if (threadIdx.x == 0) {
            result[0] = f[0];
            result[1] = f[1];
            *ticket = 0;
            __threadfence_system();
        }
    }
}

// floating signature (f1 spin-1, f2 spin-2 floating resonances) x number of cached columns
#define MIPWA_HYB_CASE(f1, f2, rc) ((f1) * 100 + (f2) * 10 + (rc))
#define MIPWA_DISPATCH_HYB(f1, f2, rc, CALL)                                                                   \
    switch (MIPWA_HYB_CASE(f1, f2, rc)) {                                                                       \
        case MIPWA_HYB_CASE(1, 0, 1): { constexpr int R1 = 1, R2 = 0, RCT = 1; CALL; } break;                  \
        case MIPWA_HYB_CASE(1, 0, 2): { constexpr int R1 = 1, R2 = 0, RCT = 2; CALL; } break;                  \
        case MIPWA_HYB_CASE(1, 0, 3): { constexpr int R1 = 1, R2 = 0, RCT = 3; CALL; } break;                  \
        case MIPWA_HYB_CASE(1, 0, 4): { constexpr int R1 = 1, R2 = 0, RCT = 4; CALL; } break;                  \
        case MIPWA_HYB_CASE(1, 0, 5): { constexpr int R1 = 1, R2 = 0, RCT = 5; CALL; } break;                  \
        case MIPWA_HYB_CASE(0, 1, 1): { constexpr int R1 = 0, R2 = 1, RCT = 1; CALL; } break;                  \
        case MIPWA_HYB_CASE(0, 1, 2): { constexpr int R1 = 0, R2 = 1, RCT = 2; CALL; } break;                  \
        case MIPWA_HYB_CASE(0, 1, 3): { constexpr int R1 = 0, R2 = 1, RCT = 3; CALL; } break;                  \
        case MIPWA_HYB_CASE(0, 1, 4): { constexpr int R1 = 0, R2 = 1, RCT = 4; CALL; } break;                  \
        case MIPWA_HYB_CASE(2, 0, 1): { constexpr int R1 = 2, R2 = 0, RCT = 1; CALL; } break;                  \
        case MIPWA_HYB_CASE(2, 0, 2): { constexpr int R1 = 2, R2 = 0, RCT = 2; CALL; } break;                  \
        case MIPWA_HYB_CASE(2, 0, 3): { constexpr int R1 = 2, R2 = 0, RCT = 3; CALL; } break;                  \
        case MIPWA_HYB_CASE(2, 0, 4): { constexpr int R1 = 2, R2 = 0, RCT = 4; CALL; } break;                  \
        case MIPWA_HYB_CASE(1, 1, 1): { constexpr int R1 = 1, R2 = 1, RCT = 1; CALL; } break;                  \
        case MIPWA_HYB_CASE(1, 1, 2): { constexpr int R1 = 1, R2 = 1, RCT = 2; CALL; } break;                  \
        case MIPWA_HYB_CASE(1, 1, 3): { constexpr int R1 = 1, R2 = 1, RCT = 3; CALL; } break;                  \
        case MIPWA_HYB_CASE(1, 1, 4): { constexpr int R1 = 1, R2 = 1, RCT = 4; CALL; } break;                  \
        default: supported = false; break;                                                                      \
    }

// the same with constexpr FL = the MIPWA_FL_EQM bit of the model flags (radii sharing needs two floating resonances
// of one spin: only the <2, 0, *> signatures)
#define MIPWA_DISPATCH_HYBFL(f1, f2, rc, fl, CALL)                                                              \
    if ((fl) & MIPWA_FL_EQM) {                                                                                  \
        if (((fl) & MIPWA_FL_SHR) && (f1) == 2) { constexpr int FL = MIPWA_FL_EQM | MIPWA_FL_SHR; MIPWA_DISPATCH_HYB(f1, f2, rc, CALL) } \
        else { constexpr int FL = MIPWA_FL_EQM; MIPWA_DISPATCH_HYB(f1, f2, rc, CALL) }                         \
    } else { constexpr int FL = 0; MIPWA_DISPATCH_HYB(f1, f2, rc, CALL) }
