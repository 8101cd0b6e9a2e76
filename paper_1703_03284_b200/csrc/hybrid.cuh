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
__device__ __forceinline__ double hybrid_abs2(const RowsSmem& sm, const DevModel& m, const HybCoef& cc, double2 s,
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

// ---- staging ring ------------------------------------------------------------------------------------------------------
// At 16 + 16 RC bytes per point this kernel needs 3-6 TB/s while the FP64 pipe is busy with the floating terms, and a
// register prefetch one tile ahead keeps only ~17 KB per SM in flight (measured: 2.8 TB/s, latency bound, slower than
// the full recompute at RC = 1).  The cache columns therefore go through a shared-memory ring filled by per-thread
// 16-byte cp.async copies MIPWA_HYB_STAGES - 1 tiles ahead: every thread copies exactly the slots it later reads, so
// cp.async.wait_group is the only synchronisation (no barrier, no mbarrier), the data in flight cost no registers,
// and (STAGES - 1) x 512 threads x 16 (1 + RC) B = 50-110 KB per SM are on their way at any time.
// threads per block (a multiple of the 256-point cache tile), resident blocks per SM, and points per thread and
// iteration: a block takes MIPWA_HYB_PTS * MIPWA_HYB_BLOCK / MIPWA_TILE tiles per iteration.  One floating resonance is
// a single dependent chain of ~100 FP64 instructions per point; with four warps per scheduler that does not fill the
// pipe (k_nll_recompute with one resonance: 0.19 ms where the instruction count says 0.14), so two independent points
// are evaluated side by side.
#define MIPWA_HYB_BLOCK 512
// points per thread and iteration: two while the ring still gets >= 3 stages (RC <= 3), else one
#define MIPWA_HYB_PTS(rct) ((rct) <= 3 ? 2 : 1)
// ring stages: as many as fit 200 KB of shared memory, at most 4, at least 2
__host__ __device__ constexpr int mipwa_hyb_stages(int rct)
{
    const size_t per_stage = (size_t)MIPWA_HYB_PTS(rct) * (1 + rct) * MIPWA_HYB_BLOCK * sizeof(double2);
    const size_t fit = (size_t)200 * 1024 / per_stage;
    return fit >= 4 ? 4 : (fit >= 2 ? (int)fit : 2);
}
#define MIPWA_HYB_STAGES(rct) mipwa_hyb_stages(rct)
__host__ __device__ constexpr size_t mipwa_hyb_ring_bytes(int rct)
{
    return (size_t)mipwa_hyb_stages(rct) * MIPWA_HYB_PTS(rct) * (1 + rct) * MIPWA_HYB_BLOCK * sizeof(double2);
}

__device__ __forceinline__ void cp_async16(double2* smem_dst, const double2* gsrc)
{
    const unsigned int sa = (unsigned int)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NPENDING) : "memory"); }

// One launch over [events | normalisation points]; one point per thread and tile.  result[0] = sum ln|A|^2,
// result[1] = sum w |A|^2 (w == NULL: weight 1).
// eseg / gseg: the stored segment pairs of the same (cell-sorted or caller's) point order the caches were built in;
// they and the weights (2 + 8 B per point) are prefetched through registers, as far ahead as the ring.
// Dynamic shared memory: mipwa_hyb_ring_bytes(RCT).
template <int R1, int R2, int RCT, int FL>
__global__ void __launch_bounds__(MIPWA_HYB_BLOCK, 1)
k_nll_hybrid(const __grid_constant__ DevModel m, const __grid_constant__ HybCoef cc,
             const double2* __restrict__ ev_cache, const unsigned short* __restrict__ eseg, long long n_ev,
             const double2* __restrict__ nm_cache, const double* __restrict__ gw,
             const unsigned short* __restrict__ gseg, long long n_norm,
             double2* __restrict__ partials, unsigned int* __restrict__ ticket, double* __restrict__ result, long long tag)
{
    extern __shared__ __align__(16) unsigned char hyb_ring_raw[];
    __shared__ RowsSmem sm;
    __shared__ double red[2 * 32];
    __shared__ bool is_last;
    asm volatile("griddepcontrol.launch_dependents;");     // mipwa_nll_batch: as k_nll_recompute (kernels.cuh); otherwise nothing
    load_rows_smem(sm, m);
    constexpr int C = 1 + RCT, ST = MIPWA_HYB_STAGES(RCT), AHEAD = ST - 1, PTS = MIPWA_HYB_PTS(RCT);
    constexpr int TPB = MIPWA_HYB_BLOCK / MIPWA_TILE;                                  // tiles per block and point slot
    constexpr int STAGE = PTS * C * MIPWA_HYB_BLOCK;                                   // double2 per ring stage
    // slot (stage, point u, column k) of this thread: ring[stage * STAGE + (u * C + k) * BLOCK]
    double2* const ring = reinterpret_cast<double2*>(hyb_ring_raw) + threadIdx.x;
    const int sub = threadIdx.x / MIPWA_TILE, lane_t = threadIdx.x % MIPWA_TILE;       // this thread's tile of the TPB, slot in it
    const int G = (int)gridDim.x * TPB * PTS;                                          // tiles per grid iteration
    LogProd lp;
    double integ = 0.0;
    // The FP64 pipe and the other instructions share the scheduler's issue slots (profiles/r1_k_nll_hybrid_ncu.md), so the
    // bookkeeping is kept to 32-bit tile counters, one compare per point and pointers advanced by a constant.
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        const double2* cache = pass == 0 ? ev_cache : nm_cache;
        const unsigned short* segs = pass == 0 ? eseg : gseg;
        const long long n = pass == 0 ? n_ev : n_norm;
        const bool has_w = pass == 1 && gw != nullptr;
        const int n_tiles = (int)((n + MIPWA_TILE - 1) / MIPWA_TILE);
        // this thread's slot of tile t holds a point iff t < lim (the last tile may be partly filled)
        const int lim = (int)(n / MIPWA_TILE) + (lane_t < (int)(n % MIPWA_TILE) ? 1 : 0);
        int tile = (int)blockIdx.x * TPB * PTS + sub;       // point u of this thread: tile + u * TPB
        // cursors of the next tile to fetch (AHEAD iterations ahead of `tile`)
        int ft = tile;
        const double2* fc = cache + (size_t)tile * C * MIPWA_TILE + lane_t;
        const unsigned short* fs = segs + (size_t)tile * MIPWA_TILE + lane_t;
        const double* fw = gw + (size_t)tile * MIPWA_TILE + lane_t;
        const size_t dcache = (size_t)G * C * MIPWA_TILE, dpts = (size_t)G * MIPWA_TILE;
        int wr = 0, rd = 0;                                   // ring offsets (double2) of the stage to fill / to read
        // one commit group per iteration (empty past the end, so that the group count stays uniform)
        auto fetch = [&](unsigned int (&sg)[PTS], double (&w)[PTS]) {
#pragma unroll
            for (int u = 0; u < PTS; ++u) {
                if (ft + u * TPB < n_tiles) {
#pragma unroll
                    for (int k = 0; k < C; ++k)
                        cp_async16(ring + wr + (u * C + k) * MIPWA_HYB_BLOCK, fc + (size_t)(u * TPB * C + k) * MIPWA_TILE);
                }
                const bool in = ft + u * TPB < lim;
                sg[u] = in ? fs[(size_t)u * TPB * MIPWA_TILE] : 0u;
                w[u] = pass == 1 && in ? (has_w ? fw[(size_t)u * TPB * MIPWA_TILE] : 1.0) : 0.0;
            }
            cp_async_commit();
            ft += G; fc += dcache; fs += dpts; fw += dpts;
            wr = wr + STAGE == ST * STAGE ? 0 : wr + STAGE;
        };
        unsigned int sgq[AHEAD][PTS];
        double wq[AHEAD][PTS];
#pragma unroll
        for (int q = 0; q < AHEAD; ++q) fetch(sgq[q], wq[q]);
        for (; tile - sub < n_tiles; tile += G) {          // block-uniform trip count
            unsigned int nsg[PTS];
            double nw[PTS];
            fetch(nsg, nw);
            cp_async_wait<AHEAD>();                                        // this iteration's group has landed
            double vv[PTS];
            bool live[PTS];
#pragma unroll
            for (int u = 0; u < PTS; ++u) {
                const double2* slot = ring + rd + u * C * MIPWA_HYB_BLOCK;
                double2 b[RCT];
                const double2 s = slot[0];
#pragma unroll
                for (int k = 0; k < RCT; ++k) b[k] = slot[(1 + k) * MIPWA_HYB_BLOCK];
                live[u] = tile + u * TPB < lim;
                // padding slots of the last tile hold (0, 0), slots of tiles past the end are stale: evaluate a
                // harmless point instead and drop its value below
                vv[u] = hybrid_abs2<R1, R2, RCT, FL>(sm, m, cc, live[u] ? s : make_double2(1.0, 1.0), sgq[0][u], b);
            }
#pragma unroll
            for (int u = 0; u < PTS; ++u) {
                if (pass == 0) lp.add_counted(live[u] ? vv[u] : 1.0);
                else integ = fma(wq[0][u], live[u] ? vv[u] : 0.0, integ);
            }
#pragma unroll
            for (int q = 0; q + 1 < AHEAD; ++q) {
#pragma unroll
                for (int u = 0; u < PTS; ++u) { sgq[q][u] = sgq[q + 1][u]; wq[q][u] = wq[q + 1][u]; }
            }
#pragma unroll
            for (int u = 0; u < PTS; ++u) { sgq[AHEAD - 1][u] = nsg[u]; wq[AHEAD - 1][u] = nw[u]; }
            rd = rd + STAGE == ST * STAGE ? 0 : rd + STAGE;
        }
        cp_async_wait<0>();                                                // nothing of this pass lands in the next pass's stages
    }
    double v[2] = { lp.value(), integ };
    block_reduce<2>(v, red);
    asm volatile("griddepcontrol.wait;" ::: "memory");     // the previous launch has left the partials and the ticket
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
            publish_result(result, tag);
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
