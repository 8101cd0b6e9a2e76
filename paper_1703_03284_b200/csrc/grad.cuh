// grad.cuh -- analytic gradient of the NLL on the recompute path (BASELINE configs[3]).
//
// With calG_k := dNLL/dRe c_k + i dNLL/dIm c_k for every complex linear coefficient c_k of A = sum_k c_k B_k,
//   calG_k = sum_i f_i conj(B_ik) + (2 n_ev / I) sum_j g_j conj(B_jk),   f_i = -2 / conj(A_i),  g_j = w_j A_j.
// The kernel never forms the dense spline basis.  On segment j the S-wave is the cubic
//   S(s) = sum_q sc[q][j] t^q,  t = s - x_j,
// and sc is a REAL linear image of the knot values y (DevModel::sc, built on the host from y and y'' = Mx y), so it
// is enough to accumulate the complex moments  M[q][j] = sum f t^q  over the points whose channel falls in segment
// j (the adjoint of the Horner evaluation); the host applies the transposed map sc -> (y, y'') -> y and the polar
// chain rule (O(N) work, one transposed tridiagonal relation via Mx^T).  Resonance coefficients get
// F_r = sum f conj(T_r(s12,s13) + T_r(s13,s12)) in per-thread registers.
//
// Scatter without atomics in the inner loop: mipwa_nll_grad works on a copy of the points SORTED BY CELL
// (cell = seg(s12) * (N-1) + seg(s13); knots are fixed, so the order is built once per mipwa_set_*).  Each warp owns
// a contiguous chunk, so consecutive iterations of a warp stay in one cell for thousands of points: the 8 complex
// moments (4 per channel) live in registers and are flushed (warp shuffle reduction, then 16 shared-memory
// adds by lane 0) only when the warp's cell changes.  A warp-iteration that straddles a cell boundary takes a
// slower path: one shuffle-reduce round per distinct cell in the group (add_mixed).
#pragma once
#include "cached.cuh"

// segment index and offset of one channel, then the Horner value (same arithmetic as spline_eval)
__device__ __forceinline__ void spline_eval_jt(const SplineSmem& sm, const DevModel& m, double s, int& j, double& t,
                                               double& re, double& im)
{
    double xj;
    j = spline_segment(sm, m, s, xj);
    t = s - xj;
    const double2 c0 = sm.sc[0][j], c1 = sm.sc[1][j], c2 = sm.sc[2][j], c3 = sm.sc[3][j];
    re = fma(t, fma(t, fma(t, c3.x, c2.x), c1.x), c0.x);
    im = fma(t, fma(t, fma(t, c3.y, c2.y), c1.y), c0.y);
}

#define MIPWA_GRAD_MAXR (MIPWA_DEV_MAX_RES)

// amplitude with the pieces the gradient needs: segment/offset of both channels and every symmetrised resonance
// term WITHOUT its coefficient (device slot order; the host multiplies by sqrt(n_R n_D))
template <int R1, int R2, int FL>
__device__ __forceinline__ void amplitude_parts(const SplineCoefSmem& sm, const DevModel& m, double s12, double s13,
                                                unsigned int seg, double& are, double& aim, int& j1, double& t1,
                                                int& j2, double& t2,
                                                double (&tr)[R1 >= 0 ? (R1 + R2 > 0 ? R1 + R2 : 1) : MIPWA_GRAD_MAXR],
                                                double (&ti)[R1 >= 0 ? (R1 + R2 > 0 ? R1 + R2 : 1) : MIPWA_GRAD_MAXR])
{
    double r1, i1, r2, i2;
    j1 = (int)(seg & 0xffu); j2 = (int)(seg >> 8);         // segment pair stored by k_validate
    t1 = s12 - sm.knots[j1]; t2 = s13 - sm.knots[j2];
    spline_eval_at(sm, s12, j1, r1, i1);
    spline_eval_at(sm, s13, j2, r2, i2);
    are = r1 + r2;
    aim = i1 + i2;
    if (R1 == 0 && R2 == 0) return;
    const Channel ca = make_channel<FL>(m, s12, s13), cb = make_channel<FL>(m, s13, s12);
    if (R1 >= 0) {
        if ((FL & MIPWA_FL_SHR) && R1 >= 2) {
            group_shared_terms<1, (R1 >= 2 ? R1 : 2)>(&m.res[0], ca, cb, &tr[0], &ti[0]);
        } else {
#pragma unroll
            for (int r = 0; r < R1; ++r) resonance_sym<1>(m.res[r], ca, cb, tr[r], ti[r]);
        }
        if ((FL & MIPWA_FL_SHR) && R2 >= 2) {
            group_shared_terms<2, (R2 >= 2 ? R2 : 2)>(&m.res[R1 > 0 ? R1 : 0], ca, cb, &tr[R1 > 0 ? R1 : 0],
                                                      &ti[R1 > 0 ? R1 : 0]);
        } else {
#pragma unroll
            for (int r = 0; r < R2; ++r) resonance_sym<2>(m.res[R1 + r], ca, cb, tr[R1 + r], ti[R1 + r]);
        }
#pragma unroll
        for (int r = 0; r < R1 + R2; ++r) {
            are = fma(m.res[r].cre, tr[r], fma(-m.res[r].cim, ti[r], are));
            aim = fma(m.res[r].cre, ti[r], fma(m.res[r].cim, tr[r], aim));
        }
    } else {
        for (int r = 0; r < m.R; ++r) {
            resonance_sym<-1>(m.res[r], ca, cb, tr[r], ti[r]);
            are = fma(m.res[r].cre, tr[r], fma(-m.res[r].cim, ti[r], are));
            aim = fma(m.res[r].cre, ti[r], fma(m.res[r].cim, tr[r], aim));
        }
    }
}

// per-warp running moments of the current cell
struct CellAcc {
    double v[16];          // [channel][q][re,im]
    int j1, j2;            // segments of the cell, -1: empty
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = 0.0;
    }
    __device__ __forceinline__ void add(double fr, double fi, double t1, double t2) {
        double p = 1.0;
#pragma unroll
        for (int q = 0; q < 4; ++q) { v[2 * q] = fma(fr, p, v[2 * q]); v[2 * q + 1] = fma(fi, p, v[2 * q + 1]); p *= t1; }
        p = 1.0;
#pragma unroll
        for (int q = 0; q < 4; ++q) { v[8 + 2 * q] = fma(fr, p, v[8 + 2 * q]); v[8 + 2 * q + 1] = fma(fi, p, v[8 + 2 * q + 1]); p *= t2; }
    }
};

// bins[(q * NS + j) * 2 + {0,1}], NS = N - 1 segments
__device__ __forceinline__ void flush_warp(CellAcc& a, double* bins, int NS)
{
    if (a.j1 >= 0) {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            double x = a.v[k];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
            a.v[k] = x;
        }
        if ((threadIdx.x & 31) == 0) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                atomicAdd(&bins[(q * NS + a.j1) * 2], a.v[2 * q]);
                atomicAdd(&bins[(q * NS + a.j1) * 2 + 1], a.v[2 * q + 1]);
                atomicAdd(&bins[(q * NS + a.j2) * 2], a.v[8 + 2 * q]);
                atomicAdd(&bins[(q * NS + a.j2) * 2 + 1], a.v[8 + 2 * q + 1]);
            }
        }
    }
    a.clear();
    a.j1 = a.j2 = -1;
}

// A warp-iteration whose 32 points fall into several cells (it straddles a cell boundary of the sorted order): one
// round per distinct cell - the lanes of that cell contribute, the others add zeros - through the same
// shuffle-reduce + lane-0 flush, instead of per-lane shared atomics that would all collide on the same bins.
// `acc` must be empty on entry and is empty on return.
__device__ __forceinline__ void add_mixed(CellAcc& acc, bool valid, int j1, int j2, double fr, double fi, double t1,
                                          double t2, double* bins, int NS)
{
    unsigned int remaining = __ballot_sync(0xffffffffu, valid);
    while (remaining) {                                                    // warp-uniform
        const int leader = __ffs(remaining) - 1;
        const int l1 = __shfl_sync(0xffffffffu, j1, leader), l2 = __shfl_sync(0xffffffffu, j2, leader);
        const bool mine = valid && j1 == l1 && j2 == l2;
        acc.j1 = l1; acc.j2 = l2;
        acc.add(mine ? fr : 0.0, mine ? fi : 0.0, t1, t2);
        flush_warp(acc, bins, NS);
        remaining &= ~__ballot_sync(0xffffffffu, mine);
    }
}

// sum over the block of one value per thread (valid in thread 0); red32: 32 doubles of shared memory
__device__ __forceinline__ double block_sum(double x, double* red32)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
    __syncthreads();                                       // red32 free again
    if (lane == 0) red32[warp] = x;
    __syncthreads();
    x = (warp == 0 && lane < nwarp) ? red32[lane] : 0.0;
    if (warp == 0) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
    }
    return x;
}

#ifndef MIPWA_GRAD_RING_STAGES
#define MIPWA_GRAD_RING_STAGES 4
#endif
#ifndef MIPWA_CP_ASYNC_DEFINED
#define MIPWA_CP_ASYNC_DEFINED
__device__ __forceinline__ void cp_async16(double2* smem_dst, const double2* gsrc)
{
    const unsigned int sa = (unsigned int)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NPENDING) : "memory"); }
#endif

template <int R1, int R2> struct GradDims {
    static constexpr int RR = R1 >= 0 ? (R1 + R2 > 0 ? R1 + R2 : 1) : MIPWA_GRAD_MAXR;
};

// one pass over a cell-sorted point set.  EV: events (f = -2/conj(A), scalar = sum ln|A|^2);
// otherwise normalisation points (f = w A, scalar = sum w |A|^2).
// MIX (EV only): background density w[i] per event and D = |A|^2 + kappa w: f = -2 A / D, scalar = sum ln D,
// qsum = sum w / D (mipwa_nll_mix_grad).
// RCT > 0 (k_grad_hybrid, grad_hybrid.cuh): `m` holds only the floating resonances; the symmetrised values of RCT
// fixed-shape resonances are read from the per-point cache of MIPWA_PATH_HYBRID (tile layout of cached.cuh, column 1 + k,
// same point order as s12/s13), enter the amplitude with the coefficients coef[k] and get their own accumulators
// Cr/Ci = sum f conj(b_k): for a cached term the basis function IS the cache column.
template <int R1, int R2, int FL, bool EV, bool MIX = false, int RCT = 0>
__device__ __forceinline__ void grad_pass(const SplineCoefSmem& sm, const DevModel& m, const double* __restrict__ s12,
                                          const double* __restrict__ s13, const double* __restrict__ w,
                                          const unsigned short* __restrict__ sgp, long long n,
                                          double2* __restrict__ fout, double kappa, double& qsum,
                                          double* bins, double& scalar, double (&Fr)[GradDims<R1, R2>::RR],
                                          double (&Fi)[GradDims<R1, R2>::RR],
                                          const double2* __restrict__ cache = nullptr, const double2* coef = nullptr,
                                          double* Cr = nullptr, double* Ci = nullptr, double2* ring = nullptr)
{
    constexpr int RR = GradDims<R1, R2>::RR;
    const int NS = m.N - 1, lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    const long long W = (long long)gridDim.x * wpb, wg = (long long)blockIdx.x * wpb + (threadIdx.x >> 5);
    const long long CH = (((n + W - 1) / W) + 31) & ~31LL;
    const long long lo = wg * CH, hi = lo + CH < n ? lo + CH : n;
    CellAcc acc;
    acc.clear();
    acc.j1 = acc.j2 = -1;
    LogProd lp;
    double integ = 0.0;
    const int nres = R1 >= 0 ? R1 + R2 : m.R;
    // Non-FP64 instructions cost the issue slots the FP64 pipe needs (profiles/r1_k_grad_recompute_ncu.md): the loop runs
    // on 32-bit offsets into this warp's chunk (CH <= 2^31 - 32: mipwa_nll_grad admits at most 2^31 - 1 points per set).
    const int cnt = lo < hi ? (int)(hi - lo) : 0;
    const double* const p12 = s12 + lo;
    const double* const p13 = s13 + lo;
    const double* const pw = w + lo;
    const unsigned short* const psg = sgp + lo;
    double2* const pf = fout + lo;
    const bool has_w = w != nullptr;
    double nx = 1.0, ny = 1.0, nw = 0.0;                                   // next iteration's point, loaded one ahead
    unsigned int nsg = 0u;
    // cache columns of the warp's 32 points: lo is a multiple of 32, so they share one 256-point tile
    constexpr int RCN = RCT > 0 ? RCT : 1, CC = 1 + RCT;
    const double2* const cbase = RCT > 0 ? cache + (size_t)(lo / MIPWA_TILE) * CC * MIPWA_TILE : nullptr;
    const int coff = (int)(lo % MIPWA_TILE);
    auto cidx = [&](int ii) { const int g = coff + ii; return (g / MIPWA_TILE) * (CC * MIPWA_TILE) + (g % MIPWA_TILE); };
    // The cache columns go through a per-thread cp.async ring (as in k_nll_hybrid: every lane copies the slots it later
    // reads, cp.async.wait_group is the only synchronisation), GRAD_RING_AHEAD warp-iterations ahead; slot (stage, k) of
    // this thread: ring[(stage * (1 + RCT) + k) * blockDim.x], `ring` already offset by threadIdx.x.  Column 0 is the
    // point (s12, s13) itself, so only the segment pair and the weight (2 + 8 B) still come through registers - two
    // iterations ahead: with the resonance arithmetic gone an iteration is too short to cover a DRAM round trip.
    constexpr int AHEAD = MIPWA_GRAD_RING_STAGES - 1;
    const int rstage = (RCT > 0 ? CC : 1) * (int)blockDim.x;
    int wr = 0, rd = 0;
    auto fetch = [&](int i_next) {                        // i_next: this lane's offset AHEAD iterations on (or past the end)
        if (RCT > 0) {
            if (i_next - lane < cnt) {                     // warp-uniform: the iteration exists
                const double2* q = cbase + cidx(i_next < cnt ? i_next : 0);
#pragma unroll
                for (int k = 0; k < CC; ++k) cp_async16(ring + wr + k * (int)blockDim.x, q + k * MIPWA_TILE);
            }
            cp_async_commit();
            wr = wr + rstage == MIPWA_GRAD_RING_STAGES * rstage ? 0 : wr + rstage;
        }
    };
    if (RCT > 0) {
#pragma unroll
        for (int q = 0; q < AHEAD; ++q) fetch(lane + 32 * q);
    }
    double n2w = 0.0;                                                      // RCT > 0: the point after the next
    unsigned int n2sg = 0u;
    auto side = [&](int i_at, unsigned int& sgo, double& wo) {            // segment pair and weight at offset i_at
        const bool in = i_at < cnt;
        const int ii = in ? i_at : 0;
        sgo = psg[ii];
        wo = 0.0;
        if (!EV) wo = in ? (has_w ? pw[ii] : 1.0) : 0.0;
        if (EV && MIX) wo = pw[ii];
    };
    if (cnt > 0) {
        if (RCT > 0) {
            side(lane, nsg, nw);
            if (32 < cnt) side(lane + 32, n2sg, n2w);
        } else {
            const int ii = lane < cnt ? lane : 0;
            nx = p12[ii]; ny = p13[ii]; nsg = psg[ii];
            if (!EV) nw = lane < cnt ? (has_w ? pw[ii] : 1.0) : 0.0;
            if (EV && MIX) nw = pw[ii];
        }
    }
    for (int base = 0; base < cnt; base += 32) {                           // warp-uniform trip count
        const int i = base + lane;
        const bool valid = i < cnt;
        double x = nx, y = ny;
        const double wv = nw;
        const unsigned int sg = nsg;
        double2 bk[RCN];
        if (RCT > 0) {
            nsg = n2sg; nw = n2w;
            if (base + 64 < cnt) side(i + 64, n2sg, n2w);
            fetch(i + 32 * AHEAD);
            cp_async_wait<AHEAD>();                        // this iteration's columns have landed
            const double2 pt = ring[rd];
            x = pt.x; y = pt.y;
#pragma unroll
            for (int k = 0; k < RCT; ++k) bk[k] = ring[rd + (1 + k) * (int)blockDim.x];
            rd = rd + rstage == MIPWA_GRAD_RING_STAGES * rstage ? 0 : rd + rstage;
        } else if (base + 32 < cnt) {
            const bool more = i + 32 < cnt;
            const int ii = more ? i + 32 : 0;
            nx = p12[ii]; ny = p13[ii]; nsg = psg[ii];
            if (!EV) nw = more ? (has_w ? pw[ii] : 1.0) : 0.0;
            if (EV && MIX) nw = pw[ii];
        }
        double are, aim, t1, t2, tr[RR], ti[RR];
        int j1, j2;
        amplitude_parts<R1, R2, FL>(sm, m, x, y, sg, are, aim, j1, t1, j2, t2, tr, ti);
        if (RCT > 0) {
#pragma unroll
            for (int k = 0; k < RCT; ++k) {
                const double2 ck = coef[k];
                are = fma(ck.x, bk[k].x, fma(-ck.y, bk[k].y, are));
                aim = fma(ck.x, bk[k].y, fma(ck.y, bk[k].x, aim));
            }
        }
        const double a2 = fma(are, are, aim * aim);
        double fr, fi;
        if (EV) {
            const double D = MIX ? fma(kappa, wv, a2) : a2;
            const double rD = fast_rcp(D);
            const double k = valid ? -2.0 * rD : 0.0;
            fr = k * are; fi = k * aim;
            lp.add(valid ? D : 1.0);
            if (MIX) qsum += valid ? wv * rD : 0.0;
        } else {
            fr = wv * are; fi = wv * aim;
            integ = fma(wv, a2, integ);
        }
        if (fout && valid) pf[i] = make_double2(fr, fi);                  // for k_grad_shape (mipwa_nll_grad_full)
        if (RCT > 0) {
#pragma unroll
            for (int k = 0; k < RCT; ++k) {
                Cr[k] = fma(fr, bk[k].x, fma(fi, bk[k].y, Cr[k]));         // f conj(b_k)
                Ci[k] = fma(fi, bk[k].x, fma(-fr, bk[k].y, Ci[k]));
            }
        }
        if (R1 >= 0) {
#pragma unroll
            for (int r = 0; r < (R1 >= 0 ? R1 + R2 : 0); ++r) {
                Fr[r] = fma(fr, tr[r], fma(fi, ti[r], Fr[r]));             // f conj(T)
                Fi[r] = fma(fi, tr[r], fma(-fr, ti[r], Fi[r]));
            }
        } else {
            for (int r = 0; r < nres; ++r) {
                Fr[r] = fma(fr, tr[r], fma(fi, ti[r], Fr[r]));
                Fi[r] = fma(fi, tr[r], fma(-fr, ti[r], Fi[r]));
            }
        }
        const bool same = !valid || (j1 == acc.j1 && j2 == acc.j2);
        if (__all_sync(0xffffffffu, same)) {
            acc.add(fr, fi, t1, t2);
        } else {
            flush_warp(acc, bins, NS);
            const int l1 = __shfl_sync(0xffffffffu, j1, 0), l2 = __shfl_sync(0xffffffffu, j2, 0);   // lane 0 is valid
            const bool uni = !valid || (j1 == l1 && j2 == l2);
            if (__all_sync(0xffffffffu, uni)) {
                acc.j1 = l1; acc.j2 = l2;
                acc.add(fr, fi, t1, t2);
            } else {
                add_mixed(acc, valid, j1, j2, fr, fi, t1, t2, bins, NS);
            }
        }
    }
    flush_warp(acc, bins, NS);
    if (RCT > 0) cp_async_wait<0>();                       // nothing of this pass lands in the next pass's stages
    scalar = EV ? lp.value() : integ;
}

// result / partial layout (doubles): [0] sum ln|A|^2, [1] sum w|A|^2, [2 + 2d + {0,1}] F_ev of device slot d,
// [2 + 2R + 2d + {0,1}] F_nm, then bins_ev[4][N-1][2], bins_nm[4][N-1][2];  NV = 2 + 4R + 16 (N-1).
#ifndef MIPWA_GRAD_BLOCK
#define MIPWA_GRAD_BLOCK 512
#endif
#ifndef MIPWA_GRAD_MINBLOCKS
#define MIPWA_GRAD_MINBLOCKS 1
#endif
template <int R1, int R2, int FL, bool MIX>
__global__ void __launch_bounds__(MIPWA_GRAD_BLOCK, MIPWA_GRAD_MINBLOCKS)
k_grad_recompute(const __grid_constant__ DevModel m,
                 const double* __restrict__ e12, const double* __restrict__ e13,
                 const unsigned short* __restrict__ eseg, const double* __restrict__ eb, double kappa, long long n_ev,
                 const double* __restrict__ g12, const double* __restrict__ g13, const double* __restrict__ gw,
                 const unsigned short* __restrict__ gseg, long long n_norm, double* __restrict__ partials,
                 double2* __restrict__ f_ev, double2* __restrict__ f_nm)
{
    constexpr int RR = GradDims<R1, R2>::RR;
    extern __shared__ double grad_bins[];                  // [2][4][N-1][2]
    __shared__ SplineCoefSmem sm;
    const int NS = m.N - 1, R = m.R, nb = 8 * NS, NV = 2 + 4 * R + 2 * nb;
    for (int k = threadIdx.x; k < 2 * nb; k += blockDim.x) grad_bins[k] = 0.0;
    load_spline_coef_smem(sm, m);                          // ends with __syncthreads()

    double* mine = partials + (size_t)blockIdx.x * NV;
    // events pass, then normalisation pass; only one set of resonance accumulators is live at a time (register
    // pressure).  After a pass every warp leaves its sums in shared memory and moves on: no block barrier between the
    // passes, so a warp that finishes its chunk early starts the next pass at once.
    __shared__ double wpart[2][MIPWA_GRAD_BLOCK / 32][1 + 2 * RR];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        double Sc = 0.0, Fr[RR], Fi[RR];
#pragma unroll
        for (int r = 0; r < RR; ++r) Fr[r] = Fi[r] = 0.0;
        double qsum = 0.0;
        if (pass == 0) grad_pass<R1, R2, FL, true, MIX>(sm, m, e12, e13, eb, eseg, n_ev, f_ev, kappa, qsum, grad_bins, Sc, Fr, Fi);
        else grad_pass<R1, R2, FL, false>(sm, m, g12, g13, gw, gseg, n_norm, f_nm, 0.0, qsum, grad_bins + nb, Sc, Fr, Fi);
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) Sc += __shfl_down_sync(0xffffffffu, Sc, off);
        if (MIX) {
            // the events-only launch of the mixture has no normalisation points: slot [1] carries sum b / D instead
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) qsum += __shfl_down_sync(0xffffffffu, qsum, off);
            if (lane == 0) {
                if (pass == 0) { wpart[0][warp][0] = Sc; wpart[1][warp][0] = qsum; }
                else wpart[1][warp][0] += Sc;
            }
        } else if (lane == 0) wpart[pass][warp][0] = Sc;
#pragma unroll
        for (int r = 0; r < RR; ++r) {
            double a = Fr[r], bq = Fi[r];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                a += __shfl_down_sync(0xffffffffu, a, off);
                bq += __shfl_down_sync(0xffffffffu, bq, off);
            }
            if (lane == 0) { wpart[pass][warp][1 + 2 * r] = a; wpart[pass][warp][2 + 2 * r] = bq; }
        }
    }
    __syncthreads();                                       // every warp has left both sets of sums
    for (int t = threadIdx.x; t < 2 * (1 + 2 * R); t += blockDim.x) {
        const int pass = t / (1 + 2 * R), k = t - pass * (1 + 2 * R);
        double v = 0.0;
        for (int w = 0; w < nwarp; ++w) v += wpart[pass][w][k];            // fixed order
        mine[k == 0 ? pass : 2 + 2 * R * pass + (k - 1)] = v;
    }
    __syncthreads();                                       // all flushes into grad_bins are done
    for (int k = threadIdx.x; k < 2 * nb; k += blockDim.x) mine[2 + 4 * R + k] = grad_bins[k];
}

// fixed-order sum of the per-block partial vectors: one warp per value, lane l adds blocks l, l+32, .. then a shuffle
// tree.  A separate tiny launch: done inside the last block of k_grad_recompute it would serialise ~NV x grid L2 reads
// on one SM while the rest of the GPU idles.
static __global__ void __launch_bounds__(256)
k_grad_finalize(const double* __restrict__ partials, int nblocks, int NV, double* __restrict__ result)
{
    const int k = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (k >= NV) return;
    double s = 0.0;
    for (int b = lane; b < nblocks; b += 32) s += partials[(size_t)b * NV + k];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
    if (lane == 0) result[k] = s;
}

// ---- cell sort (once per point set): key = seg(s12) * (N-1) + seg(s13) ---------------------------------------------
static __global__ void __launch_bounds__(MIPWA_TILE)
k_cell_keys(const unsigned short* __restrict__ seg, long long n, int NS, unsigned int* __restrict__ keys,
            unsigned int* __restrict__ idx)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const unsigned int sg = seg[i];                    // j12 | j13 << 8, stored by k_validate
        keys[i] = (sg & 0xffu) * (unsigned int)NS + (sg >> 8);
        idx[i] = (unsigned int)i;
    }
}

static __global__ void __launch_bounds__(MIPWA_TILE)
k_gather(const unsigned int* __restrict__ idx, long long n, const double* __restrict__ a, const double* __restrict__ b,
         const double* __restrict__ c, const unsigned short* __restrict__ sg, double* __restrict__ oa,
         double* __restrict__ ob, double* __restrict__ oc, unsigned short* __restrict__ osg)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const unsigned int s = idx[i];
        oa[i] = a[s]; ob[i] = b[s]; osg[i] = sg[s];
        if (c) oc[i] = c[s];
    }
}

// ---- A8 on the compact cached path (fixed shapes) -------------------------------------------------------------------
// Events only: the normalisation part of the gradient is (2 n_ev / I) (G c)_k from the Gram matrix (host, K^2 MACs).
// Streams the compact cache (16 + 16 R bytes per event, cell-sorted event order), evaluates the spline part from
// the shared-memory tables, and accumulates  f = -2/conj(A):  moments f t^q per segment (as k_grad_recompute) and
// F_r = sum f conj(B_{N+r}) per resonance.  Partial vector per block: [S, F(2R), bins(8 (N-1))].
template <int RT>
__global__ void __launch_bounds__(MIPWA_TILE, 2)
k_grad_compact(const __grid_constant__ DevModel m, const __grid_constant__ CoefDev cc,
               const double2* __restrict__ cache, long long n_ev, double* __restrict__ partials)
{
    constexpr int RC = RT > 0 ? RT : (RT == 0 ? 1 : MIPWA_GRAD_MAXR);
    extern __shared__ double grad_bins[];                  // [4][N-1][2]
    __shared__ SplineSmem sm;
    __shared__ double red32[32];
    const int R = RT >= 0 ? RT : m.R, C = 1 + R, N = cc.N, NS = N - 1, nb = 8 * NS, NV = 1 + 2 * R + nb;
    for (int k = threadIdx.x; k < nb; k += blockDim.x) grad_bins[k] = 0.0;
    load_spline_smem(sm, m);

    const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    const long long W = (long long)gridDim.x * wpb, wg = (long long)blockIdx.x * wpb + (threadIdx.x >> 5);
    const long long CH = (((n_ev + W - 1) / W) + 31) & ~31LL;
    const long long lo = wg * CH, hi = lo + CH < n_ev ? lo + CH : n_ev;
    CellAcc acc;
    acc.clear();
    acc.j1 = acc.j2 = -1;
    LogProd lp;
    double Fr[RC], Fi[RC];
#pragma unroll
    for (int r = 0; r < RC; ++r) Fr[r] = Fi[r] = 0.0;
    for (long long base = lo; base < hi; base += 32) {                     // warp-uniform trip count; base % 32 == 0
        const long long i = base + lane;
        const bool valid = i < hi;
        const long long ii = valid ? i : lo;
        const double2* p = cache + (size_t)(ii / MIPWA_TILE) * C * MIPWA_TILE + (ii % MIPWA_TILE);
        const double2 s = ld_stream(p);
        double2 b[RC];
        if (RT >= 0) {
#pragma unroll
            for (int r = 0; r < RT; ++r) b[r] = ld_stream(p + (size_t)(1 + r) * MIPWA_TILE);
        } else {
            for (int r = 0; r < R; ++r) b[r] = ld_stream(p + (size_t)(1 + r) * MIPWA_TILE);
        }
        int j1, j2;
        double t1, t2, r1, i1, r2, i2;
        spline_eval_jt(sm, m, s.x, j1, t1, r1, i1);
        spline_eval_jt(sm, m, s.y, j2, t2, r2, i2);
        double are = r1 + r2, aim = i1 + i2;
        if (RT >= 0) {
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                const double2 c = cc.c[N + r];
                are = fma(c.x, b[r].x, fma(-c.y, b[r].y, are));
                aim = fma(c.x, b[r].y, fma(c.y, b[r].x, aim));
            }
        } else {
            for (int r = 0; r < R; ++r) {
                const double2 c = cc.c[N + r];
                are = fma(c.x, b[r].x, fma(-c.y, b[r].y, are));
                aim = fma(c.x, b[r].y, fma(c.y, b[r].x, aim));
            }
        }
        const double a2 = fma(are, are, aim * aim);
        const double k = valid ? -2.0 * fast_rcp(a2) : 0.0;
        const double fr = k * are, fi = k * aim;
        lp.add(valid ? a2 : 1.0);
        if (RT >= 0) {
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                Fr[r] = fma(fr, b[r].x, fma(fi, b[r].y, Fr[r]));
                Fi[r] = fma(fi, b[r].x, fma(-fr, b[r].y, Fi[r]));
            }
        } else {
            for (int r = 0; r < R; ++r) {
                Fr[r] = fma(fr, b[r].x, fma(fi, b[r].y, Fr[r]));
                Fi[r] = fma(fi, b[r].x, fma(-fr, b[r].y, Fi[r]));
            }
        }
        const bool same = !valid || (j1 == acc.j1 && j2 == acc.j2);
        if (__all_sync(0xffffffffu, same)) {
            acc.add(fr, fi, t1, t2);
        } else {
            flush_warp(acc, grad_bins, NS);
            const int l1 = __shfl_sync(0xffffffffu, j1, 0), l2 = __shfl_sync(0xffffffffu, j2, 0);
            const bool uni = !valid || (j1 == l1 && j2 == l2);
            if (__all_sync(0xffffffffu, uni)) {
                acc.j1 = l1; acc.j2 = l2;
                acc.add(fr, fi, t1, t2);
            } else {
                add_mixed(acc, valid, j1, j2, fr, fi, t1, t2, grad_bins, NS);
            }
        }
    }
    flush_warp(acc, grad_bins, NS);

    double* mine = partials + (size_t)blockIdx.x * NV;
    double v = block_sum(lp.value(), red32);
    if (threadIdx.x == 0) mine[0] = v;
    for (int r = 0; r < R; ++r) {
        double a = 0, bb = 0;
        if (RT >= 0) {
#pragma unroll
            for (int q = 0; q < RC; ++q) if (q == r) { a = Fr[q]; bb = Fi[q]; }
        } else { a = Fr[r]; bb = Fi[r]; }
        a = block_sum(a, red32); if (threadIdx.x == 0) mine[1 + 2 * r] = a;
        bb = block_sum(bb, red32); if (threadIdx.x == 0) mine[1 + 2 * r + 1] = bb;
    }
    __syncthreads();
    for (int k2 = threadIdx.x; k2 < nb; k2 += blockDim.x) mine[1 + 2 * R + k2] = grad_bins[k2];
}


// ---- derivatives with respect to floating masses and widths (mipwa_nll_grad_full) ---------------------
// For a floating resonance in one channel, with D_R, D_D, W' = m0 Gamma(x) D_R, dD = (m0^2 - x) D_R, E = dD^2 + W'^2
// (dev_model.cuh) and u = (dD + i W') / E  (so BW = D_R u and BW m0 Gamma = W' u):
//   T'        = Z D_R rsqrt(D_R D_D) u                          (T without sqrt(n_R n_D), as everywhere in the kernels)
//   dT'/dG0   = T' (i W' / Gamma0) u
//   dT'/dm0   = T' [ a1 + u (-2 m0 D_R + i a2 W') ]             (a1, a2: ResDev::sh_a1, sh_a2)
// k_grad_recompute stores its per-point factor f (-2/conj(A) for events, w A for normalisation points) when asked to;
// this kernel streams (s12, s13, f), evaluates the two channels of every floating resonance and adds f conj(dT'_sym)
// into 4 doubles per floating resonance and pass.  The host multiplies by conj(c_r sqrt(n_R n_D)) and takes the real
// part.  One instantiation per number of floating resonances handled per launch (1..4).
#define MIPWA_SHAPE_MAXF 4
struct ShapeSel { int32_t slot[MIPWA_SHAPE_MAXF]; };       // device slots of the floating resonances of this launch

// LT = 0, 1, 2: spin known at compile time (one floating resonance per launch: the usual case); LT < 0: read from r.
template <int LT>
__device__ __forceinline__ void shape_channel(const ResDev& r, const Channel& c, double& mr, double& mi, double& gr,
                                              double& gi)
{
    double DR, DD, W, Z;
    if (LT == 0) {
        DR = 1.0; DD = 1.0; W = r.Kw * c.w[0]; Z = 1.0;
    } else if (LT == 1) {
        DR = fma(r.cR, c.ql, 1.0); DD = fma(r.cD, c.lam2, 1.0); W = r.Kw * c.w[1]; Z = c.Z[1];
    } else if (LT == 2) {
        const double zR = r.cR * c.ql, zD = r.cD * c.lam2;
        DR = fma(zR, zR + 3.0, 9.0); DD = fma(zD, zD + 3.0, 9.0); W = r.Kw * c.w[2]; Z = c.Z[2];
    } else {
        const double zR = r.cR * c.ql, zD = r.cD * c.lam2;
        DR = fma(zR, fma(zR, r.pa, r.pb), r.pc); DD = fma(zD, fma(zD, r.pa, r.pb), r.pc);
        W = r.Kw * pick(r.L, c.w); Z = pick(r.L, c.Z);
    }
    const double dD = (r.m0sq - c.x) * DR;
    const double rE = fast_rcp(fma(dD, dD, W * W));
    const double ur = dD * rE, ui = W * rE;
    const double t = Z * DR * fast_rsqrt(DR * DD);
    const double tr = t * ur, ti = t * ui;                 // T'
    const double k = r.sh_ig0 * W;                         // dT'/dG0 = T' (i k u)
    const double xr = -k * ui, xi = k * ur;
    gr = fma(tr, xr, -ti * xi); gi = fma(tr, xi, ti * xr);
    const double p = -r.sh_2m0 * DR, q = r.sh_a2 * W;      // dT'/dm0 = T' [a1 + u (p + i q)]
    const double br = r.sh_a1 + fma(ur, p, -ui * q), bi = fma(ur, q, ui * p);
    mr = fma(tr, br, -ti * bi); mi = fma(tr, bi, ti * br);
}

template <int NF, int FL, int LT = -1>
__global__ void __launch_bounds__(512, 1)
k_grad_shape(const __grid_constant__ DevModel m, const ShapeSel sel,
             const double* __restrict__ e12, const double* __restrict__ e13, const double2* __restrict__ f_ev,
             long long n_ev,
             const double* __restrict__ g12, const double* __restrict__ g13, const double2* __restrict__ f_nm,
             long long n_norm, double* __restrict__ partials)
{
    __shared__ double red32[32];
    const long long stride = (long long)gridDim.x * blockDim.x;
    double* mine = partials + (size_t)blockIdx.x * (8 * NF);
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        const double* s12 = pass == 0 ? e12 : g12;
        const double* s13 = pass == 0 ? e13 : g13;
        const double2* fp = pass == 0 ? f_ev : f_nm;
        const long long n = pass == 0 ? n_ev : n_norm;
        double acc[NF][4];
#pragma unroll
        for (int f = 0; f < NF; ++f) acc[f][0] = acc[f][1] = acc[f][2] = acc[f][3] = 0.0;
        // 32-bit trip count and cursor pointers, as in k_nll_recompute (issue slots: DESIGN.md section 6)
        const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        const int iters = n > t0 ? (int)((n - t0 + stride - 1) / stride) : 0;
        const double *pa = s12 + t0, *pb = s13 + t0;
        const double2* pf = fp + t0;
        double nx = 1.0, ny = 1.0;                         // the next point, loaded one iteration ahead
        double2 nf = make_double2(0.0, 0.0);
        if (iters > 0) { nx = *pa; ny = *pb; nf = *pf; }
        for (int it = 0; it < iters; ++it) {
            const double x = nx, y = ny, fr = nf.x, fi = nf.y;
            pa += stride; pb += stride; pf += stride;
            if (it + 1 < iters) { nx = *pa; ny = *pb; nf = *pf; }
            const Channel ca = make_channel<FL & MIPWA_FL_EQM>(m, x, y), cb = make_channel<FL & MIPWA_FL_EQM>(m, y, x);
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                const ResDev& r = m.res[sel.slot[f]];
                double amr, ami, agr, agi, bmr, bmi, bgr, bgi;
                shape_channel<LT>(r, ca, amr, ami, agr, agi);
                shape_channel<LT>(r, cb, bmr, bmi, bgr, bgi);
                const double dmr = amr + bmr, dmi = ami + bmi, dgr = agr + bgr, dgi = agi + bgi;
                acc[f][0] = fma(fr, dmr, fma(fi, dmi, acc[f][0]));      // f conj(dT'/dm0)
                acc[f][1] = fma(fi, dmr, fma(-fr, dmi, acc[f][1]));
                acc[f][2] = fma(fr, dgr, fma(fi, dgi, acc[f][2]));      // f conj(dT'/dG0)
                acc[f][3] = fma(fi, dgr, fma(-fr, dgi, acc[f][3]));
            }
        }
#pragma unroll
        for (int f = 0; f < NF; ++f)
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const double v = block_sum(acc[f][q], red32);
                if (threadIdx.x == 0) mine[(pass * NF + f) * 4 + q] = v;
            }
    }
}
