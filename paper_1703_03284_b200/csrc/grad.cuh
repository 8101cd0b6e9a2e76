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
#include <type_traits>
#include "cached.cuh"

#define MIPWA_GRAD_MAXR (MIPWA_DEV_MAX_RES)

// ---- one floating resonance in one channel, with its shape derivatives ------------------------------------------------
// With D_R, D_D, W' = m0 Gamma(x) D_R, dD = (m0^2 - x) D_R, E = dD^2 + W'^2 (dev_model.cuh) and u = (dD + i W') / E
// (so BW = D_R u and BW m0 Gamma = W' u):
//   T'        = Z D_R rsqrt(D_R D_D) u = FZ u                    (T without sqrt(n_R n_D), as everywhere in the kernels)
//   dT'/dG0   = T' (i W' / Gamma0) u
//   dT'/dm0   = T' [ a1 + u (-2 m0 D_R + i a2 W') ]             (a1, a2: ResDev::sh_a1, sh_a2)
// Input: FZ, DR, the running width W' and u of the channel.  Output: T', dT'/dm0, dT'/dG0.
__device__ __forceinline__ void shape_terms(const ResDev& r, double FZ, double DR, double W, double ur, double ui,
                                            double& tr, double& ti, double& mr, double& mi, double& gr, double& gi)
{
    tr = FZ * ur; ti = FZ * ui;
    const double k = r.sh_ig0 * W;                         // dT'/dG0 = T' (i k u)
    const double xr = -k * ui, xi = k * ur;
    gr = fma(tr, xr, -ti * xi); gi = fma(tr, xi, ti * xr);
    const double p = -r.sh_2m0 * DR, q = r.sh_a2 * W;      // dT'/dm0 = T' [a1 + u (p + i q)]
    const double br = r.sh_a1 + fma(ur, p, -ui * q), bi = fma(ur, q, ui * p);
    mr = fma(tr, br, -ti * bi); mi = fma(tr, bi, ti * br);
}

// LT = 0, 1, 2: spin known at compile time; LT < 0: read from r.
template <int LT>
__device__ __forceinline__ void shape_channel(const ResDev& r, const Channel& c, double& tr, double& ti, double& mr,
                                              double& mi, double& gr, double& gi)
{
    double DR, DD, W, Z;
    if (LT == 0) {
        DR = 1.0; DD = 1.0; W = r.Kw * c.w[0]; Z = 1.0;
    } else if (LT == 1) {
        DR = fma(r.cR, c.ql, 1.0); DD = fma(r.cD, c.lam2, 1.0); W = r.Kw * c.w[1]; Z = c.Z[1];
    } else if (LT == 2) {
        DR = fma(c.ql, fma(c.ql, r.qR2, r.qR1), 9.0); DD = fma(c.lam2, fma(c.lam2, r.qD2, r.qD1), 9.0);
        W = r.Kw * c.w[2]; Z = c.Z[2];
    } else {
        const double zR = r.cR * c.ql, zD = r.cD * c.lam2;
        DR = fma(zR, fma(zR, r.pa, r.pb), r.pc); DD = fma(zD, fma(zD, r.pa, r.pb), r.pc);
        W = r.Kw * pick(r.L, c.w); Z = pick(r.L, c.Z);
    }
    const double dD = (r.m0sq - c.x) * DR;
    const double rE = fast_rcp(fma(dD, dD, W * W));
    const double FZ = (LT == 0) ? 1.0 : Z * DR * fast_rsqrt(DR * DD);
    shape_terms(r, FZ, DR, W, dD * rE, W * rE, tr, ti, mr, mi, gr, gi);
}

// group_shared_terms (dev_model.cuh) with the shape derivatives of member 0: sh = symmetrised (dT'/dm0, dT'/dG0)
template <int LT, int NR>
__device__ __forceinline__ void group_shared_terms_shape(const ResDev* rd, const Channel& ca, const Channel& cb,
                                                         double* tr, double* ti, double (&sh)[4])
{
    double DRa, FZa, DRb, FZb;
    group_barrier<LT>(rd[0], ca, DRa, FZa);
    group_barrier<LT>(rd[0], cb, DRb, FZb);
    const double xDa = ca.x * DRa, xDb = cb.x * DRb;
    {
        const double Wa = rd[0].Kw * ca.w[LT], Wb = rd[0].Kw * cb.w[LT];
        const double da = fma(rd[0].m0sq, DRa, -xDa), db = fma(rd[0].m0sq, DRb, -xDb);
        const double ra = fast_rcp(fma(da, da, Wa * Wa)), rb = fast_rcp(fma(db, db, Wb * Wb));
        double tra, tia, mra, mia, gra, gia, trb, tib, mrb, mib, grb, gib;
        shape_terms(rd[0], FZa, DRa, Wa, da * ra, Wa * ra, tra, tia, mra, mia, gra, gia);
        shape_terms(rd[0], FZb, DRb, Wb, db * rb, Wb * rb, trb, tib, mrb, mib, grb, gib);
        tr[0] = tra + trb; ti[0] = tia + tib;
        sh[0] = mra + mrb; sh[1] = mia + mib; sh[2] = gra + grb; sh[3] = gia + gib;
    }
#pragma unroll
    for (int r = 1; r < NR; ++r) {
        const double Wa = rd[r].Kw * ca.w[LT], Wb = rd[r].Kw * cb.w[LT];
        const double da = fma(rd[r].m0sq, DRa, -xDa), db = fma(rd[r].m0sq, DRb, -xDb);
        const double ta = FZa * fast_rcp(fma(da, da, Wa * Wa)), tb = FZb * fast_rcp(fma(db, db, Wb * Wb));
        tr[r] = fma(ta, da, tb * db);
        ti[r] = fma(ta, Wa, tb * Wb);
    }
}

// T'(s12,s13) + T'(s13,s12) of one resonance with its symmetrised shape derivatives
template <int LT>
__device__ __forceinline__ void resonance_sym_shape(const ResDev& rd, const Channel& ca, const Channel& cb, double& tr,
                                                    double& ti, double (&sh)[4])
{
    double tra, tia, mra, mia, gra, gia, trb, tib, mrb, mib, grb, gib;
    shape_channel<LT>(rd, ca, tra, tia, mra, mia, gra, gia);
    shape_channel<LT>(rd, cb, trb, tib, mrb, mib, grb, gib);
    tr = tra + trb; ti = tia + tib;
    sh[0] = mra + mrb; sh[1] = mia + mib; sh[2] = gra + grb; sh[3] = gia + gib;
}

// amplitude with the pieces the gradient needs: offset t of both channels and every symmetrised resonance term WITHOUT
// its coefficient (device slot order; the host multiplies by sqrt(n_R n_D)).
// SHP = 1 / 2: the FIRST spin-1 / spin-2 device slot is a floating resonance (the host orders floating resonances first
// within their spin): its symmetrised shape derivatives come back in sh.
template <int R1, int R2, int FL, int SHP>
__device__ __forceinline__ void amplitude_parts(const RowsSmem& sm, const DevModel& m, const PointRec& p, double& are,
                                                double& aim, double& t1, double& t2,
                                                double (&tr)[R1 >= 0 ? (R1 + R2 > 0 ? R1 + R2 : 1) : MIPWA_GRAD_MAXR],
                                                double (&ti)[R1 >= 0 ? (R1 + R2 > 0 ? R1 + R2 : 1) : MIPWA_GRAD_MAXR],
                                                double (&sh)[4])
{
    double r1, i1, r2, i2;
    spline_eval_off(sm, p.s12, p.o1, r1, i1, t1);
    spline_eval_off(sm, p.s13, p.o2, r2, i2, t2);
    are = r1 + r2;
    aim = i1 + i2;
    if (R1 == 0 && R2 == 0) return;
    Channel ca, cb;
    make_channels<FL>(m, p.s12, p.s13, ca, cb);
    if (R1 >= 0) {
        constexpr int o2 = R1 > 0 ? R1 : 0;
        if ((FL & MIPWA_FL_SHR) && R1 >= 2) {
            if (SHP == 1) group_shared_terms_shape<1, (R1 >= 2 ? R1 : 2)>(&m.res[0], ca, cb, &tr[0], &ti[0], sh);
            else group_shared_terms<1, (R1 >= 2 ? R1 : 2)>(&m.res[0], ca, cb, &tr[0], &ti[0]);
        } else {
#pragma unroll
            for (int r = 0; r < R1; ++r) {
                if (SHP == 1 && r == 0) resonance_sym_shape<1>(m.res[r], ca, cb, tr[r], ti[r], sh);
                else resonance_sym<1>(m.res[r], ca, cb, tr[r], ti[r]);
            }
        }
        if ((FL & MIPWA_FL_SHR) && R2 >= 2) {
            if (SHP == 2) group_shared_terms_shape<2, (R2 >= 2 ? R2 : 2)>(&m.res[o2], ca, cb, &tr[o2], &ti[o2], sh);
            else group_shared_terms<2, (R2 >= 2 ? R2 : 2)>(&m.res[o2], ca, cb, &tr[o2], &ti[o2]);
        } else {
#pragma unroll
            for (int r = 0; r < R2; ++r) {
                if (SHP == 2 && r == 0) resonance_sym_shape<2>(m.res[R1 + r], ca, cb, tr[R1 + r], ti[R1 + r], sh);
                else resonance_sym<2>(m.res[R1 + r], ca, cb, tr[R1 + r], ti[R1 + r]);
            }
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

// per-warp running moments of the current cell: sum f t1^q (q = 0..3) and sum f t2^q (q = 1..3); the q = 0 moment
// sum f is the same number for both channels of a cell
struct CellAcc {
    double v[14];          // [0..7]: channel 1, q = 0..3, (re, im); [8..13]: channel 2, q = 1..3
    unsigned int o1, o2;   // row offsets (= segments) of the cell, 0xffffffff: empty
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int k = 0; k < 14; ++k) v[k] = 0.0;
    }
    __device__ __forceinline__ void add(double fr, double fi, double t1, double t2) {
        v[0] += fr; v[1] += fi;
        double p = t1;
#pragma unroll
        for (int q = 1; q < 4; ++q) { v[2 * q] = fma(fr, p, v[2 * q]); v[2 * q + 1] = fma(fi, p, v[2 * q + 1]); p *= t1; }
        p = t2;
#pragma unroll
        for (int q = 1; q < 4; ++q) { v[6 + 2 * q] = fma(fr, p, v[6 + 2 * q]); v[7 + 2 * q] = fma(fi, p, v[7 + 2 * q]); p *= t2; }
    }
};
#define MIPWA_NO_CELL 0xffffffffu

// bins[(q * NS + j) * 2 + {0,1}], NS = N - 1 segments: the bins of THIS WARP (shared memory, one set per warp), so the
// flush is a plain read-modify-write by lane 0 in program order: no atomics, and the block sums the warps' bins in warp
// order afterwards - the gradient is bit-reproducible call to call like the value.
__device__ __forceinline__ void flush_warp(CellAcc& a, double* bins, int NS)
{
    if (a.o1 != MIPWA_NO_CELL) {
#pragma unroll
        for (int k = 0; k < 14; ++k) {
            double x = a.v[k];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
            a.v[k] = x;
        }
        if ((threadIdx.x & 31) == 0) {
            const int j1 = (int)(a.o1 / MIPWA_ROW_BYTES), j2 = (int)(a.o2 / MIPWA_ROW_BYTES);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                bins[(q * NS + j1) * 2] += a.v[2 * q];
                bins[(q * NS + j1) * 2 + 1] += a.v[2 * q + 1];
            }
            bins[j2 * 2] += a.v[0];                        // after the j1 updates: j2 may be the same segment
            bins[j2 * 2 + 1] += a.v[1];
#pragma unroll
            for (int q = 1; q < 4; ++q) {
                bins[(q * NS + j2) * 2] += a.v[6 + 2 * q];
                bins[(q * NS + j2) * 2 + 1] += a.v[7 + 2 * q];
            }
        }
        __syncwarp();
    }
    a.clear();
    a.o1 = a.o2 = MIPWA_NO_CELL;
}

// A warp-iteration whose 32 points fall into several cells (it straddles a cell boundary of the sorted order): one
// round per distinct cell - the lanes of that cell contribute, the others add zeros - through the same
// shuffle-reduce + lane-0 flush.  `acc` must be empty on entry and is empty on return.
__device__ __forceinline__ void add_mixed(CellAcc& acc, bool valid, unsigned int o1, unsigned int o2, double fr, double fi,
                                          double t1, double t2, double* bins, int NS)
{
    unsigned int remaining = __ballot_sync(0xffffffffu, valid);
    while (remaining) {                                                    // warp-uniform
        const int leader = __ffs(remaining) - 1;
        const unsigned int l1 = __shfl_sync(0xffffffffu, o1, leader), l2 = __shfl_sync(0xffffffffu, o2, leader);
        const bool mine = valid && o1 == l1 && o2 == l2;
        acc.o1 = l1; acc.o2 = l2;
        acc.add(mine ? fr : 0.0, mine ? fi : 0.0, t1, t2);
        flush_warp(acc, bins, NS);
        remaining &= ~__ballot_sync(0xffffffffu, mine);
    }
}

// moments of one warp-iteration into the warp's running cell (flush on a cell change)
__device__ __forceinline__ void cell_accumulate(CellAcc& acc, bool valid, unsigned int o1, unsigned int o2, double fr,
                                                double fi, double t1, double t2, double* bins, int NS)
{
    const bool same = !valid || (o1 == acc.o1 && o2 == acc.o2);
    if (__all_sync(0xffffffffu, same)) {
        acc.add(fr, fi, t1, t2);
    } else {
        flush_warp(acc, bins, NS);
        const unsigned int l1 = __shfl_sync(0xffffffffu, o1, 0), l2 = __shfl_sync(0xffffffffu, o2, 0);   // lane 0 is valid
        const bool uni = !valid || (o1 == l1 && o2 == l2);
        if (__all_sync(0xffffffffu, uni)) {
            acc.o1 = l1; acc.o2 = l2;
            acc.add(fr, fi, t1, t2);
        } else {
            add_mixed(acc, valid, o1, o2, fr, fi, t1, t2, bins, NS);
        }
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

template <int R1, int R2> struct GradDims {
    static constexpr int RR = R1 >= 0 ? (R1 + R2 > 0 ? R1 + R2 : 1) : MIPWA_GRAD_MAXR;
};

// ---- A8: the gradient sums of one point set --------------------------------------------------------------------------
// ONE launch covers both sets: blocks [0, ev_blocks) walk the cell-sorted event records (f = -2/conj(A), scalar =
// sum ln|A|^2), blocks [ev_blocks, gridDim.x) the normalisation records (f = w A, scalar = sum w|A|^2); 512 threads, one
// block per SM, the second set's blocks start as the first set's finish.  A block runs exactly one of the two bodies, so
// no register is spent on choosing between them.  Warp wg of a set owns the contiguous chunk [wg CH, (wg+1) CH) of it.
// MIX (events only): background density w per event and D = |A|^2 + kappa w: f = -2 A / D, scalar = sum ln D,
// Q = sum w / D (mipwa_nll_mix_grad).
// SHP = 1 / 2: also sum f conj(dT'/dm0), f conj(dT'/dG0) of the floating resonance in the first spin-1 / spin-2 slot.
// Block partial vector (doubles): [0] scalar, [1] Q, [2 + 2d + {0,1}] F of device slot d, then bins[4][N-1][2], then
// (SHP) 4 shape sums;  NVB = 2 + 2R + 8 (N-1) + 4.  Dynamic shared memory: (blockDim / 32) x 8 (N-1) doubles.
#define MIPWA_GRAD_BLOCK 512
template <int R1, int R2, int FL, bool EV, bool MIX, int SHP>
__device__ __forceinline__ void grad_body(const RowsSmem& sm, const DevModel& m, const PointRec* __restrict__ rec,
                                          long long n, int set_block, int set_blocks, double kappa,
                                          double2* __restrict__ fout, double* bins, double2* stage,
                                          double* __restrict__ mine,
                                          double (*wpart)[2 + 2 * GradDims<R1, R2>::RR + 4])
{
    constexpr int RR = GradDims<R1, R2>::RR;
    const int NS = m.N - 1, nb = 8 * NS, lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpb = blockDim.x >> 5;
    const int nres = R1 >= 0 ? R1 + R2 : m.R;
    const long long W = (long long)set_blocks * wpb, wg = (long long)set_block * wpb + warp;
    const long long CH = (((n + W - 1) / W) + 31) & ~31LL;
    const long long lo = wg * CH, hi = lo + CH < n ? lo + CH : n;
    // 32-bit offsets into this warp's chunk (CH <= 2^31 - 32: mipwa_nll_grad admits at most 2^31 - 1 points per set)
    const int cnt = lo < hi ? (int)(hi - lo) : 0;
    double* const wbins = bins + warp * nb;
    CellAcc acc;
    acc.clear();
    acc.o1 = acc.o2 = MIPWA_NO_CELL;
    LogProd lp;
    double integ = 0.0, qsum = 0.0, Fr[RR], Fi[RR], Sh[4] = { 0.0, 0.0, 0.0, 0.0 };
#pragma unroll
    for (int r = 0; r < RR; ++r) Fr[r] = Fi[r] = 0.0;
    if (cnt > 0) {
        // The gradient's running sums leave no registers for a second record in flight, so the next iteration's 32 records
        // (1 KB, contiguous) travel through shared memory: cp.async, two 16-byte units per lane, issued one iteration
        // ahead (the scheduler's other warps run ~3 iterations meanwhile: DRAM latency is covered) and read back with two
        // conflict-free LDS.128.  Unit u = 2 * record + half of the warp's 1 KB lands in slot half * 32 + record.  The
        // record arrays are padded: the copy issued by the last iteration needs no bounds test.
        double2* const st = stage + warp * 128;            // 2 stages x 64 units
        const unsigned st0 = (unsigned)__cvta_generic_to_shared(st);
        const unsigned dst = st0 + 16u * ((lane & 1) * 32 + (lane >> 1));
        const char* g = reinterpret_cast<const char*>(rec + lo) + 16 * lane;
        auto issue = [&](unsigned sbytes) {
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + sbytes), "l"(g) : "memory");
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + sbytes + 256u), "l"(g + 512) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
            g += 1024;
        };
        issue(0u);
        unsigned cur = 0u;                                 // stage being read, in 16-byte units (0 or 64)
        int base = 0, adds = 0;                            // offset of the current iteration in the chunk; adds since the last flush
        // the record of the iteration after the one last returned (the copy of the one after that is issued behind it)
        auto next_record = [&]() {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncwarp();
            const double2 ra = st[cur + lane], rb = st[cur + 32 + lane];
            cur ^= 64u;
            issue(cur * 16u);
            PointRec r;
            r.s12 = ra.x; r.s13 = ra.y; r.w = rb.x;
            const unsigned long long ob = (unsigned long long)__double_as_longlong(rb.y);
            r.o1 = (unsigned)ob; r.o2 = (unsigned)(ob >> 32);
            return r;
        };
        // one point: amplitude, f, the scalar sums and the resonance sums - everything but the spline moments
        auto point = [&](auto masked, const PointRec& r, bool valid, double& fr, double& fi, double& t1, double& t2) {
            constexpr bool MASKED = decltype(masked)::value;   // lanes past the end evaluate a real point and add zeros
            double are, aim, tr[RR], ti[RR], sh[4];
            amplitude_parts<R1, R2, FL, SHP>(sm, m, r, are, aim, t1, t2, tr, ti, sh);
            const double a2 = fma(are, are, aim * aim);
            if (EV) {
                const double D = MIX ? fma(kappa, r.w, a2) : a2;
                const double rD = fast_rcp(D);
                const double k = !MASKED || valid ? -2.0 * rD : 0.0;
                fr = k * are; fi = k * aim;
                lp.add(!MASKED || valid ? D : 1.0);
                if (MIX) qsum += !MASKED || valid ? r.w * rD : 0.0;
            } else {
                const double wv = !MASKED || valid ? r.w : 0.0;
                fr = wv * are; fi = wv * aim;
                integ = fma(wv, a2, integ);
            }
            if (fout && (!MASKED || valid))                // for k_grad_shape (several floating resonances)
                fout[lo + base + lane] = make_double2(fr, fi);
            if (R1 >= 0) {
#pragma unroll
                for (int q = 0; q < (R1 >= 0 ? R1 + R2 : 0); ++q) {
                    Fr[q] = fma(fr, tr[q], fma(fi, ti[q], Fr[q]));         // f conj(T)
                    Fi[q] = fma(fi, tr[q], fma(-fr, ti[q], Fi[q]));
                }
            } else {
                for (int q = 0; q < nres; ++q) {
                    Fr[q] = fma(fr, tr[q], fma(fi, ti[q], Fr[q]));
                    Fi[q] = fma(fi, tr[q], fma(-fr, ti[q], Fi[q]));
                }
            }
            if (SHP) {
                Sh[0] = fma(fr, sh[0], fma(fi, sh[1], Sh[0]));             // f conj(dT'/dm0)
                Sh[1] = fma(fi, sh[0], fma(-fr, sh[1], Sh[1]));
                Sh[2] = fma(fr, sh[2], fma(fi, sh[3], Sh[2]));             // f conj(dT'/dG0)
                Sh[3] = fma(fi, sh[2], fma(-fr, sh[3], Sh[3]));
            }
        };
        // Two loops.  The HOT one takes the iterations whose 32 points all lie in the warp's current cell (cell-sorted
        // points: all but a few per warp): straight-line code, moments into the register accumulators.  Whatever else -
        // the first iteration, a cell change, an iteration that straddles cells, the partly filled last one - leaves it
        // and is handled once by the general code below (flush into the warp's bins, shuffles, masks), which then hands
        // back.  With the flush inside the one loop ptxas re-read 19 model constants per point and spilled.
        const int full = cnt & ~31;                        // iterations in which every lane has a point
        PointRec r = next_record();
        while (base < cnt) {
            const int room = LOGPROD_FLUSH - adds;         // iterations until the log-product has to be flushed
            const int stop = (full - base) >> 5 < room ? full : base + 32 * room;
            while (base < stop && __all_sync(0xffffffffu, r.o1 == acc.o1 && r.o2 == acc.o2)) {
                double fr, fi, t1, t2;
                point(std::false_type(), r, true, fr, fi, t1, t2);
                acc.add(fr, fi, t1, t2);
                base += 32; ++adds;
                r = next_record();
            }
            if (base < stop || (base == full && full < cnt)) {
                const bool valid = base + lane < cnt;
                double fr, fi, t1, t2;
                point(std::true_type(), r, valid, fr, fi, t1, t2);
                cell_accumulate(acc, valid, r.o1, r.o2, fr, fi, t1, t2, wbins, NS);
                base += 32; ++adds;
                r = next_record();
            }
            if (EV && (adds == LOGPROD_FLUSH || base >= cnt)) { lp.flush(adds); adds = 0; }
        }
    }
    flush_warp(acc, wbins, NS);

    // warp sums -> shared memory, then the block adds them in warp order (fixed order)
    constexpr int NW = 2 + 2 * RR + 4;
    double vals[NW];
    vals[0] = EV ? lp.sum : integ; vals[1] = qsum;
#pragma unroll
    for (int q = 0; q < RR; ++q) { vals[2 + 2 * q] = Fr[q]; vals[3 + 2 * q] = Fi[q]; }
#pragma unroll
    for (int q = 0; q < 4; ++q) vals[2 + 2 * RR + q] = Sh[q];
#pragma unroll
    for (int k = 0; k < NW; ++k) {
        double x = vals[k];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
        if (lane == 0) wpart[warp][k] = x;
    }
    __syncthreads();                                       // every warp has left its sums and flushed its bins
    const int R = m.R;
    for (int t = threadIdx.x; t < 2 + 2 * R + 4; t += blockDim.x) {
        const int k = t < 2 + 2 * R ? t : 2 + 2 * RR + (t - 2 - 2 * R);
        double v = 0.0;
        for (int w = 0; w < wpb; ++w) v += wpart[w][k];
        mine[t < 2 + 2 * R ? t : 2 + 2 * R + nb + (t - 2 - 2 * R)] = v;
    }
    for (int k = threadIdx.x; k < nb; k += blockDim.x) {
        double v = 0.0;
        for (int w = 0; w < wpb; ++w) v += bins[w * nb + k];
        mine[2 + 2 * R + k] = v;
    }
}

template <int R1, int R2, int FL, bool MIX, int SHP>
__global__ void __launch_bounds__(MIPWA_GRAD_BLOCK, 1)
k_grad_recompute(const __grid_constant__ DevModel m, const PointRec* __restrict__ ev, double kappa, long long n_ev,
                 const PointRec* __restrict__ nm, long long n_norm, int ev_blocks, double* __restrict__ partials,
                 double2* __restrict__ f_ev, double2* __restrict__ f_nm)
{
    constexpr int RR = GradDims<R1, R2>::RR;
    extern __shared__ __align__(16) double grad_bins[];                  // [warp][4][N-1][2]
    __shared__ RowsSmem sm;
    __shared__ double wpart[MIPWA_GRAD_BLOCK / 32][2 + 2 * RR + 4];
    const int NS = m.N - 1, nb = 8 * NS, NVB = 2 + 2 * m.R + nb + 4;
    asm volatile("griddepcontrol.launch_dependents;");     // k_grad_finalize may be scheduled behind this grid's blocks
    for (int k = threadIdx.x; k < (int)(blockDim.x >> 5) * nb; k += blockDim.x) grad_bins[k] = 0.0;
    double2* const stage = reinterpret_cast<double2*>(grad_bins + (blockDim.x >> 5) * nb);   // [warp][2][64] record halves
    load_rows_smem(sm, m);                                 // ends with __syncthreads()
    double* mine = partials + (size_t)blockIdx.x * NVB;
    if ((int)blockIdx.x < ev_blocks)
        grad_body<R1, R2, FL, true, MIX, SHP>(sm, m, ev, n_ev, (int)blockIdx.x, ev_blocks, kappa, f_ev, grad_bins, stage, mine, wpart);
    else
        grad_body<R1, R2, FL, false, false, SHP>(sm, m, nm, n_norm, (int)blockIdx.x - ev_blocks,
                                                 (int)gridDim.x - ev_blocks, 0.0, f_nm, grad_bins, stage, mine, wpart);
}

// Fixed-order sums of the per-block partial vectors, one warp per value: lane l adds blocks l, l+32, .. then a shuffle
// tree.  result[k] = sum over blocks [0, split) and, with sets = 2, result[NV + k] = sum over blocks [split, nblocks).  A separate tiny launch: done inside the last block of the gradient kernel it would serialise ~NV x grid L2
// reads on one SM while the rest of the GPU idles.
static __global__ void __launch_bounds__(256)
k_grad_finalize(const double* __restrict__ partials, int split, int nblocks, int NV, int sets,
                double* __restrict__ result, unsigned int* __restrict__ ticket, double* __restrict__ tag_word, long long tag)
{
    // launched with programmatic stream serialisation right behind the kernel that writes `partials`: its blocks may be
    // resident before that kernel has finished; nothing is read before this point
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int kk = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (kk < sets * NV) {
        const int set = kk / NV, k = kk - set * NV;
        const int b0 = set == 0 ? 0 : split, b1 = set == 0 ? split : nblocks;
        double s = 0.0;
        for (int b = b0 + lane; b < b1; b += 32) s += partials[(size_t)b * NV + k];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
        if (lane == 0) { result[kk] = s; __threadfence_system(); }
    }
    if (ticket) {
        // `result` is mapped host memory: the last block to finish writes the call's tag behind everybody's values, and the
        // host polls that word instead of sleeping in cudaStreamSynchronize (as the value kernels do, dev_model.cuh)
        __syncthreads();
        if (threadIdx.x == 0 && atomicAdd(ticket, 1u) == gridDim.x - 1) {
            *ticket = 0;
            __threadfence_system();
            *reinterpret_cast<volatile long long*>(tag_word) = tag;
        }
    }
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
// Streams the compact cache (16 + 16 R bytes per event, cell-sorted event order) and the stored segment pairs,
// evaluates the spline part from the shared-memory rows, and accumulates  f = -2/conj(A):  moments f t^q per segment
// (per-warp bins, as k_grad_recompute) and F_r = sum f conj(B_{N+r}) per resonance.
// Partial vector per block: [S, F(2R), bins(8 (N-1))].  Dynamic shared memory: (blockDim / 32) x 8 (N-1) doubles.
template <int RT>
__global__ void __launch_bounds__(MIPWA_TILE, 2)
k_grad_compact(const __grid_constant__ DevModel m, const __grid_constant__ CoefDev cc,
               const double2* __restrict__ cache, const unsigned short* __restrict__ seg, long long n_ev,
               double* __restrict__ partials)
{
    constexpr int RC = RT > 0 ? RT : (RT == 0 ? 1 : MIPWA_GRAD_MAXR);
    extern __shared__ __align__(16) double grad_bins[];                  // [warp][4][N-1][2]
    __shared__ RowsSmem sm;
    __shared__ double red32[32];
    const int R = RT >= 0 ? RT : cc.K - cc.N, C = 1 + R, N = cc.N, NS = N - 1, nb = 8 * NS, NV = 1 + 2 * R + nb;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpb = blockDim.x >> 5;
    asm volatile("griddepcontrol.launch_dependents;");     // k_grad_finalize may be scheduled behind this grid's blocks
    for (int k = threadIdx.x; k < wpb * nb; k += blockDim.x) grad_bins[k] = 0.0;
    load_rows_smem(sm, m);
    double* const wbins = grad_bins + warp * nb;

    const long long W = (long long)gridDim.x * wpb, wg = (long long)blockIdx.x * wpb + warp;
    const long long CH = (((n_ev + W - 1) / W) + 31) & ~31LL;
    const long long lo = wg * CH, hi = lo + CH < n_ev ? lo + CH : n_ev;
    CellAcc acc;
    acc.clear();
    acc.o1 = acc.o2 = MIPWA_NO_CELL;
    LogProd lp;
    int adds = 0;
    double Fr[RC], Fi[RC];
#pragma unroll
    for (int r = 0; r < RC; ++r) Fr[r] = Fi[r] = 0.0;
    for (long long base = lo; base < hi; base += 32) {                     // warp-uniform trip count; base % 32 == 0
        const long long i = base + lane;
        const bool valid = i < hi;
        const long long ii = valid ? i : lo;
        const double2* p = cache + (size_t)(ii / MIPWA_TILE) * C * MIPWA_TILE + (ii % MIPWA_TILE);
        const double2 s = ld_stream(p);
        const unsigned int sg = seg[ii], o1 = seg_off1(sg), o2 = seg_off2(sg);
        double2 b[RC];
        {   // the next iteration's lines on their way into L2 (the running sums leave no registers for a second set of
            // columns in flight: with a register prefetch ptxas spilled and the kernel lost 9 %)
            const long long nx = i + 32 < hi ? i + 32 : lo;
            const double2* q = cache + (size_t)(nx / MIPWA_TILE) * C * MIPWA_TILE + (nx % MIPWA_TILE);
#pragma unroll
            for (int r = 0; r < (RT >= 0 ? 1 + RT : 1); ++r)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(q + (size_t)r * MIPWA_TILE));
        }
        if (RT >= 0) {
#pragma unroll
            for (int r = 0; r < RT; ++r) b[r] = ld_stream(p + (size_t)(1 + r) * MIPWA_TILE);
        } else {
            for (int r = 0; r < R; ++r) b[r] = ld_stream(p + (size_t)(1 + r) * MIPWA_TILE);
        }
        double t1, t2, r1, i1, r2, i2;
        spline_eval_off(sm, s.x, o1, r1, i1, t1);
        spline_eval_off(sm, s.y, o2, r2, i2, t2);
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
        if (++adds == LOGPROD_FLUSH) { lp.flush(adds); adds = 0; }
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
        cell_accumulate(acc, valid, o1, o2, fr, fi, t1, t2, wbins, NS);
    }
    flush_warp(acc, wbins, NS);
    lp.flush(adds);

    double* mine = partials + (size_t)blockIdx.x * NV;
    double v = block_sum(lp.sum, red32);
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
    __syncthreads();                                       // every warp has flushed its bins
    for (int k2 = threadIdx.x; k2 < nb; k2 += blockDim.x) {
        double x = 0.0;
        for (int w = 0; w < wpb; ++w) x += grad_bins[w * nb + k2];         // warp order: fixed
        mine[1 + 2 * R + k2] = x;
    }
}


// ---- derivatives with respect to floating masses and widths, general case (mipwa_nll_grad_full) ---------
// Models with ONE floating resonance of spin 1 or 2 get these sums from k_grad_recompute itself (SHP).  Otherwise
// k_grad_recompute stores its per-point factor f (-2/conj(A) for events, w A for normalisation points); this kernel
// streams (s12, s13, f), evaluates the two channels of every floating resonance (shape_channel) and adds
// f conj(dT'_sym) into 4 doubles per floating resonance and pass.  The host multiplies by conj(c_r sqrt(n_R n_D)) and
// takes the real part.  One instantiation per number of floating resonances handled per launch (1..4).
#define MIPWA_SHAPE_MAXF 4
struct ShapeSel { int32_t slot[MIPWA_SHAPE_MAXF]; };       // device slots of the floating resonances of this launch

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
            Channel ca, cb;
            make_channels<FL & MIPWA_FL_EQM>(m, x, y, ca, cb);
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                const ResDev& r = m.res[sel.slot[f]];
                double atr, ati, btr, bti, amr, ami, agr, agi, bmr, bmi, bgr, bgi;
                shape_channel<LT>(r, ca, atr, ati, amr, ami, agr, agi);
                shape_channel<LT>(r, cb, btr, bti, bmr, bmi, bgr, bgi);
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
