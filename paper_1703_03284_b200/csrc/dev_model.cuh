// dev_model.cuh -- the per-call model block handed to every kernel, and the per-point amplitude device function.
//
// Operation definitions: include/mipwa.h (Eq. 1; spline PAPER.md:29; Breit-Wigner x angular factor
// PAPER.md:27; symmetrisation PAPER.md:47).  This file restates them in the form the FP64 pipe likes:
//
//   per channel x (= s12 or s13), other = y:
//     lam1 = lambda(x, m1^2, m2^2) = (x - (m1+m2)^2)(x - (m1-m2)^2)          [factored: no cancellation at threshold]
//     lam2 = lambda(M^2, x, m3^2)  = ((M-m3)^2 - x)((M+m3)^2 - x)
//     ix = 1/x,  ql = lam1 ix = 4 q^2,  pl = lam2 ix,  g = sqrt(lam1) ix / 2 = sqrt(q^2 / x)
//     Z1 = x + 2y - Sigma + kappa ix,  Z2 = Z1^2 - ql pl / 3
//   per resonance (spin L, constants prepared on the host, step A3):
//     D_R = den_L(cR ql), D_D = den_L(cD lam2), den_1(z) = 1 + z, den_2(z) = 9 + 3z + z^2
//     W'  = Kw (2g) ql^L                       [= m0 Gamma(x) D_R: the running width without its barrier denominator]
//     dD  = (m0^2 - x) D_R,  E = dD^2 + W'^2
//     F_D F_R BW = sqrt(n_R n_D) D_R (dD + i W') / (sqrt(D_R D_D) E) = sqrt(n_R n_D) D_R (dD + i W') rsqrt(D_R D_D E^2)
//   so that ONE reciprocal square root per resonance and channel replaces two square roots and three divisions.
//   sqrt(n_R n_D) is folded into the coefficient on the host.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define MIPWA_DEV_MAX_KNOTS 128
#define MIPWA_DEV_MAX_RES 16
#define MIPWA_DEV_LUT 512

struct ResDev {
    double m0sq;      // m0^2
    double cR;        // r_res^2 / 4            (z_R = cR * ql);  0 for L = 0
    double cD;        // r_parent^2 / (4 M^2)   (z_D = cD * lam2); 0 for L = 0
    double Kw;        // m0^2 Gamma0 n_R / (2 (4 q0^2)^L sqrt(q0^2))   (the 1/2 of g = sqrt(lam1)/(2x) lives here)
    double cre, cim;  // c_r * sqrt(n_R n_D)
    double pa, pb, pc;// barrier denominator den_L(z) = pc + z (pb + pa z)
    double qR1, qR2;  // L = 2: D_R = 9 + ql (qR1 + qR2 ql), qR1 = 3 cR, qR2 = cR^2 (one instruction less than via z)
    double qD1, qD2;  // L = 2: D_D = 9 + lam2 (qD1 + qD2 lam2)
    // shape derivatives (mipwa_nll_grad_full; only the pole quantities depend on m0, so these are per-call constants):
    double sh_a1;     // d ln sqrt(n_R n_D) / d m0
    double sh_a2;     // d ln(m0 Gamma(x)) / d m0 = 2/m0 - (L + 1/2) (dq0^2/dm0)/q0^2 + n_R'/n_R r^2 dq0^2/dm0
    double sh_2m0;    // 2 m0
    double sh_ig0;    // 1 / Gamma0
    int32_t L;
    int32_t fl;       // index among the floating resonances (caller's list order), -1: shape fixed
};

// One spline segment as the per-call kernels read it: MIPWA_ROW consecutive double2 in shared memory,
//   row[0] = (x_j, 0),  row[1 + q] = coefficient of t^q, t = s - x_j:  S(s) = c0 + t (c1 + t (c2 + t c3)).
// A point addresses its two rows by BYTE OFFSET (segment x MIPWA_ROW_BYTES): the offsets are a property of the point
// set (knots are fixed at mipwa_create) and sit in the 32-byte point records, so the hot loops spend no instruction on
// index arithmetic.
#define MIPWA_ROW 5
#define MIPWA_ROW_BYTES (MIPWA_ROW * 16)

// Everything a per-call kernel needs for one likelihood call; passed by value as a __grid_constant__ kernel parameter.
struct DevModel {
    int32_t N;                 // knots
    int32_t R;                 // resonances
    int32_t pad0, pad1;
    double t_lo, t_d;          // (m1+m2)^2, (m1-m2)^2
    double s_hi, s_top;        // (M-m3)^2, (M+m3)^2
    double sigma;              // M^2 + m1^2 + m2^2 + m3^2
    double kappa;              // (M^2 - m3^2)(m2^2 - m1^2)
    double k_third;            // -1/3: a constant-bank operand instead of a 64-bit immediate rebuilt for every point
    double lam2_b, lam2_c;     // lambda(M^2, x, m3^2) = x (x + lam2_b) + lam2_c: -(s_hi + s_top), s_hi s_top
    double pad2;
    ResDev res[MIPWA_DEV_MAX_RES];
    double2 rows[MIPWA_DEV_MAX_KNOTS * MIPWA_ROW];
};

// The knot search table: depends on the knots only, so it is uploaded once at mipwa_create and read through a pointer
// by the few kernels that meet points whose segment is not stored yet (boundary check, cache / Gram setup, generator).
struct DevSearch {
    int32_t N, nlut;           // knots; buckets in lut
    int32_t lut_exact, pad;    // 1: every bucket holds at most one knot (xk), so the segment needs no search
    double lut_off, lut_inv;   // bucket = floor(s * lut_inv + lut_off), lut_off = -x_0 * lut_inv
    double knots[MIPWA_DEV_MAX_KNOTS];
    uint8_t lut[MIPWA_DEV_LUT];           // segment that contains the left edge of each bucket
    double xk[MIPWA_DEV_LUT];             // the interior knot inside bucket b (+inf if none); valid iff lut_exact
};

// Shared-memory copy of the segment rows (divergent lookups: constant memory would serialise them).
struct RowsSmem {
    double2 rows[MIPWA_DEV_MAX_KNOTS * MIPWA_ROW];
};

// The model arrives as a __grid_constant__ kernel parameter.  Read as a parameter (LDC from the constant bank) the copy is
// slow either way: a thread-indexed LDC is replayed once per distinct address (~20 us per block), and a warp-uniform one
// walks the table in dependent constant-cache misses (1.0 us at N = 40 in a 512-thread block, 3 us in a 256-thread block,
// 10 us at N = 128: a quarter of a likelihood call at the paper's sample size).  So the table is read through the
// GENERIC address of the parameter block with plain 16-byte loads, one entry per thread, all in flight together
// (0.5 us whatever N is).  `m` must be the kernel's own __grid_constant__ parameter.
__device__ __forceinline__ void load_rows_smem(RowsSmem& sm, const DevModel& m)
{
    const double2* g = m.rows;
    const int n = m.N * MIPWA_ROW;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        double2 v;
        asm volatile("ld.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(g + i));
        sm.rows[i] = v;
    }
    __syncthreads();
}

// ---- fp64 reciprocal / reciprocal square root: MUFU seed + ONE third-order correction step ----------------------
// The seeds (MUFU.RCP64H / MUFU.RSQ64H) look only at the upper 32 bits of the argument: relative error <= ~2^-20.
// With e = 1 - x y (resp. 1 - x y^2, |e| <= ~2^-19) the series 1/(1-e) = 1 + e + e^2 + O(e^3) and
// (1-e)^(-1/2) = 1 + e/2 + 3e^2/8 + O(e^3) leave a truncation error below 2^-57, under the rounding of the last fma:
// results are good to ~1 ulp.  Arguments here are finite, normal and positive (x >= (m1+m2)^2 > 0; denominators
// are sums of squares plus positive constants), so the special-case paths of the library routines are not needed.
__device__ __forceinline__ double fast_rcp(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    return fma(y, fma(e, e, e), y);
}

__device__ __forceinline__ double fast_rsqrt(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x * y, y, 1.0);
    return fma(y * e, fma(0.375, e, 0.5), y);
}

// The value kernels deliver their totals through mapped pinned host memory; the host may poll instead of blocking in
// cudaStreamSynchronize (a wake-up costs more than a small likelihood call).  Slot 2 of `result` gets the call's tag
// AFTER the totals are visible system-wide.
#define MIPWA_RESULT_TAG 2
__device__ __forceinline__ void publish_result(double* result, long long tag)
{
    __threadfence_system();
    *reinterpret_cast<volatile long long*>(result + MIPWA_RESULT_TAG) = tag;
}

// Shared-memory copy of the search table (setup kernels only).
struct SearchSmem {
    int32_t N, nlut, lut_exact, pad;
    double lut_off, lut_inv;
    double knots[MIPWA_DEV_MAX_KNOTS];
    uint8_t lut[MIPWA_DEV_LUT];
    double xk[MIPWA_DEV_LUT];
};

__device__ __forceinline__ void load_search_smem(SearchSmem& ss, const DevSearch* __restrict__ g)
{
    if (threadIdx.x == 0) {
        ss.N = g->N; ss.nlut = g->nlut; ss.lut_exact = g->lut_exact; ss.pad = 0;
        ss.lut_off = g->lut_off; ss.lut_inv = g->lut_inv;
    }
    for (int i = threadIdx.x; i < g->N; i += blockDim.x) ss.knots[i] = g->knots[i];
    for (int i = threadIdx.x; i < g->nlut; i += blockDim.x) { ss.lut[i] = g->lut[i]; ss.xk[i] = g->xk[i]; }
    __syncthreads();
}

// segment index j with x_j <= s < x_{j+1}, clamped to [0, N-2] (beyond the end knots the end cubic is used).
// Buckets are narrower than the smallest knot spacing (lut_exact), so one compare against the single knot a bucket
// can hold replaces a search: two dependent shared-memory reads (bucket entry, then the knot) and no branch.
// A point within rounding of a bucket edge or a knot may land in the neighbouring segment; the spline is C^2, so
// the neighbouring cubic differs there by O(distance^3) - far below one ulp.  Knot tables too dense for the
// MIPWA_DEV_LUT buckets fall back to the search.
__device__ __forceinline__ int spline_segment(const SearchSmem& ss, double s)
{
    int b = __double2int_rd(fma(s, ss.lut_inv, ss.lut_off));     // lut_off = -lut_x0 * lut_inv
    b = max(0, min(b, ss.nlut - 1));
    int j = ss.lut[b];
    if (ss.lut_exact) return j + (s >= ss.xk[b] ? 1 : 0);
    double xj = ss.knots[j], xn = ss.knots[j + 1];
    while (s >= xn && j < ss.N - 2) { ++j; xj = xn; xn = ss.knots[j + 1]; }
    if (s < xj && j > 0) --j;                               // guards the rounding of the bucket index
    return j;
}

// spline value on the segment whose row starts `off` bytes into the shared-memory rows
__device__ __forceinline__ void spline_eval_off(const RowsSmem& sm, double s, unsigned int off, double& re, double& im,
                                                double& t)
{
    const double2* row = reinterpret_cast<const double2*>(reinterpret_cast<const char*>(sm.rows) + off);
    t = s - row[0].x;
    const double2 c0 = row[1], c1 = row[2], c2 = row[3], c3 = row[4];
    re = fma(t, fma(t, fma(t, c3.x, c2.x), c1.x), c0.x);
    im = fma(t, fma(t, fma(t, c3.y, c2.y), c1.y), c0.y);
}

// the stored segment pair of a point (one uint16 per point, j12 | j13 << 8, written by k_validate) as row offsets
__device__ __forceinline__ unsigned int seg_off1(unsigned int seg) { return (seg & 0xffu) * MIPWA_ROW_BYTES; }
__device__ __forceinline__ unsigned int seg_off2(unsigned int seg) { return (seg >> 8) * MIPWA_ROW_BYTES; }

// One point of a point set as the recompute kernels stream it: 32 bytes, one 256-bit load.
//   w   normalisation points: weight w_j (1 if the caller gave none); events: background density b_i of the mixture
//       likelihood (0 if none)
//   o1, o2   byte offsets of the spline rows of s12 and s13 in RowsSmem
struct __align__(32) PointRec {
    double s12, s13, w;
    unsigned int o1, o2;
};

__device__ __forceinline__ PointRec ld_rec(const PointRec* p)
{
    PointRec r;
    double d;
    asm("ld.global.nc.L1::no_allocate.v4.f64 {%0, %1, %2, %3}, [%4];"
        : "=d"(r.s12), "=d"(r.s13), "=d"(r.w), "=d"(d) : "l"(p));
    r.o1 = (unsigned int)__double2loint(d);
    r.o2 = (unsigned int)__double2hiint(d);
    return r;
}

// per-channel kinematic quantities shared by all resonances
struct Channel {
    double x, lam2, ql;
    double w[3];      // w[L] = g ql^L: the running-width factor of a spin-L resonance
    double Z[3];      // Zemach factors Z_0 = 1, Z_1, Z_2
};

// Model flags a kernel can be specialised on (decided on the host once per model, mipwa_create):
//   MIPWA_FL_EQM  m1 == m2 (pi+pi-pi+, K+K-K+): lam1 = x (x - 4 m^2), so ql = x - 4 m^2 needs no reciprocal, kappa = 0,
//                 and 2g = sqrt(ql / x) = ql rsqrt(ql x): the channel needs no 1/x at all
//                 (Z2's ql pl = ql lam2 / x = (2g)^2 lam2)
//   MIPWA_FL_SHR  every resonance of one spin has the same r_res and r_parent (the usual choice, e.g. 1.5 and
//                 5 GeV^-1 for all): the barrier denominators D_R, D_D and rsqrt(D_R D_D) are per spin and channel
#define MIPWA_FL_EQM 1
#define MIPWA_TINY 0x1p-996
#define MIPWA_FL_SHR 2

// x: the channel's mass squared; z1: Z_1 of the equal-mass case, x + 2 y - Sigma (y = the other channel), which the
// caller forms for both channels from one shared sum.
// lam2 in expanded form: two instructions instead of three; its absolute error (~1e-15) only matters where lam2 itself
// vanishes, at the edge x = (M - m3)^2, and there it enters as 1 + c_D lam2 and as a term of Z_2.
template <int FL = 0>
__device__ __forceinline__ Channel make_channel(const DevModel& m, double x, double z1)
{
    Channel c;
    c.x = x;
    c.lam2 = fma(x, x + m.lam2_b, m.lam2_c);
    c.Z[0] = 1.0;
    if (FL & MIPWA_FL_EQM) {
        // |ql| x + 2^-996 under the root: a point within rounding of the threshold (the boundary check admits a
        // relative 1e-12) gives a width of rounding size, not NaN or infinity.  (2^-996 ~ 1.5e-300 has a zero low
        // word, so it is an immediate operand; 1e-300 took two moves per point.)
        c.ql = x - m.t_lo;
        const double lc = fma(fabs(c.ql), x, MIPWA_TINY);
        double y0;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(lc));
        const double u = c.ql * y0, e = fma(-(lc * y0), y0, 1.0);      // ql rsqrt(lc), refinement merged in
        c.w[0] = fma(u * e, fma(0.375, e, 0.5), u);
        c.w[1] = c.w[0] * c.ql;
        c.w[2] = c.w[1] * c.ql;
        c.Z[1] = z1;
        c.Z[2] = fma(c.Z[1], c.Z[1], (c.w[0] * c.w[0]) * (c.lam2 * m.k_third));
        return c;
    }
    const double lam1 = (x - m.t_lo) * (x - m.t_d);
    const double ix = fast_rcp(x);
    c.ql = lam1 * ix;
    const double pl = c.lam2 * ix;
    // sqrt(lam1) = l rsqrt(l) with l = max(lam1, tiny): no branch, ~1e-150 instead of 0 at threshold where the
    // width vanishes anyway
    // (rsqrt refinement merged with the product: sqrt(l) = h + h e p(e), h = l y0, e = 1 - h y0, p = 1/2 + 3e/8;
    // the factor 1/2 of g is folded into Kw on the host)
    const double lc = fmax(lam1, MIPWA_TINY);
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(lc));
    const double h = lc * y0, e = fma(-h, y0, 1.0);
    const double sq = fma(h * e, fma(0.375, e, 0.5), h);
    c.w[0] = sq * ix;
    c.w[1] = c.w[0] * c.ql;
    c.w[2] = c.w[1] * c.ql;
    c.Z[1] = fma(m.kappa, ix, z1);
    c.Z[2] = fma(c.Z[1], c.Z[1], m.k_third * (c.ql * pl));
    return c;
}

// both channels of a point: Z_1 = x + 2 y - Sigma = (s12 + s13 - Sigma) + y, the bracket shared by the two
template <int FL = 0>
__device__ __forceinline__ void make_channels(const DevModel& m, double s12, double s13, Channel& ca, Channel& cb)
{
    const double u = (s12 + s13) - m.sigma;
    ca = make_channel<FL>(m, s12, u + s13);
    cb = make_channel<FL>(m, s13, u + s12);
}

__device__ __forceinline__ double pick(int L, const double (&v)[3]) { return L == 0 ? v[0] : (L == 1 ? v[1] : v[2]); }

// One resonance in one channel: F_D F_R Z_L BW / sqrt(n_R n_D) = t (dD + i W) as the three real factors (the caller
// symmetrises with fused multiply-adds); c_r sqrt(n_R n_D) is applied later.
// LT = 0, 1, 2: spin known at compile time (no selects, unused factors vanish).  LT < 0: spin read from the model,
// branch-free: den_L(z) = pc + z (pb + pa z) with (pa, pb, pc) = (0,0,1), (0,1,1), (1,3,9), factors selected.
template <int LT>
__device__ __forceinline__ void resonance_channel(const ResDev& r, const Channel& c, double& t, double& dD, double& W)
{
    double DR, DD, Z;
    if (LT == 0) {
        DR = 1.0; DD = 1.0; W = r.Kw * c.w[0]; Z = 1.0;
    } else if (LT == 1) {
        DR = fma(r.cR, c.ql, 1.0);
        DD = fma(r.cD, c.lam2, 1.0);
        W = r.Kw * c.w[1];
        Z = c.Z[1];
    } else if (LT == 2) {
        DR = fma(c.ql, fma(c.ql, r.qR2, r.qR1), 9.0);
        DD = fma(c.lam2, fma(c.lam2, r.qD2, r.qD1), 9.0);
        W = r.Kw * c.w[2];
        Z = c.Z[2];
    } else {
        const double zR = r.cR * c.ql, zD = r.cD * c.lam2;
        DR = fma(zR, fma(zR, r.pa, r.pb), r.pc);
        DD = fma(zD, fma(zD, r.pa, r.pb), r.pc);
        W = r.Kw * pick(r.L, c.w);
        Z = pick(r.L, c.Z);
    }
    dD = (r.m0sq - c.x) * DR;
    const double E = fma(dD, dD, W * W);
    const double rs = fast_rsqrt((DR * DD) * (E * E));
    t = (LT == 0 ? rs : Z * DR * rs);
}

// Bose-symmetrised term T_r(s12,s13) + T_r(s13,s12) without its coefficient (and without sqrt(n_R n_D))
template <int LT>
__device__ __forceinline__ void resonance_sym(const ResDev& rd, const Channel& ca, const Channel& cb, double& tr,
                                              double& ti)
{
    double ta, da, Wa, tb, db, Wb;
    resonance_channel<LT>(rd, ca, ta, da, Wa);
    resonance_channel<LT>(rd, cb, tb, db, Wb);
    tr = fma(ta, da, tb * db);
    ti = fma(ta, Wa, tb * Wb);
}

template <int LT>
__device__ __forceinline__ void add_resonance(const ResDev& rd, const Channel& ca, const Channel& cb, double& are,
                                              double& aim)
{
    double tr, ti;
    resonance_sym<LT>(rd, ca, cb, tr, ti);
    are = fma(rd.cre, tr, fma(-rd.cim, ti, are));
    aim = fma(rd.cre, ti, fma(rd.cim, tr, aim));
}

// MIPWA_FL_SHR: NR >= 2 resonances of spin LT (1 or 2) with common radii.  Per channel ONE barrier block
// (D_R, D_D, rsqrt(D_R D_D), times Z_L D_R), then per resonance F_D F_R Z BW / sqrt(n_R n_D) = [Z D_R rsqrt(D_R D_D)]
// (dD + i W') / E with one reciprocal of E = dD^2 + W'^2 (three DFMAs after the seed) instead of the five-instruction
// reciprocal square root of D_R D_D E^2.
template <int LT>
__device__ __forceinline__ void group_barrier(const ResDev& r, const Channel& c, double& DR, double& FZ)
{
    double DD;
    if (LT == 1) {
        DR = fma(r.cR, c.ql, 1.0);
        DD = fma(r.cD, c.lam2, 1.0);
    } else {
        DR = fma(c.ql, fma(c.ql, r.qR2, r.qR1), 9.0);
        DD = fma(c.lam2, fma(c.lam2, r.qD2, r.qD1), 9.0);
    }
    FZ = (c.Z[LT] * DR) * fast_rsqrt(DR * DD);
}

// symmetrised terms T_r(s12,s13) + T_r(s13,s12) (without coefficient and sqrt(n_R n_D)) of the NR group members
template <int LT, int NR>
__device__ __forceinline__ void group_shared_terms(const ResDev* rd, const Channel& ca, const Channel& cb,
                                                   double* tr, double* ti)
{
    double DRa, FZa, DRb, FZb;
    group_barrier<LT>(rd[0], ca, DRa, FZa);
    group_barrier<LT>(rd[0], cb, DRb, FZb);
    const double xDa = ca.x * DRa, xDb = cb.x * DRb;       // (m0^2 - x) D_R = m0^2 D_R - x D_R: one product for the group
#pragma unroll
    for (int r = 0; r < NR; ++r) {
        const double Wa = rd[r].Kw * ca.w[LT], Wb = rd[r].Kw * cb.w[LT];
        const double da = fma(rd[r].m0sq, DRa, -xDa), db = fma(rd[r].m0sq, DRb, -xDb);
        const double ta = FZa * fast_rcp(fma(da, da, Wa * Wa)), tb = FZb * fast_rcp(fma(db, db, Wb * Wb));
        tr[r] = fma(ta, da, tb * db);
        ti[r] = fma(ta, Wa, tb * Wb);
    }
}

template <int LT, int NR>
__device__ __forceinline__ void add_group_shared(const ResDev* rd, const Channel& ca, const Channel& cb, double& are,
                                                 double& aim)
{
    double tr[NR], ti[NR];
    group_shared_terms<LT, NR>(rd, ca, cb, tr, ti);
#pragma unroll
    for (int r = 0; r < NR; ++r) {
        are = fma(rd[r].cre, tr[r], fma(-rd[r].cim, ti[r], are));
        aim = fma(rd[r].cre, ti[r], fma(rd[r].cim, tr[r], aim));
    }
}

// A(s12,s13) = S(s12) + S(s13) + sum_r c_r [T_r(s12,s13) + T_r(s13,s12)]
// Model signature <R1, R2>: the host orders the resonances spin 1 first (R1 of them), then spin 2 (R2), so that
// the whole sum unrolls with compile-time spins and constants straight from the parameter bank (2 (R1 + R2)
// independent chains).  <-1, -1>: any list (incl. spin 0), run-time loop over m.R.  FL: MIPWA_FL_* of the model.
template <int R1, int R2, int FL = 0>
__device__ __forceinline__ void add_resonances(const DevModel& m, double s12, double s13, double& are, double& aim)
{
    if (R1 == 0 && R2 == 0) return;
    Channel ca, cb;
    make_channels<FL>(m, s12, s13, ca, cb);
    if (R1 >= 0) {
        if ((FL & MIPWA_FL_SHR) && R1 >= 2) {
            add_group_shared<1, (R1 >= 2 ? R1 : 2)>(&m.res[0], ca, cb, are, aim);
        } else {
#pragma unroll
            for (int r = 0; r < R1; ++r) add_resonance<1>(m.res[r], ca, cb, are, aim);
        }
        if ((FL & MIPWA_FL_SHR) && R2 >= 2) {
            add_group_shared<2, (R2 >= 2 ? R2 : 2)>(&m.res[R1 > 0 ? R1 : 0], ca, cb, are, aim);
        } else {
#pragma unroll
            for (int r = 0; r < R2; ++r) add_resonance<2>(m.res[R1 + r], ca, cb, are, aim);
        }
    } else {
        for (int r = 0; r < m.R; ++r) add_resonance<-1>(m.res[r], ca, cb, are, aim);
    }
}

// A at a point whose spline rows are known (byte offsets o1, o2 into the shared-memory rows)
template <int R1, int R2, int FL = 0>
__device__ __forceinline__ void amplitude_off(const RowsSmem& sm, const DevModel& m, double s12, double s13,
                                              unsigned int o1, unsigned int o2, double& are, double& aim)
{
    double r1, i1, r2, i2, t;
    spline_eval_off(sm, s12, o1, r1, i1, t);
    spline_eval_off(sm, s13, o2, r2, i2, t);
    are = r1 + r2;
    aim = i1 + i2;
    add_resonances<R1, R2, FL>(m, s12, s13, are, aim);
}

// the same from the stored segment pair (seg = j12 | j13 << 8)
template <int R1, int R2, int FL = 0>
__device__ __forceinline__ void amplitude_seg(const RowsSmem& sm, const DevModel& m, double s12, double s13,
                                              unsigned int seg, double& are, double& aim)
{
    amplitude_off<R1, R2, FL>(sm, m, s12, s13, seg_off1(seg), seg_off2(seg), are, aim);
}

// the same for a point met for the first time (generator, setup): segment search in the knot table
template <int R1, int R2, int FL = 0>
__device__ __forceinline__ void amplitude_search(const RowsSmem& sm, const SearchSmem& ss, const DevModel& m, double s12,
                                                 double s13, double& are, double& aim)
{
    amplitude_off<R1, R2, FL>(sm, m, s12, s13, spline_segment(ss, s12) * MIPWA_ROW_BYTES,
                              spline_segment(ss, s13) * MIPWA_ROW_BYTES, are, aim);
}

#define MIPWA_SIG_MAX1 4
#define MIPWA_SIG_MAX2 2
// run CALL with constexpr R1, R2 matching the model signature (n0, n1, n2 = resonances of spin 0, 1, 2)
#define MIPWA_DISPATCH_SIG(n0, n1, n2, CALL)                                                      \
    switch (((n0) == 0 && (n1) <= MIPWA_SIG_MAX1 && (n2) <= MIPWA_SIG_MAX2) ? (n1) * 8 + (n2) : -1) { \
        case 0: { constexpr int R1 = 0, R2 = 0; CALL; } break;                                    \
        case 1: { constexpr int R1 = 0, R2 = 1; CALL; } break;                                    \
        case 2: { constexpr int R1 = 0, R2 = 2; CALL; } break;                                    \
        case 8: { constexpr int R1 = 1, R2 = 0; CALL; } break;                                    \
        case 9: { constexpr int R1 = 1, R2 = 1; CALL; } break;                                    \
        case 10: { constexpr int R1 = 1, R2 = 2; CALL; } break;                                   \
        case 16: { constexpr int R1 = 2, R2 = 0; CALL; } break;                                   \
        case 17: { constexpr int R1 = 2, R2 = 1; CALL; } break;                                   \
        case 18: { constexpr int R1 = 2, R2 = 2; CALL; } break;                                   \
        case 24: { constexpr int R1 = 3, R2 = 0; CALL; } break;                                   \
        case 25: { constexpr int R1 = 3, R2 = 1; CALL; } break;                                   \
        case 26: { constexpr int R1 = 3, R2 = 2; CALL; } break;                                   \
        case 32: { constexpr int R1 = 4, R2 = 0; CALL; } break;                                   \
        case 33: { constexpr int R1 = 4, R2 = 1; CALL; } break;                                   \
        case 34: { constexpr int R1 = 4, R2 = 2; CALL; } break;                                   \
        default: { constexpr int R1 = -1, R2 = -1; CALL; } break;                                 \
    }

// As MIPWA_DISPATCH_SIG, with constexpr FL = the model's MIPWA_FL_* flags as far as the signature can use them
// (MIPWA_FL_SHR only where a spin group has two or more members; none on the run-time <-1,-1> form).
#define MIPWA_FL_CASES(r1, r2, fl, CALL)                                                          \
    {                                                                                             \
        constexpr int R1 = (r1), R2 = (r2);                                                       \
        constexpr bool shr_useful = (r1) >= 2 || (r2) >= 2;                                       \
        switch (shr_useful ? ((fl) & 3) : ((fl) & MIPWA_FL_EQM)) {                                \
            case 0: { constexpr int FL = 0; CALL; } break;                                        \
            case 1: { constexpr int FL = MIPWA_FL_EQM; CALL; } break;                             \
            case 2: { constexpr int FL = shr_useful ? MIPWA_FL_SHR : 0; CALL; } break;            \
            default: { constexpr int FL = shr_useful ? (MIPWA_FL_EQM | MIPWA_FL_SHR) : MIPWA_FL_EQM; CALL; } break; \
        }                                                                                         \
    }
#define MIPWA_DISPATCH_SIGFL(n0, n1, n2, fl, CALL)                                                \
    switch (((n0) == 0 && (n1) <= MIPWA_SIG_MAX1 && (n2) <= MIPWA_SIG_MAX2) ? (n1) * 8 + (n2) : -1) { \
        case 0: MIPWA_FL_CASES(0, 0, 0, CALL) break;                                              \
        case 1: MIPWA_FL_CASES(0, 1, fl, CALL) break;                                             \
        case 2: MIPWA_FL_CASES(0, 2, fl, CALL) break;                                             \
        case 8: MIPWA_FL_CASES(1, 0, fl, CALL) break;                                             \
        case 9: MIPWA_FL_CASES(1, 1, fl, CALL) break;                                             \
        case 10: MIPWA_FL_CASES(1, 2, fl, CALL) break;                                            \
        case 16: MIPWA_FL_CASES(2, 0, fl, CALL) break;                                            \
        case 17: MIPWA_FL_CASES(2, 1, fl, CALL) break;                                            \
        case 18: MIPWA_FL_CASES(2, 2, fl, CALL) break;                                            \
        case 24: MIPWA_FL_CASES(3, 0, fl, CALL) break;                                            \
        case 25: MIPWA_FL_CASES(3, 1, fl, CALL) break;                                            \
        case 26: MIPWA_FL_CASES(3, 2, fl, CALL) break;                                            \
        case 32: MIPWA_FL_CASES(4, 0, fl, CALL) break;                                            \
        case 33: MIPWA_FL_CASES(4, 1, fl, CALL) break;                                            \
        case 34: MIPWA_FL_CASES(4, 2, fl, CALL) break;                                            \
        default: { constexpr int R1 = -1, R2 = -1, FL = 0; CALL; } break;                         \
    }
