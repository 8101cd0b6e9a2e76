// gen.cuh -- toy Monte-Carlo generation on the device ("samples of 100K signal events are
// generated from a Dalitz plot PDF").  Accept-reject against a piecewise-constant envelope, the recipe of DESIGN.md
// reading P22 and of paper_1703_03284_b200/inputs.py (Envelope, accept_reject), restated here for the device:
//
//   envelope   n_coarse x n_coarse cells over the bounding square [lo, hi]^2; env(cell) = 1.2 x max |A|^2 over the
//              cell centres of an n_side x n_side fine grid that lie inside the Dalitz boundary and in that coarse
//              cell (an empty coarse cell takes its largest neighbour: done on the host, O(n_coarse^2))
//   candidate  i uses uniforms 4i .. 4i+3 of the counter-based stream `key`: coarse cell by inverse CDF over
//              env, uniform position inside the cell, kept iff inside the boundary and u_3 env(cell) < |A|^2
//   events     the first n accepted candidates IN COUNTER ORDER (stream compaction per batch), so the sample depends
//              on (model, parameters, key, n, n_side, n_coarse) only - not on grid size, batch size or timing.
//
// The generator is the splitmix64 counter scheme of inputs.py (every side implements the same one); the placement
// arithmetic uses explicit round-to-nearest intrinsics so that no fused multiply-add changes a coordinate's last bit.
#pragma once
#include "dev_model.cuh"

struct GenKin { double M2, a, b, c, lo, hi; };            // M^2, m1^2, m2^2, m3^2, (m1+m2)^2, (M-m3)^2

__device__ __forceinline__ unsigned long long gen_mix(unsigned long long z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

// uniform in [0, 1) of counter ctr of the stream key
__device__ __forceinline__ double gen_uniform(unsigned long long key, unsigned long long ctr)
{
    const unsigned long long x = gen_mix(gen_mix(ctr * 0x9E3779B97F4A7C15ULL + key) ^ key);
    return (double)(x >> 11) * (1.0 / 9007199254740992.0);
}

__device__ __forceinline__ double gen_lam(double a, double b, double c)
{
    const double sq = __dadd_rn(__dadd_rn(__dmul_rn(a, a), __dmul_rn(b, b)), __dmul_rn(c, c));
    const double cr = __dadd_rn(__dadd_rn(__dmul_rn(a, b), __dmul_rn(a, c)), __dmul_rn(b, c));
    return __dsub_rn(sq, __dmul_rn(2.0, cr));
}

// lo <= s12 <= hi and |s13 - centre(s12)| <= half(s12), centre and half as in SURVEY 8(c) O1 (product form)
__device__ __forceinline__ bool gen_inside(const GenKin& k, double s12, double s13)
{
    if (!(s12 >= k.lo && s12 <= k.hi)) return false;
    const double two_s = __dmul_rn(2.0, s12);
    const double num = __dmul_rn(__dsub_rn(__dadd_rn(s12, k.a), k.b), __dsub_rn(__dsub_rn(k.M2, s12), k.c));
    const double centre = __dadd_rn(__dadd_rn(k.a, k.c), __ddiv_rn(num, two_s));
    const double prod = __dmul_rn(gen_lam(s12, k.a, k.b), gen_lam(k.M2, s12, k.c));
    const double half = __ddiv_rn(__dsqrt_rn(fmax(prod, 0.0)), two_s);
    return fabs(__dsub_rn(s13, centre)) <= half;
}

__device__ __forceinline__ double gen_abs2(const RowsSmem& sm, const SearchSmem& ss, const DevModel& m, double x, double y)
{
    double re, im;
    amplitude_search<-1, -1, 0>(sm, ss, m, x, y, re, im);
    return fma(re, re, im * im);
}

// fine grid pass: own[cx * nc + cy] = max |A|^2 (as the bit pattern of a non-negative double: ordered like integers)
static __global__ void __launch_bounds__(256)
k_gen_envelope(const __grid_constant__ DevModel m, const DevSearch* __restrict__ srch, const GenKin k, int n_side,
               double h, double H, int nc, unsigned long long* __restrict__ own)
{
    __shared__ RowsSmem sm;
    __shared__ SearchSmem ss;
    load_search_smem(ss, srch);
    load_rows_smem(sm, m);
    const long long total = (long long)n_side * n_side, stride = (long long)gridDim.x * blockDim.x;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += stride) {
        const int i = (int)(t / n_side), j = (int)(t % n_side);
        const double x = __dadd_rn(k.lo, __dmul_rn((double)i + 0.5, h)), y = __dadd_rn(k.lo, __dmul_rn((double)j + 0.5, h));
        if (!gen_inside(k, x, y)) continue;
        const double a2 = gen_abs2(sm, ss, m, x, y);
        const int cx = min((int)__ddiv_rn(__dsub_rn(x, k.lo), H), nc - 1), cy = min((int)__ddiv_rn(__dsub_rn(y, k.lo), H), nc - 1);
        if (a2 > 0.0) atomicMax(&own[cx * nc + cy], (unsigned long long)__double_as_longlong(a2));
    }
}

// candidates ctr0 .. ctr0 + count - 1: position and accept flag
static __global__ void __launch_bounds__(256)
k_gen_candidates(const __grid_constant__ DevModel m, const DevSearch* __restrict__ srch, const GenKin k,
                 unsigned long long key, long long ctr0, long long count, int nc, double H,
                 const double* __restrict__ cum, const double* __restrict__ env,
                 double* __restrict__ c12, double* __restrict__ c13, unsigned char* __restrict__ flag)
{
    __shared__ RowsSmem sm;
    __shared__ SearchSmem ss;
    load_search_smem(ss, srch);
    load_rows_smem(sm, m);
    const long long stride = (long long)gridDim.x * blockDim.x;
    const int ncell = nc * nc;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < count; t += stride) {
        const unsigned long long c4 = 4ULL * (unsigned long long)(ctr0 + t);
        const double u0 = gen_uniform(key, c4), u1 = gen_uniform(key, c4 + 1), u2 = gen_uniform(key, c4 + 2),
                     u3 = gen_uniform(key, c4 + 3);
        int lo = 0, hi = ncell;                            // first index with cum[idx] > u0
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (cum[mid] > u0) hi = mid; else lo = mid + 1;
        }
        const int cell = min(lo, ncell - 1), cx = cell / nc, cy = cell % nc;
        const double x = __dadd_rn(k.lo, __dmul_rn(__dadd_rn((double)cx, u1), H));
        const double y = __dadd_rn(k.lo, __dmul_rn(__dadd_rn((double)cy, u2), H));
        bool acc = gen_inside(k, x, y);
        if (acc) acc = __dmul_rn(u3, env[cell]) < gen_abs2(sm, ss, m, x, y);
        c12[t] = x; c13[t] = y; flag[t] = acc ? 1 : 0;
    }
}
