// kernels.cuh -- the recompute path: fused amplitude + log-sum / normalisation reduction,
// the per-point test hook, and the boundary check.  sm_100a only.
#pragma once
#include "dev_model.cuh"

#ifndef MIPWA_BLOCK
#define MIPWA_BLOCK 256
#endif
// launch shape of k_nll_recompute (measured, profiles/r1_recompute_shape.md): ONE block of 512 threads per SM with up
// to 128 registers per thread, one point per thread and iteration.  With 128 registers the model constants stay in
// registers instead of being re-read from the constant bank every point, and one big block per SM beat two or three
// smaller ones at the same warp count (0.265 ms against 0.298 ms for 2 x 256 threads, 0.299 ms for 3 x 256 threads
// at 80 registers, config 3).
#ifndef MIPWA_REC_BLOCK
#define MIPWA_REC_BLOCK 512
#endif
#ifndef MIPWA_REC_MINBLOCKS
#define MIPWA_REC_MINBLOCKS 1
#endif
#ifndef MIPWA_REC_PTS
#define MIPWA_REC_PTS 1
#endif

// ---- deterministic block reduction of NV doubles per thread: warp shuffles, then shared memory -------------------
template <int NV>
__device__ __forceinline__ void block_reduce(double (&v)[NV], double* red /* [NV][32] in smem */)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], off);
        if (lane == 0) red[k * 32 + warp] = v[k];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            double x = lane < nwarp ? red[k * 32 + lane] : 0.0;
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
            v[k] = x;                                   // valid in thread 0
        }
    }
    __syncthreads();
}

// Running product of |A|^2 with the exponents peeled off by integer operations: ln prod = ln(mantissa product)
// + (exponent sum) ln 2.  One DMUL per event instead of a ~30-instruction fp64 log; the log is taken once per
// LOGPROD_FLUSH events per thread.  Zero, denormal, inf and NaN values take the plain log so that IEEE specials
// propagate exactly as in -sum ln|A|^2.
#define LOGPROD_FLUSH 512
struct LogProd {
    double prod = 1.0, sum = 0.0;
    int esum = 0, cnt = 0;
    __device__ __forceinline__ void flush()
    {
        // ln2 split hi/lo so that esum * ln2 carries no rounding of its own
        sum += fma((double)esum, 6.93147180369123816490e-01, fma((double)esum, 1.90821492927058770002e-10, log(prod)));
        prod = 1.0; esum = 0; cnt = 0;
    }
    __device__ __forceinline__ void add(double v)
    {
        const int hi = __double2hiint(v);
        const int ex = (hi >> 20) & 0x7ff;               // v >= 0 or NaN: the sign bit lands in the NaN branch
        if (ex == 0 || ex == 0x7ff || hi < 0) {
            sum += log(v);
        } else {
            esum += ex - 1023;
            prod *= __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(v));
            if (++cnt == LOGPROD_FLUSH) flush();
        }
    }
    __device__ __forceinline__ double value() { flush(); return sum; }
};

// ---- A4-A6: one launch over [events | normalisation points] ------------------------------------------------------
// Persistent grid (a multiple of the SM count).  Per thread: grid-stride over events (coalesced 8-byte loads of
// s12[i], s13[i], the next point's pair prefetched before the current one is evaluated; nothing is written per
// event), then over normalisation points.  Block partials go to partials[block] = (sum ln|A|^2, sum w|A|^2); the
// last block to finish adds them in block order (fixed order: bit-reproducible for a given grid) and writes the
// two totals to `result` (mapped pinned host memory).
// MIX = true (mipwa_nll_mix, signal + background mixture): the events carry a background density eb[i] and the sum is
// over ln(|A_i|^2 + kappa eb[i]) with kappa = I (1 - f_s) / f_s from a first, normalisation-only launch.
template <int R1, int R2, int FL, bool MIX>
__global__ void __launch_bounds__(MIPWA_REC_BLOCK, MIPWA_REC_MINBLOCKS)
k_nll_recompute(const __grid_constant__ DevModel m,
                const double* __restrict__ e12, const double* __restrict__ e13, const unsigned short* __restrict__ eseg,
                const double* __restrict__ eb, double kappa, long long n_ev,
                const double* __restrict__ g12, const double* __restrict__ g13, const double* __restrict__ gw,
                const unsigned short* __restrict__ gseg, long long n_norm, double2* __restrict__ partials, unsigned int* __restrict__ ticket,
                double* __restrict__ result)
{
    __shared__ SplineCoefSmem sm;
    __shared__ double red[2 * 32];
    __shared__ bool is_last;
    load_spline_coef_smem(sm, m);

    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;

    // PTS points per thread and iteration: independent dependency chains for the FP64 pipe.  Out-of-range slots
    // evaluate a harmless in-range point and contribute ln 1 = 0 (events) or weight 0 (normalisation).
    // a pure S-wave model (R = 0) is bound by memory latency, not arithmetic: four points in flight per thread
    constexpr int PTS = (R1 == 0 && R2 == 0) ? 4 : MIPWA_REC_PTS;
    LogProd lp;
    double integ = 0.0;
    if constexpr (PTS == 1) {
        // One point per thread and iteration.  Every non-FP64 instruction costs the issue slot an FP64 instruction
        // could have used (cycles per warp-point ~ 2 x FP64 + others, profiles/r1_k_nll_recompute_ncu.md), so the loop
        // bookkeeping is a 32-bit trip count, cursors advanced by a constant and no tail predicates: all `iters` points
        // of a thread exist, and the prefetch of the last iteration is skipped, its registers never read.
        {
            const long long rem = n_ev - t0;
            const int iters = rem > 0 ? (int)((rem + stride - 1) / stride) : 0;
            const double *pa = e12 + t0, *pb = e13 + t0, *pk = eb + t0;
            const unsigned short* ps = eseg + t0;
            double a = 1.0, b = 1.0, bk = 0.0;
            unsigned int sg = 0u;
            if (iters > 0) { a = *pa; b = *pb; sg = *ps; if (MIX) bk = *pk; }
            double na = a, nb = b, nbk = bk;
            unsigned int ns = sg;
            for (int it = 0; it < iters; ++it) {
                pa += stride; pb += stride; ps += stride;
                if (MIX) pk += stride;
                if (it + 1 < iters) { na = *pa; nb = *pb; ns = *ps; if (MIX) nbk = *pk; }
                double re, im;
                amplitude_seg<R1, R2, FL>(sm, m, a, b, sg, re, im);
                double v = fma(re, re, im * im);
                if (MIX) v = fma(kappa, bk, v);
                lp.add(v);
                a = na; b = nb; sg = ns;
                if (MIX) bk = nbk;
            }
        }
        {
            const long long rem = n_norm - t0;
            const int iters = rem > 0 ? (int)((rem + stride - 1) / stride) : 0;
            const bool has_w = gw != nullptr;
            const double *pa = g12 + t0, *pb = g13 + t0, *pw = gw + t0;
            const unsigned short* ps = gseg + t0;
            double a = 1.0, b = 1.0, w = 1.0;
            unsigned int sg = 0u;
            if (iters > 0) { a = *pa; b = *pb; sg = *ps; if (has_w) w = *pw; }
            double na = a, nb = b, nw = w;
            unsigned int ns = sg;
            for (int it = 0; it < iters; ++it) {
                pa += stride; pb += stride; ps += stride; pw += stride;
                if (it + 1 < iters) { na = *pa; nb = *pb; ns = *ps; if (has_w) nw = *pw; }
                double re, im;
                amplitude_seg<R1, R2, FL>(sm, m, a, b, sg, re, im);
                integ = fma(w, fma(re, re, im * im), integ);
                a = na; b = nb; w = nw; sg = ns;
            }
        }
    } else {
    {
        double a[PTS], b[PTS], bk[PTS];
        unsigned int sg[PTS];
#pragma unroll
        for (int q = 0; q < PTS; ++q) {
            const long long i = t0 + q * stride;
            a[q] = 1.0; b[q] = 1.0; sg[q] = 0u; bk[q] = 0.0;
            if (i < n_ev) { a[q] = e12[i]; b[q] = e13[i]; sg[q] = eseg[i]; if (MIX) bk[q] = eb[i]; }
        }
        for (long long i = t0; i < n_ev; i += PTS * stride) {
            double na[PTS], nb[PTS], nbk[PTS];
            unsigned int ns[PTS];
#pragma unroll
            for (int q = 0; q < PTS; ++q) {
                const long long nx = i + (PTS + q) * stride;
                na[q] = 1.0; nb[q] = 1.0; ns[q] = 0u; nbk[q] = 0.0;
                if (nx < n_ev) { na[q] = e12[nx]; nb[q] = e13[nx]; ns[q] = eseg[nx]; if (MIX) nbk[q] = eb[nx]; }
            }
            double v[PTS];
#pragma unroll
            for (int q = 0; q < PTS; ++q) {
                double re, im;
                amplitude_seg<R1, R2, FL>(sm, m, a[q], b[q], sg[q], re, im);
                v[q] = fma(re, re, im * im);
                if (MIX) v[q] = fma(kappa, bk[q], v[q]);
            }
#pragma unroll
            for (int q = 0; q < PTS; ++q) {
                lp.add(i + q * stride < n_ev ? v[q] : 1.0);
                a[q] = na[q]; b[q] = nb[q]; sg[q] = ns[q];
                if (MIX) bk[q] = nbk[q];
            }
        }
    }
    {
        double a[PTS], b[PTS], w[PTS];
        unsigned int sg[PTS];
#pragma unroll
        for (int q = 0; q < PTS; ++q) {
            const long long j = t0 + q * stride;
            a[q] = 1.0; b[q] = 1.0; w[q] = 0.0; sg[q] = 0u;
            if (j < n_norm) { a[q] = g12[j]; b[q] = g13[j]; w[q] = gw ? gw[j] : 1.0; sg[q] = gseg[j]; }
        }
        for (long long j = t0; j < n_norm; j += PTS * stride) {
            double na[PTS], nb[PTS], nw[PTS];
            unsigned int ns[PTS];
#pragma unroll
            for (int q = 0; q < PTS; ++q) {
                const long long nx = j + (PTS + q) * stride;
                na[q] = 1.0; nb[q] = 1.0; nw[q] = 0.0; ns[q] = 0u;
                if (nx < n_norm) { na[q] = g12[nx]; nb[q] = g13[nx]; nw[q] = gw ? gw[nx] : 1.0; ns[q] = gseg[nx]; }
            }
#pragma unroll
            for (int q = 0; q < PTS; ++q) {
                double re, im;
                amplitude_seg<R1, R2, FL>(sm, m, a[q], b[q], sg[q], re, im);
                integ = fma(w[q], fma(re, re, im * im), integ);
            }
#pragma unroll
            for (int q = 0; q < PTS; ++q) { a[q] = na[q]; b[q] = nb[q]; w[q] = nw[q]; sg[q] = ns[q]; }
        }
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
        for (int b = threadIdx.x; b < gridDim.x; b += blockDim.x) {
            const double2 p = __ldcg(&partials[b]);
            f[0] += p.x; f[1] += p.y;
        }
        block_reduce<2>(f, red);
        if (threadIdx.x == 0) {
            result[0] = f[0];
            result[1] = f[1];
            *ticket = 0;                                  // ready for the next call
            __threadfence_system();
        }
    }
}

// ---- test hook: |A|^2 per point from the same device function ---------------------------------------------------
template <int R1, int R2, int FL>
__global__ void __launch_bounds__(MIPWA_BLOCK)
k_abs2(const __grid_constant__ DevModel m, const double* __restrict__ s12, const double* __restrict__ s13,
       const unsigned short* __restrict__ seg, long long n, double* __restrict__ out)
{
    __shared__ SplineCoefSmem sm;
    load_spline_coef_smem(sm, m);
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        double re, im;
        amplitude_seg<R1, R2, FL>(sm, m, s12[i], s13[i], seg[i], re, im);
        out[i] = fma(re, re, im * im);
    }
}

// ---- boundary check of mipwa_set_events / mipwa_set_norm_points ---------------------------------------------------
// inside iff (m1+m2)^2 <= s12 <= (M-m3)^2 and |s13 - centre(s12)| <= half(s12); a relative slack of 1e-12 keeps
// points that the caller's own fp64 boundary test placed exactly on the edge.  Counts offenders into *bad.
struct DevKin { double M2, m1s, m2s, m3s, t_lo, t_d, s_hi, s_top; };

// Also stores the spline segment pair of every point, seg[i] = j12 | j13 << 8 (knots are fixed at mipwa_create, so
// the pair is a property of the point set): the per-call kernels then index the coefficient tables directly.
static __global__ void __launch_bounds__(MIPWA_BLOCK)
k_validate(const DevKin k, const __grid_constant__ DevModel m, const double* __restrict__ s12,
           const double* __restrict__ s13, long long n, unsigned short* __restrict__ seg,
           unsigned long long* __restrict__ bad)
{
    __shared__ SplineSmem sm;
    load_spline_smem(sm, m);
    const long long stride = (long long)gridDim.x * blockDim.x;
    unsigned int mine = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const double x = s12[i], y = s13[i];
        const double slack = 1e-12;
        bool ok = x >= k.t_lo * (1.0 - slack) && x <= k.s_hi * (1.0 + slack);
        if (ok) {
            const double centre = k.m1s + k.m3s + (x + k.m1s - k.m2s) * (k.M2 - x - k.m3s) / (2.0 * x);
            const double prod = ((x - k.t_lo) * (x - k.t_d)) * ((k.s_hi - x) * (k.s_top - x));
            const double half = sqrt(fmax(prod, 0.0)) / (2.0 * x);
            ok = fabs(y - centre) <= half + slack * (fabs(centre) + half) + 1e-13;
        }
        mine += ok ? 0u : 1u;                             // NaN compares false above -> counted as bad
        double xj;
        const int j1 = spline_segment(sm, m, x, xj), j2 = spline_segment(sm, m, y, xj);
        seg[i] = (unsigned short)(j1 | (j2 << 8));
    }
    mine = __reduce_add_sync(0xffffffffu, mine);
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(bad, (unsigned long long)mine);
}

// ---- FP64 peak: register-resident dependent-chain DFMA loop, 8 independent chains per thread --------------------
static __global__ void __launch_bounds__(256)
k_dfma_peak(double* __restrict__ out, long long iters, double a, double b)
{
    double x0 = threadIdx.x * 1e-3, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (long long i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456) out[0] = s;                          // keeps the chains alive
}
