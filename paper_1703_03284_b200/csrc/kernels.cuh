// kernels.cuh -- the recompute path: fused amplitude + log-sum / normalisation reduction,
// the per-point test hook, and the boundary check.  sm_100a only.
#pragma once
#include "dev_model.cuh"

#define MIPWA_BLOCK 256
// launch shape of k_nll_recompute (measured, profiles/r1_recompute_shape.md): ONE block of 512 threads per SM with up
// to 128 registers per thread, one point per thread and iteration.  With 128 registers the model constants stay in
// registers instead of being re-read from the constant bank every point, and one big block per SM beat two or three
// smaller ones at the same warp count.
#define MIPWA_REC_BLOCK 512

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
// + (exponent sum) ln 2.  One DMUL per event instead of a ~30-instruction fp64 log; the caller takes the log (flush)
// at least once per LOGPROD_FLUSH values (mantissas are in [1, 2): the product cannot overflow).  Zero, denormal,
// negative, inf and NaN values take the plain log so that IEEE specials propagate exactly as in -sum ln|A|^2.
// Per value: one compare for the specials, one shift-add of the raw biased exponent, one mask; the bias is removed
// at the flush (every add, special or not, counts 1023 into eacc).
#define LOGPROD_FLUSH 512
struct LogProd {
    double prod = 1.0, sum = 0.0;
    int eacc = 0;
    __device__ __forceinline__ void flush(int count)       // count = adds since the last flush
    {
        // ln2 split hi/lo so that esum * ln2 carries no rounding of its own
        const double es = (double)(eacc - 1023 * count);
        sum += fma(es, 6.93147180369123816490e-01, fma(es, 1.90821492927058770002e-10, log(prod)));
        prod = 1.0; eacc = 0;
    }
    __device__ __forceinline__ void add(double v)
    {
        const int hi = __double2hiint(v);
        if ((unsigned int)(hi - 0x00100000) >= 0x7fe00000u) {              // exponent 0 or 0x7ff, or sign set
            sum += log(v);
            eacc += 1023;
        } else {
            eacc += (int)((unsigned int)hi >> 20);
            prod *= __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(v));
        }
    }
    // The same without a branch, for the hot loop of the full-recompute kernel: a special value is skipped here
    // (mantissa 1, exponent 0) and only remembered in `bad`; the kernel then walks the thread's values a second time and
    // adds the plain logs of the special ones (add_special).  With the log's slow path inside the loop ptxas keeps the ~23
    // model constants of the loop in vector registers instead of uniform ones, and every DFMA that reads one becomes a
    // three-register DFMA (3 instead of 2 issue cycles of the FP64 pipe): 22 per point.
    bool bad = false;
    static __device__ __forceinline__ bool special(double v)
    {
        return (unsigned int)(__double2hiint(v) - 0x00100000) >= 0x7fe00000u;   // exponent 0 or 0x7ff, or sign set
    }
    __device__ __forceinline__ void add_fast(double v)
    {
        const int hi = __double2hiint(v);
        const bool sp = special(v);
        bad |= sp;
        eacc += sp ? 1023 : (int)((unsigned int)hi >> 20);
        prod *= sp ? 1.0 : __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(v));
    }
    __device__ __forceinline__ void add_special(double v) { if (special(v)) sum += log(v); }
    // for loops without a trip count of their own: counts the adds and flushes every LOGPROD_FLUSH of them
    int cnt = 0;
    __device__ __forceinline__ void add_counted(double v)
    {
        add(v);
        if (++cnt == LOGPROD_FLUSH) { flush(cnt); cnt = 0; }
    }
    __device__ __forceinline__ double value() { flush(cnt); cnt = 0; return sum; }
};

// ---- point records (once per point set) ---------------------------------------------------------------------------
// rec[i] = (s12, s13, w or 1, row offsets) of point idx[i] (idx == nullptr: i).  The array is over-allocated by the
// caller and the tail zero-filled: the hot loops prefetch one record past their last point without a bounds test.
static __global__ void __launch_bounds__(MIPWA_BLOCK)
k_make_records(const double* __restrict__ s12, const double* __restrict__ s13, const double* __restrict__ w,
               double w_default, const unsigned short* __restrict__ seg, long long n, PointRec* __restrict__ rec)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const unsigned int sg = seg[i];
        PointRec r;
        r.s12 = s12[i]; r.s13 = s13[i]; r.w = w ? w[i] : w_default;
        r.o1 = seg_off1(sg); r.o2 = seg_off2(sg);
        rec[i] = r;
    }
}

// tail [n, n + pad): copies of record 0 with weight 0 - a harmless point for lanes that run past the end of a chunk
static __global__ void __launch_bounds__(MIPWA_BLOCK)
k_pad_records(PointRec* __restrict__ rec, long long n, long long pad)
{
    PointRec r = rec[0];
    r.w = 0.0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < pad; i += stride) rec[n + i] = r;
}

// ---- A4-A6: one launch over [events | normalisation points] ------------------------------------------------------
// Persistent grid (one 512-thread block per SM).  Per thread: grid-stride over the event records, then over the
// normalisation records; one 256-bit load per point, issued one iteration ahead; nothing is written per point.  Block
// partials go to partials[block] = (sum ln|A|^2, sum w|A|^2); the last block to finish adds them in block order (fixed
// order: bit-reproducible for a given grid) and writes the two totals to `result` (mapped pinned host memory).
// Every non-FP64 instruction costs the issue slot an FP64 instruction could have used (cycles per warp-point ~ 2 x FP64
// + others, profiles/r2_k_nll_recompute_ncu.md), hence: 32-bit trip counts, one cursor, no tail predicates (all
// `iters` points of a thread exist; the record arrays are padded so that the last prefetch stays in bounds).
// MIX = true (mipwa_nll_mix, signal + background mixture): the event records carry a background density w and the sum
// is over ln(|A_i|^2 + kappa w_i) with kappa = I (1 - f_s) / f_s from a first, normalisation-only launch.
template <int R1, int R2, int FL, bool MIX>
__global__ void __launch_bounds__(MIPWA_REC_BLOCK, 1)
k_nll_recompute(const __grid_constant__ DevModel m, const PointRec* __restrict__ ev, double kappa, long long n_ev,
                const PointRec* __restrict__ nm, long long n_norm, double2* __restrict__ partials,
                unsigned int* __restrict__ ticket, double* __restrict__ result, long long tag,
                const double* __restrict__ integral_src)
{
    __shared__ RowsSmem sm;
    __shared__ double red[2 * 32];
    __shared__ bool is_last;
    // Launched with programmatic stream serialisation (mipwa_nll_batch: the same kernel enqueued back to back) the next
    // launch's blocks may be scheduled as this one's leave their SMs, before the last block's epilogue is over; they read
    // only the point records and their own parameter block until griddepcontrol.wait below.  Both instructions do nothing
    // in an ordinary launch.
    asm volatile("griddepcontrol.launch_dependents;");
    const unsigned int stride = gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const PointRec* p = ev + t0;
    PointRec r = ld_rec(p);                                // the first record is on its way while the rows are copied
    load_rows_smem(sm, m);
    // MIX with integral_src: the integral of the normalisation launch that ran just before on this stream is read from device
    // memory (no host round trip between the two launches of mipwa_nll_mix); `kappa` then carries (1 - f_s) / f_s x weight scale
    if (MIX && integral_src) kappa *= __ldcg(integral_src);

    LogProd lp;
    double integ = 0.0;
    {
        const long long rem = n_ev - t0;
        int left = rem > 0 ? (int)((rem + stride - 1) / stride) : 0;
        while (left > 0) {
            const int chunk = left < LOGPROD_FLUSH ? left : LOGPROD_FLUSH;
#pragma unroll 2
            for (int it = 0; it < chunk; ++it) {
                p += stride;
                const PointRec nx = ld_rec(p);
                double re, im;
                amplitude_off<R1, R2, FL>(sm, m, r.s12, r.s13, r.o1, r.o2, re, im);
                double v = fma(re, re, im * im);
                if (MIX) v = fma(kappa, r.w, v);
                lp.add_fast(v);
                r = nx;
            }
            lp.flush(chunk);
            left -= chunk;
        }
    }
    {
        const long long rem = n_norm - t0;
        const int iters = rem > 0 ? (int)((rem + stride - 1) / stride) : 0;
        p = nm + t0;
        r = ld_rec(p);
#pragma unroll 2
        for (int it = 0; it < iters; ++it) {
            p += stride;
            const PointRec nx = ld_rec(p);
            double re, im;
            amplitude_off<R1, R2, FL>(sm, m, r.s12, r.s13, r.o1, r.o2, re, im);
            integ = fma(r.w, fma(re, re, im * im), integ);
            r = nx;
        }
    }

    if (lp.bad) {
        // some |A|^2 of this thread was zero, denormal, negative, infinite or NaN (a degenerate model, a point on a pole
        // of zero width): the thread walks its events again and adds the plain logs of those values, so that IEEE
        // specials reach the NLL exactly as in -sum ln|A|^2
        p = ev + t0;
        for (long long i = t0; i < n_ev; i += stride, p += stride) {
            const PointRec q = ld_rec(p);
            double re, im;
            amplitude_off<R1, R2, FL>(sm, m, q.s12, q.s13, q.o1, q.o2, re, im);
            double v = fma(re, re, im * im);
            if (MIX) v = fma(kappa, q.w, v);
            lp.add_special(v);
        }
    }
    double v[2] = { lp.sum, integ };
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
        for (int b = threadIdx.x; b < gridDim.x; b += blockDim.x) {
            const double2 p = __ldcg(&partials[b]);
            f[0] += p.x; f[1] += p.y;
        }
        block_reduce<2>(f, red);
        if (threadIdx.x == 0) {
            result[0] = f[0];
            result[1] = MIX && integral_src ? __ldcg(integral_src) : f[1];   // the mixture's event launch hands the integral on
            *ticket = 0;                                  // ready for the next call
            publish_result(result, tag);
        }
    }
}

// ---- test hook: |A|^2 per point from the same device function ---------------------------------------------------
template <int R1, int R2, int FL>
__global__ void __launch_bounds__(MIPWA_BLOCK)
k_abs2(const __grid_constant__ DevModel m, const double* __restrict__ s12, const double* __restrict__ s13,
       const unsigned short* __restrict__ seg, long long n, double* __restrict__ out)
{
    __shared__ RowsSmem sm;
    load_rows_smem(sm, m);
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
// the pair is a property of the point set): the per-call kernels then index the coefficient rows directly.  With `rec` it
// also writes the 32-byte records the recompute kernels stream (what k_make_records does on first use otherwise).
static __global__ void __launch_bounds__(MIPWA_BLOCK)
k_validate(const DevKin k, const DevSearch* __restrict__ srch, const double* __restrict__ s12,
           const double* __restrict__ s13, const double* __restrict__ w, double w_default, long long n,
           unsigned short* __restrict__ seg, PointRec* __restrict__ rec, unsigned long long* __restrict__ bad)
{
    __shared__ SearchSmem ss;
    load_search_smem(ss, srch);
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
        const int j1 = spline_segment(ss, x), j2 = spline_segment(ss, y);
        seg[i] = (unsigned short)(j1 | (j2 << 8));
        if (rec) {                                        // the record of the point, while it is in registers anyway
            PointRec r;
            r.s12 = x; r.s13 = y; r.w = w ? w[i] : w_default;
            r.o1 = j1 * MIPWA_ROW_BYTES; r.o2 = j2 * MIPWA_ROW_BYTES;
            rec[i] = r;
        }
    }
    mine = __reduce_add_sync(0xffffffffu, mine);
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(bad, (unsigned long long)mine);
}

// ---- sharded likelihood on the device (mipwa_nll_parts_device / mipwa_combine_parts_device) ---------------------------
// this rank's (S, I, n_ev) from the totals a value kernel left in device memory
static __global__ void k_pack_parts(const double* __restrict__ totals, double i_scale, double n_ev, double* __restrict__ parts)
{
    parts[0] = totals[0];
    parts[1] = totals[1] * i_scale;
    parts[2] = n_ev;
}

// A7 over all ranks' pieces, added in rank order (every rank forms the same bits): result = (S, I, tag, NLL, n)
static __global__ void k_combine_parts(const double* __restrict__ all, int n_ranks, double* __restrict__ result, long long tag)
{
    double S = 0.0, I = 0.0, n = 0.0;
    for (int r = 0; r < n_ranks; ++r) { S += all[3 * r]; I += all[3 * r + 1]; n += all[3 * r + 2]; }
    result[0] = S; result[1] = I;
    result[3] = n > 0.0 ? -S + n * log(I) : 0.0;
    result[4] = n;
    publish_result(result, tag);
}

// ---- timing aid: keeps the GPU busy for `ns` nanoseconds ---------------------------------------------------------------
// With kernel timing on (mipwa_enable_timing) this runs in front of the first event record, so that the host has
// submitted [event, kernel, event] before the first event executes: the two timestamps then bracket the kernel's
// execution, not the host's launch call (8-13 us for a 12 KB parameter block, 3-5 % of a config-3 likelihood call).
static __global__ void k_spacer(unsigned long long ns)
{
    unsigned long long t0, t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    do { asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); } while (t - t0 < ns);
}

// ---- FP64 peak: register-resident dependent-chain loops, 8 independent chains per thread ---------------------------
// MODE 0: DFMA with three distinct register operands (x = x a + b).  The operand fetch of this form costs the pipe
//         ~8 % (profiles/r1_fp64_microbench.md: 58.8 of 64 instructions per clock and SM).
// MODE 1: DFMA with an immediate and a repeated register operand (x = x 2^-60 + x, which leaves x unchanged: a stable
//         chain), the form most FP64 instructions of the likelihood kernels have: it issues every 2 clk, the pipe's
//         demonstrated rate (63.4 of 64).  Two flops per instruction in both modes.
template <int MODE>
static __global__ void __launch_bounds__(256)
k_fp64_peak(double* __restrict__ out, long long iters, double a, double b)
{
    double x[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) x[u] = threadIdx.x * 1e-3 + u;
    for (long long i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                if (MODE == 0) x[u] = fma(x[u], a, b);
                else x[u] = fma(x[u], 0x1p-60, x[u]);
            }
        }
    }
    const double s = ((x[0] + x[1]) + (x[2] + x[3])) + ((x[4] + x[5]) + (x[6] + x[7]));
    if (s == 123.456) out[0] = s;                          // keeps the chains alive
}
