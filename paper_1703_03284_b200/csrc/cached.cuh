// cached.cuh -- the fixed-shape path (BASELINE.json north_star (d)): when no resonance mass or
// width floats, A(s12,s13) = sum_k c_k B_k(s12,s13) is linear in c = [y_0..y_{N-1}, c_0..c_{R-1}], so
//   A9  (once)      B_ik for every event, G_kl = sum_j w_j conj(B_jk) B_jl over the normalisation points
//   A10 (per call)  A_i = sum_k c_k B_ik, sum ln|A_i|^2, I = c^H G c            -- one streaming pass, HBM bound.
// k < N:  B_k = beta_k(s12) + beta_k(s13), beta_k = cardinal natural spline of knot k (real);
// k >= N: B_k = T_r(s12,s13) + T_r(s13,s12), r = k - N, in the caller's resonance order.
//
// HBM layout of the cache: tiles of MIPWA_TILE = 256 consecutive events; inside a tile column-major,
//   cache[(tile * C + col) * 256 + e]  (double2),  C columns per event:
//   dense   (MIPWA_PATH_CACHED):          C = K,      col k = B_k                       -> 16 K bytes per event
//   compact (MIPWA_PATH_CACHED_COMPACT):  C = 1 + R,  col 0 = (s12, s13), col 1+r = B_{N+r} -> 16 + 16 R bytes per event
// so a block streams one contiguous C x 4 KiB chunk per tile and a warp reads 512 contiguous bytes per column.
// The compact form re-evaluates the spline part from the per-call segment coefficients in shared memory.
#pragma once
#include "kernels.cuh"

#define MIPWA_TILE 256
#define MIPWA_MAX_K (MIPWA_DEV_MAX_KNOTS + MIPWA_DEV_MAX_RES)

struct CoefDev {                    // the linear coefficients of one call, a __grid_constant__ kernel parameter
    int32_t K, N;
    double2 c[MIPWA_MAX_K];
};

struct BasisAux {
    const double* Mx;               // N x N row-major: y''_j = sum_k Mx[j*N + k] y_k (natural spline, knots only)
    uint8_t col_of_slot[MIPWA_DEV_MAX_RES];   // device slot d holds the caller's resonance col_of_slot[d]
    int32_t nonres_col;             // caller's index of the constant non-resonant term (its basis function is 1), -1: none
    int32_t n_res_cols;             // resonance columns of the basis (the caller's list length: m.R + the constant term)
};

// ---- NR-form local weights: S(s) = A y_j + B y_j+1 + C y''_j + D y''_j+1 -----------------------------------------
struct SplW { int j; double A, B, C, D; };

__device__ __forceinline__ SplW spline_weights(const SearchSmem& ss, double s)
{
    SplW r;
    r.j = spline_segment(ss, s);
    const double xj = ss.knots[r.j], xn = ss.knots[r.j + 1], h = xn - xj;
    r.A = (xn - s) / h;
    r.B = 1.0 - r.A;
    const double h6 = h * h / 6.0;
    r.C = (r.A * r.A * r.A - r.A) * h6;
    r.D = (r.B * r.B * r.B - r.B) * h6;
    return r;
}

__device__ __forceinline__ double cardinal_one(const double* __restrict__ Mx, int N, const SplW& a, int k)
{
    double v = fma(a.C, __ldg(Mx + (size_t)a.j * N + k), a.D * __ldg(Mx + (size_t)(a.j + 1) * N + k));
    if (k == a.j) v += a.A;
    if (k == a.j + 1) v += a.B;
    return v;
}

// Basis row of one point: emit(k, B_k) for the spline columns k = k0, k0+kstep, .. < N and the resonance slots
// d = k0, k0+kstep, .. < R.  `m` must be the UNIT-coefficient model (cre = sqrt(n_R n_D), cim = 0).
template <class Emit>
__device__ __forceinline__ void basis_point(const SearchSmem& ss, const DevModel& m, const BasisAux& aux, double s12,
                                            double s13, int k0, int kstep, bool spline_cols, Emit emit)
{
    if (spline_cols) {
        const SplW a = spline_weights(ss, s12), b = spline_weights(ss, s13);
        for (int k = k0; k < m.N; k += kstep)
            emit(k, make_double2(cardinal_one(aux.Mx, m.N, a, k) + cardinal_one(aux.Mx, m.N, b, k), 0.0));
    }
    if (m.R > 0) {
        Channel ca, cb;
        make_channels(m, s12, s13, ca, cb);
        for (int d = k0; d < m.R; d += kstep) {
            double tr, ti;
            resonance_sym<-1>(m.res[d], ca, cb, tr, ti);
            emit(m.N + aux.col_of_slot[d], make_double2(m.res[d].cre * tr, m.res[d].cre * ti));
        }
    }
    // the constant term: a column of ones in the dense basis; the compact layouts carry it in the spline tables
    // (mipwa.cu: build_model) and keep a column of zeros in its place
    if (aux.nonres_col >= 0 && k0 == 0) emit(m.N + aux.nonres_col, make_double2(spline_cols ? 1.0 : 0.0, 0.0));
}

// ---- A9: build the per-event cache -------------------------------------------------------------------------------
template <bool COMPACT>
__global__ void __launch_bounds__(MIPWA_TILE)
k_basis_build(const __grid_constant__ DevModel m, const DevSearch* __restrict__ srch, const BasisAux aux,
              const double* __restrict__ s12, const double* __restrict__ s13, long long n, double2* __restrict__ cache)
{
    __shared__ SearchSmem sm;
    load_search_smem(sm, srch);
    const int C = COMPACT ? 1 + aux.n_res_cols : m.N + aux.n_res_cols;
    const long long n_tiles = (n + MIPWA_TILE - 1) / MIPWA_TILE;
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const long long i = tile * MIPWA_TILE + threadIdx.x;
        double2* col0 = cache + (size_t)tile * C * MIPWA_TILE + threadIdx.x;
        if (i < n) {
            const double x = s12[i], y = s13[i];
            if (COMPACT) col0[0] = make_double2(x, y);
            basis_point(sm, m, aux, x, y, 0, 1, !COMPACT, [&](int k, double2 v) {
                col0[(size_t)(COMPACT ? k - m.N + 1 : k) * MIPWA_TILE] = v;
            });
        } else {
            for (int k = 0; k < C; ++k) col0[(size_t)k * MIPWA_TILE] = make_double2(0.0, 0.0);
        }
    }
}

// ---- test hook: basis rows, row-major out[i*K + k] ----------------------------------------------------------------
static __global__ void __launch_bounds__(MIPWA_TILE)
k_basis_rows(const __grid_constant__ DevModel m, const DevSearch* __restrict__ srch, const BasisAux aux,
             const double* __restrict__ s12, const double* __restrict__ s13, long long first, long long n,
             double2* __restrict__ out)
{
    __shared__ SearchSmem sm;
    load_search_smem(sm, srch);
    const int K = m.N + aux.n_res_cols;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        basis_point(sm, m, aux, s12[first + i], s13[first + i], 0, 1, true,
                    [&](int k, double2 v) { out[(size_t)i * K + k] = v; });
}

// ---- grid-wide deterministic sum: block partials, last block adds them in block order ----------------------------
// Returns true in every thread of the last block to arrive; there v[] (valid in thread 0) holds the grid totals.
// The caller's thread 0 then writes its results and resets *ticket to 0.
template <int NV>
__device__ __forceinline__ bool grid_reduce(double (&v)[NV], double* __restrict__ partials,
                                            unsigned int* __restrict__ ticket, double* red, bool* flag)
{
    block_reduce<NV>(v, red);
    asm volatile("griddepcontrol.wait;" ::: "memory");     // an overlapped launch (k_nll_compact): the previous one is done with these
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) partials[(size_t)blockIdx.x * NV + k] = v[k];
        __threadfence();
        *flag = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!*flag) return false;
    __threadfence();
    double f[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) f[k] = 0.0;
    for (int b = threadIdx.x; b < gridDim.x; b += blockDim.x) {
#pragma unroll
        for (int k = 0; k < NV; ++k) f[k] += __ldcg(&partials[(size_t)b * NV + k]);
    }
    block_reduce<NV>(f, red);
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] = f[k];
    return true;
}

// I = c^H G c = sum_kl conj(c_k) G_kl c_l (real for Hermitian G); whole block, result valid in thread 0
__device__ __forceinline__ double quadratic_form(const CoefDev& cc, const double2* __restrict__ G, double* red)
{
    const int K = cc.K;
    double acc[1] = { 0.0 };
    // c_k, c_l through the generic address of the parameter block: indexed by thread, a constant-bank read would be
    // replayed once per distinct address (dev_model.cuh: load_rows_smem)
    const double2* cg = cc.c;
    auto coef = [&](int k) {
        double2 v;
        asm volatile("ld.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(cg + k));
        return v;
    };
    for (int idx = threadIdx.x; idx < K * K; idx += blockDim.x) {
        const int k = idx / K, l = idx - k * K;
        const double2 g = G[idx], a = coef(k), b = coef(l);
        const double gr = g.x * b.x - g.y * b.y, gi = g.x * b.y + g.y * b.x;     // G_kl c_l
        acc[0] += a.x * gr + a.y * gi;                                          // Re(conj(c_k) ...)
    }
    block_reduce<1>(acc, red);
    return acc[0];
}

// streaming 16-byte load: the cache is read once per call and is far larger than L2 -> evict-first
__device__ __forceinline__ double2 ld_stream(const double2* p)
{
    double2 v;
    asm volatile("ld.global.cs.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}

// ---- A10 dense: A_i = sum_k c_k B_ik -------------------------------------------------------------------------------
// One event per thread and tile, K independent 16-byte loads per thread (unrolled by 8: >= 128 B in flight per
// thread), four FMA chains.  Events past n_ev (the padding of the last tile) contribute ln 1 = 0.
// result[0] = sum ln|A_i|^2, result[1] = c^H G c.
static __global__ void __launch_bounds__(MIPWA_TILE, 4)
k_nll_dense(const __grid_constant__ CoefDev cc, const double2* __restrict__ cache, long long n_ev,
            const double2* __restrict__ G, double* __restrict__ partials, unsigned int* __restrict__ ticket,
            double* __restrict__ result, long long tag)
{
    __shared__ double red[2 * 32];
    __shared__ bool is_last;
    const int K = cc.K;
    const long long n_tiles = (n_ev + MIPWA_TILE - 1) / MIPWA_TILE;
    LogProd lp;
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const double2* p = cache + (size_t)tile * K * MIPWA_TILE + threadIdx.x;
        double r0 = 0.0, r1 = 0.0, i0 = 0.0, i1 = 0.0;
        int k = 0;
        for (; k + 8 <= K; k += 8) {
            double2 b[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) b[u] = ld_stream(p + (size_t)(k + u) * MIPWA_TILE);
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const double2 c = cc.c[k + u];
                r0 = fma(c.x, b[u].x, r0); r1 = fma(-c.y, b[u].y, r1);
                i0 = fma(c.x, b[u].y, i0); i1 = fma(c.y, b[u].x, i1);
            }
        }
        for (; k < K; ++k) {
            const double2 b = ld_stream(p + (size_t)k * MIPWA_TILE), c = cc.c[k];
            r0 = fma(c.x, b.x, r0); r1 = fma(-c.y, b.y, r1);
            i0 = fma(c.x, b.y, i0); i1 = fma(c.y, b.x, i1);
        }
        const double re = r0 + r1, im = i0 + i1;
        lp.add_counted(tile * MIPWA_TILE + threadIdx.x < n_ev ? fma(re, re, im * im) : 1.0);
    }
    double v[1] = { lp.value() };
    if (grid_reduce<1>(v, partials, ticket, red, &is_last)) {
        const double sum_log = v[0];
        __syncthreads();
        const double integ = quadratic_form(cc, G, red);
        if (threadIdx.x == 0) {
            result[0] = sum_log;
            result[1] = integ;
            *ticket = 0;
            publish_result(result, tag);
        }
    }
}

// ---- A10 dense with REAL spline columns (SURVEY 8(d) bytes table, row "cached, real spline columns") ------------------
// The spline columns B_k = beta_k(s12) + beta_k(s13), k < N, are real: storing them as complex (BASELINE.json's layout,
// k_nll_dense) spends 8 of every 16 bytes on zeros.  Here a tile of 256 events holds N real columns followed by R complex
// ones:   MIPWA_PATH_CACHED_REAL  fp64 columns, 8 N + 16 R bytes per event, exact;
//         MIPWA_PATH_CACHED_F32   the same columns stored as fp32 (4 N + 8 R bytes per event), accumulated in fp64:
//                                 OPT-IN, outside the 1e-12 contract (each column carries a relative 6e-8 rounding).
// TS / TR: storage types of a spline / resonance column element (double, double2 or float, float2).
template <class TS, class TR> struct RealTile {
    static __host__ __device__ constexpr size_t bytes(int N, int R) { return (size_t)MIPWA_TILE * (N * sizeof(TS) + R * sizeof(TR)); }
};

template <class T> __device__ __forceinline__ T ld_stream_t(const T* p);
template <> __device__ __forceinline__ double ld_stream_t<double>(const double* p)
{
    double v; asm volatile("ld.global.cs.f64 %0, [%1];" : "=d"(v) : "l"(p)); return v;
}
template <> __device__ __forceinline__ float ld_stream_t<float>(const float* p)
{
    float v; asm volatile("ld.global.cs.f32 %0, [%1];" : "=f"(v) : "l"(p)); return v;
}
template <> __device__ __forceinline__ double2 ld_stream_t<double2>(const double2* p)
{
    double2 v; asm volatile("ld.global.cs.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p)); return v;
}
template <> __device__ __forceinline__ float2 ld_stream_t<float2>(const float2* p)
{
    float2 v; asm volatile("ld.global.cs.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p)); return v;
}

template <class TS, class TR>
__global__ void __launch_bounds__(MIPWA_TILE)
k_basis_build_real(const __grid_constant__ DevModel m, const DevSearch* __restrict__ srch, const BasisAux aux,
                   const double* __restrict__ s12, const double* __restrict__ s13, long long n,
                   unsigned char* __restrict__ cache)
{
    __shared__ SearchSmem sm;
    load_search_smem(sm, srch);
    const int N = m.N, R = aux.n_res_cols;
    const size_t tile_bytes = RealTile<TS, TR>::bytes(N, R);
    const long long n_tiles = (n + MIPWA_TILE - 1) / MIPWA_TILE;
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const long long i = tile * MIPWA_TILE + threadIdx.x;
        TS* sp = reinterpret_cast<TS*>(cache + (size_t)tile * tile_bytes) + threadIdx.x;
        TR* rs = reinterpret_cast<TR*>(cache + (size_t)tile * tile_bytes + (size_t)MIPWA_TILE * N * sizeof(TS)) + threadIdx.x;
        if (i < n) {
            basis_point(sm, m, aux, s12[i], s13[i], 0, 1, true, [&](int k, double2 v) {
                if (k < N) sp[(size_t)k * MIPWA_TILE] = (TS)v.x;
                else { TR t; t.x = v.x; t.y = v.y; rs[(size_t)(k - N) * MIPWA_TILE] = t; }
            });
        } else {
            for (int k = 0; k < N; ++k) sp[(size_t)k * MIPWA_TILE] = (TS)0;
            for (int r = 0; r < R; ++r) { TR t; t.x = 0; t.y = 0; rs[(size_t)r * MIPWA_TILE] = t; }
        }
    }
}

// One event per thread and tile; the N spline loads are unrolled by 8 (8 independent loads in flight per thread).
template <class TS, class TR>
__global__ void __launch_bounds__(MIPWA_TILE, 4)
k_nll_dense_real(const __grid_constant__ CoefDev cc, const unsigned char* __restrict__ cache, long long n_ev,
                 const double2* __restrict__ G, double* __restrict__ partials, unsigned int* __restrict__ ticket,
                 double* __restrict__ result, long long tag)
{
    __shared__ double red[2 * 32];
    __shared__ bool is_last;
    const int N = cc.N, R = cc.K - cc.N;
    const size_t tile_bytes = RealTile<TS, TR>::bytes(N, R);
    const long long n_tiles = (n_ev + MIPWA_TILE - 1) / MIPWA_TILE;
    LogProd lp;
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const TS* sp = reinterpret_cast<const TS*>(cache + (size_t)tile * tile_bytes) + threadIdx.x;
        const TR* rs = reinterpret_cast<const TR*>(cache + (size_t)tile * tile_bytes + (size_t)MIPWA_TILE * N * sizeof(TS)) + threadIdx.x;
        double r0 = 0.0, r1 = 0.0, i0 = 0.0, i1 = 0.0;
        int k = 0;
        for (; k + 8 <= N; k += 8) {
            TS b[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) b[u] = ld_stream_t<TS>(sp + (size_t)(k + u) * MIPWA_TILE);
#pragma unroll
            for (int u = 0; u < 8; u += 2) {
                const double2 c0 = cc.c[k + u], c1 = cc.c[k + u + 1];
                r0 = fma(c0.x, (double)b[u], r0); i0 = fma(c0.y, (double)b[u], i0);
                r1 = fma(c1.x, (double)b[u + 1], r1); i1 = fma(c1.y, (double)b[u + 1], i1);
            }
        }
        for (; k < N; ++k) {
            const double b = (double)ld_stream_t<TS>(sp + (size_t)k * MIPWA_TILE);
            r0 = fma(cc.c[k].x, b, r0); i0 = fma(cc.c[k].y, b, i0);
        }
        for (int r = 0; r < R; ++r) {
            const TR t = ld_stream_t<TR>(rs + (size_t)r * MIPWA_TILE);
            const double2 c = cc.c[N + r];
            r1 = fma(c.x, (double)t.x, fma(-c.y, (double)t.y, r1));
            i1 = fma(c.x, (double)t.y, fma(c.y, (double)t.x, i1));
        }
        const double re = r0 + r1, im = i0 + i1;
        lp.add_counted(tile * MIPWA_TILE + threadIdx.x < n_ev ? fma(re, re, im * im) : 1.0);
    }
    double v[1] = { lp.value() };
    if (grid_reduce<1>(v, partials, ticket, red, &is_last)) {
        const double sum_log = v[0];
        __syncthreads();
        const double integ = quadratic_form(cc, G, red);
        if (threadIdx.x == 0) {
            result[0] = sum_log;
            result[1] = integ;
            *ticket = 0;
            publish_result(result, tag);
        }
    }
}

// ---- A10 compact: A_i = S(s12_i) + S(s13_i) + sum_r c_r B_{i,N+r} ----------------------------------------------------
// Streams 16 + 16 R bytes per event; the spline part comes from the per-call segment coefficients in shared memory
// (same Horner evaluation as the recompute path).  cc.c[N + r] = c_r in the caller's resonance order.
template <int RT>      // RT >= 0: number of resonances known at compile time; -1: run-time
__global__ void __launch_bounds__(MIPWA_TILE, 4)
k_nll_compact(const __grid_constant__ DevModel m, const __grid_constant__ CoefDev cc,
              const double2* __restrict__ cache, const unsigned short* __restrict__ seg, long long n_ev,
              const double2* __restrict__ G,
              double* __restrict__ partials, unsigned int* __restrict__ ticket, double* __restrict__ result, long long tag)
{
    __shared__ RowsSmem sm;
    __shared__ double red[2 * 32];
    __shared__ bool is_last;
    asm volatile("griddepcontrol.launch_dependents;");     // mipwa_nll_batch: as k_nll_recompute (kernels.cuh); otherwise nothing
    load_rows_smem(sm, m);
    const int R = RT >= 0 ? RT : cc.K - cc.N, C = 1 + R, N = cc.N;
    const long long n_tiles = (n_ev + MIPWA_TILE - 1) / MIPWA_TILE;
    LogProd lp;
    if (RT >= 0) {
        // two tiles per iteration: all 2 (1 + R) loads are in flight before the first value is used
        constexpr int RC = RT > 0 ? RT : 1;
        for (long long tile = blockIdx.x; tile < n_tiles; tile += 2LL * gridDim.x) {
            const long long tiles[2] = { tile, tile + gridDim.x };
            double2 s[2], b[2][RC];
            unsigned int sg[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const long long tt = tiles[u] < n_tiles ? tiles[u] : tile;
                const double2* p = cache + (size_t)tt * C * MIPWA_TILE + threadIdx.x;
                s[u] = ld_stream(p);
                const long long ii = tt * MIPWA_TILE + threadIdx.x;
                sg[u] = ii < n_ev ? seg[ii] : 0u;          // padding slots hold (0, 0): any segment will do
#pragma unroll
                for (int r = 0; r < RT; ++r) b[u][r] = ld_stream(p + (size_t)(1 + r) * MIPWA_TILE);
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                double r1, i1, r2, i2, t;
                spline_eval_off(sm, s[u].x, seg_off1(sg[u]), r1, i1, t);
                spline_eval_off(sm, s[u].y, seg_off2(sg[u]), r2, i2, t);
                double re = r1 + r2, im = i1 + i2;
#pragma unroll
                for (int r = 0; r < RT; ++r) {
                    const double2 c = cc.c[N + r];
                    re = fma(c.x, b[u][r].x, fma(-c.y, b[u][r].y, re));
                    im = fma(c.x, b[u][r].y, fma(c.y, b[u][r].x, im));
                }
                const bool live = tiles[u] < n_tiles && tiles[u] * MIPWA_TILE + threadIdx.x < n_ev;
                lp.add_counted(live ? fma(re, re, im * im) : 1.0);
            }
        }
    } else {
        for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            const double2* p = cache + (size_t)tile * C * MIPWA_TILE + threadIdx.x;
            const double2 s = ld_stream(p);
            const long long ii = tile * MIPWA_TILE + threadIdx.x;
            const unsigned int sg = ii < n_ev ? seg[ii] : 0u;
            double r1, i1, r2, i2, t;
            spline_eval_off(sm, s.x, seg_off1(sg), r1, i1, t);
            spline_eval_off(sm, s.y, seg_off2(sg), r2, i2, t);
            double re = r1 + r2, im = i1 + i2;
            for (int r = 0; r < R; ++r) {
                const double2 b = ld_stream(p + (size_t)(1 + r) * MIPWA_TILE), c = cc.c[N + r];
                re = fma(c.x, b.x, fma(-c.y, b.y, re));
                im = fma(c.x, b.y, fma(c.y, b.x, im));
            }
            lp.add_counted(tile * MIPWA_TILE + threadIdx.x < n_ev ? fma(re, re, im * im) : 1.0);
        }
    }
    double v[1] = { lp.value() };
    if (grid_reduce<1>(v, partials, ticket, red, &is_last)) {
        const double sum_log = v[0];
        __syncthreads();
        const double integ = quadratic_form(cc, G, red);
        if (threadIdx.x == 0) {
            result[0] = sum_log;
            result[1] = integ;
            *ticket = 0;
            publish_result(result, tag);
        }
    }
}

// ---- A9: Gram matrix G_kl = sum_j w_j conj(B_jk) B_jl over the normalisation points -------------------------------
// The one dense contraction of the path (Hermitian rank-n update, 4 K^2 n flops), run once per set of
// normalisation points, so it is kept simple: per block, GRAM_P points at a time are expanded into a shared-memory
// tile Bs[k][p] (the basis of the normalisation points is never written to HBM); every thread owns TPT 4 x 4
// register tiles of the upper triangle and sweeps the GRAM_P points.  Block partials go to
// partial[block][K*K]; k_gram_reduce adds them in block order and mirrors the lower triangle.
#define GRAM_P 32
#define GRAM_LD (GRAM_P + 1)

// HESS = true (mipwa_nll_hessian): the same sweep over the EVENTS with the complex weight 1 / A_i^2, A_i = sum_k c_k B_ik,
// and WITHOUT the conjugate: M_kl = sum_i B_ik B_il / A_i^2, the event part of d2NLL / dc_k dc_l (complex symmetric).
template <int TPT, bool HESS>
__global__ void __launch_bounds__(MIPWA_TILE, 1)
k_gram(const __grid_constant__ DevModel m, const DevSearch* __restrict__ srch, const BasisAux aux,
       const __grid_constant__ CoefDev cc, const double* __restrict__ g12, const double* __restrict__ g13,
       const double* __restrict__ gw, long long n, double w_default, double2* __restrict__ partial)
{
    extern __shared__ double2 gram_smem[];
    __shared__ SearchSmem sm;
    __shared__ double ws[GRAM_P], wsi[GRAM_P];
    load_search_smem(sm, srch);
    const int K = m.N + aux.n_res_cols, nt = (K + 3) / 4, ntile = nt * (nt + 1) / 2, rows = 4 * nt;
    double2* Bs = gram_smem;                                       // [rows][GRAM_LD]
    for (int idx = threadIdx.x; idx < rows * GRAM_LD; idx += blockDim.x) Bs[idx] = make_double2(0.0, 0.0);

    int ta[TPT], tb[TPT];
#pragma unroll
    for (int u = 0; u < TPT; ++u) {                                // tile t -> (a, b), a <= b, row-major upper triangle
        int t = threadIdx.x + u * MIPWA_TILE, a = 0;
        if (t >= ntile) { ta[u] = -1; tb[u] = -1; continue; }
        while (t >= nt - a) { t -= nt - a; ++a; }
        ta[u] = a; tb[u] = a + t;
    }
    double2 acc[TPT][4][4];
#pragma unroll
    for (int u = 0; u < TPT; ++u)
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[u][i][j] = make_double2(0.0, 0.0);
    __syncthreads();

    const int p = threadIdx.x & 31, slice = threadIdx.x >> 5;     // phase 1: 32 points x 8 column slices
    for (long long base = (long long)blockIdx.x * GRAM_P; base < n; base += (long long)gridDim.x * GRAM_P) {
        const long long j = base + p;
        if (j < n) {
            basis_point(sm, m, aux, g12[j], g13[j], slice, MIPWA_TILE / 32, true,
                        [&](int k, double2 v) { Bs[k * GRAM_LD + p] = v; });
            if (slice == 0 && !HESS) ws[p] = gw ? gw[j] : w_default;
        } else if (slice == 0) {
            ws[p] = 0.0; wsi[p] = 0.0;                             // stale columns of an absent point get weight 0
        }
        __syncthreads();
        if (HESS) {
            if (slice == 0 && j < n) {                             // A = sum_k c_k B_k of point p, weight 1 / A^2
                double ar = 0.0, ai = 0.0;
                for (int k = 0; k < K; ++k) {
                    const double2 b = Bs[k * GRAM_LD + p], c = cc.c[k];
                    ar = fma(c.x, b.x, fma(-c.y, b.y, ar));
                    ai = fma(c.x, b.y, fma(c.y, b.x, ai));
                }
                const double qr = ar * ar - ai * ai, qi = 2.0 * ar * ai, d = 1.0 / (qr * qr + qi * qi);
                ws[p] = qr * d; wsi[p] = -qi * d;
            }
            __syncthreads();
        }
#pragma unroll
        for (int u = 0; u < TPT; ++u) {
            if (ta[u] < 0) continue;
            const double2* ra = Bs + (4 * ta[u]) * GRAM_LD;
            const double2* rb = Bs + (4 * tb[u]) * GRAM_LD;
            for (int q = 0; q < GRAM_P; ++q) {
                const double w = ws[q], wi = HESS ? wsi[q] : 0.0;
                double2 x[4], y[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    x[i] = ra[i * GRAM_LD + q];
                    const double2 t = rb[i * GRAM_LD + q];
                    if (HESS) y[i] = make_double2(fma(w, t.x, -wi * t.y), fma(w, t.y, wi * t.x));
                    else y[i] = make_double2(t.x * w, t.y * w);
                }
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int l = 0; l < 4; ++l) {                  // conj(x_i) * y_l   (HESS: x_i * y_l)
                        const double xi = HESS ? -x[i].y : x[i].y;
                        acc[u][i][l].x = fma(x[i].x, y[l].x, fma(xi, y[l].y, acc[u][i][l].x));
                        acc[u][i][l].y = fma(x[i].x, y[l].y, fma(-xi, y[l].x, acc[u][i][l].y));
                    }
            }
        }
        __syncthreads();
    }
    double2* out = partial + (size_t)blockIdx.x * K * K;
#pragma unroll
    for (int u = 0; u < TPT; ++u) {
        if (ta[u] < 0) continue;
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int l = 0; l < 4; ++l) {
                const int k = 4 * ta[u] + i, c = 4 * tb[u] + l;
                if (k < K && c < K) out[k * K + c] = acc[u][i][l];
            }
    }
}

// hermitian = 1: G (lower triangle = conjugate, real diagonal); 0: the complex symmetric M of mipwa_nll_hessian
static __global__ void k_gram_reduce(const double2* __restrict__ partial, int nblocks, int K, double2* __restrict__ G,
                                     int hermitian)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= K * K) return;
    const int k = idx / K, l = idx - k * K;
    if (k > l) return;
    double2 s = make_double2(0.0, 0.0);
    for (int b = 0; b < nblocks; ++b) {
        const double2 v = partial[(size_t)b * K * K + idx];
        s.x += v.x; s.y += v.y;
    }
    if (k == l && hermitian) s.y = 0.0;
    G[k * K + l] = s;
    G[l * K + k] = make_double2(s.x, hermitian ? -s.y : s.y);
}
