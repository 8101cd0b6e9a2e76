// mipwa.cu -- host side of libmipwa: context, per-call model preparation (A1-A3), launches, C ABI (include/mipwa.h).
// No CPU fallback: every numeric result comes from the kernels in kernels.cuh / cached.cuh / grad.cuh.
#include "../../include/mipwa.h"

#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "launch.h"
#include "kernels.cuh"
#include "cached.cuh"
#include "grad.cuh"
#include "hybrid.cuh"
#include "gen.cuh"

#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_select.cuh>

static_assert(MIPWA_DEV_MAX_KNOTS == MIPWA_MAX_KNOTS, "capacity mismatch");
static_assert(MIPWA_DEV_MAX_RES == MIPWA_MAX_RESONANCES, "capacity mismatch");
static_assert(sizeof(DevModel) < 32000, "DevModel must fit the kernel parameter space");

namespace {

struct Slot {                       // events or normalisation points
    const double* s12 = nullptr;
    const double* s13 = nullptr;
    const double* w = nullptr;
    const unsigned short* seg = nullptr;   // spline segment pair per point, j12 | j13 << 8 (always library-owned)
    const PointRec* rec = nullptr;  // 32-byte records of the recompute kernels (built on first use, library-owned)
    int64_t n = -1;                 // -1: not set
    void* owned[5] = { nullptr, nullptr, nullptr, nullptr, nullptr };   // s12, s13, w, seg, rec
};

// RAII range for profilers: shows the C-ABI entry points on an Nsight timeline; costs nothing
// when no tool is attached
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

}  // namespace

struct mipwa_ctx {
    mipwa_kinematics kin;
    // N: knots of the spline tables the kernels use (>= 2); Np: knots in the parameter vector (the caller's n_knots: 0
    // for an Isobar model, whose constant term rides on a two-knot table); R: resonance-list entries, the constant
    // non-resonant one (index nr_idx, -1: none) included; F: floating shapes
    int N = 0, Np = 0, R = 0, F = 0, nr_idx = -1;
    int n_par() const { return 2 * Np + 2 * R + 2 * F; }   // length of the parameter vector
    int pb() const { return 2 * Np; }                      // first entry of the resonance block
    std::vector<double> knots;
    std::vector<mipwa_resonance> res;
    int n_spin[3] = { 0, 0, 0 };   // resonances of spin 0, 1, 2 (the kernel signature)
    int model_flags = 0;           // MIPWA_FL_*: equal daughter masses m1 == m2; radii shared within each spin
    std::vector<int> perm;          // device slot d holds resonance perm[d]: spin 1 first, then spin 2, then spin 0
    double *parts_ev = nullptr, *parts_nm = nullptr;   // mipwa_nll_grad_parts: host outputs of the running call
    double parts_S = 0.0, parts_I = 0.0;
    int device = 0;
    int sm_count = 0;
    cudaStream_t stream = nullptr;
    cudaStream_t copy_stream = nullptr;   // host -> device uploads of mipwa_set_*, overlapped with the boundary check
    cudaEvent_t copy_done[2] = { nullptr, nullptr };
    int path = MIPWA_PATH_AUTO;

    // natural-spline system (A2): the tridiagonal matrix depends on the knots only -> factor once
    std::vector<double> sp_sub, sp_inv, sp_cp;     // sub-diagonal, 1/pivot, modified super-diagonal
    DevSearch search;               // knot search table (knots only): host copy, uploaded once to d_search
    DevSearch* d_search = nullptr;

    Slot ev, nm;

    // workspaces
    int blocks_per_sm = 0;
    double2* d_partials = nullptr;
    unsigned int* d_ticket = nullptr;
    double* h_result = nullptr;     // mapped pinned: [0] sum ln|A|^2, [1] sum w|A|^2, [2] tag of the call that wrote them
    double* d_result = nullptr;     // device alias of h_result
    long long tag = 0;              // number of value-kernel launches: what publish_result writes into slot 2
    double* result_dst = nullptr;   // where the value kernels write their totals: d_result, or d_dev_result (device mode)
    double* d_dev_result = nullptr; // device memory, 8 doubles: totals of a call that stays on the device
    bool async_result = false;      // device mode (mipwa_nll_parts_device): do not wait, do not read h_result
    double* h_batch = nullptr;      // mapped pinned, 4 doubles per slot (S, I, tag, -): totals of mipwa_nll_batch's calls
    double* d_batch = nullptr;      // device alias of h_batch
    int64_t batch_cap = 0;          // slots
    long long grad_tag = 0;         // tag of the last k_grad_finalize launch (wait_grad)
    bool overlap_launch = false;    // mipwa_nll_batch, vectors 1..: the value kernel may start while its predecessor drains
    unsigned long long* h_bad = nullptr;
    unsigned long long* d_bad = nullptr;

    DevModel model;                 // staging for the current call
    std::vector<double> y_re, y_im;          // knot values a_k e^{i phi_k} of the call (zero for the two stand-in knots)
    std::vector<double> ys_re, ys_im;        // the values the tables are built from: y_k + c_nr / 2
    std::vector<double> ypp_re, ypp_im;

    // fixed-shape path (A9, A10)
    std::vector<double> Mx;         // N x N: y'' = Mx y (knots only)
    double* d_Mx = nullptr;
    void* d_cache = nullptr;        // per-event cache in use (owned or the caller's buffer)
    void* owned_cache = nullptr;
    int64_t owned_cache_bytes = 0;
    void* user_cache = nullptr;
    int64_t user_cache_bytes = 0;
    int cache_kind = 0;             // MIPWA_PATH_CACHED / _COMPACT / _REAL / _F32, valid iff cache_valid
    bool cache_valid = false;
    double2* d_gram = nullptr;
    std::vector<double> h_gram;     // host copy (K x K complex, row-major) for the cached-path gradient
    bool gram_valid = false;
    int dense_blocks_per_sm = 0, compact_blocks_per_sm = 0;

    // hybrid path: floating resonances recomputed, fixed ones cached (events and normalisation points)
    const std::vector<int>* active = nullptr;   // resonances (caller's indices, device-slot order) build_model packs; null: perm
    std::vector<int> hyb_float, hyb_fixed;      // floating: spin 1 first, then spin 2; fixed: caller's order
    int hyb_f1 = 0, hyb_f2 = 0;
    bool hyb_ok = false;                        // a k_nll_hybrid instantiation exists for this model
    void* d_hyb_ev = nullptr; void* d_hyb_nm = nullptr;
    int64_t hyb_ev_bytes = 0, hyb_nm_bytes = 0;
    bool hyb_ev_valid = false, hyb_nm_valid = false;
    int hyb_blocks_per_sm = 0;

    // gradient (A8): cell-sorted copies of both point sets, per-block partial vectors
    Slot ev_sorted, nm_sorted;
    bool ev_sorted_valid = false, nm_sorted_valid = false;
    size_t grad_smem_set[2][3] = { { 0, 0, 0 }, { 0, 0, 0 } };   // dynamic shared memory granted to k_grad_recompute<mix, shp>
    size_t gcompact_smem_set = 0;
    double* d_gpartials = nullptr;
    size_t gpartials_len = 0;
    double2* d_f_ev = nullptr; double2* d_f_nm = nullptr;   // per-point gradient factors for k_grad_shape
    int64_t f_ev_len = 0, f_nm_len = 0;
    double res_fold[MIPWA_MAX_RESONANCES];   // sqrt(n_R n_D) of device slot d for the current call

    bool timing = false;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    float last_ms = 0.f;
    int64_t launches = 0;
    std::string err;
};

namespace {

int fail(mipwa_ctx* c, int code, const std::string& msg)
{
    if (c) c->err = msg;
    return code;
}

#define CU(ctx, call)                                                                             \
    do {                                                                                          \
        cudaError_t e__ = (call);                                                                 \
        if (e__ != cudaSuccess)                                                                   \
            return fail(ctx, e__ == cudaErrorMemoryAllocation ? MIPWA_ERR_NOMEM : MIPWA_ERR_CUDA, \
                        std::string(#call) + ": " + cudaGetErrorString(e__));                     \
    } while (0)

double lam(double a, double b, double c) { return (a - b - c) * (a - b - c) - 4.0 * b * c; }

double barrier_num(int L, double z0) { return L == 0 ? 1.0 : (L == 1 ? 1.0 + z0 : 9.0 + 3.0 * z0 + z0 * z0); }

// A3: constants of one resonance for the device formulas of dev_model.cuh
int resonance_constants(mipwa_ctx* c, int r, double m0, double g0, double cmag, double carg, ResDev* out, double* fold)
{
    const mipwa_kinematics& k = c->kin;
    const mipwa_resonance& d = c->res[r];
    if (!(m0 > k.m1 + k.m2) || !(m0 < k.m_parent - k.m3) || !(g0 > 0.0) || !std::isfinite(m0) || !std::isfinite(g0))
        return fail(c, MIPWA_ERR_ARG, "resonance " + std::to_string(r) + ": need m1+m2 < mass < M-m3 and width > 0");
    const double M2 = k.m_parent * k.m_parent, m0sq = m0 * m0;
    const double q0sq = lam(m0sq, k.m1 * k.m1, k.m2 * k.m2) / (4.0 * m0sq);
    const double p0sq = lam(M2, m0sq, k.m3 * k.m3) / (4.0 * M2);
    const int L = d.spin;
    const double nR = barrier_num(L, d.r_res * d.r_res * q0sq), nD = barrier_num(L, d.r_parent * d.r_parent * p0sq);
    out->m0sq = m0sq;
    out->cR = L ? 0.25 * d.r_res * d.r_res : 0.0;
    out->cD = L ? d.r_parent * d.r_parent / (4.0 * M2) : 0.0;
    out->Kw = 0.5 * m0sq * g0 * nR / (std::pow(4.0 * q0sq, L) * std::sqrt(q0sq));
    const double f = cmag * std::sqrt(nR * nD);
    if (fold) *fold = std::sqrt(nR * nD);
    out->cre = f * std::cos(carg);
    out->cim = f * std::sin(carg);
    out->pa = L == 2 ? 1.0 : 0.0;
    out->pb = L == 2 ? 3.0 : (L == 1 ? 1.0 : 0.0);
    out->pc = L == 2 ? 9.0 : 1.0;
    out->qR1 = 3.0 * out->cR; out->qR2 = out->cR * out->cR;
    out->qD1 = 3.0 * out->cD; out->qD2 = out->cD * out->cD;
    out->L = L;
    out->fl = -1;
    // shape derivatives: only q0^2 and p0*^2 depend on m0 (include/mipwa.h, mipwa_nll_grad_full)
    {
        const double m1s = k.m1 * k.m1, m2s = k.m2 * k.m2, m3s = k.m3 * k.m3;
        const double dq0 = 0.5 * m0 * (1.0 - (m1s - m2s) * (m1s - m2s) / (m0sq * m0sq));
        const double dp0 = m0 * (m0sq - M2 - m3s) / M2;
        auto dlog_num = [L](double z0) { return L == 0 ? 0.0 : (L == 1 ? 1.0 / (1.0 + z0) : (3.0 + 2.0 * z0) / (9.0 + 3.0 * z0 + z0 * z0)); };
        const double rr = d.r_res * d.r_res, rp = d.r_parent * d.r_parent;
        const double dlnFR = 0.5 * dlog_num(rr * q0sq) * rr * dq0, dlnFD = 0.5 * dlog_num(rp * p0sq) * rp * dp0;
        out->sh_a1 = dlnFR + dlnFD;
        out->sh_a2 = 2.0 / m0 - (L + 0.5) * dq0 / q0sq + 2.0 * dlnFR;
        out->sh_2m0 = 2.0 * m0;
        out->sh_ig0 = 1.0 / g0;
    }
    return MIPWA_OK;
}

// A2: second derivatives of the natural spline through (x_k, y_k) with the pre-factored tridiagonal system
void spline_solve(const mipwa_ctx* c, const double* y, double* ypp)
{
    const int n = c->N;
    const double* x = c->knots.data();
    for (int i = 0; i < n; ++i) ypp[i] = 0.0;
    const int m = n - 2;
    if (m < 1) return;
    std::vector<double> d(m);
    for (int i = 0; i < m; ++i) {
        const double rhs = (y[i + 2] - y[i + 1]) / (x[i + 2] - x[i + 1]) - (y[i + 1] - y[i]) / (x[i + 1] - x[i]);
        d[i] = (i == 0 ? rhs : rhs - c->sp_sub[i] * d[i - 1]) * c->sp_inv[i];
    }
    ypp[m] = d[m - 1];
    for (int i = m - 2; i >= 0; --i) ypp[i + 1] = d[i] - c->sp_cp[i] * ypp[i + 2];
}

void spline_factor(mipwa_ctx* c)
{
    const int n = c->N, m = n - 2;
    const double* x = c->knots.data();
    c->sp_sub.assign(std::max(m, 0), 0.0); c->sp_inv.assign(std::max(m, 0), 0.0); c->sp_cp.assign(std::max(m, 0), 0.0);
    for (int i = 0; i < m; ++i) {
        const double sub = (x[i + 1] - x[i]) / 6.0, dia = (x[i + 2] - x[i]) / 3.0, sup = (x[i + 2] - x[i + 1]) / 6.0;
        const double piv = i == 0 ? dia : dia - sub * c->sp_cp[i - 1];
        c->sp_sub[i] = sub;
        c->sp_inv[i] = 1.0 / piv;
        c->sp_cp[i] = sup / piv;
    }
    // bucket table for the segment lookup: lut[b] = segment containing the left edge of bucket b, xk[b] = the
    // interior knot inside bucket b.  Buckets no wider than 0.9 x the smallest knot spacing hold at most one knot.
    DevSearch& t = c->search;
    std::memset(&t, 0, sizeof(t));
    double minsp = x[1] - x[0];
    for (int i = 1; i < n - 1; ++i) minsp = std::min(minsp, x[i + 1] - x[i]);
    const double range = x[n - 1] - x[0];
    const double want = std::ceil(range / (0.9 * minsp));
    t.N = n;
    t.nlut = (int)std::min<double>(MIPWA_DEV_LUT, std::max<double>(64.0, want));
    t.lut_exact = range / t.nlut <= 0.9 * minsp ? 1 : 0;
    t.lut_inv = t.nlut / range;
    t.lut_off = -x[0] * t.lut_inv;
    for (int i = 0; i < n; ++i) t.knots[i] = x[i];
    for (int b = 0; b < t.nlut; ++b) {
        const double lo = x[0] + b / t.lut_inv, hi = x[0] + (b + 1) / t.lut_inv;
        int j = 0;
        while (j < n - 2 && lo >= x[j + 1]) ++j;
        t.lut[b] = (uint8_t)j;
        t.xk[b] = (j + 1 <= n - 2 && x[j + 1] < hi) ? x[j + 1] : HUGE_VAL;
    }
}

// the parameter-independent part of DevModel (kinematics, knot positions of the rows)
void fill_static_model(mipwa_ctx* c)
{
    DevModel& m = c->model;
    const mipwa_kinematics& k = c->kin;
    m.N = c->N; m.R = c->R;
    m.t_lo = (k.m1 + k.m2) * (k.m1 + k.m2);
    m.t_d = (k.m1 - k.m2) * (k.m1 - k.m2);
    m.s_hi = (k.m_parent - k.m3) * (k.m_parent - k.m3);
    m.s_top = (k.m_parent + k.m3) * (k.m_parent + k.m3);
    m.sigma = k.m_parent * k.m_parent + k.m1 * k.m1 + k.m2 * k.m2 + k.m3 * k.m3;
    m.kappa = (k.m_parent * k.m_parent - k.m3 * k.m3) * (k.m2 * k.m2 - k.m1 * k.m1);
    m.k_third = -1.0 / 3.0;
    m.lam2_b = -(m.s_hi + m.s_top); m.lam2_c = m.s_hi * m.s_top;
    for (int i = 0; i < c->N; ++i) m.rows[i * MIPWA_ROW] = make_double2(c->knots[i], 0.0);
}

// A1-A3: parameters -> DevModel
int build_model(mipwa_ctx* c, const double* p, int64_t n_params)
{
    const int N = c->N, Np = c->Np, R = c->R, pb = c->pb();
    if (n_params != c->n_par()) return fail(c, MIPWA_ERR_ARG, "n_params must be " + std::to_string(c->n_par()));
    for (int64_t i = 0; i < n_params; ++i)
        if (!std::isfinite(p[i])) return fail(c, MIPWA_ERR_ARG, "non-finite parameter " + std::to_string(i));
    DevModel& m = c->model;
    for (int i = 0; i < Np; ++i) {
        c->y_re[i] = p[i] * std::cos(p[Np + i]);           // y_k = a_k e^{i phi_k}
        c->y_im[i] = p[i] * std::sin(p[Np + i]);
    }
    // The constant non-resonant term c_nr rides on the spline tables: the natural spline through
    // y_k + c_nr / 2 is S + c_nr / 2 (constant data have no curvature), and the two channels add up to S(s12) + S(s13)
    // + c_nr.  No kernel knows about it; the gradient of c_nr is half the sum of the knot gradients (polar_chain).
    double off_re = 0.0, off_im = 0.0;
    if (c->nr_idx >= 0) {
        off_re = 0.5 * p[pb + 2 * c->nr_idx] * std::cos(p[pb + 2 * c->nr_idx + 1]);
        off_im = 0.5 * p[pb + 2 * c->nr_idx] * std::sin(p[pb + 2 * c->nr_idx + 1]);
    }
    for (int i = 0; i < N; ++i) { c->ys_re[i] = c->y_re[i] + off_re; c->ys_im[i] = c->y_im[i] + off_im; }
    spline_solve(c, c->ys_re.data(), c->ypp_re.data());
    spline_solve(c, c->ys_im.data(), c->ypp_im.data());
    for (int j = 0; j < N - 1; ++j) {                       // cubic in t = s - x_j on segment j
        const double h = c->knots[j + 1] - c->knots[j];
        const double* Y[2] = { c->ys_re.data(), c->ys_im.data() };
        const double* P[2] = { c->ypp_re.data(), c->ypp_im.data() };
        double co[4][2];
        for (int q = 0; q < 2; ++q) {
            co[0][q] = Y[q][j];
            co[1][q] = (Y[q][j + 1] - Y[q][j]) / h - h * (2.0 * P[q][j] + P[q][j + 1]) / 6.0;
            co[2][q] = 0.5 * P[q][j];
            co[3][q] = (P[q][j + 1] - P[q][j]) / (6.0 * h);
        }
        for (int q = 0; q < 4; ++q) m.rows[j * MIPWA_ROW + 1 + q] = make_double2(co[q][0], co[q][1]);
    }
    for (int q = 0; q < 4; ++q) m.rows[(N - 1) * MIPWA_ROW + 1 + q] = make_double2(0.0, 0.0);
    std::vector<int> fidx(R, -1);
    for (int r = 0, f = 0; r < R; ++r) if (c->res[r].shape_floats) fidx[r] = f++;
    const std::vector<int>& slots = c->active ? *c->active : c->perm;
    m.R = (int)slots.size();
    for (int d = 0; d < (int)slots.size(); ++d) {
        const int r = slots[d];
        double m0 = c->res[r].mass, g0 = c->res[r].width;
        if (fidx[r] >= 0) { m0 = p[pb + 2 * R + 2 * fidx[r]]; g0 = p[pb + 2 * R + 2 * fidx[r] + 1]; }
        const int rc = resonance_constants(c, r, m0, g0, p[pb + 2 * r], p[pb + 2 * r + 1], &m.res[d], &c->res_fold[d]);
        if (rc) return rc;
        m.res[d].fl = fidx[r];
    }
    return MIPWA_OK;
}

int use_device(mipwa_ctx* c)
{
    CU(c, cudaSetDevice(c->device));
    (void)cudaGetLastError();                              // a stale error of an earlier, unchecked call is not ours to report
    return MIPWA_OK;
}

int grid_for(const mipwa_ctx* c, int64_t n, int blocks_per_sm)
{
    const int64_t full = (int64_t)c->sm_count * blocks_per_sm;
    const int64_t need = (n + MIPWA_BLOCK - 1) / MIPWA_BLOCK;
    return (int)std::max<int64_t>(1, std::min(full, need));
}

void free_slot(Slot& s)
{
    for (void*& p : s.owned) { if (p) cudaFree(p); p = nullptr; }
    s = Slot();
}

void drop_records(Slot& s)
{
    if (s.owned[4]) cudaFree(s.owned[4]);
    s.owned[4] = nullptr; s.rec = nullptr;
}

// records past the end of a point set that the prefetching loops may LOAD (never evaluate), in records
int64_t record_pad(const mipwa_ctx* c) { return (int64_t)c->sm_count * 2048; }

// The 32-byte records of a point set (kernels.cuh: k_make_records), built on first use.  w_default: the weight of a
// normalisation point without weights (1: the caller of the kernel divides by n), 0 for events without background
// densities.  The tail [n, n + pad) holds copies of record 0 with weight 0 (zeros if the set is empty).
int ensure_records(mipwa_ctx* c, Slot& s, double w_default)
{
    if (s.rec) return MIPWA_OK;
    const int64_t pad = record_pad(c), n = std::max<int64_t>(s.n, 0);
    if (!s.owned[4]) CU(c, cudaMalloc(&s.owned[4], (size_t)(n + pad) * sizeof(PointRec)));
    PointRec* rec = (PointRec*)s.owned[4];
    CU(c, cudaMemsetAsync(rec + n, 0, (size_t)pad * sizeof(PointRec), c->stream));
    if (n > 0) {
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)c->sm_count * 8, (n + MIPWA_BLOCK - 1) / MIPWA_BLOCK));
        k_make_records<<<grid, MIPWA_BLOCK, 0, c->stream>>>(s.s12, s.s13, s.w, w_default, s.seg, n, rec);
        ++c->launches;
        CU(c, cudaGetLastError());
        k_pad_records<<<(int)std::min<int64_t>(c->sm_count, (pad + MIPWA_BLOCK - 1) / MIPWA_BLOCK), MIPWA_BLOCK, 0, c->stream>>>(rec, n, pad);
        ++c->launches;
        CU(c, cudaGetLastError());
    }
    s.rec = rec;
    return MIPWA_OK;
}

}  // namespace


// the library's working view of a point set: the cell-sorted copy once mipwa_prepare / mipwa_nll_grad built it
static inline Slot& evs(mipwa_ctx* c) { return c->ev_sorted_valid ? c->ev_sorted : c->ev; }
static inline Slot& nms(mipwa_ctx* c) { return c->nm_sorted_valid ? c->nm_sorted : c->nm; }

// tag of the next value-kernel launch; clears the word the kernel will publish it in (a gradient call may have left
// anything there)
static long long next_tag(mipwa_ctx* c)
{
    *reinterpret_cast<volatile long long*>(c->h_result + MIPWA_RESULT_TAG) = 0;
    return ++c->tag;
}

// k_grad_finalize right behind the kernel that writes the block partials, launched with programmatic stream serialisation:
// its launch latency runs under the producer's tail (the kernel itself waits in griddepcontrol.wait, grad.cuh)
#define MIPWA_GRAD_TAG_SLOT 4095                           // h_result word the gradient's tag goes to (the vectors end below 4030)
static cudaError_t launch_finalize(mipwa_ctx* c, int blocks, const double* partials, int split, int nblocks, int NV, int sets,
                                   double* result)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks); cfg.blockDim = dim3(256); cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    // the tag of this call behind the values: d_ticket + 1 is the finalize kernel's own counter
    *reinterpret_cast<volatile long long*>(c->h_result + MIPWA_GRAD_TAG_SLOT) = 0;
    c->grad_tag = ++c->tag;
    return cudaLaunchKernelEx(&cfg, k_grad_finalize, partials, split, nblocks, NV, sets, result, c->d_ticket + 1,
                              c->d_result + MIPWA_GRAD_TAG_SLOT, c->grad_tag);
}

// wait for the gradient sums of the call launch_finalize just enqueued (polls the tag, then falls back to the stream)
static int wait_grad(mipwa_ctx* c)
{
    if (c->timing) {
        CU(c, cudaEventRecord(c->ev1, c->stream));
        CU(c, cudaEventSynchronize(c->ev1));
        CU(c, cudaEventElapsedTime(&c->last_ms, c->ev0, c->ev1));
        return MIPWA_OK;
    }
    volatile long long* flag = reinterpret_cast<volatile long long*>(c->h_result + MIPWA_GRAD_TAG_SLOT);
    for (int spin = 0; spin < 400000; ++spin) {
        if (*flag == c->grad_tag) return MIPWA_OK;
        if ((spin & 0x3fff) == 0x3fff) {
            const cudaError_t e = cudaStreamQuery(c->stream);
            if (e != cudaSuccess && e != cudaErrorNotReady) return fail(c, MIPWA_ERR_CUDA, cudaGetErrorString(e));
        }
    }
    CU(c, cudaStreamSynchronize(c->stream));
    return MIPWA_OK;
}

// start of the timed region of a call (timing mode only): spacer kernel, then the first event (kernels.cuh: k_spacer)
static int timing_begin(mipwa_ctx* c)
{
    if (!c->timing) return MIPWA_OK;
    k_spacer<<<1, 1, 0, c->stream>>>(40000ULL);
    CU(c, cudaGetLastError());
    CU(c, cudaEventRecord(c->ev0, c->stream));
    return MIPWA_OK;
}

// Wait for the value kernel that carries `tag`: its last block writes the totals into mapped pinned memory and then the
// tag (publish_result).  Polling that word for a while before blocking saves the wake-up latency of
// cudaStreamSynchronize, which at the paper's sample sizes (1e4-1e5 events) is as long as the kernel itself.
static int wait_result(mipwa_ctx* c, long long tag)
{
    if (c->async_result) return MIPWA_OK;                  // device mode: the totals stay on the device
    if (c->timing) {
        CU(c, cudaEventRecord(c->ev1, c->stream));
        CU(c, cudaEventSynchronize(c->ev1));
        CU(c, cudaEventElapsedTime(&c->last_ms, c->ev0, c->ev1));
        return MIPWA_OK;
    }
    volatile long long* flag = reinterpret_cast<volatile long long*>(c->h_result + MIPWA_RESULT_TAG);
    for (int spin = 0; spin < 200000; ++spin) {
        if (*flag == tag) return MIPWA_OK;
        if ((spin & 0x3fff) == 0x3fff) {                   // a faulted kernel never publishes: ask the driver now and then
            const cudaError_t e = cudaStreamQuery(c->stream);
            if (e != cudaSuccess && e != cudaErrorNotReady) return fail(c, MIPWA_ERR_CUDA, cudaGetErrorString(e));
        }
    }
    CU(c, cudaStreamSynchronize(c->stream));
    return MIPWA_OK;
}

// sustained rate of one of the k_fp64_peak loops (kernels.cuh), best launch over about `seconds` seconds
template <int MODE>
static int fp64_rate(const cudaDeviceProp& prop, double seconds, double* tflops)
{
    double* d = nullptr;
    cudaEvent_t a, b;
    if (cudaMalloc(&d, 64) != cudaSuccess || cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return MIPWA_ERR_CUDA;
    const int grid = prop.multiProcessorCount * 8, block = 256;
    long long iters = 2000;
    double best = 0, spent = 0;
    for (int rep = 0; rep < 64 && spent < seconds; ++rep) {
        cudaEventRecord(a);
        k_fp64_peak<MODE><<<grid, block>>>(d, iters, MODE == 0 ? 0.999999 : 0x1p-60, 1e-9);
        cudaEventRecord(b);
        if (cudaEventSynchronize(b) != cudaSuccess) { cudaFree(d); return MIPWA_ERR_CUDA; }
        float ms = 0;
        cudaEventElapsedTime(&ms, a, b);
        const double fl = 2.0 * 64.0 * (double)iters * grid * block;   // 64 DFMAs per thread and iteration
        if (rep > 0) { best = std::max(best, fl / (ms * 1e-3) * 1e-12); spent += ms * 1e-3; }
        if (ms < 50.0f) iters *= 2;                        // grow each launch to ~0.1 s
    }
    cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(d);
    *tflops = best;
    return MIPWA_OK;
}

// =================================================================================================================
// C ABI
// =================================================================================================================
extern "C" {

const char* mipwa_version(void) { return "mipwa-b200 0.1 (sm_100a)"; }

const char* mipwa_last_error(const mipwa_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int mipwa_create(const mipwa_kinematics* kin, const double* knots, int32_t n_knots, const mipwa_resonance* res,
                 int32_t n_res, int32_t device, mipwa_ctx** out)
{
    if (!out) return MIPWA_ERR_ARG;
    *out = nullptr;
    if (!kin || (n_knots > 0 && !knots) || n_knots < 0 || n_knots == 1 || n_knots > MIPWA_MAX_KNOTS || n_res < 0 ||
        n_res > MIPWA_MAX_RESONANCES || (n_res > 0 && !res) || n_knots + n_res == 0)
        return MIPWA_ERR_ARG;
    if (!(kin->m1 > 0 && kin->m2 > 0 && kin->m3 > 0) || kin->m2 != kin->m3 || !(kin->m_parent > kin->m1 + kin->m2 + kin->m3))
        return MIPWA_ERR_ARG;
    for (int i = 0; i < n_knots; ++i)
        if (!std::isfinite(knots[i]) || (i > 0 && !(knots[i] > knots[i - 1]))) return MIPWA_ERR_ARG;
    int nr_idx = -1;
    for (int r = 0; r < n_res; ++r) {
        if (res[r].spin == MIPWA_SPIN_NONRES) {            // the constant term: one at most, nothing to float
            if (nr_idx >= 0 || res[r].shape_floats) return MIPWA_ERR_ARG;
            nr_idx = r;
            continue;
        }
        if (res[r].spin < 0 || res[r].spin > 2 || !(res[r].r_res >= 0) || !(res[r].r_parent >= 0) ||
            !(res[r].mass > kin->m1 + kin->m2) || !(res[r].mass < kin->m_parent - kin->m3) || !(res[r].width > 0))
            return MIPWA_ERR_ARG;
    }

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return MIPWA_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return MIPWA_ERR_CUDA;
    if (prop.major != 10) return MIPWA_ERR_CUDA;          // built for sm_100a only
    if (cudaSetDevice(device) != cudaSuccess) return MIPWA_ERR_CUDA;

    mipwa_ctx* c = new (std::nothrow) mipwa_ctx();
    if (!c) return MIPWA_ERR_NOMEM;
    c->kin = *kin;
    c->Np = n_knots; c->R = n_res; c->nr_idx = nr_idx;
    if (n_knots >= 2) {
        c->N = n_knots;
        c->knots.assign(knots, knots + n_knots);
    } else {                                               // no spline S-wave: a two-knot table carries the constant term
        c->N = 2;
        c->knots = { (kin->m1 + kin->m2) * (kin->m1 + kin->m2), (kin->m_parent - kin->m3) * (kin->m_parent - kin->m3) };
    }
    n_knots = c->N;
    if (n_res) c->res.assign(res, res + n_res);
    for (int r = 0; r < n_res; ++r) c->F += res[r].shape_floats ? 1 : 0;
    // device slots: spin 1, then spin 2, then spin 0; within a spin the floating resonances first (k_grad_recompute
    // folds the shape derivatives of the FIRST slot of a spin into its pass), then the caller's order
    for (int L : { 1, 2, 0 })
        for (int fl : { 1, 0 })
            for (int r = 0; r < n_res; ++r)
                if (res[r].spin == L && (res[r].shape_floats ? 1 : 0) == fl) { c->perm.push_back(r); ++c->n_spin[L]; }
    for (int L : { 1, 2 })
        for (int r = 0; r < n_res; ++r)
            if (res[r].shape_floats && res[r].spin == L) { c->hyb_float.push_back(r); (L == 1 ? c->hyb_f1 : c->hyb_f2)++; }
    for (int r = 0; r < n_res; ++r) if (!res[r].shape_floats && res[r].spin >= 0) c->hyb_fixed.push_back(r);
    {
        bool supported = (int)c->hyb_float.size() == c->F && c->F > 0 && !c->hyb_fixed.empty();   // no floating spin 0
        if (supported) supported = mipwa_hybrid_supported(c->hyb_f1, c->hyb_f2, (int)c->hyb_fixed.size());
        c->hyb_ok = supported;
    }
    if (kin->m1 == kin->m2) c->model_flags |= MIPWA_FL_EQM;
    {
        bool shared = true;
        for (int a = 0; a < n_res; ++a)
            for (int b = a + 1; b < n_res; ++b)
                if (res[a].spin >= 0 && res[a].spin == res[b].spin &&
                    (res[a].r_res != res[b].r_res || res[a].r_parent != res[b].r_parent))
                    shared = false;
        if (shared) c->model_flags |= MIPWA_FL_SHR;
    }
    c->device = device;
    c->sm_count = prop.multiProcessorCount;
    c->y_re.assign(n_knots, 0.0); c->y_im.assign(n_knots, 0.0); c->ys_re.resize(n_knots); c->ys_im.resize(n_knots);
    c->ypp_re.resize(n_knots); c->ypp_im.resize(n_knots);
    spline_factor(c);
    std::memset(&c->model, 0, sizeof(DevModel));
    fill_static_model(c);
    c->Mx.assign((size_t)n_knots * n_knots, 0.0);          // column k = second derivatives of the cardinal spline k
    {
        std::vector<double> e(n_knots), pp(n_knots);
        for (int k = 0; k < n_knots; ++k) {
            for (int j = 0; j < n_knots; ++j) e[j] = j == k ? 1.0 : 0.0;
            spline_solve(c, e.data(), pp.data());
            for (int j = 0; j < n_knots; ++j) c->Mx[(size_t)j * n_knots + k] = pp[j];
        }
    }

    bool ok = true;
    c->blocks_per_sm = 1;                                  // k_nll_recompute: one 512-thread block per SM
    const size_t max_grid = (size_t)c->sm_count * 16;
    ok = ok && cudaMalloc(&c->d_partials, max_grid * sizeof(double2) * 64) == cudaSuccess;
    ok = ok && cudaMalloc(&c->d_ticket, 64) == cudaSuccess && cudaMemset(c->d_ticket, 0, 64) == cudaSuccess;
    ok = ok && cudaHostAlloc(&c->h_result, 4096 * sizeof(double), cudaHostAllocMapped) == cudaSuccess;
    ok = ok && cudaHostGetDevicePointer(&c->d_result, c->h_result, 0) == cudaSuccess;
    if (ok) std::memset(c->h_result, 0, 4096 * sizeof(double));   // recycled pinned memory: no stale tag of an older context
    c->result_dst = c->d_result;
    ok = ok && cudaMalloc(&c->d_dev_result, 64) == cudaSuccess;
    ok = ok && cudaHostAlloc(&c->h_bad, 64, cudaHostAllocMapped) == cudaSuccess;
    ok = ok && cudaHostGetDevicePointer(&c->d_bad, c->h_bad, 0) == cudaSuccess;
    ok = ok && cudaEventCreate(&c->ev0) == cudaSuccess && cudaEventCreate(&c->ev1) == cudaSuccess;
    ok = ok && cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&c->copy_done[0], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&c->copy_done[1], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaMalloc(&c->d_Mx, c->Mx.size() * sizeof(double)) == cudaSuccess &&
         cudaMemcpy(c->d_Mx, c->Mx.data(), c->Mx.size() * sizeof(double), cudaMemcpyHostToDevice) == cudaSuccess;
    ok = ok && cudaMalloc(&c->d_gram, (size_t)(n_knots + n_res) * (n_knots + n_res) * sizeof(double2)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->d_search, sizeof(DevSearch)) == cudaSuccess &&
         cudaMemcpy(c->d_search, &c->search, sizeof(DevSearch), cudaMemcpyHostToDevice) == cudaSuccess;
    if (!ok) { mipwa_destroy(c); return MIPWA_ERR_CUDA; }
    *out = c;
    return MIPWA_OK;
}

void mipwa_destroy(mipwa_ctx* c)
{
    if (!c) return;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    free_slot(c->ev); free_slot(c->nm);
    if (c->d_partials) cudaFree(c->d_partials);
    if (c->d_ticket) cudaFree(c->d_ticket);
    if (c->d_Mx) cudaFree(c->d_Mx);
    if (c->d_search) cudaFree(c->d_search);
    if (c->d_dev_result) cudaFree(c->d_dev_result);
    if (c->owned_cache) cudaFree(c->owned_cache);
    if (c->d_gram) cudaFree(c->d_gram);
    if (c->d_gpartials) cudaFree(c->d_gpartials);
    if (c->d_f_ev) cudaFree(c->d_f_ev);
    if (c->d_f_nm) cudaFree(c->d_f_nm);
    if (c->d_hyb_ev) cudaFree(c->d_hyb_ev);
    if (c->d_hyb_nm) cudaFree(c->d_hyb_nm);
    free_slot(c->ev_sorted); free_slot(c->nm_sorted);
    if (c->h_result) cudaFreeHost(c->h_result);
    if (c->h_batch) cudaFreeHost(c->h_batch);
    if (c->h_bad) cudaFreeHost(c->h_bad);
    if (c->copy_stream) { cudaStreamSynchronize(c->copy_stream); cudaStreamDestroy(c->copy_stream); }
    for (cudaEvent_t e : c->copy_done) if (e) cudaEventDestroy(e);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    delete c;
}

int mipwa_set_stream(mipwa_ctx* c, void* s)
{
    if (!c) return MIPWA_ERR_ARG;
    c->stream = (cudaStream_t)s;
    return MIPWA_OK;
}

int mipwa_enable_timing(mipwa_ctx* c, int32_t on)
{
    if (!c) return MIPWA_ERR_ARG;
    c->timing = on != 0;
    return MIPWA_OK;
}

static int set_slot(mipwa_ctx* c, Slot& slot, const double* s12, const double* s13, const double* w, int64_t n,
                    int32_t mem, bool allow_empty)
{
    if (!c) return MIPWA_ERR_ARG;
    if (n < (allow_empty ? 0 : 1) || (n > 0 && (!s12 || !s13)) || (mem != MIPWA_MEM_HOST && mem != MIPWA_MEM_DEVICE))
        return fail(c, MIPWA_ERR_ARG, "bad pointer, count or mem flag");
    int rc = use_device(c);
    if (rc) return rc;
    CU(c, cudaStreamSynchronize(c->stream));
    Slot s;
    if (n > 0 && slot.n == n) {                            // same size as before: reuse the library-owned storage
        if (mem == MIPWA_MEM_HOST && slot.owned[0] && slot.owned[1]) {
            for (int q = 0; q < 3; ++q) { s.owned[q] = slot.owned[q]; slot.owned[q] = nullptr; }
            if (!w && s.owned[2]) { cudaFree(s.owned[2]); s.owned[2] = nullptr; }
        }
        s.owned[3] = slot.owned[3]; slot.owned[3] = nullptr;                                    // segment pairs
        s.owned[4] = slot.owned[4]; slot.owned[4] = nullptr;                                    // records (rebuilt on use)
    }
    free_slot(slot);
    if (mem == MIPWA_MEM_HOST && n > 0) {
        const double* src[3] = { s12, s13, w };
        for (int q = 0; q < 3; ++q) {
            if (!src[q] || s.owned[q]) continue;
            const cudaError_t e = cudaMalloc(&s.owned[q], (size_t)n * sizeof(double));
            if (e != cudaSuccess) {
                free_slot(s);
                return fail(c, e == cudaErrorMemoryAllocation ? MIPWA_ERR_NOMEM : MIPWA_ERR_CUDA, cudaGetErrorString(e));
            }
        }
        s.s12 = (const double*)s.owned[0]; s.s13 = (const double*)s.owned[1]; s.w = (const double*)s.owned[2];
    } else {
        s.s12 = s12; s.s13 = s13; s.w = w;
    }
    s.n = n;
    if (n > 0 && !s.owned[3]) {
        cudaError_t e = cudaMalloc(&s.owned[3], (size_t)n * sizeof(unsigned short));
        if (e != cudaSuccess) {
            free_slot(s);
            return fail(c, e == cudaErrorMemoryAllocation ? MIPWA_ERR_NOMEM : MIPWA_ERR_CUDA, cudaGetErrorString(e));
        }
    }
    s.seg = (const unsigned short*)s.owned[3];
    if (n > 0) {
        // Boundary check on the device (north_star invariant), which also stores the segment pairs and - when the slot
        // keeps record storage from an earlier set of the same size (a caller that re-sends its sample every step) -
        // the 32-byte records, so that the likelihood call that follows finds everything in place.
        // Host arrays go up in chunks on a second stream: chunk k + 1 is on the bus while chunk k is checked.
        const mipwa_kinematics& k = c->kin;
        DevKin dk = { k.m_parent * k.m_parent, k.m1 * k.m1, k.m2 * k.m2, k.m3 * k.m3,
                      (k.m1 + k.m2) * (k.m1 + k.m2), (k.m1 - k.m2) * (k.m1 - k.m2),
                      (k.m_parent - k.m3) * (k.m_parent - k.m3), (k.m_parent + k.m3) * (k.m_parent + k.m3) };
        *c->h_bad = 0;
        PointRec* rec = (PointRec*)s.owned[4];             // may be null: records are then built on first use
        const double w_default = allow_empty ? 0.0 : 1.0;  // events carry no weight, unweighted normalisation points 1
        const bool host = mem == MIPWA_MEM_HOST;
        const int64_t chunk = host ? (int64_t)1 << 21 : n; // 16 MB per array and chunk
        cudaError_t e = cudaSuccess;
        int slot_ev = 0;
        for (int64_t lo = 0; lo < n && e == cudaSuccess; lo += chunk) {
            const int64_t len = std::min(chunk, n - lo);
            if (host) {
                const double* src[3] = { s12, s13, w };
                for (int q = 0; q < 3 && e == cudaSuccess; ++q)
                    if (src[q])
                        e = cudaMemcpyAsync((double*)s.owned[q] + lo, src[q] + lo, (size_t)len * sizeof(double),
                                            cudaMemcpyHostToDevice, c->copy_stream);
                if (e == cudaSuccess) e = cudaEventRecord(c->copy_done[slot_ev], c->copy_stream);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(c->stream, c->copy_done[slot_ev], 0);
                slot_ev ^= 1;
            }
            if (e != cudaSuccess) break;
            k_validate<<<grid_for(c, len, 8), MIPWA_BLOCK, 0, c->stream>>>(dk, c->d_search, s.s12 + lo, s.s13 + lo,
                                                                       s.w ? s.w + lo : nullptr, w_default, len,
                                                                       (unsigned short*)s.owned[3] + lo,
                                                                       rec ? rec + lo : nullptr, c->d_bad);
            ++c->launches;
            e = cudaGetLastError();
        }
        if (e == cudaSuccess && rec) {
            const int64_t pad = record_pad(c);
            k_pad_records<<<(int)std::min<int64_t>(c->sm_count, (pad + MIPWA_BLOCK - 1) / MIPWA_BLOCK), MIPWA_BLOCK, 0, c->stream>>>(rec, n, pad);
            ++c->launches;
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) { cudaStreamSynchronize(c->copy_stream); free_slot(s); return fail(c, MIPWA_ERR_CUDA, cudaGetErrorString(e)); }
        if (*c->h_bad) {
            const unsigned long long nb = *c->h_bad;
            free_slot(s);
            return fail(c, MIPWA_ERR_DOMAIN, std::to_string(nb) + " point(s) outside the Dalitz boundary");
        }
        s.rec = rec;
    }
    slot = s;
    return MIPWA_OK;
}

int mipwa_set_events(mipwa_ctx* c, const double* s12, const double* s13, int64_t n, int32_t mem)
{
    if (!c) return MIPWA_ERR_ARG;
    NvtxRange range("mipwa_set_events");
    c->cache_valid = false; c->ev_sorted_valid = false; c->hyb_ev_valid = false;
    return set_slot(c, c->ev, s12, s13, nullptr, n, mem, true);
}

int mipwa_set_norm_points(mipwa_ctx* c, const double* s12, const double* s13, const double* w, int64_t n, int32_t mem)
{
    if (!c) return MIPWA_ERR_ARG;
    NvtxRange range("mipwa_set_norm_points");
    c->gram_valid = false; c->nm_sorted_valid = false; c->hyb_nm_valid = false;
    return set_slot(c, c->nm, s12, s13, w, n, mem, false);
}

int mipwa_n_params(const mipwa_ctx* c, int64_t* n)
{
    if (!c || !n) return MIPWA_ERR_ARG;
    *n = c->n_par();
    return MIPWA_OK;
}

int mipwa_set_path(mipwa_ctx* c, int32_t path)
{
    if (!c) return MIPWA_ERR_ARG;
    if (path < MIPWA_PATH_AUTO || path > MIPWA_PATH_CACHED_F32) return fail(c, MIPWA_ERR_ARG, "unknown path");
    if (path == MIPWA_PATH_HYBRID && !c->hyb_ok)
        return fail(c, MIPWA_ERR_STATE, "the hybrid path needs 1-2 floating spin-1/2 resonances and 1-5 fixed ones");
    if ((path == MIPWA_PATH_CACHED || path == MIPWA_PATH_CACHED_COMPACT || path == MIPWA_PATH_CACHED_REAL ||
         path == MIPWA_PATH_CACHED_F32) && c->F > 0)
        return fail(c, MIPWA_ERR_STATE, "cached paths need fixed resonance shapes");
    c->path = path;
    return MIPWA_OK;
}

// grid of the recompute kernels: one 512-thread block per SM, fewer for small samples
static int recompute_grid(const mipwa_ctx* c, int64_t n)
{
    const int64_t need = (n + MIPWA_REC_BLOCK - 1) / MIPWA_REC_BLOCK;
    return (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)c->sm_count * c->blocks_per_sm, need));
}

static int nll_recompute(mipwa_ctx* c, double* sum_log, double* integral)
{
    Slot& E = evs(c);
    Slot& G = nms(c);
    int rc = ensure_records(c, E, 0.0);
    if (rc) return rc;
    rc = ensure_records(c, G, 1.0);
    if (rc) return rc;
    const int grid = recompute_grid(c, std::max(E.n, G.n));
    { const int trc = timing_begin(c); if (trc) return trc; }
    const long long tag = next_tag(c);
    const cudaError_t le = c->overlap_launch
        ? mipwa_launch_nll_recompute_overlapped(c->n_spin, c->model_flags, grid, c->stream, c->model, E.rec, E.n, G.rec, G.n,
                                                c->d_partials, c->d_ticket, c->result_dst, tag)
        : mipwa_launch_nll_recompute(c->n_spin, c->model_flags, false, grid, c->stream, c->model, E.rec, 0.0,
                                     E.n, G.rec, G.n, c->d_partials, c->d_ticket, c->result_dst, tag);
    ++c->launches;
    CU(c, le);
    rc = wait_result(c, tag);
    if (rc) return rc;
    *sum_log = c->h_result[0];
    *integral = c->nm.w ? c->h_result[1] : c->h_result[1] / (double)c->nm.n;
    return MIPWA_OK;
}

// ---- fixed-shape path: host side of A9 / A10 ---------------------------------------------------------------------
static int effective_path(const mipwa_ctx* c)
{
    if (c->path != MIPWA_PATH_AUTO) return c->path;
    if (c->F == 0) return MIPWA_PATH_CACHED_COMPACT;
    return c->hyb_ok ? MIPWA_PATH_HYBRID : MIPWA_PATH_RECOMPUTE;
}

static int64_t cache_bytes_for(const mipwa_ctx* c, int kind, int64_t n)
{
    const int64_t tiles = (n + MIPWA_TILE - 1) / MIPWA_TILE;
    if (kind == MIPWA_PATH_CACHED_REAL) return tiles * (int64_t)RealTile<double, double2>::bytes(c->N, c->R);
    if (kind == MIPWA_PATH_CACHED_F32) return tiles * (int64_t)RealTile<float, float2>::bytes(c->N, c->R);
    const int64_t cols = kind == MIPWA_PATH_CACHED ? c->N + c->R : 1 + c->R;
    return tiles * MIPWA_TILE * cols * (int64_t)sizeof(double2);
}

// unit-coefficient model (a_k = 1, phi_k = 0, c_r = 1) with the shapes of `params` (or the listed ones) -> c->model
static int build_unit_model(mipwa_ctx* c, const double* params)
{
    const int Np = c->Np, R = c->R, pb = c->pb();
    std::vector<double> p(c->n_par(), 0.0);
    for (int i = 0; i < Np; ++i) p[i] = 1.0;
    for (int r = 0; r < R; ++r) p[pb + 2 * r] = r == c->nr_idx ? 0.0 : 1.0;   // the basis kernels emit the constant column themselves
    for (int r = 0, f = 0; r < R; ++r)
        if (c->res[r].shape_floats) {
            p[pb + 2 * R + 2 * f] = params ? params[pb + 2 * R + 2 * f] : c->res[r].mass;
            p[pb + 2 * R + 2 * f + 1] = params ? params[pb + 2 * R + 2 * f + 1] : c->res[r].width;
            ++f;
        }
    return build_model(c, p.data(), (int64_t)p.size());
}

static BasisAux basis_aux(const mipwa_ctx* c)
{
    BasisAux a;
    a.Mx = c->d_Mx;
    std::memset(a.col_of_slot, 0, sizeof(a.col_of_slot));
    if (c->active) for (int d = 0; d < (int)c->active->size(); ++d) a.col_of_slot[d] = (uint8_t)d;   // subset: own order
    else for (int d = 0; d < (int)c->perm.size(); ++d) a.col_of_slot[d] = (uint8_t)c->perm[d];
    a.nonres_col = c->active ? -1 : c->nr_idx;             // the hybrid caches hold fixed-shape resonances only
    a.n_res_cols = c->active ? (int)c->active->size() : c->R;
    return a;
}

static int ensure_cache(mipwa_ctx* c, int kind)
{
    if (c->cache_valid && c->cache_kind == kind) return MIPWA_OK;
    const int64_t need = cache_bytes_for(c, kind, c->ev.n);
    c->cache_valid = false;
    if (c->user_cache && c->user_cache_bytes >= need) {
        c->d_cache = c->user_cache;
    } else {
        if (c->owned_cache_bytes < need) {
            if (c->owned_cache) cudaFree(c->owned_cache);
            c->owned_cache = nullptr; c->owned_cache_bytes = 0;
            if (need > 0) CU(c, cudaMalloc(&c->owned_cache, (size_t)need));
            c->owned_cache_bytes = need;
        }
        c->d_cache = c->owned_cache;
    }
    if (c->ev.n > 0) {
        int rc = build_unit_model(c, nullptr);
        if (rc) return rc;
        const int64_t tiles = (c->ev.n + MIPWA_TILE - 1) / MIPWA_TILE;
        const int grid = (int)std::min<int64_t>(tiles, (int64_t)c->sm_count * 8);
        if (kind == MIPWA_PATH_CACHED)
            k_basis_build<false><<<grid, MIPWA_TILE, 0, c->stream>>>(c->model, c->d_search, basis_aux(c), evs(c).s12,
                                                                      evs(c).s13, c->ev.n, (double2*)c->d_cache);
        else if (kind == MIPWA_PATH_CACHED_REAL)
            k_basis_build_real<double, double2><<<grid, MIPWA_TILE, 0, c->stream>>>(
                c->model, c->d_search, basis_aux(c), evs(c).s12, evs(c).s13, c->ev.n, (unsigned char*)c->d_cache);
        else if (kind == MIPWA_PATH_CACHED_F32)
            k_basis_build_real<float, float2><<<grid, MIPWA_TILE, 0, c->stream>>>(
                c->model, c->d_search, basis_aux(c), evs(c).s12, evs(c).s13, c->ev.n, (unsigned char*)c->d_cache);
        else
            k_basis_build<true><<<grid, MIPWA_TILE, 0, c->stream>>>(c->model, c->d_search, basis_aux(c), evs(c).s12,
                                                                     evs(c).s13, c->ev.n, (double2*)c->d_cache);
        ++c->launches;
        CU(c, cudaGetLastError());
        CU(c, cudaStreamSynchronize(c->stream));
    }
    c->cache_kind = kind;
    c->cache_valid = true;
    return MIPWA_OK;
}

// shapes: parameter vector whose floating masses and widths the basis is built with (mipwa_nll_hessian_full: the Gram
// matrix is then rebuilt on every call); nullptr: the listed shapes, built once per set of normalisation points
static int ensure_gram(mipwa_ctx* c, const double* shapes = nullptr)
{
    if (c->gram_valid && !(shapes && c->F > 0)) return MIPWA_OK;
    c->gram_valid = false;
    int rc = build_unit_model(c, shapes);
    if (rc) return rc;
    const int K = c->N + c->R, nt = (K + 3) / 4, ntile = nt * (nt + 1) / 2;
    const int tpt = (ntile + MIPWA_TILE - 1) / MIPWA_TILE;
    const int grid = (int)std::min<int64_t>((c->nm.n + GRAM_P - 1) / GRAM_P, c->sm_count);
    const size_t smem = (size_t)4 * nt * GRAM_LD * sizeof(double2);
    double2* partial = nullptr;
    CU(c, cudaMalloc(&partial, (size_t)grid * K * K * sizeof(double2)));
    const double wd = 1.0 / (double)c->nm.n;
    CoefDev cdummy{};                                      // unused by the Gram instantiation
    cdummy.K = K; cdummy.N = c->N;
    cudaError_t e = cudaSuccess;
#define MIPWA_GRAM_LAUNCH(T)                                                                                         \
    do {                                                                                                             \
        e = cudaFuncSetAttribute(k_gram<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);          \
        if (e == cudaSuccess)                                                                                        \
            k_gram<T, false><<<grid, MIPWA_TILE, smem, c->stream>>>(c->model, c->d_search, basis_aux(c), cdummy,     \
                                                                     nms(c).s12, nms(c).s13, nms(c).w, c->nm.n, wd,  \
                                                                     partial);                                       \
    } while (0)
    if (tpt <= 1) MIPWA_GRAM_LAUNCH(1); else if (tpt == 2) MIPWA_GRAM_LAUNCH(2); else MIPWA_GRAM_LAUNCH(3);
#undef MIPWA_GRAM_LAUNCH
    ++c->launches;
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) {
        k_gram_reduce<<<(K * K + 255) / 256, 256, 0, c->stream>>>(partial, grid, K, c->d_gram, 1);
        ++c->launches;
        e = cudaGetLastError();
    }
    c->h_gram.resize((size_t)2 * K * K);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(c->h_gram.data(), c->d_gram, (size_t)K * K * sizeof(double2), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(partial);
    if (e != cudaSuccess) return fail(c, MIPWA_ERR_CUDA, std::string("gram: ") + cudaGetErrorString(e));
    c->gram_valid = !(shapes && c->F > 0);
    return MIPWA_OK;
}

// A1 for the cached kernels: c = [y_0 .. y_{N-1}, c_0 .. c_{R-1}] (caller's resonance order); needs build_model first
static void fill_coef(const mipwa_ctx* c, const double* p, CoefDev* cc)
{
    const int N = c->N, R = c->R, pb = c->pb();
    cc->K = N + R; cc->N = N;
    for (int k = 0; k < N; ++k) cc->c[k] = make_double2(c->y_re[k], c->y_im[k]);
    for (int r = 0; r < R; ++r)                             // the constant term included: its dense column is 1
        cc->c[N + r] = make_double2(p[pb + 2 * r] * std::cos(p[pb + 2 * r + 1]), p[pb + 2 * r] * std::sin(p[pb + 2 * r + 1]));
}

static int nll_cached(mipwa_ctx* c, int kind, const double* params, double* sum_log, double* integral)
{
    // both callers have built c->model from `params`; a cache or Gram (re)build overwrites it with the unit model
    const bool rebuilt = !(c->cache_valid && c->cache_kind == kind && c->gram_valid);
    int rc = ensure_cache(c, kind);
    if (rc) return rc;
    rc = ensure_gram(c);
    if (rc) return rc;
    if (rebuilt) {
        rc = build_model(c, params, c->n_par());
        if (rc) return rc;
    }
    CoefDev cc;
    fill_coef(c, params, &cc);
    const int64_t tiles = (c->ev.n + MIPWA_TILE - 1) / MIPWA_TILE;
    const double2* cache = (const double2*)c->d_cache;
    { const int trc = timing_begin(c); if (trc) return trc; }
    const long long tag = next_tag(c);
    if (kind == MIPWA_PATH_CACHED) {
        if (!c->dense_blocks_per_sm) {
            CU(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->dense_blocks_per_sm, k_nll_dense, MIPWA_TILE, 0));
            if (c->dense_blocks_per_sm < 1) c->dense_blocks_per_sm = 1;
        }
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(tiles, (int64_t)c->sm_count * c->dense_blocks_per_sm));
        k_nll_dense<<<grid, MIPWA_TILE, 0, c->stream>>>(cc, cache, c->ev.n, c->d_gram, (double*)c->d_partials,
                                                         c->d_ticket, c->result_dst, tag);
    } else if (kind == MIPWA_PATH_CACHED_REAL || kind == MIPWA_PATH_CACHED_F32) {
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(tiles, (int64_t)c->sm_count * 8));
        if (kind == MIPWA_PATH_CACHED_REAL)
            k_nll_dense_real<double, double2><<<grid, MIPWA_TILE, 0, c->stream>>>(
                cc, (const unsigned char*)c->d_cache, c->ev.n, c->d_gram, (double*)c->d_partials, c->d_ticket, c->result_dst, tag);
        else
            k_nll_dense_real<float, float2><<<grid, MIPWA_TILE, 0, c->stream>>>(
                cc, (const unsigned char*)c->d_cache, c->ev.n, c->d_gram, (double*)c->d_partials, c->d_ticket, c->result_dst, tag);
    } else {
        if (!c->compact_blocks_per_sm) {
            CU(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->compact_blocks_per_sm, k_nll_compact<-1>, MIPWA_TILE, 0));
            if (c->compact_blocks_per_sm < 1) c->compact_blocks_per_sm = 1;
        }
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(tiles, (int64_t)c->sm_count * c->compact_blocks_per_sm));
        // overlap_launch (mipwa_nll_batch, vectors 1..): programmatic stream serialisation, as for k_nll_recompute
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(MIPWA_TILE); cfg.stream = c->stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr; cfg.numAttrs = c->overlap_launch ? 1 : 0;
        const unsigned short* segp = evs(c).seg;
        const long long n_ev_ll = c->ev.n;
        const double2* gram = c->d_gram;
        double* parts = (double*)c->d_partials;
#define MIPWA_COMPACT_LAUNCH(T)                                                                                   \
    (void)cudaLaunchKernelEx(&cfg, k_nll_compact<T>, c->model, cc, cache, segp, n_ev_ll, gram, parts, c->d_ticket, \
                             c->result_dst, tag)
        switch (c->R) {
            case 0: MIPWA_COMPACT_LAUNCH(0); break;
            case 1: MIPWA_COMPACT_LAUNCH(1); break;
            case 2: MIPWA_COMPACT_LAUNCH(2); break;
            case 3: MIPWA_COMPACT_LAUNCH(3); break;
            case 4: MIPWA_COMPACT_LAUNCH(4); break;
            case 6: MIPWA_COMPACT_LAUNCH(6); break;
            default: MIPWA_COMPACT_LAUNCH(-1); break;
        }
#undef MIPWA_COMPACT_LAUNCH
    }
    ++c->launches;
    CU(c, cudaGetLastError());
    rc = wait_result(c, tag);
    if (rc) return rc;
    *sum_log = c->h_result[0];
    *integral = c->h_result[1];
    return MIPWA_OK;
}

// ---- hybrid path: fixed-shape resonances cached per point, floating ones and the spline re-evaluated ---------------------
static int64_t hyb_bytes_for(const mipwa_ctx* c, int64_t n)
{
    const int64_t tiles = (n + MIPWA_TILE - 1) / MIPWA_TILE;
    return tiles * MIPWA_TILE * (1 + (int64_t)c->hyb_fixed.size()) * (int64_t)sizeof(double2);
}

static int ensure_hyb_cache(mipwa_ctx* c, const Slot& pts, void** buf, int64_t* have, bool* valid)
{
    if (*valid) return MIPWA_OK;
    const int64_t need = hyb_bytes_for(c, pts.n);
    if (*have < need) {
        if (*buf) cudaFree(*buf);
        *buf = nullptr; *have = 0;
        if (need > 0) CU(c, cudaMalloc(buf, (size_t)need));
        *have = need;
    }
    if (pts.n > 0) {
        c->active = &c->hyb_fixed;                         // unit model of the fixed resonances only
        int rc = build_unit_model(c, nullptr);
        const BasisAux aux = basis_aux(c);
        c->active = nullptr;
        if (rc) return rc;
        const int64_t tiles = (pts.n + MIPWA_TILE - 1) / MIPWA_TILE;
        const int grid = (int)std::min<int64_t>(tiles, (int64_t)c->sm_count * 8);
        k_basis_build<true><<<grid, MIPWA_TILE, 0, c->stream>>>(c->model, c->d_search, aux, pts.s12, pts.s13, pts.n,
                                                                 (double2*)*buf);
        ++c->launches;
        CU(c, cudaGetLastError());
        CU(c, cudaStreamSynchronize(c->stream));
    }
    *valid = true;
    return MIPWA_OK;
}

static int nll_hybrid(mipwa_ctx* c, const double* params, int64_t n_params, double* sum_log, double* integral)
{
    int rc = ensure_hyb_cache(c, evs(c), &c->d_hyb_ev, &c->hyb_ev_bytes, &c->hyb_ev_valid);
    if (rc) return rc;
    rc = ensure_hyb_cache(c, nms(c), &c->d_hyb_nm, &c->hyb_nm_bytes, &c->hyb_nm_valid);
    if (rc) return rc;
    c->active = &c->hyb_float;                             // spline tables + the floating resonances of this call
    rc = build_model(c, params, n_params);
    c->active = nullptr;
    if (rc) return rc;
    const int pb = c->pb(), RC = (int)c->hyb_fixed.size();
    HybCoef cc;
    cc.RC = RC; cc.pad = 0;
    for (int k = 0; k < RC; ++k) {
        const int r = c->hyb_fixed[k];
        cc.c[k] = make_double2(params[pb + 2 * r] * std::cos(params[pb + 2 * r + 1]),
                               params[pb + 2 * r] * std::sin(params[pb + 2 * r + 1]));
    }
    bool supported = true;
    if (!c->hyb_blocks_per_sm) {
        supported = mipwa_occupancy_nll_hybrid(c->hyb_f1, c->hyb_f2, RC, c->model_flags, &c->hyb_blocks_per_sm) == cudaSuccess;
        if (!supported) return fail(c, MIPWA_ERR_CUDA, "hybrid: occupancy query failed");
        if (c->hyb_blocks_per_sm < 1) c->hyb_blocks_per_sm = 1;
    }
    const int64_t tpb = mipwa_hybrid_tiles_per_block(RC);
    const int64_t tiles = (std::max(c->ev.n, c->nm.n) + MIPWA_TILE - 1) / MIPWA_TILE;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((tiles + tpb - 1) / tpb, (int64_t)c->sm_count * c->hyb_blocks_per_sm));
    { const int trc = timing_begin(c); if (trc) return trc; }
    const long long tag = next_tag(c);
    const cudaError_t le = mipwa_launch_nll_hybrid(c->hyb_f1, c->hyb_f2, RC, c->model_flags, grid, c->stream, c->model, cc,
                                                   (const double2*)c->d_hyb_ev, evs(c).seg, c->ev.n,
                                                   (const double2*)c->d_hyb_nm, nms(c).w, nms(c).seg, c->nm.n,
                                                   c->d_partials, c->d_ticket, c->result_dst, tag, c->overlap_launch);
    ++c->launches;
    CU(c, le);
    rc = wait_result(c, tag);
    if (rc) return rc;
    *sum_log = c->h_result[0];
    *integral = c->nm.w ? c->h_result[1] : c->h_result[1] / (double)c->nm.n;
    return MIPWA_OK;
}

int mipwa_nll_parts(mipwa_ctx* c, const double* params, int64_t n_params, double* nll, double* sum_log, double* integral)
{
    if (!c || !params || !nll) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    NvtxRange range("mipwa_nll");
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    int rc = use_device(c);
    if (rc) return rc;
    rc = build_model(c, params, n_params);                 // validates n_params and the parameter values
    if (rc) return rc;
    double S = 0, I = 0;
    const int path = effective_path(c);
    if (path == MIPWA_PATH_RECOMPUTE) rc = nll_recompute(c, &S, &I);
    else if (path == MIPWA_PATH_HYBRID) rc = nll_hybrid(c, params, n_params, &S, &I);
    else rc = nll_cached(c, path, params, &S, &I);
    if (rc) return rc;
    *nll = -S + (double)c->ev.n * std::log(I);             // A7
    if (sum_log) *sum_log = S;
    if (integral) *integral = I;
    return MIPWA_OK;
}

int mipwa_nll(mipwa_ctx* c, const double* params, int64_t n_params, double* nll)
{
    return mipwa_nll_parts(c, params, n_params, nll, nullptr, nullptr);
}

// n_batch likelihood values of the same sample, pipelined: every call's kernel is enqueued behind the previous one without
// waiting, its last block writes (S, I, tag) into the call's own slot of a mapped host block, and the host waits once, for
// the last slot (the stream runs the kernels in order).  Same kernels, same grid, same bits as n_batch mipwa_nll calls.
int mipwa_nll_batch(mipwa_ctx* c, const double* params, int64_t n_params, int32_t n_batch, double* nll, double* sum_log,
                    double* integral)
{
    if (!c || !params || !nll || n_batch < 0) return c ? fail(c, MIPWA_ERR_ARG, "bad argument") : MIPWA_ERR_ARG;
    NvtxRange range("mipwa_nll_batch");
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    if (n_params != c->n_par()) return fail(c, MIPWA_ERR_ARG, "n_params must be " + std::to_string(c->n_par()));
    if (n_batch == 0) return MIPWA_OK;
    int rc = use_device(c);
    if (rc) return rc;
    if (c->batch_cap < n_batch) {
        if (c->h_batch) cudaFreeHost(c->h_batch);
        c->h_batch = nullptr; c->d_batch = nullptr; c->batch_cap = 0;
        const int64_t cap = std::max<int64_t>(256, n_batch);
        CU(c, cudaHostAlloc(&c->h_batch, (size_t)cap * 4 * sizeof(double), cudaHostAllocMapped));
        CU(c, cudaHostGetDevicePointer(&c->d_batch, c->h_batch, 0));
        c->batch_cap = cap;
    }
    std::memset(c->h_batch, 0, (size_t)n_batch * 4 * sizeof(double));     // no stale tag in any slot
    const int path = effective_path(c);
    const bool timing = c->timing;
    c->timing = false; c->async_result = true;
    long long last_tag = 0;
    int32_t launched = 0;
    for (int32_t b = 0; b < n_batch && rc == MIPWA_OK; ++b) {
        const double* p = params + (size_t)b * n_params;
        rc = build_model(c, p, n_params);
        if (rc) break;
        double S = 0, I = 0;
        c->result_dst = c->d_batch + 4 * (size_t)b;
        c->overlap_launch = b > 0;                         // its predecessor on the stream is the same kernel on the same records
        if (path == MIPWA_PATH_RECOMPUTE) rc = nll_recompute(c, &S, &I);
        else if (path == MIPWA_PATH_HYBRID) rc = nll_hybrid(c, p, n_params, &S, &I);
        else rc = nll_cached(c, path, p, &S, &I);
        if (rc == MIPWA_OK) { last_tag = c->tag; ++launched; }
    }
    c->timing = timing; c->async_result = false; c->result_dst = c->d_result; c->overlap_launch = false;
    if (launched > 0) {                                    // also after an error: nothing of this call stays in flight
        volatile long long* flag = reinterpret_cast<volatile long long*>(c->h_batch + 4 * (size_t)(launched - 1) + MIPWA_RESULT_TAG);
        bool seen = false;
        for (long long spin = 0; spin < 4000000 && !seen; ++spin) {
            seen = *flag == last_tag;
            if (!seen && (spin & 0xffff) == 0xffff) {
                const cudaError_t e = cudaStreamQuery(c->stream);
                if (e == cudaSuccess) break;
                if (e != cudaErrorNotReady) return fail(c, MIPWA_ERR_CUDA, cudaGetErrorString(e));
            }
        }
        if (!seen) CU(c, cudaStreamSynchronize(c->stream));
    }
    if (rc) return rc;
    const bool raw = path == MIPWA_PATH_RECOMPUTE || path == MIPWA_PATH_HYBRID;   // sum |A|^2 without its 1/n when unweighted
    for (int32_t b = 0; b < n_batch; ++b) {
        const double S = c->h_batch[4 * (size_t)b];
        const double I = raw && !c->nm.w ? c->h_batch[4 * (size_t)b + 1] / (double)c->nm.n : c->h_batch[4 * (size_t)b + 1];
        nll[b] = -S + (double)c->ev.n * std::log(I);       // A7
        if (sum_log) sum_log[b] = S;
        if (integral) integral[b] = I;
    }
    return MIPWA_OK;
}

// ---- sharded likelihood without a host round trip --------------------------------------------------------
// rank-local pieces left in DEVICE memory: dev_parts[0..2] = (sum ln|A|^2, sum w|A|^2, n_ev); nothing is waited for
int mipwa_nll_parts_device(mipwa_ctx* c, const double* params, int64_t n_params, double* dev_parts)
{
    if (!c || !params || !dev_parts) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    NvtxRange range("mipwa_nll_parts_device");
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    int rc = use_device(c);
    if (rc) return rc;
    rc = build_model(c, params, n_params);
    if (rc) return rc;
    double S = 0, I = 0;
    const int path = effective_path(c);
    const bool timing = c->timing;
    c->timing = false; c->async_result = true; c->result_dst = c->d_dev_result;
    if (path == MIPWA_PATH_RECOMPUTE) rc = nll_recompute(c, &S, &I);
    else if (path == MIPWA_PATH_HYBRID) rc = nll_hybrid(c, params, n_params, &S, &I);
    else rc = nll_cached(c, path, params, &S, &I);
    c->timing = timing; c->async_result = false; c->result_dst = c->d_result;
    if (rc) return rc;
    // the recompute and hybrid kernels leave sum |A|^2 without its 1/n when the points have no weights
    const bool raw = path == MIPWA_PATH_RECOMPUTE || path == MIPWA_PATH_HYBRID;
    k_pack_parts<<<1, 1, 0, c->stream>>>(c->d_dev_result, raw && !c->nm.w ? 1.0 / (double)c->nm.n : 1.0, (double)c->ev.n, dev_parts);
    ++c->launches;
    CU(c, cudaGetLastError());
    return MIPWA_OK;
}

// A7 over the gathered pieces of all ranks, on the device: rank-ordered sums, NLL = -S + n ln I; the four numbers come
// back through the mapped result block like any likelihood value
int mipwa_combine_parts_device(mipwa_ctx* c, const double* dev_parts_all, int32_t n_ranks, double* nll, double* sum_log,
                               double* integral, int64_t* n_ev)
{
    if (!c || !dev_parts_all || n_ranks < 1 || !nll) return c ? fail(c, MIPWA_ERR_ARG, "bad argument") : MIPWA_ERR_ARG;
    int rc = use_device(c);
    if (rc) return rc;
    const long long tag = next_tag(c);
    k_combine_parts<<<1, 1, 0, c->stream>>>(dev_parts_all, n_ranks, c->d_result, tag);
    ++c->launches;
    CU(c, cudaGetLastError());
    const bool timing = c->timing;
    c->timing = false;
    rc = wait_result(c, tag);
    c->timing = timing;
    if (rc) return rc;
    *nll = c->h_result[3];
    if (sum_log) *sum_log = c->h_result[0];
    if (integral) *integral = c->h_result[1];
    if (n_ev) *n_ev = (int64_t)c->h_result[4];
    return MIPWA_OK;
}

// A7 on the host over gathered pieces (parts[3 r + {0,1,2}] = S_r, I_r, n_r): the same rank-ordered sums; needs no GPU
int mipwa_combine_parts(int32_t n_ranks, const double* parts, double* nll, double* sum_log, double* integral, int64_t* n_ev)
{
    if (n_ranks < 1 || !parts || !nll) return MIPWA_ERR_ARG;
    double S = 0.0, I = 0.0, n = 0.0;
    for (int r = 0; r < n_ranks; ++r) { S += parts[3 * r]; I += parts[3 * r + 1]; n += parts[3 * r + 2]; }
    *nll = n > 0.0 ? -S + n * std::log(I) : 0.0;
    if (sum_log) *sum_log = S;
    if (integral) *integral = I;
    if (n_ev) *n_ev = (int64_t)n;
    return MIPWA_OK;
}

// A7 at every vector of a batch from gathered rows parts[r] = (S_r[0..B), I_r[0..B), n_r): the same rank-ordered sums as
// mipwa_combine_parts, hence the same bits per vector
int mipwa_combine_parts_batch(int32_t n_ranks, int32_t n_batch, const double* parts, double* nll)
{
    if (n_ranks < 1 || n_batch < 0 || !parts || (!nll && n_batch > 0)) return MIPWA_ERR_ARG;
    const size_t row = 2 * (size_t)n_batch + 1;
    for (int32_t b = 0; b < n_batch; ++b) {
        double S = 0.0, I = 0.0, n = 0.0;
        for (int r = 0; r < n_ranks; ++r) { S += parts[r * row + b]; I += parts[r * row + n_batch + b]; n += parts[r * row + 2 * (size_t)n_batch]; }
        nll[b] = n > 0.0 ? -S + n * std::log(I) : 0.0;
    }
    return MIPWA_OK;
}

// whole-sample NLL and gradient from the gathered mipwa_nll_grad_parts pieces, parts[r] = (S_r, I_r, n_r, grad_ev_r[P],
// grad_nm_r[P]): NLL = -sum S_r + n ln I, grad = sum grad_ev_r + (n / I) sum grad_nm_r, every sum in rank order
int mipwa_combine_grad_parts(int32_t n_ranks, int64_t n_params, const double* parts, double* nll, double* grad,
                             double* sum_log, double* integral, int64_t* n_ev)
{
    if (n_ranks < 1 || n_params < 0 || !parts || !nll || (n_params > 0 && !grad)) return MIPWA_ERR_ARG;
    const int64_t P = n_params, stride = 3 + 2 * P;
    double S = 0.0, I = 0.0, n = 0.0;
    for (int r = 0; r < n_ranks; ++r) { S += parts[r * stride]; I += parts[r * stride + 1]; n += parts[r * stride + 2]; }
    for (int64_t k = 0; k < P; ++k) {
        double ge = 0.0, gn = 0.0;
        for (int r = 0; r < n_ranks; ++r) { ge += parts[r * stride + 3 + k]; gn += parts[r * stride + 3 + P + k]; }
        grad[k] = n > 0.0 ? ge + (n / I) * gn : 0.0;
    }
    *nll = n > 0.0 ? -S + n * std::log(I) : 0.0;
    if (sum_log) *sum_log = S;
    if (integral) *integral = I;
    if (n_ev) *n_ev = (int64_t)n;
    return MIPWA_OK;
}

int mipwa_eval_abs2(mipwa_ctx* c, const double* params, int64_t n_params, int32_t which, double* out, int64_t n)
{
    if (!c || !params || (which != 0 && which != 1)) return c ? fail(c, MIPWA_ERR_ARG, "bad argument") : MIPWA_ERR_ARG;
    const Slot& s = which == 0 ? c->ev : c->nm;
    if (s.n < 0) return fail(c, MIPWA_ERR_STATE, "slot not set");
    if (n != s.n || (n > 0 && !out)) return fail(c, MIPWA_ERR_ARG, "n must equal the slot size");
    int rc = use_device(c);
    if (rc) return rc;
    rc = build_model(c, params, n_params);
    if (rc) return rc;
    if (n == 0) return MIPWA_OK;
    double* d_out = nullptr;
    CU(c, cudaMalloc(&d_out, (size_t)n * sizeof(double)));
    cudaError_t e = mipwa_launch_abs2(c->n_spin, c->model_flags, grid_for(c, n, 4), c->stream, c->model, s.s12, s.s13,
                                      s.seg, n, d_out);
    ++c->launches;
    if (e == cudaSuccess) e = cudaMemcpyAsync(out, d_out, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(d_out);
    if (e != cudaSuccess) return fail(c, MIPWA_ERR_CUDA, cudaGetErrorString(e));
    return MIPWA_OK;
}

int mipwa_last_kernel_ms(const mipwa_ctx* c, float* ms)
{
    if (!c || !ms) return MIPWA_ERR_ARG;
    *ms = c->last_ms;
    return MIPWA_OK;
}

int64_t mipwa_launch_count(const mipwa_ctx* c) { return c ? c->launches : -1; }

int mipwa_measure_fp64_peak(int32_t device, double seconds, double* tflops, double* tflops_3reg)
{
    if (!tflops || !(seconds > 0)) return MIPWA_ERR_ARG;
    cudaDeviceProp prop;
    if (cudaSetDevice(device) != cudaSuccess || cudaGetDeviceProperties(&prop, device) != cudaSuccess) return MIPWA_ERR_CUDA;
    int rc = fp64_rate<1>(prop, tflops_3reg ? 0.5 * seconds : seconds, tflops);
    if (rc == MIPWA_OK && tflops_3reg) rc = fp64_rate<0>(prop, 0.5 * seconds, tflops_3reg);
    return rc;
}

}  // extern "C"


extern "C" {

int64_t mipwa_basis_bytes(const mipwa_ctx* c)
{
    if (!c) return MIPWA_ERR_ARG;
    const int path = effective_path(c);
    if (path == MIPWA_PATH_RECOMPUTE) return 0;
    if (c->ev.n < 0) return MIPWA_ERR_STATE;
    if (path == MIPWA_PATH_HYBRID) return hyb_bytes_for(c, c->ev.n) + (c->nm.n > 0 ? hyb_bytes_for(c, c->nm.n) : 0);
    return cache_bytes_for(c, path, c->ev.n);
}

int mipwa_set_basis_buffer(mipwa_ctx* c, void* dev, int64_t bytes)
{
    if (!c) return MIPWA_ERR_ARG;
    if ((dev && bytes <= 0) || ((uintptr_t)dev & 255)) return fail(c, MIPWA_ERR_ARG, "buffer must be 256-byte aligned with bytes > 0");
    int rc = use_device(c);
    if (rc) return rc;
    CU(c, cudaStreamSynchronize(c->stream));
    c->user_cache = dev;
    c->user_cache_bytes = dev ? bytes : 0;
    c->cache_valid = false;
    return MIPWA_OK;
}

int mipwa_eval_basis(mipwa_ctx* c, const double* params, int64_t n_params, int32_t which, int64_t first, int64_t n,
                     double* out)
{
    if (!c || !params || (which != 0 && which != 1)) return c ? fail(c, MIPWA_ERR_ARG, "bad argument") : MIPWA_ERR_ARG;
    const Slot& s = which == 0 ? c->ev : c->nm;
    if (s.n < 0) return fail(c, MIPWA_ERR_STATE, "slot not set");
    if (first < 0 || n < 0 || first + n > s.n || (n > 0 && !out)) return fail(c, MIPWA_ERR_ARG, "bad range");
    if (n_params != c->n_par()) return fail(c, MIPWA_ERR_ARG, "wrong n_params");
    int rc = use_device(c);
    if (rc) return rc;
    rc = build_unit_model(c, params);
    if (rc) return rc;
    if (n == 0) return MIPWA_OK;
    const int K = c->N + c->R;
    double2* d_out = nullptr;
    CU(c, cudaMalloc(&d_out, (size_t)n * K * sizeof(double2)));
    k_basis_rows<<<grid_for(c, n, 4), MIPWA_TILE, 0, c->stream>>>(c->model, c->d_search, basis_aux(c), s.s12, s.s13, first, n,
                                                                  d_out);
    ++c->launches;
    cudaError_t e = cudaGetLastError();
    const int skip = c->N - c->Np;                         // stand-in knots of a model without spline: not the caller's columns
    std::vector<double> tmp;
    double* dst = out;
    if (skip) { tmp.resize((size_t)n * K * 2); dst = tmp.data(); }
    if (e == cudaSuccess) e = cudaMemcpyAsync(dst, d_out, (size_t)n * K * sizeof(double2), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(d_out);
    if (e != cudaSuccess) return fail(c, MIPWA_ERR_CUDA, cudaGetErrorString(e));
    if (skip)
        for (int64_t i = 0; i < n; ++i)
            std::memcpy(out + (size_t)i * (K - skip) * 2, tmp.data() + ((size_t)i * K + skip) * 2, (size_t)(K - skip) * 2 * sizeof(double));
    return MIPWA_OK;
}

// adjoint of the map knot values y -> segment coefficients sc (build_model): from calG of sc[q][j] (Gsc[(q*NS+j)*2+ri])
// to calG of y_k (Gy[2k+ri]).  sc0 = y_j; sc1 = (y_j+1 - y_j)/h - h (2 P_j + P_j+1)/6; sc2 = P_j/2;
// sc3 = (P_j+1 - P_j)/(6h); P = Mx y  =>  Gy = g_y + Mx^T g_P.
static void spline_adjoint(const mipwa_ctx* c, const double* Gsc, double* Gy)
{
    const int N = c->N, NS = N - 1;
    std::vector<double> gy(2 * N, 0.0), gP(2 * N, 0.0);
    for (int j = 0; j < NS; ++j) {
        const double hj = c->knots[j + 1] - c->knots[j];
        for (int q = 0; q < 2; ++q) {                                  // re, im
            const double G0 = Gsc[(0 * NS + j) * 2 + q], G1 = Gsc[(1 * NS + j) * 2 + q];
            const double G2 = Gsc[(2 * NS + j) * 2 + q], G3 = Gsc[(3 * NS + j) * 2 + q];
            gy[2 * j + q] += G0 - G1 / hj;
            gy[2 * (j + 1) + q] += G1 / hj;
            gP[2 * j + q] += -G1 * hj / 3.0 + 0.5 * G2 - G3 / (6.0 * hj);
            gP[2 * (j + 1) + q] += -G1 * hj / 6.0 + G3 / (6.0 * hj);
        }
    }
    for (int k = 0; k < N; ++k) {
        double gr = gy[2 * k], gi = gy[2 * k + 1];
        for (int j = 0; j < N; ++j) {
            const double mjk = c->Mx[(size_t)j * N + k];
            gr += mjk * gP[2 * j]; gi += mjk * gP[2 * j + 1];
        }
        Gy[2 * k] = gr; Gy[2 * k + 1] = gi;
    }
}

// polar chain rule: c = rho e^{i theta}: d/drho = Re(calG e^{-i theta}), d/dtheta = Re(calG conj(i c)).
// Gy: calG of the knot values (2N), Gr: calG of the resonance coefficients in the caller's order (2R).
static void polar_chain(const mipwa_ctx* c, const double* params, const double* Gy, const double* Gr, double* grad)
{
    const int Np = c->Np, R = c->R, pb = c->pb();
    for (int k = 0; k < Np; ++k) {
        const double ph = params[Np + k];
        grad[k] = Gy[2 * k] * std::cos(ph) + Gy[2 * k + 1] * std::sin(ph);
        grad[Np + k] = -Gy[2 * k] * c->y_im[k] + Gy[2 * k + 1] * c->y_re[k];
    }
    for (int r = 0; r < R; ++r) {
        const double mag = params[pb + 2 * r], th = params[pb + 2 * r + 1];
        grad[pb + 2 * r] = Gr[2 * r] * std::cos(th) + Gr[2 * r + 1] * std::sin(th);
        grad[pb + 2 * r + 1] = mag * (-Gr[2 * r] * std::sin(th) + Gr[2 * r + 1] * std::cos(th));
    }
}

// The constant non-resonant term enters the kernels as an offset c_nr / 2 of every knot value (build_model), so its calG
// is half the sum of the knot calGs of the SPLINE-TABLE parametrisation (Gy: what spline_adjoint returns).  Sets Gr of
// the constant's slot; nothing to do for a model without one.
static void offset_rule(const mipwa_ctx* c, const double* Gy, double* Gr)
{
    if (c->nr_idx < 0) return;
    double sr = 0.0, si = 0.0;
    for (int k = 0; k < c->N; ++k) { sr += Gy[2 * k]; si += Gy[2 * k + 1]; }
    Gr[2 * c->nr_idx] = 0.5 * sr;
    Gr[2 * c->nr_idx + 1] = 0.5 * si;
}

// ---- A8: gradient on the recompute path ---------------------------------------------------------------------------
// cell-sorted copy of a point set (keys from the knots only: valid until the next mipwa_set_* on that slot)
static int ensure_sorted(mipwa_ctx* c, const Slot& src, Slot& dst, bool& valid)
{
    if (valid) return MIPWA_OK;
    free_slot(dst);
    const int64_t n = src.n;
    if (n > 0x7fffffffLL) return fail(c, MIPWA_ERR_ARG, "mipwa_nll_grad supports at most 2^31-1 points per set");
    if (n > 0) {
        unsigned int* buf = nullptr;                       // keys in, keys out, index in, index out
        CU(c, cudaMalloc(&buf, (size_t)n * 4 * sizeof(unsigned int)));
        unsigned int *k0 = buf, *k1 = buf + n, *i0 = buf + 2 * n, *i1 = buf + 3 * n;
        void* tmp = nullptr;
        size_t tmp_bytes = 0;
        int bits = 1;
        while ((1LL << bits) < (int64_t)(c->N - 1) * (c->N - 1)) ++bits;
        cudaError_t e = cudaSuccess;
        k_cell_keys<<<grid_for(c, n, 8), MIPWA_TILE, 0, c->stream>>>(src.seg, n, c->N - 1, k0, i0);
        ++c->launches;
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, k0, k1, i0, i1, (int)n, 0, bits, c->stream);
        if (e == cudaSuccess) e = cudaMalloc(&tmp, tmp_bytes ? tmp_bytes : 16);
        if (e == cudaSuccess) e = cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, k0, k1, i0, i1, (int)n, 0, bits, c->stream);
        for (int q = 0; q < 3 && e == cudaSuccess; ++q)
            if (q < 2 || src.w) e = cudaMalloc(&dst.owned[q], (size_t)n * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc(&dst.owned[3], (size_t)n * sizeof(unsigned short));
        if (e == cudaSuccess) {
            k_gather<<<grid_for(c, n, 8), MIPWA_TILE, 0, c->stream>>>(i1, n, src.s12, src.s13, src.w, src.seg,
                                                                      (double*)dst.owned[0], (double*)dst.owned[1],
                                                                      (double*)dst.owned[2], (unsigned short*)dst.owned[3]);
            ++c->launches;
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        if (tmp) cudaFree(tmp);
        cudaFree(buf);
        if (e != cudaSuccess) {
            free_slot(dst);
            return fail(c, e == cudaErrorMemoryAllocation ? MIPWA_ERR_NOMEM : MIPWA_ERR_CUDA, std::string("cell sort: ") + cudaGetErrorString(e));
        }
        dst.s12 = (const double*)dst.owned[0]; dst.s13 = (const double*)dst.owned[1]; dst.w = (const double*)dst.owned[2];
        dst.seg = (const unsigned short*)dst.owned[3];
    }
    dst.n = n;
    valid = true;
    return MIPWA_OK;
}

// cell-sorted copies of both point sets; every kernel then reads them instead of the caller's arrays
static int prepare_sorted(mipwa_ctx* c)
{
    if (c->ev_sorted_valid && c->nm_sorted_valid) return MIPWA_OK;
    int rc = build_unit_model(c, nullptr);                 // knots and bucket table for k_cell_keys
    if (rc) return rc;
    if (!c->ev_sorted_valid) {
        rc = ensure_sorted(c, c->ev, c->ev_sorted, c->ev_sorted_valid);
        if (rc) return rc;
        c->cache_valid = false;                            // the per-event caches follow the event order
        c->hyb_ev_valid = false;
    }
    if (!c->nm_sorted_valid) c->hyb_nm_valid = false;
    return ensure_sorted(c, c->nm, c->nm_sorted, c->nm_sorted_valid);
}

int mipwa_prepare(mipwa_ctx* c)
{
    if (!c) return MIPWA_ERR_ARG;
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    int rc = use_device(c);
    if (rc) return rc;
    return prepare_sorted(c);
}

// A8 on the compact cached path: events through k_grad_compact, normalisation part from the Gram matrix
static int nll_grad_compact(mipwa_ctx* c, const double* params, int64_t n_params, double* nll, double* grad)
{
    int rc = ensure_cache(c, MIPWA_PATH_CACHED_COMPACT);
    if (rc) return rc;
    rc = ensure_gram(c);
    if (rc) return rc;
    rc = build_model(c, params, n_params);                 // spline tables of this call (after ensure_*: they use c->model)
    if (rc) return rc;
    CoefDev cc;
    fill_coef(c, params, &cc);
    const int N = c->N, R = c->R, K = N + R, NS = N - 1, nb = 8 * NS, NV = 1 + 2 * R + nb;
    const size_t smem = (size_t)(MIPWA_TILE / 32) * nb * sizeof(double);   // one set of segment bins per warp
    const int grid = grid_for(c, c->ev.n, 2);
    if (c->gpartials_len < (size_t)grid * NV) {
        if (c->d_gpartials) cudaFree(c->d_gpartials);
        c->d_gpartials = nullptr; c->gpartials_len = 0;
        CU(c, cudaMalloc(&c->d_gpartials, (size_t)grid * NV * sizeof(double)));
        c->gpartials_len = (size_t)grid * NV;
    }
    const double2* cache = (const double2*)c->d_cache;
    { const int trc = timing_begin(c); if (trc) return trc; }
#define MIPWA_GC_LAUNCH(T)                                                                                             \
    do {                                                                                                               \
        if (c->gcompact_smem_set < smem) {                                                                             \
            CU(c, cudaFuncSetAttribute(k_grad_compact<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));   \
            c->gcompact_smem_set = smem;                                                                               \
        }                                                                                                              \
        k_grad_compact<T><<<grid, MIPWA_TILE, smem, c->stream>>>(c->model, cc, cache, evs(c).seg, c->ev.n, c->d_gpartials); \
    } while (0)
    switch (R) {
        case 0: MIPWA_GC_LAUNCH(0); break;
        case 1: MIPWA_GC_LAUNCH(1); break;
        case 2: MIPWA_GC_LAUNCH(2); break;
        case 3: MIPWA_GC_LAUNCH(3); break;
        case 4: MIPWA_GC_LAUNCH(4); break;
        case 6: MIPWA_GC_LAUNCH(6); break;
        default: MIPWA_GC_LAUNCH(-1); break;
    }
#undef MIPWA_GC_LAUNCH
    ++c->launches;
    CU(c, cudaGetLastError());
    (void)launch_finalize(c, (NV + 7) / 8, c->d_gpartials, grid, grid, NV, 1, c->d_result);
    ++c->launches;
    CU(c, cudaGetLastError());

    // host, while the kernels run: g = G c, I = Re(c^H g) (K^2 complex MACs); after the wait the adjoint maps
    const double* h = c->h_result;
    const double* G = c->h_gram.data();
    std::vector<double> gc(2 * K, 0.0);
    double I = 0.0;
    for (int k = 0; k < K; ++k) {
        double gr = 0.0, gi = 0.0;
        for (int l = 0; l < K; ++l) {
            const double a = G[2 * ((size_t)k * K + l)], b = G[2 * ((size_t)k * K + l) + 1];
            gr += a * cc.c[l].x - b * cc.c[l].y;
            gi += a * cc.c[l].y + b * cc.c[l].x;
        }
        gc[2 * k] = gr; gc[2 * k + 1] = gi;
        I += cc.c[k].x * gr + cc.c[k].y * gi;
    }
    { const int wrc = wait_grad(c); if (wrc) return wrc; }
    const double S = h[0], n_ev = (double)c->ev.n;
    *nll = -S + n_ev * std::log(I);
    const double scale = c->ev.n > 0 ? 2.0 * n_ev / I : 0.0;
    std::vector<double> Gy(2 * N), Gr(2 * std::max(R, 1));
    // event part: the spline tables carry the constant term (offset rule); normalisation part: I = c^H G c in the dense
    // parametrisation, where the constant has a column (and a coefficient) of its own
    spline_adjoint(c, h + 1 + 2 * R, Gy.data());
    for (int r = 0; r < R; ++r) { Gr[2 * r] = h[1 + 2 * r]; Gr[2 * r + 1] = h[1 + 2 * r + 1]; }   // caller's order, fold included
    offset_rule(c, Gy.data(), Gr.data());
    for (int k = 0; k < 2 * N; ++k) Gy[k] += scale * gc[k];
    for (int r = 0; r < 2 * R; ++r) Gr[r] += scale * gc[2 * N + r];
    polar_chain(c, params, Gy.data(), Gr.data(), grad);
    if (c->parts_ev) {                                     // mipwa_nll_grad_parts: d(-S)/dtheta and dI/dtheta = 2 G c apart
        spline_adjoint(c, h + 1 + 2 * R, Gy.data());
        for (int r = 0; r < R; ++r) { Gr[2 * r] = h[1 + 2 * r]; Gr[2 * r + 1] = h[1 + 2 * r + 1]; }
        offset_rule(c, Gy.data(), Gr.data());
        polar_chain(c, params, Gy.data(), Gr.data(), c->parts_ev);
        for (int k = 0; k < 2 * N; ++k) Gy[k] = 2.0 * gc[k];
        for (int r = 0; r < 2 * R; ++r) Gr[r] = 2.0 * gc[2 * N + r];
        polar_chain(c, params, Gy.data(), Gr.data(), c->parts_nm);
        c->parts_S = S; c->parts_I = I;
    }
    return MIPWA_OK;
}

// ---- A8 on the recompute path -----------------------------------------------------------------------------------------
// One launch of k_grad_recompute over both cell-sorted record sets and one of k_grad_finalize; the totals land in
// h_result as [event vector | normalisation vector], each of NVB = 2 + 2R + 8 (N-1) + 4 doubles laid out like the block
// partials of grad.cuh.  n_ev / n_norm = 0 leaves that set out (the two launches of the mixture likelihood).
struct GradTotals {
    int NVB, nb;
    const double *ev, *nm;                                 // the two vectors
    const double* F(const double* v) const { return v + 2; }
    const double* bins(const double* v, int R) const { return v + 2 + 2 * R; }
    const double* shape(const double* v, int R) const { return v + 2 + 2 * R + nb; }
};

static int launch_grad_recompute(mipwa_ctx* c, bool mix, int shp, double kappa, bool with_ev, bool with_nm, bool want_f,
                                 GradTotals* out)
{
    Slot& E = c->ev_sorted;
    Slot& G = c->nm_sorted;
    int rc = ensure_records(c, E, 0.0);
    if (rc) return rc;
    rc = ensure_records(c, G, 1.0);
    if (rc) return rc;
    const int N = c->N, R = (int)c->perm.size(), NS = N - 1, nb = 8 * NS, NVB = 2 + 2 * R + nb + 4;   // R: device slots
    const int64_t n_ev = with_ev ? E.n : 0, n_nm = with_nm ? G.n : 0;
    const int ev_blocks = n_ev > 0 ? recompute_grid(c, n_ev) : 0, nm_blocks = n_nm > 0 ? recompute_grid(c, n_nm) : 0;
    const int grid = std::max(1, ev_blocks + nm_blocks);
    // per-warp segment bins + per-warp record staging (2 stages x 32 records x 32 B), grad.cuh: grad_body
    const size_t smem = (size_t)(MIPWA_GRAD_BLOCK / 32) * (nb * sizeof(double) + 2 * 32 * sizeof(PointRec));
    if (smem > 200 * 1024) return fail(c, MIPWA_ERR_ARG, "mipwa_nll_grad: too many knots for the per-warp segment bins");
    if (c->grad_smem_set[mix ? 1 : 0][shp] < std::max<size_t>(smem, 1)) {
        if (mipwa_grad_set_smem(c->n_spin, c->model_flags, mix, shp, smem) != cudaSuccess)
            return fail(c, MIPWA_ERR_CUDA, "k_grad_recompute: shared-memory request refused");
        c->grad_smem_set[mix ? 1 : 0][shp] = std::max<size_t>(smem, 1);
    }
    if (c->gpartials_len < (size_t)grid * NVB) {
        if (c->d_gpartials) cudaFree(c->d_gpartials);
        c->d_gpartials = nullptr; c->gpartials_len = 0;
        CU(c, cudaMalloc(&c->d_gpartials, (size_t)grid * NVB * sizeof(double)));
        c->gpartials_len = (size_t)grid * NVB;
    }
    const cudaError_t le = mipwa_launch_grad_recompute(c->n_spin, c->model_flags, mix, shp, grid, ev_blocks, smem, c->stream,
                                                       c->model, E.rec, kappa, n_ev, G.rec, n_nm, c->d_gpartials,
                                                       want_f ? c->d_f_ev : nullptr, want_f ? c->d_f_nm : nullptr);
    ++c->launches;
    CU(c, le);
    (void)launch_finalize(c, (2 * NVB + 7) / 8, c->d_gpartials, ev_blocks, ev_blocks + nm_blocks, NVB, 2, c->d_result);
    ++c->launches;
    CU(c, cudaGetLastError());
    out->NVB = NVB; out->nb = nb;
    out->ev = c->h_result; out->nm = c->h_result + NVB;
    return MIPWA_OK;
}

// the floating resonance whose shape sums k_grad_recompute can fold into its pass: exactly one, of spin 1 or 2, in a
// model with a compile-time signature.  Returns its spin (the SHP template argument) or 0.
static int foldable_shape(const mipwa_ctx* c)
{
    if (c->F != 1 || c->n_spin[0] != 0 || c->n_spin[1] > MIPWA_SIG_MAX1 || c->n_spin[2] > MIPWA_SIG_MAX2) return 0;
    for (int r = 0; r < c->R; ++r)
        if (c->res[r].shape_floats) return c->res[r].spin == 1 || c->res[r].spin == 2 ? c->res[r].spin : 0;
    return 0;
}

// value + gradient on the recompute path.  full: also d/d(mass, width) of every floating resonance (grad has n_params
// entries then); one floating resonance of spin 1 or 2 costs no extra pass (SHP), otherwise k_grad_shape runs afterwards.
static int nll_grad_recompute(mipwa_ctx* c, const double* params, int64_t n_params, bool full, double* nll, double* grad)
{
    int rc = build_model(c, params, n_params);
    if (rc) return rc;
    const int N = c->N, R = c->R, Rd = (int)c->perm.size(), F = c->F, pb = c->pb();
    const int shp = full ? foldable_shape(c) : 0;
    const bool want_f = full && F > 0 && !shp;
    if (want_f) {                                          // room for the per-point factors k_grad_shape reads
        if (c->f_ev_len < c->ev.n) {
            if (c->d_f_ev) cudaFree(c->d_f_ev);
            c->d_f_ev = nullptr; c->f_ev_len = 0;
            CU(c, cudaMalloc(&c->d_f_ev, (size_t)std::max<int64_t>(c->ev.n, 1) * sizeof(double2)));
            c->f_ev_len = c->ev.n;
        }
        if (c->f_nm_len < c->nm.n) {
            if (c->d_f_nm) cudaFree(c->d_f_nm);
            c->d_f_nm = nullptr; c->f_nm_len = 0;
            CU(c, cudaMalloc(&c->d_f_nm, (size_t)c->nm.n * sizeof(double2)));
            c->f_nm_len = c->nm.n;
        }
    }
    { const int trc = timing_begin(c); if (trc) return trc; }
    GradTotals t;
    rc = launch_grad_recompute(c, false, shp, 0.0, true, true, want_f, &t);
    if (rc) return rc;
    rc = wait_grad(c);
    if (rc) return rc;

    // ---- host: O(N + R) combine (A7) and adjoint of the coefficient maps ----------------------------------------------
    const double wn = c->nm.w ? 1.0 : 1.0 / (double)c->nm.n;          // w == NULL: the records carry weight 1
    const double S = t.ev[0], I = t.nm[0] * wn;
    const double n_ev = (double)c->ev.n;
    *nll = -S + n_ev * std::log(I);
    const double scale = c->ev.n > 0 ? 2.0 * n_ev / I * wn : 0.0;
    const double *Fe = t.F(t.ev), *Fn = t.F(t.nm), *Be = t.bins(t.ev, Rd), *Bn = t.bins(t.nm, Rd);
    std::vector<double> Gsc(t.nb), Gy(2 * N), Gr(2 * std::max(R, 1), 0.0);
    auto emit = [&](double se, double sn, double* out) {   // out = se * (event part) + sn * (normalisation part)
        for (int k = 0; k < t.nb; ++k) Gsc[k] = se * Be[k] + sn * Bn[k];
        spline_adjoint(c, Gsc.data(), Gy.data());
        for (int d = 0; d < Rd; ++d) {
            const int r = c->perm[d];
            Gr[2 * r] = c->res_fold[d] * (se * Fe[2 * d] + sn * Fn[2 * d]);
            Gr[2 * r + 1] = c->res_fold[d] * (se * Fe[2 * d + 1] + sn * Fn[2 * d + 1]);
        }
        offset_rule(c, Gy.data(), Gr.data());
        polar_chain(c, params, Gy.data(), Gr.data(), out);
    };
    emit(1.0, scale, grad);
    if (c->parts_ev) {                                     // mipwa_nll_grad_parts: d(-S)/dtheta and dI/dtheta apart
        emit(1.0, 0.0, c->parts_ev);
        emit(0.0, 2.0 * wn, c->parts_nm);
        c->parts_S = S; c->parts_I = I;
    }
    if (!full || F == 0) return MIPWA_OK;

    // ---- d/d(mass, width): sums of f conj(dT'/dm0), f conj(dT'/dG0) per floating resonance and set -----------------------
    auto put = [&](int f, const ResDev& rd, const double* e, const double* g) {   // e, g: [dm_re, dm_im, dG_re, dG_im]
        for (int q = 0; q < 2; ++q) {                      // q = 0: mass, 1: width
            const double dr = e[2 * q] + scale * g[2 * q], di = e[2 * q + 1] + scale * g[2 * q + 1];
            grad[pb + 2 * R + 2 * f + q] = rd.cre * dr + rd.cim * di;             // Re(conj(c sqrt(n_R n_D)) D)
            if (c->parts_ev) {
                c->parts_ev[pb + 2 * R + 2 * f + q] = rd.cre * e[2 * q] + rd.cim * e[2 * q + 1];
                c->parts_nm[pb + 2 * R + 2 * f + q] = 2.0 * wn * (rd.cre * g[2 * q] + rd.cim * g[2 * q + 1]);
            }
        }
    };
    if (shp) {                                             // folded into the pass: first device slot of that spin
        put(0, c->model.res[shp == 1 ? 0 : c->n_spin[1]], t.shape(t.ev, Rd), t.shape(t.nm, Rd));
        return MIPWA_OK;
    }
    constexpr int SHAPE_OFF = 3900;                        // in h_result, clear of the main gradient's 2 NVB <= 2144 values
    std::vector<int> slots;                                // device slot of each floating resonance, list order
    for (int f = 0; f < F; ++f)
        for (int d = 0; d < c->model.R; ++d)
            if (c->model.res[d].fl == f) slots.push_back(d);
    if ((int)slots.size() != F) return fail(c, MIPWA_ERR_STATE, "floating resonance not found in the device model");
    const int64_t need = (std::max(c->ev.n, c->nm.n) + 511) / 512;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)c->sm_count, need));
    const size_t want = (size_t)grid * 8 * MIPWA_SHAPE_MAXF;
    if (c->gpartials_len < want) {
        if (c->d_gpartials) cudaFree(c->d_gpartials);
        c->d_gpartials = nullptr; c->gpartials_len = 0;
        CU(c, cudaMalloc(&c->d_gpartials, want * sizeof(double)));
        c->gpartials_len = want;
    }
    const Slot& E = c->ev_sorted;
    const Slot& G = c->nm_sorted;
    float ms_total = c->last_ms;
    for (int f0 = 0; f0 < F; f0 += MIPWA_SHAPE_MAXF) {
        const int nf = std::min(MIPWA_SHAPE_MAXF, F - f0);
        ShapeSel sel;
        for (int q = 0; q < MIPWA_SHAPE_MAXF; ++q) sel.slot[q] = slots[f0 + std::min(q, nf - 1)];
        { const int trc = timing_begin(c); if (trc) return trc; }
#define MIPWA_SHAPE_LAUNCH(NF, LT)                                                                                 \
    do {                                                                                                           \
        if (c->model_flags & MIPWA_FL_EQM)                                                                         \
            k_grad_shape<NF, MIPWA_FL_EQM, LT><<<grid, 512, 0, c->stream>>>(c->model, sel, E.s12, E.s13, c->d_f_ev, E.n, \
                                                                            G.s12, G.s13, c->d_f_nm, G.n, c->d_gpartials); \
        else                                                                                                       \
            k_grad_shape<NF, 0, LT><<<grid, 512, 0, c->stream>>>(c->model, sel, E.s12, E.s13, c->d_f_ev, E.n, G.s12, \
                                                                 G.s13, c->d_f_nm, G.n, c->d_gpartials);           \
    } while (0)
        switch (nf) {
            case 1:                                        // one floating resonance: its spin is a template argument
                switch (c->model.res[sel.slot[0]].L) {
                    case 0: MIPWA_SHAPE_LAUNCH(1, 0); break;
                    case 1: MIPWA_SHAPE_LAUNCH(1, 1); break;
                    default: MIPWA_SHAPE_LAUNCH(1, 2); break;
                }
                break;
            case 2: MIPWA_SHAPE_LAUNCH(2, -1); break;
            case 3: MIPWA_SHAPE_LAUNCH(3, -1); break;
            default: MIPWA_SHAPE_LAUNCH(4, -1); break;
        }
#undef MIPWA_SHAPE_LAUNCH
        ++c->launches;
        CU(c, cudaGetLastError());
        k_grad_finalize<<<(8 * nf + 7) / 8, 256, 0, c->stream>>>(c->d_gpartials, grid, grid, 8 * nf, 1, c->d_result + SHAPE_OFF,
                                                                 nullptr, nullptr, 0);
        ++c->launches;
        CU(c, cudaGetLastError());
        if (c->timing) CU(c, cudaEventRecord(c->ev1, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
        if (c->timing) { float ms = 0.f; CU(c, cudaEventElapsedTime(&ms, c->ev0, c->ev1)); ms_total += ms; }
        const double* D = c->h_result + SHAPE_OFF;         // [pass][f][dm_re, dm_im, dG_re, dG_im]
        for (int q = 0; q < nf; ++q) put(f0 + q, c->model.res[slots[f0 + q]], D + (0 * nf + q) * 4, D + (1 * nf + q) * 4);
    }
    c->last_ms = ms_total;
    return MIPWA_OK;
}

static int nll_grad_any(mipwa_ctx* c, const double* params, int64_t n_params, bool full, double* nll, double* grad)
{
    if (!c || !params || !nll || !grad) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    int rc = use_device(c);
    if (rc) return rc;
    rc = prepare_sorted(c);
    if (rc) return rc;
    if (effective_path(c) == MIPWA_PATH_CACHED_COMPACT) return nll_grad_compact(c, params, n_params, nll, grad);
    return nll_grad_recompute(c, params, n_params, full, nll, grad);
}

int mipwa_nll_grad(mipwa_ctx* c, const double* params, int64_t n_params, double* nll, double* grad)
{
    NvtxRange range("mipwa_nll_grad");
    return nll_grad_any(c, params, n_params, false, nll, grad);
}

// value + gradient over ALL n_params parameters: the 2N + 2R linear-coefficient parameters, then (mass, width) of every
// floating resonance (layout of grad = layout of params)
int mipwa_nll_grad_full(mipwa_ctx* c, const double* params, int64_t n_params, double* nll, double* grad)
{
    NvtxRange range("mipwa_nll_grad_full");
    return nll_grad_any(c, params, n_params, true, nll, grad);
}

// the pieces one rank of a sharded likelihood contributes (include/mipwa.h): same launches as
// mipwa_nll_grad_full, the host combine run once more per piece
int mipwa_nll_grad_parts(mipwa_ctx* c, const double* params, int64_t n_params, double* sum_log, double* integral,
                         double* grad_ev, double* grad_nm)
{
    if (!c) return MIPWA_ERR_ARG;
    if (!params || !sum_log || !integral || !grad_ev || !grad_nm) return fail(c, MIPWA_ERR_ARG, "null argument");
    if (n_params != c->n_par()) return fail(c, MIPWA_ERR_ARG, "wrong n_params");
    NvtxRange range("mipwa_nll_grad_parts");
    std::vector<double> total((size_t)std::max<int64_t>(n_params, 1));
    double nll = 0.0;
    c->parts_ev = grad_ev; c->parts_nm = grad_nm;
    const int rc = nll_grad_any(c, params, n_params, true, &nll, total.data());
    c->parts_ev = c->parts_nm = nullptr;
    if (rc) return rc;
    *sum_log = c->parts_S; *integral = c->parts_I;
    return MIPWA_OK;
}

// ---- signal + background mixture (include/mipwa.h): recompute path, two launches -----------------------------------
int mipwa_set_event_background(mipwa_ctx* c, const double* b, int32_t mem)
{
    if (!c) return MIPWA_ERR_ARG;
    if (c->ev.n < 0) return fail(c, MIPWA_ERR_STATE, "set the events first");
    if (mem != MIPWA_MEM_HOST && mem != MIPWA_MEM_DEVICE) return fail(c, MIPWA_ERR_ARG, "bad mem flag");
    int rc = use_device(c);
    if (rc) return rc;
    CU(c, cudaStreamSynchronize(c->stream));
    Slot& s = c->ev;
    if (s.owned[2]) { cudaFree(s.owned[2]); s.owned[2] = nullptr; }
    s.w = nullptr;
    drop_records(s);                                       // the event records carry the densities
    c->ev_sorted_valid = false;                            // the cell-sorted copy carries the densities along
    c->cache_valid = false; c->hyb_ev_valid = false;       // the caches follow the event order of the sorted copy
    if (!b || s.n == 0) return MIPWA_OK;                   // NULL clears
    if (mem == MIPWA_MEM_HOST || ((uintptr_t)b & 7u)) {
        CU(c, cudaMalloc(&s.owned[2], (size_t)s.n * sizeof(double)));
        CU(c, cudaMemcpyAsync(s.owned[2], b, (size_t)s.n * sizeof(double), cudaMemcpyDefault, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
        s.w = (const double*)s.owned[2];
    } else {
        s.w = b;
    }
    return MIPWA_OK;
}

// I from a normalisation-only launch, then the event sum of ln(|A|^2 + kappa b), kappa = I (1 - f_s) / f_s:
// NLL = -sum_i ln(f_s |A_i|^2 / I + (1 - f_s) b_i) = -sum_i ln(|A_i|^2 + kappa b_i) - n_ev ln(f_s / I)
int mipwa_nll_mix(mipwa_ctx* c, const double* params, int64_t n_params, double f_sig, double* nll)
{
    if (!c || !params || !nll) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    if (c->ev.n > 0 && !c->ev.w) return fail(c, MIPWA_ERR_STATE, "set the background densities (mipwa_set_event_background)");
    if (!(f_sig > 0.0 && f_sig <= 1.0)) return fail(c, MIPWA_ERR_ARG, "signal fraction must be in (0, 1]");
    NvtxRange range("mipwa_nll_mix");
    int rc = use_device(c);
    if (rc) return rc;
    rc = build_model(c, params, n_params);
    if (rc) return rc;
    Slot& E = evs(c);
    Slot& G = nms(c);
    rc = ensure_records(c, E, 0.0);
    if (rc) return rc;
    rc = ensure_records(c, G, 1.0);
    if (rc) return rc;
    const int grid = recompute_grid(c, std::max(E.n, G.n));
    const bool timing = c->timing;
    { const int trc = timing_begin(c); if (trc) return trc; }
    c->timing = false;                                     // wait_result polls: one pair of events spans both launches
    // Launch 1: the normalisation points alone; with events to follow its totals stay in DEVICE memory and launch 2 (events,
    // D_i = |A_i|^2 + kappa b_i) reads the integral from there: kappa = I (1 - f_s) / f_s is formed on the device, the host
    // waits once, and launch 2 hands the integral on beside its own sum.
    const double wn = c->nm.w ? 1.0 : 1.0 / (double)c->nm.n;
    long long tag = next_tag(c);
    cudaError_t le = mipwa_launch_nll_recompute(c->n_spin, c->model_flags, false, grid, c->stream, c->model, E.rec, 0.0, 0,
                                                G.rec, G.n, c->d_partials, c->d_ticket,
                                                E.n > 0 ? c->d_dev_result : c->result_dst, tag);
    ++c->launches;
    double S = 0.0;
    if (le == cudaSuccess && E.n > 0) {
        tag = next_tag(c);
        le = mipwa_launch_nll_recompute_mix(c->n_spin, c->model_flags, grid, c->stream, c->model, E.rec,
                                            wn * (1.0 - f_sig) / f_sig, E.n, G.rec, 0, c->d_partials, c->d_ticket,
                                            c->result_dst, tag, c->d_dev_result + 1);
        ++c->launches;
    }
    if (le == cudaSuccess) rc = wait_result(c, tag);
    if (E.n > 0) S = c->h_result[0];
    const double I = c->h_result[1] * wn;
    c->timing = timing;
    CU(c, le);
    if (rc) return rc;
    if (timing) {
        CU(c, cudaEventRecord(c->ev1, c->stream));
        CU(c, cudaEventSynchronize(c->ev1));
        CU(c, cudaEventElapsedTime(&c->last_ms, c->ev0, c->ev1));
    }
    *nll = -S - (double)c->ev.n * std::log(f_sig / I);
    return MIPWA_OK;
}

// value + gradient of the mixture: k_grad_recompute twice.  Launch 1 over the normalisation points alone gives I, F_nm
// and the normalisation moments; launch 2 over the events alone with kappa = I (1 - f_s) / f_s gives sum ln D_i,
// Q = sum b_i / D_i (D_i = |A_i|^2 + kappa b_i), F_ev and the event moments, f_i = -2 A_i / D_i.  Then
//   NLL = -sum ln D_i - n ln(f_s / I),  calG = G_ev + (2 / I) (n - kappa Q) G_nm,  dNLL/df_s = -(n - I Q / f_s) / f_s.
int mipwa_nll_mix_grad(mipwa_ctx* c, const double* params, int64_t n_params, double f_sig, double* nll, double* grad,
                       double* dnll_dfsig)
{
    if (!c || !params || !nll || !grad) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    if (c->ev.n > 0 && !c->ev.w) return fail(c, MIPWA_ERR_STATE, "set the background densities (mipwa_set_event_background)");
    if (!(f_sig > 0.0 && f_sig <= 1.0)) return fail(c, MIPWA_ERR_ARG, "signal fraction must be in (0, 1]");
    NvtxRange range("mipwa_nll_mix_grad");
    int rc = use_device(c);
    if (rc) return rc;
    rc = prepare_sorted(c);
    if (rc) return rc;
    rc = build_model(c, params, n_params);
    if (rc) return rc;
    const int N = c->N, R = c->R, Rd = (int)c->perm.size();
    const double wn = c->nm.w ? 1.0 : 1.0 / (double)c->nm.n;
    { const int trc = timing_begin(c); if (trc) return trc; }
    GradTotals t;
    rc = launch_grad_recompute(c, false, 0, 0.0, false, true, false, &t);      // normalisation points alone
    if (rc) return rc;
    CU(c, cudaStreamSynchronize(c->stream));
    std::vector<double> hn(t.nm, t.nm + t.NVB), he(t.NVB, 0.0);
    const double I = hn[0] * wn, n_ev = (double)c->ev.n, kappa = I * (1.0 - f_sig) / f_sig;
    if (c->ev.n > 0) {
        rc = launch_grad_recompute(c, true, 0, kappa, true, false, false, &t); // events alone, D = |A|^2 + kappa b
        if (rc) return rc;
    }
    if (c->timing) CU(c, cudaEventRecord(c->ev1, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    if (c->timing) CU(c, cudaEventElapsedTime(&c->last_ms, c->ev0, c->ev1));
    if (c->ev.n > 0) he.assign(t.ev, t.ev + t.NVB);

    const double S = he[0], Q = he[1];
    *nll = -S - n_ev * std::log(f_sig / I);
    if (dnll_dfsig) *dnll_dfsig = -(n_ev - I * Q / f_sig) / f_sig;
    const double scale = 2.0 * (n_ev - kappa * Q) / I * wn;
    const double *Fe = t.F(he.data()), *Fn = t.F(hn.data()), *Be = t.bins(he.data(), Rd), *Bn = t.bins(hn.data(), Rd);
    std::vector<double> Gsc(t.nb), Gy(2 * N), Gr(2 * std::max(R, 1), 0.0);
    for (int k = 0; k < t.nb; ++k) Gsc[k] = Be[k] + scale * Bn[k];
    spline_adjoint(c, Gsc.data(), Gy.data());
    for (int d = 0; d < Rd; ++d) {
        const int r = c->perm[d];
        Gr[2 * r] = c->res_fold[d] * (Fe[2 * d] + scale * Fn[2 * d]);
        Gr[2 * r + 1] = c->res_fold[d] * (Fe[2 * d + 1] + scale * Fn[2 * d + 1]);
    }
    offset_rule(c, Gy.data(), Gr.data());
    polar_chain(c, params, Gy.data(), Gr.data(), grad);
    return MIPWA_OK;
}

// ---- sharded mixture likelihood (include/mipwa.h): the event sum needs the integral of the WHOLE sample, so a call is two
// phases with one exchange between them -----------------------------------------------------------------------------------
// phase 1: this rank's I_r = sum_j w_j |A_j|^2 and dI_r/dtheta over the 2N + 2R linear-coefficient parameters
int mipwa_norm_parts(mipwa_ctx* c, const double* params, int64_t n_params, double* integral, double* grad_nm)
{
    if (!c || !params || !integral) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    NvtxRange range("mipwa_norm_parts");
    int rc = use_device(c);
    if (rc) return rc;
    rc = prepare_sorted(c);
    if (rc) return rc;
    rc = build_model(c, params, n_params);
    if (rc) return rc;
    const int N = c->N, R = c->R, Rd = (int)c->perm.size();
    const double wn = c->nm.w ? 1.0 : 1.0 / (double)c->nm.n;
    GradTotals t;
    rc = launch_grad_recompute(c, false, 0, 0.0, false, true, false, &t);
    if (rc) return rc;
    CU(c, cudaStreamSynchronize(c->stream));
    *integral = t.nm[0] * wn;
    if (!grad_nm) return MIPWA_OK;
    const double *Fn = t.F(t.nm), *Bn = t.bins(t.nm, Rd);
    std::vector<double> Gsc(t.nb), Gy(2 * N), Gr(2 * std::max(R, 1), 0.0);
    for (int k = 0; k < t.nb; ++k) Gsc[k] = 2.0 * wn * Bn[k];
    spline_adjoint(c, Gsc.data(), Gy.data());
    for (int d = 0; d < Rd; ++d) {
        const int r = c->perm[d];
        Gr[2 * r] = c->res_fold[d] * 2.0 * wn * Fn[2 * d];
        Gr[2 * r + 1] = c->res_fold[d] * 2.0 * wn * Fn[2 * d + 1];
    }
    offset_rule(c, Gy.data(), Gr.data());
    polar_chain(c, params, Gy.data(), Gr.data(), grad_nm);
    return MIPWA_OK;
}

// phase 2, with I of the whole sample: S_r = sum_i ln(|A_i|^2 + kappa b_i), Q_r = sum_i b_i / D_i and d(-S_r)/dtheta at
// fixed kappa = I (1 - f_s) / f_s, over this rank's events
int mipwa_nll_mix_parts(mipwa_ctx* c, const double* params, int64_t n_params, double f_sig, double integral_total,
                        double* sum_log, double* q, double* grad_ev)
{
    if (!c || !params || !sum_log || !q) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    if (c->ev.n > 0 && !c->ev.w) return fail(c, MIPWA_ERR_STATE, "set the background densities (mipwa_set_event_background)");
    if (!(f_sig > 0.0 && f_sig <= 1.0) || !(integral_total > 0.0)) return fail(c, MIPWA_ERR_ARG, "need 0 < f_sig <= 1 and I > 0");
    NvtxRange range("mipwa_nll_mix_parts");
    int rc = use_device(c);
    if (rc) return rc;
    rc = prepare_sorted(c);
    if (rc) return rc;
    rc = build_model(c, params, n_params);
    if (rc) return rc;
    const int N = c->N, R = c->R, Rd = (int)c->perm.size(), P = 2 * c->Np + 2 * R;
    *sum_log = 0.0; *q = 0.0;
    if (grad_ev) for (int k = 0; k < P; ++k) grad_ev[k] = 0.0;
    if (c->ev.n == 0) return MIPWA_OK;
    const double kappa = integral_total * (1.0 - f_sig) / f_sig;
    GradTotals t;
    rc = launch_grad_recompute(c, true, 0, kappa, true, false, false, &t);
    if (rc) return rc;
    CU(c, cudaStreamSynchronize(c->stream));
    *sum_log = t.ev[0]; *q = t.ev[1];
    if (!grad_ev) return MIPWA_OK;
    const double *Fe = t.F(t.ev), *Be = t.bins(t.ev, Rd);
    std::vector<double> Gy(2 * N), Gr(2 * std::max(R, 1), 0.0);
    spline_adjoint(c, Be, Gy.data());
    for (int d = 0; d < Rd; ++d) {
        const int r = c->perm[d];
        Gr[2 * r] = c->res_fold[d] * Fe[2 * d];
        Gr[2 * r + 1] = c->res_fold[d] * Fe[2 * d + 1];
    }
    offset_rule(c, Gy.data(), Gr.data());
    polar_chain(c, params, Gy.data(), Gr.data(), grad_ev);
    return MIPWA_OK;
}

// whole-sample mixture likelihood from the gathered pieces, sums in rank order:
//   norm_parts[r] = (I_r, dI_r/dtheta[P]),  ev_parts[r] = (S_r, Q_r, n_r, d(-S_r)/dtheta[P]);  I = sum I_r must be the
//   value phase 2 was given.   NLL = -S - n ln(f_s / I),  grad = sum grad_ev + ((n - kappa Q) / I) sum dI/dtheta,
//   dNLL/df_s = -(n - I Q / f_s) / f_s.  Host only.
int mipwa_combine_mix_parts(int32_t n_ranks, int64_t n_lin, double f_sig, const double* norm_parts, const double* ev_parts,
                            double* nll, double* grad, double* dnll_dfsig)
{
    if (n_ranks < 1 || n_lin < 0 || !norm_parts || !ev_parts || !nll || !(f_sig > 0.0 && f_sig <= 1.0)) return MIPWA_ERR_ARG;
    const int64_t P = n_lin, sn = 1 + P, se = 3 + P;
    double I = 0.0, S = 0.0, Q = 0.0, n = 0.0;
    for (int r = 0; r < n_ranks; ++r) {
        I += norm_parts[r * sn];
        S += ev_parts[r * se]; Q += ev_parts[r * se + 1]; n += ev_parts[r * se + 2];
    }
    const double kappa = I * (1.0 - f_sig) / f_sig;
    *nll = -S - n * std::log(f_sig / I);
    if (dnll_dfsig) *dnll_dfsig = -(n - I * Q / f_sig) / f_sig;
    if (grad)
        for (int64_t k = 0; k < P; ++k) {
            double ge = 0.0, gn = 0.0;
            for (int r = 0; r < n_ranks; ++r) { ge += ev_parts[r * se + 3 + k]; gn += norm_parts[r * sn + 1 + k]; }
            grad[k] = ge + (n - kappa * Q) / I * gn;
        }
    return MIPWA_OK;
}

// ---- Hessian in the linear-coefficient parameters, fixed shapes (include/mipwa.h) ---------------------------------------
// Dense parametrisation: c = [y_k (knot values), c_r (list order, the constant term with its column of ones)], K = N + R
// entries; a model without spline has two stand-in knots in its tables (k < N - Np) that are no parameters.
int64_t mipwa_hessian_parts_len(const mipwa_ctx* c) { return c ? 2 * (int64_t)(c->N + c->R) * (c->N + c->R) : MIPWA_ERR_ARG; }

// this rank's sums: M_kl = sum_i B_ik B_il / A_i^2 over ITS events (k_gram in HESS mode) and the Gram matrix G over ITS
// normalisation points; both K x K complex, row-major, (re, im) interleaved.  Summed over the ranks they are the
// whole-sample matrices mipwa_hessian_assemble takes.
static int hessian_parts_at(mipwa_ctx* c, const double* params, int64_t n_params, double* M, double* G)
{
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    const int K = c->N + c->R;
    int rc = use_device(c);
    if (rc) return rc;
    rc = ensure_gram(c, params);                           // floating shapes: the basis at the shapes of `params`
    if (rc) return rc;
    rc = build_model(c, params, n_params);                 // y_k of this call for fill_coef
    if (rc) return rc;
    CoefDev cc;
    fill_coef(c, params, &cc);
    rc = build_unit_model(c, params);                      // the basis kernels evaluate the unit-coefficient model
    if (rc) return rc;
    const Slot& E = evs(c);
    const int nt = (K + 3) / 4, ntile = nt * (nt + 1) / 2, tpt = (ntile + MIPWA_TILE - 1) / MIPWA_TILE;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((E.n + GRAM_P - 1) / GRAM_P, c->sm_count));
    const size_t smem = (size_t)4 * nt * GRAM_LD * sizeof(double2);
    double2 *partial = nullptr, *d_M = nullptr;
    for (size_t t = 0; t < (size_t)2 * K * K; ++t) M[t] = 0.0;
    cudaError_t e = cudaMalloc(&partial, (size_t)grid * K * K * sizeof(double2));
    if (e == cudaSuccess) e = cudaMalloc(&d_M, (size_t)K * K * sizeof(double2));
    if (e == cudaSuccess && E.n > 0) {
#define MIPWA_HESS_LAUNCH(T)                                                                                         \
    do {                                                                                                             \
        e = cudaFuncSetAttribute(k_gram<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);           \
        if (e == cudaSuccess)                                                                                        \
            k_gram<T, true><<<grid, MIPWA_TILE, smem, c->stream>>>(c->model, c->d_search, basis_aux(c), cc, E.s12,   \
                                                                    E.s13, nullptr, E.n, 0.0, partial);              \
    } while (0)
        if (tpt <= 1) MIPWA_HESS_LAUNCH(1); else if (tpt == 2) MIPWA_HESS_LAUNCH(2); else MIPWA_HESS_LAUNCH(3);
#undef MIPWA_HESS_LAUNCH
        ++c->launches;
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) {
            k_gram_reduce<<<(K * K + 255) / 256, 256, 0, c->stream>>>(partial, grid, K, d_M, 0);
            ++c->launches;
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(M, d_M, (size_t)K * K * sizeof(double2), cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    }
    if (partial) cudaFree(partial);
    if (d_M) cudaFree(d_M);
    if (e != cudaSuccess)
        return fail(c, e == cudaErrorMemoryAllocation ? MIPWA_ERR_NOMEM : MIPWA_ERR_CUDA, std::string("hessian: ") + cudaGetErrorString(e));
    std::memcpy(G, c->h_gram.data(), (size_t)2 * K * K * sizeof(double));
    return MIPWA_OK;
}

int mipwa_hessian_parts(mipwa_ctx* c, const double* params, int64_t n_params, double* M, double* G)
{
    if (!c || !params || !M || !G) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    if (c->F > 0) return fail(c, MIPWA_ERR_STATE, "the analytic Hessian needs fixed resonance shapes");
    return hessian_parts_at(c, params, n_params, M, G);
}

// Hessian of the whole sample from the summed pieces: M, G (mipwa_hessian_parts, added over the ranks), the event count
// and the polar gradient of the whole sample (mipwa_nll_grad, or the combined mipwa_nll_grad_parts).  Host only.
// the block of the linear-coefficient parameters of a P x P matrix (P = n_params: the rows and columns of floating masses
// and widths, if any, are left at zero)
static int hessian_assemble_at(mipwa_ctx* c, const double* params, int64_t n_params, int64_t n_ev_total, const double* hM,
                               const double* hG, const double* gpol, double* hess)
{
    const int N = c->N, Np = c->Np, R = c->R, K = N + R, P = c->n_par(), pb = c->pb(), k0 = N - Np;
    int rc = build_model(c, params, n_params);
    if (rc) return rc;
    CoefDev cc;
    fill_coef(c, params, &cc);
    // ---- host: O(K^2) assembly.  Wirtinger blocks from M, G, c, then the polar chain rule -------------------------------
    typedef std::complex<double> cx;
    auto Gm = [&](int k, int l) { return cx(hG[2 * ((size_t)k * K + l)], hG[2 * ((size_t)k * K + l) + 1]); };
    auto Mm = [&](int k, int l) { return cx(hM[2 * ((size_t)k * K + l)], hM[2 * ((size_t)k * K + l) + 1]); };
    std::vector<cx> cv(K), cG(K), Gc(K), e1(K), g(K);
    std::vector<int> ir(K, 0), ip(K, 0);
    for (int k = 0; k < K; ++k) cv[k] = cx(cc.c[k].x, cc.c[k].y);
    for (int k = k0; k < K; ++k) {
        ir[k] = k < N ? k : pb + 2 * (k - N);
        ip[k] = k < N ? Np + k : pb + 2 * (k - N) + 1;
        e1[k] = cx(std::cos(params[ip[k]]), std::sin(params[ip[k]]));
        if (!(std::fabs(params[ir[k]]) > 0.0))
            return fail(c, MIPWA_ERR_ARG, "mipwa_hessian_assemble: a zero magnitude makes the polar Hessian singular");
    }
    cx Iq = 0.0;
    for (int k = 0; k < K; ++k) {
        cx a = 0.0, b = 0.0;
        for (int l = 0; l < K; ++l) { a += std::conj(cv[l]) * Gm(l, k); b += Gm(k, l) * cv[l]; }
        cG[k] = a; Gc[k] = b;
    }
    for (int k = 0; k < K; ++k) Iq += std::conj(cv[k]) * Gc[k];
    const double I = Iq.real(), nev = (double)n_ev_total;
    // dNLL/dc_k from the polar gradient: dNLL/drho = 2 Re(g e^{i phi}), dNLL/dphi = 2 Re(g i c) = -2 rho Im(g e^{i phi})
    for (int k = k0; k < K; ++k) {
        const double rho = params[ir[k]];
        g[k] = 0.5 * cx(gpol[ir[k]], -gpol[ip[k]] / rho) * std::conj(e1[k]);
    }
    for (int t = 0; t < P * P; ++t) hess[t] = 0.0;
    for (int k = k0; k < K; ++k)
        for (int l = k0; l < K; ++l) {
            const cx hcc = Mm(k, l) - nev * cG[k] * cG[l] / (I * I);
            const cx hcb = nev * Gm(l, k) / I - nev * cG[k] * Gc[l] / (I * I);
            const cx dk[2] = { e1[k], cx(0.0, 1.0) * cv[k] }, dl[2] = { e1[l], cx(0.0, 1.0) * cv[l] };
            const int ik[2] = { ir[k], ip[k] }, il[2] = { ir[l], ip[l] };
            for (int a = 0; a < 2; ++a)
                for (int b = 0; b < 2; ++b)
                    hess[(size_t)ik[a] * P + il[b]] += 2.0 * (hcc * dk[a] * dl[b] + hcb * dk[a] * std::conj(dl[b])).real();
        }
    for (int k = k0; k < K; ++k) {
        const double rp = 2.0 * (g[k] * cx(0.0, 1.0) * e1[k]).real(), pp = 2.0 * (g[k] * (-cv[k])).real();
        hess[(size_t)ir[k] * P + ip[k]] += rp;
        hess[(size_t)ip[k] * P + ir[k]] += rp;
        hess[(size_t)ip[k] * P + ip[k]] += pp;
    }
    return MIPWA_OK;
}


int mipwa_hessian_assemble(mipwa_ctx* c, const double* params, int64_t n_params, int64_t n_ev_total, const double* hM,
                           const double* hG, const double* gpol, double* hess)
{
    if (!c || !params || !hM || !hG || !gpol || !hess) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    if (c->F > 0) return fail(c, MIPWA_ERR_STATE, "the analytic Hessian needs fixed resonance shapes");
    return hessian_assemble_at(c, params, n_params, n_ev_total, hM, hG, gpol, hess);
}

// Hessian over ALL n_params parameters ("correlations between the parameters").  The block of
// the linear coefficients is the analytic one, evaluated with the basis at the CURRENT masses and widths; the rows and
// columns of the floating masses and widths are central differences of the analytic gradient (mipwa_nll_grad_full) in
// that one parameter, Richardson-extrapolated from the steps h and h / 2, h = 1e-3 x the resonance's width: four
// gradient calls per floating shape parameter, relative accuracy ~1e-8.
int mipwa_nll_hessian_full(mipwa_ctx* c, const double* params, int64_t n_params, double* nll, double* grad, double* hess)
{
    if (!c || !params || !nll || !hess) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    if (c->F == 0) return mipwa_nll_hessian(c, params, n_params, nll, grad, hess);
    NvtxRange range("mipwa_nll_hessian_full");
    const int P = c->n_par(), K = c->N + c->R, Pl = c->pb() + 2 * c->R;
    std::vector<double> g0(P), M((size_t)2 * K * K), G((size_t)2 * K * K);
    int rc = mipwa_nll_grad_full(c, params, n_params, nll, g0.data());
    if (rc) return rc;
    if (grad) std::memcpy(grad, g0.data(), P * sizeof(double));
    rc = hessian_parts_at(c, params, n_params, M.data(), G.data());
    if (rc) return rc;
    rc = hessian_assemble_at(c, params, n_params, c->ev.n, M.data(), G.data(), g0.data(), hess);
    if (rc) return rc;
    std::vector<double> p(params, params + P), gp(P), gm(P), row(P);
    for (int s = 0; s < 2 * c->F; ++s) {
        const int idx = Pl + s;
        const double h = 1e-3 * params[Pl + (s | 1)];      // the width of that resonance sets the scale of both
        for (int k = 0; k < P; ++k) row[k] = 0.0;
        for (int level = 0; level < 2; ++level) {
            const double hh = level == 0 ? h : 0.5 * h, wgt = level == 0 ? -1.0 / 3.0 : 4.0 / 3.0;
            double dummy;
            p[idx] = params[idx] + hh;
            rc = mipwa_nll_grad_full(c, p.data(), n_params, &dummy, gp.data());
            if (rc) return rc;
            p[idx] = params[idx] - hh;
            rc = mipwa_nll_grad_full(c, p.data(), n_params, &dummy, gm.data());
            if (rc) return rc;
            p[idx] = params[idx];
            for (int k = 0; k < P; ++k) row[k] += wgt * (gp[k] - gm[k]) / (2.0 * hh);
        }
        for (int k = 0; k < P; ++k) {
            if (k >= Pl && k < idx) {                      // shape-shape pair met from both sides: the mean of the two
                hess[(size_t)idx * P + k] = hess[(size_t)k * P + idx] = 0.5 * (hess[(size_t)k * P + idx] + row[k]);
            } else {
                hess[(size_t)idx * P + k] = hess[(size_t)k * P + idx] = row[k];
            }
        }
    }
    return MIPWA_OK;
}

// NLL, gradient and Hessian of one context's own sample
int mipwa_nll_hessian(mipwa_ctx* c, const double* params, int64_t n_params, double* nll, double* grad, double* hess)
{
    if (!c || !params || !nll || !hess) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    if (c->F > 0) return fail(c, MIPWA_ERR_STATE, "mipwa_nll_hessian needs fixed resonance shapes");
    NvtxRange range("mipwa_nll_hessian");
    const int P = c->n_par(), K = c->N + c->R;
    std::vector<double> gpol(P), M((size_t)2 * K * K), G((size_t)2 * K * K);
    int rc = mipwa_nll_grad(c, params, n_params, nll, gpol.data());
    if (rc) return rc;
    if (grad) std::memcpy(grad, gpol.data(), P * sizeof(double));
    rc = mipwa_hessian_parts(c, params, n_params, M.data(), G.data());
    if (rc) return rc;
    return mipwa_hessian_assemble(c, params, n_params, c->ev.n, M.data(), G.data(), gpol.data(), hess);
}

// ---- toy generation on the device (gen.cuh) -------------------------------------------------------------------------
namespace {
struct GenScratch {                 // device scratch of one mipwa_generate call; freed on every exit path
    unsigned long long* own = nullptr;
    double *cum = nullptr, *env = nullptr, *c12 = nullptr, *c13 = nullptr, *o12 = nullptr, *o13 = nullptr;
    unsigned char* flag = nullptr;
    int* nsel = nullptr;
    void* tmp = nullptr;
    ~GenScratch()
    {
        for (void* p : { (void*)own, (void*)cum, (void*)env, (void*)c12, (void*)c13, (void*)o12, (void*)o13,
                         (void*)flag, (void*)nsel, tmp })
            if (p) cudaFree(p);
    }
};
}  // namespace

int mipwa_generate(mipwa_ctx* c, const double* params, int64_t n_params, uint64_t key, int64_t n, int32_t n_side,
                   int32_t n_coarse, double* s12, double* s13, int32_t mem, int64_t* n_candidates)
{
    if (!c || !params) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    if (n < 0 || (n > 0 && (!s12 || !s13)) || n_side < 1 || n_side > 16384 || n_coarse < 1 || n_coarse > 1024 ||
        (mem != MIPWA_MEM_HOST && mem != MIPWA_MEM_DEVICE))
        return fail(c, MIPWA_ERR_ARG, "mipwa_generate: bad count, grid size, pointer or mem flag");
    int rc = use_device(c);
    if (rc) return rc;
    rc = build_model(c, params, n_params);
    if (rc) return rc;
    if (n_candidates) *n_candidates = 0;
    if (n == 0) return MIPWA_OK;
    const mipwa_kinematics& kk = c->kin;
    const GenKin gk = { kk.m_parent * kk.m_parent, kk.m1 * kk.m1, kk.m2 * kk.m2, kk.m3 * kk.m3,
                        (kk.m1 + kk.m2) * (kk.m1 + kk.m2), (kk.m_parent - kk.m3) * (kk.m_parent - kk.m3) };
    const int nc = n_coarse, ncell = nc * nc;
    const double h = (gk.hi - gk.lo) / n_side, H = (gk.hi - gk.lo) / nc;
    const int64_t batch = 1 << 21;
    GenScratch g;
    size_t tmp_bytes = 0;
    CU(c, cudaMalloc(&g.own, ncell * sizeof(unsigned long long)));
    CU(c, cudaMemsetAsync(g.own, 0, ncell * sizeof(unsigned long long), c->stream));
    CU(c, cudaMalloc(&g.cum, ncell * sizeof(double)));
    CU(c, cudaMalloc(&g.env, ncell * sizeof(double)));
    CU(c, cudaMalloc(&g.c12, batch * sizeof(double)));
    CU(c, cudaMalloc(&g.c13, batch * sizeof(double)));
    CU(c, cudaMalloc(&g.flag, batch));
    CU(c, cudaMalloc(&g.nsel, sizeof(int)));
    CU(c, cudaMalloc(&g.o12, (size_t)(n + batch) * sizeof(double)));
    CU(c, cudaMalloc(&g.o13, (size_t)(n + batch) * sizeof(double)));
    CU(c, cub::DeviceSelect::Flagged(nullptr, tmp_bytes, g.c12, g.flag, g.o12, g.nsel, (int)batch, c->stream));
    CU(c, cudaMalloc(&g.tmp, tmp_bytes ? tmp_bytes : 16));

    // envelope: fine-grid maxima per coarse cell on the device, neighbour fill and CDF on the host (O(n_coarse^2))
    const int64_t fine = (int64_t)n_side * n_side;
    k_gen_envelope<<<grid_for(c, fine, 8), 256, 0, c->stream>>>(c->model, c->d_search, gk, n_side, h, H, nc, g.own);
    ++c->launches;
    CU(c, cudaGetLastError());
    std::vector<unsigned long long> own_bits(ncell);
    CU(c, cudaMemcpyAsync(own_bits.data(), g.own, ncell * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    std::vector<double> own(ncell), env(ncell), cum(ncell);
    for (int t = 0; t < ncell; ++t) std::memcpy(&own[t], &own_bits[t], sizeof(double));
    for (int cx = 0; cx < nc; ++cx)
        for (int cy = 0; cy < nc; ++cy) {
            double v = own[cx * nc + cy];
            if (!(v > 0.0))
                for (int dx = -1; dx <= 1; ++dx)
                    for (int dy = -1; dy <= 1; ++dy) {
                        const int x = cx + dx, y = cy + dy;
                        if (x >= 0 && x < nc && y >= 0 && y < nc) v = std::max(v, own[x * nc + y]);
                    }
            env[cx * nc + cy] = 1.2 * v;
        }
    double run = 0.0;
    for (int t = 0; t < ncell; ++t) { run += env[t]; cum[t] = run; }
    if (!(run > 0.0) || !std::isfinite(run))
        return fail(c, MIPWA_ERR_DOMAIN, "mipwa_generate: |A|^2 vanishes or is not finite on the envelope grid");
    for (int t = 0; t < ncell; ++t) cum[t] /= run;
    CU(c, cudaMemcpyAsync(g.cum, cum.data(), ncell * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(g.env, env.data(), ncell * sizeof(double), cudaMemcpyHostToDevice, c->stream));

    int64_t have = 0, ctr = 0;
    while (have < n) {
        k_gen_candidates<<<grid_for(c, batch, 8), 256, 0, c->stream>>>(c->model, c->d_search, gk, (unsigned long long)key,
                                                                     ctr, batch, nc, H, g.cum, g.env, g.c12, g.c13, g.flag);
        ++c->launches;
        CU(c, cudaGetLastError());
        CU(c, cub::DeviceSelect::Flagged(g.tmp, tmp_bytes, g.c12, g.flag, g.o12 + have, g.nsel, (int)batch, c->stream));
        CU(c, cub::DeviceSelect::Flagged(g.tmp, tmp_bytes, g.c13, g.flag, g.o13 + have, g.nsel, (int)batch, c->stream));
        int nsel = 0;
        CU(c, cudaMemcpyAsync(&nsel, g.nsel, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
        have += nsel; ctr += batch;
        if (ctr > ((int64_t)1 << 40))
            return fail(c, MIPWA_ERR_DOMAIN, "mipwa_generate: acceptance below 1e-6, giving up");
    }
    const cudaMemcpyKind kind = mem == MIPWA_MEM_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    CU(c, cudaMemcpyAsync(s12, g.o12, (size_t)n * sizeof(double), kind, c->stream));
    CU(c, cudaMemcpyAsync(s13, g.o13, (size_t)n * sizeof(double), kind, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    if (n_candidates) *n_candidates = ctr;
    return MIPWA_OK;
}

}  // extern "C"

// ---- allocation-free likelihood pieces (mipwa_nll_parts_static) --------------------------------------------------------
// For callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses that forbid
// cudaMalloc): k_nll_recompute needs one partial pair per block, a ticket counter and a block for its totals.  Here they
// live in a file-scope device array instead of the context's cudaMalloc'ed buffers: MIPWA_STATIC_SCRATCH_BYTES on every
// GPU that loads the library, until the process exits.  Layout: [0, 256) ticket, [256, 512) totals (S, I, tag),
// [512, ..) double2 partials of up to MIPWA_STATIC_MAX_BLOCKS blocks.
// In HOST code the array's name is a host-side stand-in, not a device address: the address is taken once per device,
// with that device current, by cudaGetSymbolAddress, and only that pointer goes to the kernels.
#define MIPWA_STATIC_SCRATCH_BYTES (512 + MIPWA_STATIC_MAX_BLOCKS * 16)
#define MIPWA_STATIC_MAX_DEVICES 64
static __device__ __align__(256) unsigned char g_static_scratch[MIPWA_STATIC_SCRATCH_BYTES];

// The array keeps what the last call (of any context) left: ticket and totals start every call at zero.  Device code names
// the array directly.
static __global__ void k_static_clear()
{
    reinterpret_cast<unsigned long long*>(g_static_scratch)[threadIdx.x] = 0ULL;   // 64 threads x 8 B = [0, 512)
}

namespace {
unsigned char* g_static_scratch_ptr[MIPWA_STATIC_MAX_DEVICES];   // device address of g_static_scratch, per device ordinal

int static_scratch(mipwa_ctx* c, unsigned char** out)           // the context's device must be current
{
    if (c->device < 0 || c->device >= MIPWA_STATIC_MAX_DEVICES)
        return fail(c, MIPWA_ERR_ARG, "mipwa_nll_parts_static: device ordinal beyond " + std::to_string(MIPWA_STATIC_MAX_DEVICES - 1));
    unsigned char* p = __atomic_load_n(&g_static_scratch_ptr[c->device], __ATOMIC_ACQUIRE);
    if (!p) {                                              // two threads may both ask: they get the same answer
        void* q = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&q, g_static_scratch);
        if (e != cudaSuccess || !q)
            return fail(c, MIPWA_ERR_CUDA, std::string("cudaGetSymbolAddress(g_static_scratch): ") + cudaGetErrorString(e));
        p = (unsigned char*)q;
        __atomic_store_n(&g_static_scratch_ptr[c->device], p, __ATOMIC_RELEASE);
    }
    *out = p;
    return MIPWA_OK;
}
}  // namespace

extern "C" int mipwa_nll_parts_static(mipwa_ctx* c, const double* params, int64_t n_params, int32_t blocks, double* dev_parts)
{
    if (!c || !params || !dev_parts) return c ? fail(c, MIPWA_ERR_ARG, "null argument") : MIPWA_ERR_ARG;
    NvtxRange range("mipwa_nll_parts_static");
    if (c->ev.n < 0 || c->nm.n < 1) return fail(c, MIPWA_ERR_STATE, "set events and normalisation points first");
    if (blocks < 0) return fail(c, MIPWA_ERR_ARG, "mipwa_nll_parts_static: blocks must be >= 0");
    Slot& E = evs(c);
    Slot& G = nms(c);
    const int grid = blocks > 0 ? blocks : recompute_grid(c, std::max(E.n, G.n));
    if (grid > MIPWA_STATIC_MAX_BLOCKS)
        return fail(c, MIPWA_ERR_ARG, "mipwa_nll_parts_static: " + std::to_string(grid) + " blocks need more than the " +
                    std::to_string(MIPWA_STATIC_SCRATCH_BYTES) + "-byte static scratch (at most " +
                    std::to_string(MIPWA_STATIC_MAX_BLOCKS) + " blocks)");
    // every thread loads the record at its own index before it looks at the counts: the grid must stay inside the padding
    if ((int64_t)grid * MIPWA_REC_BLOCK > record_pad(c))
        return fail(c, MIPWA_ERR_ARG, "mipwa_nll_parts_static: at most " + std::to_string(record_pad(c) / MIPWA_REC_BLOCK) +
                    " blocks on this GPU (4 per SM: the padding of the record arrays)");
    if (!E.rec || !G.rec)                                  // building them would allocate
        return fail(c, MIPWA_ERR_STATE, "mipwa_nll_parts_static: point records not built yet; call mipwa_nll or "
                                        "mipwa_nll_parts_device once on the recompute path after mipwa_set_* (they allocate)");
    int rc = use_device(c);
    if (rc) return rc;
    unsigned char* scratch = nullptr;
    rc = static_scratch(c, &scratch);
    if (rc) return rc;
    rc = build_model(c, params, n_params);
    if (rc) return rc;
    k_static_clear<<<1, 64, 0, c->stream>>>();
    ++c->launches;
    CU(c, cudaGetLastError());
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
    double* totals = reinterpret_cast<double*>(scratch + 256);
    double2* partials = reinterpret_cast<double2*>(scratch + 512);
    const cudaError_t le = mipwa_launch_nll_recompute(c->n_spin, c->model_flags, false, grid, c->stream, c->model, E.rec, 0.0,
                                                      E.n, G.rec, G.n, partials, ticket, totals, ++c->tag);
    ++c->launches;
    CU(c, le);
    k_pack_parts<<<1, 1, 0, c->stream>>>(totals, c->nm.w ? 1.0 : 1.0 / (double)c->nm.n, (double)c->ev.n, dev_parts);
    ++c->launches;
    CU(c, cudaGetLastError());
    return MIPWA_OK;
}
