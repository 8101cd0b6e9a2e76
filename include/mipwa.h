/* mipwa.h -- C ABI of libmipwa: the B200 (sm_100a) hot path of a model-independent partial wave analysis fit.
 *
 * What it computes (arXiv:1703.03284 = /root/reference/PAPER.md; readings in DESIGN.md section 3):
 *
 *   A(s12,s13) = S(s12) + S(s13) + sum_r c_r [ T_r(s12,s13) + T_r(s13,s12) ]
 *       Eq. 1 truncated at L = 2, Bose-symmetrised in s12 <-> s13.
 *       S   = natural cubic spline through N knots in m^2, S(s_k) = a_k exp(i phi_k), Re and Im splined
 *             separately; the S-wave is one object without a coefficient of its own.
 *       T_r = F_D F_R Z_L BW: relativistic Breit-Wigner with running width times Blatt-Weisskopf barrier factors
 *             and the Zemach angular factor (PAPER.md:27 + its ref. [5]; forms fixed in DESIGN.md readings P9, P10).
 *   NLL = - sum_i ln |A(event_i)|^2 + n_ev ln I,   I = sum_j w_j |A(norm_j)|^2
 *       unbinned likelihood with the PDF normalised to unit integral every call.
 *
 * All arithmetic is IEEE fp64 and runs in CUDA kernels on one GPU; there is no CPU fallback: every entry point
 * fails with MIPWA_ERR_CUDA when no usable device exists.  Plain C, no exceptions, nothing printed.
 *
 * Conventions
 *   - Units: masses GeV, s12/s13/knots GeV^2, radii GeV^-1.
 *   - Particle 1 is the odd-charge one; 2 and 3 are the identical pair (m2 == m3 required).
 *     s12 = m^2(1,2), s13 = m^2(1,3).
 *   - Parameter vector (HOST pointer, length mipwa_n_params()):
 *       [ a_0 .. a_{N-1} | phi_0 .. phi_{N-1} | (|c_0|, arg c_0) .. (|c_{R-1}|, arg c_{R-1}) |
 *         (mass, width) of every resonance created with shape_floats = 1, in list order ]
 *   - Ownership: a `mem` argument says where the caller's arrays live.  MIPWA_MEM_HOST: the library copies them
 *     into device memory it owns.  MIPWA_MEM_DEVICE: the library BORROWS the device pointers (zero copy, e.g.
 *     torch tensors); the caller keeps them alive and unchanged until the next mipwa_set_* call on the same slot or
 *     mipwa_destroy.  Outputs are caller-allocated HOST memory unless stated otherwise.
 *   - Errors: every function returns MIPWA_OK (0) or a negative code; mipwa_last_error() gives the text of the
 *     last failure on that context.  A |A|^2 of zero or a non-finite value propagates as IEEE inf/NaN in the
 *     result with status MIPWA_OK.
 *   - Threads: a context must not be used from two threads at once; distinct contexts are independent.
 *   - Synchrony: mipwa_nll / mipwa_nll_grad / mipwa_eval_abs2 return when their result is in host memory.
 *     Kernels are launched on the stream given to mipwa_set_stream (default: the legacy default stream).
 */
#ifndef MIPWA_H
#define MIPWA_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mipwa_ctx mipwa_ctx;                 /* opaque, owned by the library */

typedef struct {
    double m_parent, m1, m2, m3;                    /* GeV; m2 == m3 */
} mipwa_kinematics;

/* spin of the list entry that stands for the CONSTANT NON-RESONANT amplitude of the Isobar model ("a sum of
 * a constant non-resonant term and Breit-Wigner functions"): it contributes c_r x 1 over the whole Dalitz
 * plot (not doubled by the symmetrisation: DESIGN.md reading P27); its mass, width and radii are ignored, its
 * (|c_r|, arg c_r) sit in the parameter vector like those of a resonance.  At most one per model, never floating. */
#define MIPWA_SPIN_NONRES (-1)

typedef struct {
    double  mass, width;                            /* m0, Gamma0 in GeV (initial values when shape_floats = 1) */
    int32_t spin;                                   /* L = 0, 1, 2 or MIPWA_SPIN_NONRES; else MIPWA_ERR_ARG */
    int32_t shape_floats;                           /* 1: (mass, width) are read from the parameter vector */
    double  r_res, r_parent;                        /* Blatt-Weisskopf radii, GeV^-1 */
} mipwa_resonance;

enum { MIPWA_OK = 0, MIPWA_ERR_ARG = -1, MIPWA_ERR_DOMAIN = -2, MIPWA_ERR_STATE = -3, MIPWA_ERR_CUDA = -4,
       MIPWA_ERR_NOMEM = -5 };
enum { MIPWA_MEM_HOST = 0, MIPWA_MEM_DEVICE = 1 };
enum { MIPWA_PATH_AUTO = 0,            /* no shape floats: cached-compact; some float: hybrid if supported; else recompute */
       MIPWA_PATH_RECOMPUTE = 1,       /* every call re-evaluates every amplitude term (FP64-ALU bound) */
       MIPWA_PATH_CACHED = 2,          /* fixed shapes: dense n_ev x K complex basis + K x K Gram (HBM bound) */
       MIPWA_PATH_CACHED_COMPACT = 3,  /* fixed shapes: R complex resonance values per event; spline re-evaluated */
       MIPWA_PATH_HYBRID = 4,          /* some shapes float: their terms and the spline are recomputed, the fixed-shape
                                          resonance terms are cached per event AND per normalisation point */
       MIPWA_PATH_CACHED_REAL = 5,     /* fixed shapes: dense basis with the N spline columns stored as REAL numbers (they
                                          are): 8 N + 16 R bytes per event instead of 16 (N + R); exact like CACHED */
       MIPWA_PATH_CACHED_F32 = 6 };    /* OPT-IN, outside the 1e-12 contract: the columns of CACHED_REAL stored as fp32
                                          (4 N + 8 R bytes per event), every sum still in fp64; |A|^2 good to ~1e-7 */

#define MIPWA_MAX_KNOTS      128
#define MIPWA_MAX_RESONANCES 16

/* Create a context for one model on CUDA device `device`.
 *   knots: n_knots strictly increasing positions in m^2 (HOST), 2 <= n_knots <= MIPWA_MAX_KNOTS;
 *          n_knots = 0 (knots may be NULL): no spline S-wave - the Isobar comparison model of PAPER.md:27, whose
 *          S-wave is scalar (spin 0) Breit-Wigners plus the MIPWA_SPIN_NONRES term
 *   res:   n_res resonance descriptions (HOST), 0 <= n_res <= MIPWA_MAX_RESONANCES;
 *          n_knots + n_res >= 1
 * Errors: MIPWA_ERR_ARG (bad masses / knots / spin / radii / counts), MIPWA_ERR_CUDA (no device, not sm_100). */
int mipwa_create(const mipwa_kinematics* kin, const double* knots, int32_t n_knots,
                 const mipwa_resonance* res, int32_t n_res, int32_t device, mipwa_ctx** out);
void mipwa_destroy(mipwa_ctx* ctx);

/* Use `cuda_stream` (a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream; NULL = default stream). */
int mipwa_set_stream(mipwa_ctx* ctx, void* cuda_stream);

/* Data events: n pairs (s12[i], s13[i]).  Every point is checked ON THE DEVICE against the Dalitz boundary
 * ((m1+m2)^2 <= s12 <= (M-m3)^2 and s13 inside its band); a point outside -> MIPWA_ERR_DOMAIN and the slot is
 * left empty.  n = 0 is allowed (the NLL is then 0).  Invalidates the cached basis.
 * The same pass stores, in library-owned memory, the spline segment of s12[i] and of s13[i] as one uint16 per point
 * (knots are fixed at mipwa_create, so the pair is a property of the point set; +2 B per point): the per-call kernels
 * index the spline tables with it.  Borrowed (MIPWA_MEM_DEVICE) arrays must therefore not change while they are set
 * (they must be 8-byte aligned, as any array of doubles is).  The full-recompute kernels stream a library-owned copy of
 * the set as 32-byte records (s12, s13, weight, segment rows), built on first use: + 32 B per point. */
int mipwa_set_events(mipwa_ctx* ctx, const double* s12, const double* s13, int64_t n, int32_t mem);

/* Normalisation points with weights w (NULL: w_j = 1/n).  I = sum_j w_j |A_j|^2 stands for the integral of
 * |A|^2 over the Dalitz plot ("calculated numerically based on evenly distributed grid points").
 * Same boundary check and ownership rules as mipwa_set_events; n >= 1.  Invalidates the cached Gram matrix. */
int mipwa_set_norm_points(mipwa_ctx* ctx, const double* s12, const double* s13, const double* w, int64_t n,
                          int32_t mem);

/* Optional, once per point set, for fits that evaluate the same sample many times ("in each fit
 * iteration"): makes library-owned copies of the current events and normalisation points SORTED BY SPLINE CELL
 * (segment of s12, segment of s13; +16 B per event, +16/24 B per normalisation point).  Every kernel then reads
 * the copies: all lanes of a warp look up the same spline segment, so the shared-memory table reads become
 * broadcasts.  Results change only by summation order.  The test hooks keep the caller's order.  Undone for a slot
 * by the next mipwa_set_* on it; implied by mipwa_nll_grad.  Errors: MIPWA_ERR_STATE before both mipwa_set_*. */
int mipwa_prepare(mipwa_ctx* ctx);

/* Length of the parameter vector: 2N + 2R + 2F (F = resonances with shape_floats). */
int mipwa_n_params(const mipwa_ctx* ctx, int64_t* n);

/* Select the evaluation path.  CACHED* with F > 0 -> MIPWA_ERR_STATE; HYBRID needs 1-2 floating
 * resonances of spin 1 or 2 and 1-5 fixed-shape ones (else MIPWA_ERR_STATE; AUTO then recomputes). */
int mipwa_set_path(mipwa_ctx* ctx, int32_t path);

/* Bytes of device memory the current path needs for its per-event cache with the current events, n_ev rounded up
 * to a multiple of 256 (dense: n_ev * K * 16; real: n_ev * (8 N + 16 R); f32: n_ev * (4 N + 8 R); compact:
 * n_ev * (R * 16 + 16); hybrid: (n_ev + n_norm) * (16 + 16 x fixed resonances), library-owned; recompute: 0), or a negative error
 * code (MIPWA_ERR_STATE before mipwa_set_events). */
int64_t mipwa_basis_bytes(const mipwa_ctx* ctx);

/* Optional caller-provided DEVICE storage for that cache (borrowed; >= mipwa_basis_bytes(), 256-byte aligned).
 * Without it the library allocates on first use. */
int mipwa_set_basis_buffer(mipwa_ctx* ctx, void* dev, int64_t bytes);

/* One likelihood evaluation (what a minimiser calls once per step):  *nll = -sum ln|A|^2 + n_ev ln I.
 * params: HOST, n_params doubles.  Errors: MIPWA_ERR_STATE before both mipwa_set_* calls, MIPWA_ERR_ARG on a
 * wrong n_params or a non-positive floating mass/width. */
int mipwa_nll(mipwa_ctx* ctx, const double* params, int64_t n_params, double* nll);

/* n_batch likelihood evaluations of the SAME sample at n_batch parameter vectors (what a minimiser's finite-difference
 * derivatives, a likelihood scan or a profile need: steps A3-A7 of every vector are independent).  The kernels of all
 * vectors are enqueued back to back on the context's stream, every one delivers its totals into its own slot of a mapped
 * host block, and the host waits ONCE, for the last: the launch and result latency of a blocking mipwa_nll (20 us of a
 * 0.26 ms call at 10 M + 10 M points, most of a call at the paper's 10^5 events) is paid once per batch instead of once
 * per vector.  Same kernels, same launch shape: nll[b] has the bits of mipwa_nll(params + b n_params).
 *   params    HOST, n_batch x n_params doubles, vector b at params + b * n_params
 *   nll       HOST, n_batch doubles; sum_log, integral: HOST, n_batch doubles each, or NULL (the pieces S and I of A7)
 * The first call allocates the mapped block (256 slots, grown on demand).  Errors as mipwa_nll; a bad vector b fails
 * the whole call (vectors before it have run, none of the outputs is written). */
int mipwa_nll_batch(mipwa_ctx* ctx, const double* params, int64_t n_params, int32_t n_batch, double* nll, double* sum_log,
                    double* integral);

/* Same, also returning the two pieces: sum_i ln|A_i|^2 and I (either pointer may be NULL). */
int mipwa_nll_parts(mipwa_ctx* ctx, const double* params, int64_t n_params, double* nll, double* sum_log,
                    double* integral);

/* NLL and its analytic gradient with respect to the first 2N + 2R parameters (the linear coefficients in polar
 * form; reading P16; mipwa_nll_grad_full adds the derivatives with respect to floating masses/widths).
 * grad: HOST, 2N + 2R doubles, laid out like params.  Works on cell-sorted copies of the points (implies
 * mipwa_prepare).  With fixed shapes and the path MIPWA_PATH_CACHED_COMPACT (or AUTO) the events are streamed from
 * the compact cache and the normalisation part comes from the Gram matrix; otherwise every term is recomputed
 * (k_grad_recompute; MIPWA_PATH_HYBRID caches terms for the VALUE only).  Two calls with the same arguments return
 * the same bits: every sum is taken in a fixed order (no floating-point atomics). */
int mipwa_nll_grad(mipwa_ctx* ctx, const double* params, int64_t n_params, double* nll, double* grad);

/* NLL and its gradient with respect to ALL n_params parameters: the 2N + 2R entries of mipwa_nll_grad followed by
 * (d/dmass, d/dwidth) of every shape_floats resonance in list order (not in the paper).  With
 * T = F_D F_R Z / D, D = m0^2 - x - i m0 Gamma(x) (readings P9/P10), only the pole quantities q0^2 = q^2(m0^2) and
 * p0*^2 = p*^2(m0^2) depend on m0:
 *     dT/dGamma0 = T (i m0 Gamma(x) / Gamma0) / D
 *     dT/dm0     = T d ln(F_R F_D)/dm0 - T (2 m0 - i m0 Gamma(x) d ln(m0 Gamma(x))/dm0) / D
 *     dNLL/dtheta = -2 sum_i Re(conj(A_i) dA_i)/|A_i|^2 + (2 n_ev / I) sum_j w_j Re(conj(A_j) dA_j),
 *     dA = c_r [dT_r(s12,s13) + dT_r(s13,s12)].
 * grad: HOST, n_params doubles.  With ONE floating resonance of spin 1 or 2 the extra sums are folded into the gradient
 * pass itself; several floating resonances (or a floating spin-0 one) cost one more pass over both point sets
 * (k_grad_shape).  Identical to mipwa_nll_grad when no shape floats.  Errors as mipwa_nll_grad. */
int mipwa_nll_grad_full(mipwa_ctx* ctx, const double* params, int64_t n_params, double* nll, double* grad);

/* The pieces ONE RANK of a sharded likelihood contributes (events and normalisation points are
 * independent units, so rank g holds a slice of each, with normalisation weights of the WHOLE sample):
 *     *sum_log = S = sum_i ln|A_i|^2,   *integral = I = sum_j w_j |A_j|^2,
 *     grad_ev = d(-S)/dtheta,           grad_nm = dI/dtheta,
 * over all n_params parameters in the layout of mipwa_nll_grad_full.  Summed over the ranks (S, I, n_ev and both
 * vectors: 3 + 2 n_params doubles per rank and call),
 *     NLL = -S + n_ev ln I,             dNLL/dtheta = grad_ev + (n_ev / I) grad_nm.
 * A per-rank mipwa_nll_grad cannot be combined that way: it already holds its own rank's n_ev / I.
 * grad_ev, grad_nm: HOST, n_params doubles each.  Same launches, paths and errors as mipwa_nll_grad_full. */
int mipwa_nll_grad_parts(mipwa_ctx* ctx, const double* params, int64_t n_params, double* sum_log, double* integral,
                         double* grad_ev, double* grad_nm);

/* The sharded likelihood without a host round trip.  One call per rank and step:
 *   mipwa_nll_parts_device   launches this rank's kernel and leaves (S_r, I_r, n_r) in DEVICE memory `dev_parts` (3
 *                            doubles, caller-owned, e.g. a slice of a torch tensor); returns without waiting.  The
 *                            caller all-gathers the 3 doubles on the SAME stream (NCCL over NVLink) into 3 n_ranks doubles
 *   mipwa_combine_parts_device  one tiny kernel adds the gathered pieces IN RANK ORDER (every rank forms the same bits),
 *                            forms NLL = -S + n ln I (A7) and delivers it through the mapped result block; returns when
 *                            the value is on the host.  sum_log, integral, n_ev may be NULL.
 * The normalisation weights must be those of the whole sample.  mipwa_combine_parts / mipwa_combine_grad_parts are the
 * same rank-ordered sums on HOST data (no GPU needed): parts[r] = (S_r, I_r, n_r) resp. (S_r, I_r, n_r, grad_ev_r[n_params],
 * grad_nm_r[n_params]) as mipwa_nll_grad_parts returns them; grad = sum grad_ev_r + (n / I) sum grad_nm_r. */
int mipwa_nll_parts_device(mipwa_ctx* ctx, const double* params, int64_t n_params, double* dev_parts);
int mipwa_combine_parts_device(mipwa_ctx* ctx, const double* dev_parts_all, int32_t n_ranks, double* nll, double* sum_log,
                               double* integral, int64_t* n_ev);
int mipwa_combine_parts(int32_t n_ranks, const double* parts, double* nll, double* sum_log, double* integral, int64_t* n_ev);
/* the same for a batch (mipwa_nll_batch with its pieces): parts[r] = (S_r[0..n_batch), I_r[0..n_batch), n_r), 2 n_batch + 1
 * doubles per rank; nll: n_batch doubles.  Same sums, same bits per vector as mipwa_combine_parts. */
int mipwa_combine_parts_batch(int32_t n_ranks, int32_t n_batch, const double* parts, double* nll);
int mipwa_combine_grad_parts(int32_t n_ranks, int64_t n_params, const double* parts, double* nll, double* grad,
                             double* sum_log, double* integral, int64_t* n_ev);

/* mipwa_nll_parts_device for callers that cannot allocate device memory (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the same likelihood kernel (steps A4-A6 on the full-recompute path, whatever
 * mipwa_set_path says), but its scratch memory - one partial pair per block, the ticket counter, the totals - is a
 * file-scope device array of 512 + 16 * MIPWA_STATIC_MAX_BLOCKS bytes (8.5 KB) that every GPU holds from the moment it
 * loads the library until the process exits.  The call makes NO cudaMalloc / cudaFree and calls no allocating library
 * routine; it enqueues three launches on the context's stream and returns without waiting.
 *   params     HOST, n_params doubles, as mipwa_nll
 *   blocks     thread blocks (of 512 threads) to run on: 0 = one per SM as mipwa_nll does, otherwise the caller's number
 *              (part of the GPU); more than MIPWA_STATIC_MAX_BLOCKS, either way, or more than 4 per SM (the padding
 *              of the record arrays covers that many threads) -> MIPWA_ERR_ARG, nothing launched
 *   dev_parts  DEVICE, 3 doubles, caller-owned: (S, I, n_ev) as mipwa_nll_parts_device leaves them; valid once the
 *              context's stream has reached this point (mipwa_combine_parts_device on the same context waits for it)
 * The 32-byte point records must exist already (building them allocates): one mipwa_nll / mipwa_nll_parts_device on
 * the recompute path after the mipwa_set_* calls does that, else MIPWA_ERR_STATE.  The first call on each device asks
 * the runtime for the array's address (no allocation): make it before a capture starts.
 * ALL calls, of all contexts on a GPU, share the one array: calls that overlap on the GPU (two streams, two contexts,
 * two threads) race on it and give garbage; calls on one stream are safe, each clears the ticket and totals first.
 * Other errors as mipwa_nll. */
#define MIPWA_STATIC_MAX_BLOCKS 512
int mipwa_nll_parts_static(mipwa_ctx* ctx, const double* params, int64_t n_params, int32_t blocks, double* dev_parts);

/* Signal + background mixture ("signal purity 90 %"): per event the PDF is
 *     f_s |A_i|^2 / I + (1 - f_s) b_i ,      NLL = - sum_i ln( f_s |A_i|^2 / I + (1 - f_s) b_i ),
 * with b_i the background density at event i (normalised over the Dalitz plot, supplied by the caller) and f_s the
 * signal fraction.  Detector efficiency enters through the weights of the normalisation points, as for mipwa_nll.
 *   mipwa_set_event_background: b = n_ev doubles (HOST: copied; DEVICE: borrowed), in the order of the arrays given
 *     to the last mipwa_set_events, which it must follow (a new mipwa_set_events drops the densities); NULL clears.
 *   mipwa_nll_mix: recompute path, two launches (normalisation integral first: the event sum needs I).
 *   mipwa_nll_mix_grad: also the gradient over the 2N + 2R linear-coefficient parameters (layout of mipwa_nll_grad)
 *     and dNLL/df_s (dnll_dfsig may be NULL).  Implies mipwa_prepare.
 * Errors: MIPWA_ERR_STATE before the point sets or the densities are set, MIPWA_ERR_ARG unless 0 < f_sig <= 1. */
int mipwa_set_event_background(mipwa_ctx* ctx, const double* b, int32_t mem);
int mipwa_nll_mix(mipwa_ctx* ctx, const double* params, int64_t n_params, double f_sig, double* nll);
int mipwa_nll_mix_grad(mipwa_ctx* ctx, const double* params, int64_t n_params, double f_sig, double* nll, double* grad,
                       double* dnll_dfsig);

/* The mixture likelihood of a SHARDED sample: the event sum needs the integral I of the whole sample, so a step is two
 * phases with one exchange of 1 + P doubles between them (P = 2N + 2R) and one of 3 + P after:
 *   mipwa_norm_parts         this rank's I_r = sum_j w_j |A_j|^2 and dI_r/dtheta (grad_nm: HOST, P doubles, may be NULL)
 *   mipwa_nll_mix_parts      with integral_total = sum_r I_r: S_r = sum_i ln(|A_i|^2 + kappa b_i), Q_r = sum_i b_i / D_i,
 *                            D_i = |A_i|^2 + kappa b_i, kappa = I (1 - f_s) / f_s, and grad_ev = d(-S_r)/dtheta at fixed
 *                            kappa (HOST, P doubles, may be NULL)
 *   mipwa_combine_mix_parts  HOST: norm_parts[r] = (I_r, grad_nm_r[P]), ev_parts[r] = (S_r, Q_r, n_r, grad_ev_r[P]) ->
 *                            NLL = -S - n ln(f_s / I), grad = sum grad_ev_r + ((n - kappa Q) / I) sum grad_nm_r,
 *                            dNLL/df_s = -(n - I Q / f_s) / f_s; every sum in rank order.  grad, dnll_dfsig may be NULL.
 * Errors as mipwa_nll_mix_grad. */
int mipwa_norm_parts(mipwa_ctx* ctx, const double* params, int64_t n_params, double* integral, double* grad_nm);
int mipwa_nll_mix_parts(mipwa_ctx* ctx, const double* params, int64_t n_params, double f_sig, double integral_total,
                        double* sum_log, double* q, double* grad_ev);
int mipwa_combine_mix_parts(int32_t n_ranks, int64_t n_lin, double f_sig, const double* norm_parts, const double* ev_parts,
                            double* nll, double* grad, double* dnll_dfsig);

/* NLL, gradient and HESSIAN with respect to the 2N + 2R linear-coefficient parameters, for fixed resonance shapes
 * (the parameter errors and correlations PAPER.md:29 alludes to are the inverse of this matrix at the
 * minimum).  With c = [y_k, c_r], A_i = sum_k c_k B_ik, I = c^H G c and Wirtinger derivatives:
 *     d2NLL/dc_k dc_l       = sum_i B_ik B_il / A_i^2 - n_ev (c^H G)_k (c^H G)_l / I^2
 *     d2NLL/dc_k dconj(c_l) = n_ev G_lk / I - n_ev (c^H G)_k (G c)_l / I^2
 * followed by the polar chain rule.  The K x K event sum is one more sweep of the Gram kernel over the events (complex
 * weights 1/A_i^2, no conjugate: 4 K^2 flops per event); G comes from the Gram matrix of the cached paths.
 *   grad: HOST, 2N + 2R doubles, may be NULL;  hess: HOST, (2N + 2R)^2 doubles, row-major, symmetric.
 * Errors: MIPWA_ERR_STATE if a shape floats or before both mipwa_set_*; MIPWA_ERR_ARG if a magnitude is zero (the
 * polar parametrisation is singular there). */
int mipwa_nll_hessian(mipwa_ctx* ctx, const double* params, int64_t n_params, double* nll, double* grad, double* hess);

/* The Hessian over ALL n_params parameters, floating masses and widths included (the full error matrix of a fit whose
 * resonance shapes float).  Block of the linear coefficients: the formulas above with the basis at the current masses and
 * widths.  Rows and columns of a floating mass or width: central differences of the analytic gradient
 * (mipwa_nll_grad_full) in that parameter, Richardson-extrapolated from the steps h and h / 2 with h = 1e-3 x the width
 * (four gradient calls per floating shape parameter; relative accuracy ~1e-8).  Identical to mipwa_nll_hessian when no
 * shape floats.  grad: HOST, n_params doubles, may be NULL;  hess: HOST, n_params^2 doubles, row-major, symmetric. */
int mipwa_nll_hessian_full(mipwa_ctx* ctx, const double* params, int64_t n_params, double* nll, double* grad, double* hess);

/* The same Hessian for a SHARDED sample.  Both sums of the formulas above are sums over points:
 *   mipwa_hessian_parts      this rank's M_kl = sum_i B_ik B_il / A_i^2 (its events) and G_kl (its normalisation points,
 *                            whole-sample weights): HOST, mipwa_hessian_parts_len() doubles each = K x K complex, row-major,
 *                            (re, im) interleaved; K counts the columns of the dense basis
 *   mipwa_hessian_assemble   HOST arithmetic only: from M and G added over the ranks, the whole-sample event count and the
 *                            whole-sample polar gradient (mipwa_combine_grad_parts) to hess ((2N + 2R)^2, row-major). */
int64_t mipwa_hessian_parts_len(const mipwa_ctx* ctx);
int mipwa_hessian_parts(mipwa_ctx* ctx, const double* params, int64_t n_params, double* M, double* G);
int mipwa_hessian_assemble(mipwa_ctx* ctx, const double* params, int64_t n_params, int64_t n_ev_total, const double* M,
                           const double* G, const double* grad, double* hess);

/* Toy Monte-Carlo generation on the device ("samples of 100K signal events are generated from a Dalitz
 * plot PDF"): n events with density |A(params)|^2 / integral inside the Dalitz boundary, by
 * accept-reject against a piecewise-constant envelope (reading P22): n_coarse x n_coarse cells over the
 * bounding square [(m1+m2)^2, (M-m3)^2]^2, each 1.2 x the maximum of |A|^2 over the centres of an n_side x n_side
 * fine grid that fall into it.  Candidate i uses uniforms 4i .. 4i+3 of the counter-based splitmix64 stream `key`
 * (the scheme of paper_1703_03284_b200/inputs.py); the events are the first n accepted candidates in counter order,
 * so the sample is a function of (model, params, key, n, n_side, n_coarse) only.
 *   s12, s13: n doubles each, HOST or DEVICE according to mem (caller-allocated).
 *   n_candidates (may be NULL): candidates drawn.  Independent of the event / normalisation slots.
 * Errors: MIPWA_ERR_ARG (sizes, pointers), MIPWA_ERR_DOMAIN (|A|^2 zero or non-finite on the whole envelope grid,
 * or acceptance below 1e-6), MIPWA_ERR_CUDA / MIPWA_ERR_NOMEM. */
int mipwa_generate(mipwa_ctx* ctx, const double* params, int64_t n_params, uint64_t key, int64_t n, int32_t n_side,
                   int32_t n_coarse, double* s12, double* s13, int32_t mem, int64_t* n_candidates);

/* TEST HOOK: per-point |A|^2 from the same device function the NLL kernels use.
 *   which = 0: the events slot, 1: the normalisation slot; out: HOST, n doubles, n = that slot's size. */
int mipwa_eval_abs2(mipwa_ctx* ctx, const double* params, int64_t n_params, int32_t which, double* out, int64_t n);

/* TEST HOOK: the cached basis row of `n` points of slot `which` as the CACHED path builds it:
 *   out[(i*K + k)*2 + {0,1}] = Re, Im of B_ik, K = N + R (HOST, n*K*2 doubles), points i = first .. first+n-1. */
int mipwa_eval_basis(mipwa_ctx* ctx, const double* params, int64_t n_params, int32_t which, int64_t first,
                     int64_t n, double* out);

/* Kernel timing (off by default: two extra event records per call).  When on, mipwa_last_kernel_ms returns the
 * device time of the kernels of the last mipwa_nll / mipwa_nll_parts / mipwa_nll_grad call on this context in
 * milliseconds, measured with CUDA events on the context's stream (for the benchmark's roofline numbers). */
int mipwa_enable_timing(mipwa_ctx* ctx, int32_t on);
int mipwa_last_kernel_ms(const mipwa_ctx* ctx, float* ms);

/* Number of kernel launches issued by this context since creation (the benchmark's gpu_launches claim). */
int64_t mipwa_launch_count(const mipwa_ctx* ctx);

/* Measure the sustained FP64 FMA rate of the device with register-resident DFMA loops on every SM for about
 * `seconds` seconds in all; 2 flops per DFMA.
 *   *tflops       DFMAs with an immediate and a repeated register operand: the rate the FP64 pipe demonstrably issues
 *                 at (the denominator of the ALU roofline)
 *   *tflops_3reg  (may be NULL) DFMAs with three distinct register operands, which the operand fetch holds ~8 % lower */
int mipwa_measure_fp64_peak(int32_t device, double seconds, double* tflops, double* tflops_3reg);

const char* mipwa_last_error(const mipwa_ctx* ctx);   /* valid until the next call on ctx; "" if none */
const char* mipwa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MIPWA_H */
