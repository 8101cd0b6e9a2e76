// mipwa_oracle.cpp -- CPU ORACLE for the MIPWA NLL hot path.  TEST INFRASTRUCTURE ONLY.
//
// This file is the plain, slow, "obviously correct" definition of what the CUDA library in
// paper_1703_03284_b200/csrc computes.  Only tests/, __graft_entry__.smoke() and the cpu_baseline /
// --impl reference legs of bench.py may load it.  It shares no code, header, table or constant with
// the CUDA path and neither includes the other.
//
// Source of the definition: arXiv:1703.03284 as read in SURVEY.md 8(c):
//   Eq. 1   PAPER.md:25   A(s12,s13) = sum_L sum_k c_k^L A_k^L(s12,s13), truncated at L = 2
//   S-wave  PAPER.md:29   N knots s_k, A_0(s_k) = a_k exp(i phi_k), cubic spline [Numerical Recipes] "in the
//                         complex plane" between them; the S-wave is ONE object, no extra coefficient
//   P,D     PAPER.md:27   relativistic Breit-Wigner x real spin-dependent angular factor (ref [5]); the formulas are
//                         NOT printed in the paper -> readings P9/P10 of SURVEY 8(c) (PDG/CLEO-standard forms)
//   Bose    PAPER.md:47   "the Dalitz plot is symmetrised along the two axes" -> plain sum over s12 <-> s13
//   NLL     PAPER.md:47   PDF normalised to unit integral by a numerical sum over points in the Dalitz plane
//
// PARITY UNPINNED at paper level: the paper prints no amplitude, NLL, parameter or input value.  Every function
// below is instead pinned in tests/test_oracle_*.py by closed forms, invariants, library special cases
// (scipy natural CubicSpline, spherical Hankel functions), independent four-vector kinematics and finite
// differences; see DESIGN.md "Oracle pins".  The shape derivatives (O10) are pinned by Richardson-extrapolated central
// differences of the separately pinned resonance term and NLL.
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (no fast-math).  Arithmetic is IEEE double, evaluated
// formula by formula in the order written; sums over events use long double Neumaier-compensated accumulators.

#include <cmath>
#include <complex>
#include <cstdint>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;

extern "C" {
typedef struct { double M, m1, m2, m3; } orc_kin;            // particle 1 = odd-charge; 2,3 = identical pair
typedef struct { double mass, width; int32_t spin; int32_t shape_floats; double r_res, r_parent; } orc_res;
}

namespace {

// ---------------------------------------------------------------------------------------------------------------
// O1  Kinematics (three-body kinematics; problem statement PAPER.md:23, :27)
// ---------------------------------------------------------------------------------------------------------------
// Kaellen function lambda(a,b,c) = a^2 + b^2 + c^2 - 2ab - 2ac - 2bc.
double kallen(double a, double b, double c) { return a * a + b * b + c * c - 2.0 * a * b - 2.0 * a * c - 2.0 * b * c; }

double sigma_sum(const orc_kin& k) { return k.M * k.M + k.m1 * k.m1 + k.m2 * k.m2 + k.m3 * k.m3; }

// Limits of s13 at fixed s12: s13 = m1^2 + m3^2 + 2(E1* E3* -+ p1* p3*) in the (12) rest frame, written in the
// product form s13c +- h with h = sqrt(lambda(s12,m1^2,m2^2) lambda(M^2,s12,m3^2)) / (2 s12).
void s13_limits(const orc_kin& k, double s12, double* centre, double* half)
{
    const double m1s = k.m1 * k.m1, m2s = k.m2 * k.m2, m3s = k.m3 * k.m3, Ms = k.M * k.M;
    const double E1 = (s12 + m1s - m2s) / (2.0 * std::sqrt(s12));        // energy of 1 in the (12) frame
    const double E3 = (Ms - s12 - m3s) / (2.0 * std::sqrt(s12));         // energy of 3 in the (12) frame
    *centre = m1s + m3s + 2.0 * E1 * E3;
    const double l1 = kallen(s12, m1s, m2s), l2 = kallen(Ms, s12, m3s);
    *half = (l1 > 0.0 && l2 > 0.0) ? std::sqrt(l1 * l2) / (2.0 * s12) : 0.0;
}

bool inside(const orc_kin& k, double s12, double s13)
{
    const double lo = (k.m1 + k.m2) * (k.m1 + k.m2), hi = (k.M - k.m3) * (k.M - k.m3);
    if (!(s12 >= lo && s12 <= hi)) return false;
    double c, h;
    s13_limits(k, s12, &c, &h);
    return std::fabs(s13 - c) <= h;
}

// ---------------------------------------------------------------------------------------------------------------
// O3  Natural cubic spline, Numerical-Recipes form (PAPER.md:29 cites [6]; end condition: reading P2 = natural)
//     y''_0 = y''_{N-1} = 0 and for i = 1..N-2
//     (x_i-x_{i-1})/6 y''_{i-1} + (x_{i+1}-x_{i-1})/3 y''_i + (x_{i+1}-x_i)/6 y''_{i+1}
//         = (y_{i+1}-y_i)/(x_{i+1}-x_i) - (y_i-y_{i-1})/(x_i-x_{i-1}),     solved by the Thomas algorithm.
// ---------------------------------------------------------------------------------------------------------------
void spline_second_derivs(int n, const double* x, const double* y, double* ypp)
{
    for (int i = 0; i < n; ++i) ypp[i] = 0.0;
    if (n < 3) return;                                                    // N = 2: straight line
    const int m = n - 2;                                                  // unknowns y''_1 .. y''_{N-2}
    std::vector<double> sub(m), dia(m), sup(m), rhs(m);
    for (int i = 1; i <= m; ++i) {
        sub[i - 1] = (x[i] - x[i - 1]) / 6.0;
        dia[i - 1] = (x[i + 1] - x[i - 1]) / 3.0;
        sup[i - 1] = (x[i + 1] - x[i]) / 6.0;
        rhs[i - 1] = (y[i + 1] - y[i]) / (x[i + 1] - x[i]) - (y[i] - y[i - 1]) / (x[i] - x[i - 1]);
    }
    for (int i = 1; i < m; ++i) {                                         // forward elimination
        const double w = sub[i] / dia[i - 1];
        dia[i] -= w * sup[i - 1];
        rhs[i] -= w * rhs[i - 1];
    }
    ypp[m] = rhs[m - 1] / dia[m - 1];                                     // back substitution
    for (int i = m - 2; i >= 0; --i) ypp[i + 1] = (rhs[i] - sup[i] * ypp[i + 2]) / dia[i];
}

// O4  segment index: x_j <= s < x_{j+1}, clamped to [0, N-2] (reading P3: beyond the ends use the end cubic)
int spline_segment(int n, const double* x, double s)
{
    int j = 0;
    while (j < n - 2 && s >= x[j + 1]) ++j;
    return j;
}

// O4  local weights of S(s) = A y_j + B y_{j+1} + C y''_j + D y''_{j+1}
void spline_weights(int n, const double* x, double s, int* j_out, double w[4])
{
    const int j = spline_segment(n, x, s);
    const double h = x[j + 1] - x[j];
    const double A = (x[j + 1] - s) / h;
    const double B = 1.0 - A;
    w[0] = A;
    w[1] = B;
    w[2] = (A * A * A - A) * (h * h) / 6.0;
    w[3] = (B * B * B - B) * (h * h) / 6.0;
    *j_out = j;
}

cplx spline_eval(int n, const double* x, const cplx* y, const cplx* ypp, double s)
{
    if (n == 0) return cplx(0.0, 0.0);                                    // no MIPWA S-wave (Isobar model, O6b)
    int j;
    double w[4];
    spline_weights(n, x, s, &j, w);
    return w[0] * y[j] + w[1] * y[j + 1] + (w[2] * ypp[j] + w[3] * ypp[j + 1]);
}

// ---------------------------------------------------------------------------------------------------------------
// O5  Resonance term T_r(x, y) for a spin-L resonance in the pair whose mass^2 is x; y = mass^2 of the other
//     odd-charge pair ("relativistic Breit-Wigner ... multiplied by a real spin-dependent angular
//     factor [5]"; formulas are readings P9, P10 of SURVEY 8(c); barrier radii from BASELINE.json configs[0]).
// ---------------------------------------------------------------------------------------------------------------
// daughter momentum^2 in the resonance frame: q^2(x) = lambda(x, m1^2, m2^2) / (4x)
double q2_of(const orc_kin& k, double x) { return kallen(x, k.m1 * k.m1, k.m2 * k.m2) / (4.0 * x); }

// bachelor momentum^2 in the PARENT rest frame ("in the rest frame of the D"): lambda(M^2,x,m3^2)/(4M^2)
double pstar2_of(const orc_kin& k, double x) { return kallen(k.M * k.M, x, k.m3 * k.m3) / (4.0 * k.M * k.M); }

// Blatt-Weisskopf barrier normalised to 1 at the pole; z = r^2 k^2, z0 = r^2 k0^2
double barrier(int L, double z, double z0)
{
    if (L == 0) return 1.0;
    if (L == 1) return std::sqrt((1.0 + z0) / (1.0 + z));
    return std::sqrt((9.0 + 3.0 * z0 + z0 * z0) / (9.0 + 3.0 * z + z * z));
}

// running width Gamma(x) = Gamma0 (q^2/q0^2)^L sqrt(q^2/q0^2) (m0/sqrt(x)) F_R^2
double running_width(const orc_kin& k, const orc_res& r, double x)
{
    const double m0s = r.mass * r.mass;
    const double q2 = q2_of(k, x), q02 = q2_of(k, m0s);
    const double ratio = q2 / q02;
    const double FR = barrier(r.spin, r.r_res * r.r_res * q2, r.r_res * r.r_res * q02);
    double pw = 1.0;
    for (int l = 0; l < r.spin; ++l) pw *= ratio;
    return r.width * pw * std::sqrt(ratio) * (r.mass / std::sqrt(x)) * FR * FR;
}

// propagator BW(x) = 1 / (m0^2 - x - i m0 Gamma(x))
cplx breit_wigner(const orc_kin& k, const orc_res& r, double x)
{
    return 1.0 / cplx(r.mass * r.mass - x, -r.mass * running_width(k, r, x));
}

// Zemach angular factor in mass-squared form (ref [5] of the paper); s23 = Sigma - x - y
double zemach(const orc_kin& k, int L, double x, double y)
{
    if (L == 0) return 1.0;
    const double Ms = k.M * k.M, m1s = k.m1 * k.m1, m2s = k.m2 * k.m2, m3s = k.m3 * k.m3;
    const double s23 = sigma_sum(k) - x - y;
    const double Z1 = y - s23 + (Ms - m3s) * (m2s - m1s) / x;
    if (L == 1) return Z1;
    return Z1 * Z1 - (1.0 / 3.0) * (kallen(Ms, x, m3s) / x) * (kallen(x, m1s, m2s) / x);
}

cplx resonance_term(const orc_kin& k, const orc_res& r, double x, double y)
{
    const double m0s = r.mass * r.mass;
    const double FR = barrier(r.spin, r.r_res * r.r_res * q2_of(k, x), r.r_res * r.r_res * q2_of(k, m0s));
    const double FD = barrier(r.spin, r.r_parent * r.r_parent * pstar2_of(k, x),
                              r.r_parent * r.r_parent * pstar2_of(k, m0s));
    return FD * FR * zemach(k, r.spin, x, y) * breit_wigner(k, r, x);
}

// O10 (not in the paper)  Derivatives of T_r(x, y) with respect to the pole mass m0 and the pole width
//     Gamma0, from the definitions above written out.  With D = m0^2 - x - i W, W = m0 Gamma(x), T = F_D F_R Z / D:
//       dT/dGamma0 = T (i W / Gamma0) / D                                   (W is proportional to Gamma0)
//       dT/dm0     = T [ dlnF_R/dm0 + dlnF_D/dm0 ] - T (2 m0 - i W dlnW/dm0) / D
//     where only the pole quantities q0^2 = q^2(m0^2), p0*^2 = p*^2(m0^2) depend on m0:
//       ln F = (1/2) [ln n_L(z0) - ln n_L(z)], n_1(z) = 1 + z, n_2(z) = 9 + 3z + z^2, z0 = r^2 k0^2
//       dlnF_R/dm0 = (1/2) n_L'(z0R)/n_L(z0R) r_R^2 dq0^2/dm0,   dlnF_D/dm0 likewise with r_D, p0*^2
//       ln W = 2 ln m0 + ln Gamma0 + (L + 1/2) (ln q^2 - ln q0^2) - (1/2) ln x + 2 ln F_R
//       dlnW/dm0 = 2/m0 - (L + 1/2) (dq0^2/dm0)/q0^2 + 2 dlnF_R/dm0
//       q0^2 = [s0 - 2(m1^2 + m2^2) + (m1^2 - m2^2)^2 / s0] / 4  (s0 = m0^2):  dq0^2/dm0 = 2 m0 [1 - (m1^2-m2^2)^2/s0^2]/4
//       p0*^2 = lambda(M^2, s0, m3^2)/(4 M^2):                                 dp0*^2/dm0 = 2 m0 (2 s0 - 2 M^2 - 2 m3^2)/(4 M^2)
double barrier_num_dlog(int L, double z0)   // n_L'(z0) / n_L(z0)
{
    if (L == 0) return 0.0;
    if (L == 1) return 1.0 / (1.0 + z0);
    return (3.0 + 2.0 * z0) / (9.0 + 3.0 * z0 + z0 * z0);
}

void resonance_term_dshape(const orc_kin& k, const orc_res& r, double x, double y, cplx* dT_dm0, cplx* dT_dG0)
{
    const double m0 = r.mass, s0 = m0 * m0, L = (double)r.spin;
    const double m1s = k.m1 * k.m1, m2s = k.m2 * k.m2, m3s = k.m3 * k.m3, Ms = k.M * k.M;
    const cplx T = resonance_term(k, r, x, y);
    const double W = m0 * running_width(k, r, x);
    const cplx D(s0 - x, -W);
    const double q02 = q2_of(k, s0), p02 = pstar2_of(k, s0);
    const double dq02 = 2.0 * m0 * (1.0 - (m1s - m2s) * (m1s - m2s) / (s0 * s0)) / 4.0;
    const double dp02 = 2.0 * m0 * (2.0 * s0 - 2.0 * Ms - 2.0 * m3s) / (4.0 * Ms);
    const double dlnFR = 0.5 * barrier_num_dlog(r.spin, r.r_res * r.r_res * q02) * r.r_res * r.r_res * dq02;
    const double dlnFD = 0.5 * barrier_num_dlog(r.spin, r.r_parent * r.r_parent * p02) * r.r_parent * r.r_parent * dp02;
    const double dlnW = 2.0 / m0 - (L + 0.5) * dq02 / q02 + 2.0 * dlnFR;
    *dT_dG0 = T * cplx(0.0, W / r.width) / D;
    *dT_dm0 = T * (dlnFR + dlnFD) - T * cplx(2.0 * m0, -W * dlnW) / D;
}

// ---------------------------------------------------------------------------------------------------------------
// Model = kinematics + knots + resonance list; parameter vector layout:
//   [a_0..a_{N-1} | phi_0..phi_{N-1} | (|c_r|, arg c_r) r = 0..R-1 | (mass, width) of each shape_floats resonance]
// O2  unpack: y_k = a_k (cos phi_k + i sin phi_k), c_r = |c_r| (cos, sin)
// ---------------------------------------------------------------------------------------------------------------
struct Model {
    orc_kin kin;
    int n;                      // knots
    std::vector<double> x;      // knot positions in m^2 (reading P4)
    int R;
    std::vector<orc_res> res;   // shapes as given at construction
};

struct Unpacked {
    std::vector<cplx> y, ypp, c;
    std::vector<orc_res> res;   // with floating (mass,width) substituted
};

int n_params_of(const Model& m)
{
    int F = 0;
    for (int r = 0; r < m.R; ++r) F += m.res[r].shape_floats ? 1 : 0;
    return 2 * m.n + 2 * m.R + 2 * F;
}

Unpacked unpack(const Model& m, const double* p)
{
    Unpacked u;
    u.y.resize(m.n); u.ypp.resize(m.n); u.c.resize(m.R); u.res = m.res;
    for (int k = 0; k < m.n; ++k) u.y[k] = cplx(p[k] * std::cos(p[m.n + k]), p[k] * std::sin(p[m.n + k]));
    for (int r = 0; r < m.R; ++r) {
        const double mag = p[2 * m.n + 2 * r], arg = p[2 * m.n + 2 * r + 1];
        u.c[r] = cplx(mag * std::cos(arg), mag * std::sin(arg));
    }
    int f = 0;
    for (int r = 0; r < m.R; ++r)
        if (m.res[r].shape_floats) {
            u.res[r].mass = p[2 * m.n + 2 * m.R + 2 * f];
            u.res[r].width = p[2 * m.n + 2 * m.R + 2 * f + 1];
            ++f;
        }
    // O3 for Re and Im separately (reading P1: Re and Im of y_k are splined, same real matrix)
    std::vector<double> yr(m.n), yi(m.n), pr(m.n), pi(m.n);
    for (int k = 0; k < m.n; ++k) { yr[k] = u.y[k].real(); yi[k] = u.y[k].imag(); }
    spline_second_derivs(m.n, m.x.data(), yr.data(), pr.data());
    spline_second_derivs(m.n, m.x.data(), yi.data(), pi.data());
    for (int k = 0; k < m.n; ++k) u.ypp[k] = cplx(pr[k], pi[k]);
    return u;
}

// O6b Isobar-model pieces ("the S-wave is represented by a sum of a constant non-resonant term and
//     Breit-Wigner functions"; "a constant nonresonant amplitude"; reading P27):
//     a list entry with spin = ORC_SPIN_NONRES is the constant term: its basis function is 1 over the whole Dalitz
//     plot (one term, not doubled by the symmetrisation: a constant is its own mirror image and any factor is
//     absorbed by its coefficient); mass, width and radii of that entry are not used.  Scalar Breit-Wigners are the
//     spin-0 case of O5 (F_R = F_D = Z_0 = 1).  n = 0 knots switches the spline S-wave off.
const int ORC_SPIN_NONRES = -1;

cplx symmetrised_term(const orc_kin& k, const orc_res& r, double s12, double s13)
{
    if (r.spin == ORC_SPIN_NONRES) return cplx(1.0, 0.0);
    return resonance_term(k, r, s12, s13) + resonance_term(k, r, s13, s12);
}

// O6  A(s12,s13) = S(s12) + S(s13) + sum_r c_r [T_r(s12,s13) + T_r(s13,s12)]
//     (Eq. 1; symmetrisation PAPER.md:47, reading P8 plain sum; S-wave has no coefficient PAPER.md:37)
cplx amplitude(const Model& m, const Unpacked& u, double s12, double s13)
{
    cplx A = spline_eval(m.n, m.x.data(), u.y.data(), u.ypp.data(), s12)
           + spline_eval(m.n, m.x.data(), u.y.data(), u.ypp.data(), s13);
    for (int r = 0; r < m.R; ++r) A += u.c[r] * symmetrised_term(m.kin, u.res[r], s12, s13);
    return A;
}

// long double Neumaier-compensated accumulator (summation error far below the 1e-10 NLL tolerance)
struct Acc {
    long double s = 0.0L, c = 0.0L;
    void add(long double v)
    {
        const long double t = s + v;
        if (fabsl(s) >= fabsl(v)) c += (s - t) + v; else c += (v - t) + s;
        s = t;
    }
    long double value() const { return s + c; }
};

Model make_model(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res)
{
    Model m;
    m.kin = *kin; m.n = n; m.x.assign(knots, knots + n); m.R = R; m.res.assign(res, res + R);
    return m;
}

// cardinal spline beta_k(s): the spline through the unit vector e_k (O8).  M = T^{-1} D column by column.
std::vector<double> cardinal_second_derivs(const Model& m)
{
    std::vector<double> Mx((size_t)m.n * m.n), e(m.n), pp(m.n);          // Mx[j*n + k] = y''_j of beta_k
    for (int k = 0; k < m.n; ++k) {
        for (int j = 0; j < m.n; ++j) e[j] = (j == k) ? 1.0 : 0.0;
        spline_second_derivs(m.n, m.x.data(), e.data(), pp.data());
        for (int j = 0; j < m.n; ++j) Mx[(size_t)j * m.n + k] = pp[j];
    }
    return Mx;
}

}  // namespace

// ===============================================================================================================
// C ABI of the oracle (loaded with ctypes by oracle/oracle.py).  All pointers are host pointers.
// ===============================================================================================================
extern "C" {

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// ---- pieces, exported so that the tests can pin each one separately -------------------------------------------
double orc_kallen(double a, double b, double c) { return kallen(a, b, c); }
int orc_inside(const orc_kin* k, double s12, double s13) { return inside(*k, s12, s13) ? 1 : 0; }
void orc_s13_limits(const orc_kin* k, double s12, double* lo, double* hi)
{
    double c, h;
    s13_limits(*k, s12, &c, &h);
    *lo = c - h; *hi = c + h;
}
double orc_q2(const orc_kin* k, double x) { return q2_of(*k, x); }
double orc_pstar2(const orc_kin* k, double x) { return pstar2_of(*k, x); }
double orc_barrier(int L, double z, double z0) { return barrier(L, z, z0); }
double orc_running_width(const orc_kin* k, const orc_res* r, double x) { return running_width(*k, *r, x); }
void orc_breit_wigner(const orc_kin* k, const orc_res* r, double x, double* re, double* im)
{
    const cplx b = breit_wigner(*k, *r, x);
    *re = b.real(); *im = b.imag();
}
double orc_zemach(const orc_kin* k, int L, double x, double y) { return zemach(*k, L, x, y); }
void orc_resonance_term(const orc_kin* k, const orc_res* r, double x, double y, double* re, double* im)
{
    const cplx t = resonance_term(*k, *r, x, y);
    *re = t.real(); *im = t.imag();
}
void orc_spline_second_derivs(int n, const double* x, const double* y, double* ypp) { spline_second_derivs(n, x, y, ypp); }
// evaluates the complex spline through (x_k, yre_k + i yim_k) at ns points
void orc_spline_eval(int n, const double* x, const double* yre, const double* yim, int64_t ns, const double* s,
                     double* out_re, double* out_im)
{
    std::vector<double> pr(n), pi(n);
    spline_second_derivs(n, x, yre, pr.data());
    spline_second_derivs(n, x, yim, pi.data());
    std::vector<cplx> y(n), ypp(n);
    for (int k = 0; k < n; ++k) { y[k] = cplx(yre[k], yim[k]); ypp[k] = cplx(pr[k], pi[k]); }
    for (int64_t i = 0; i < ns; ++i) {
        const cplx v = spline_eval(n, x, y.data(), ypp.data(), s[i]);
        out_re[i] = v.real(); out_im[i] = v.imag();
    }
}

int orc_n_params(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res)
{
    return n_params_of(make_model(kin, n, knots, R, res));
}

// ---- O6: amplitude and |A|^2 at n points ------------------------------------------------------------------------
void orc_amplitude(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res, const double* params,
                   int64_t npts, const double* s12, const double* s13, double* out_re, double* out_im)
{
    const Model m = make_model(kin, n, knots, R, res);
    const Unpacked u = unpack(m, params);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < npts; ++i) {
        const cplx A = amplitude(m, u, s12[i], s13[i]);
        out_re[i] = A.real(); out_im[i] = A.imag();
    }
}

void orc_abs2(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res, const double* params,
              int64_t npts, const double* s12, const double* s13, double* out)
{
    const Model m = make_model(kin, n, knots, R, res);
    const Unpacked u = unpack(m, params);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < npts; ++i) out[i] = std::norm(amplitude(m, u, s12[i], s13[i]));
}

// ---- O7: NLL = - sum_i ln|A(x_i)|^2 + n_ev ln I,  I = sum_j w_j |A(x_j)|^2 (w == NULL: w_j = 1/n_norm) -----------
// Also returns the two pieces (tolerance P14 needs them).  OpenMP: static contiguous chunks, per-thread
// compensated long double partials, combined in thread order.
void orc_nll(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res, const double* params,
             int64_t n_ev, const double* e12, const double* e13,
             int64_t n_norm, const double* g12, const double* g13, const double* w,
             double* nll, double* sum_log, double* integral)
{
    const Model m = make_model(kin, n, knots, R, res);
    const Unpacked u = unpack(m, params);
    const int T = orc_num_threads();
    std::vector<Acc> accS(T), accI(T);
#pragma omp parallel num_threads(T)
    {
#ifdef _OPENMP
        const int t = omp_get_thread_num();
#else
        const int t = 0;
#endif
        Acc s, q;
#pragma omp for schedule(static) nowait
        for (int64_t i = 0; i < n_ev; ++i) s.add(std::log(std::norm(amplitude(m, u, e12[i], e13[i]))));
#pragma omp for schedule(static)
        for (int64_t j = 0; j < n_norm; ++j) {
            const double a2 = std::norm(amplitude(m, u, g12[j], g13[j]));
            q.add(w ? (long double)w[j] * a2 : (long double)a2);
        }
        accS[t] = s; accI[t] = q;
    }
    Acc S, I;
    for (int t = 0; t < T; ++t) { S.add(accS[t].value()); I.add(accI[t].value()); }
    long double Iv = I.value();
    if (!w) Iv /= (long double)n_norm;
    const long double Sv = S.value();
    *sum_log = (double)Sv;
    *integral = (double)Iv;
    *nll = (double)(-Sv + (long double)n_ev * logl(Iv));
}

// ---- O8: basis row B_k(s12,s13), K = N + R.  k < N: beta_k(s12) + beta_k(s13) (real);  k >= N: T_r sym. ---------
// With c = [y_0..y_{N-1}, c_0..c_{R-1}]:  A = sum_k c_k B_k  (the amplitude is linear in the complex coefficients).
static void basis_row(const Model& m, const std::vector<orc_res>& res, const std::vector<double>& Mx,
                      double s12, double s13, cplx* B)
{
    for (int k = 0; k < m.n; ++k) B[k] = 0.0;
    const double ss[2] = { s12, s13 };
    for (int ch = 0; ch < 2 && m.n > 0; ++ch) {
        int j;
        double w[4];
        spline_weights(m.n, m.x.data(), ss[ch], &j, w);
        for (int k = 0; k < m.n; ++k) {
            double b = w[2] * Mx[(size_t)j * m.n + k] + w[3] * Mx[(size_t)(j + 1) * m.n + k];
            if (k == j) b += w[0];
            if (k == j + 1) b += w[1];
            B[k] += b;
        }
    }
    for (int r = 0; r < m.R; ++r) B[m.n + r] = symmetrised_term(m.kin, res[r], s12, s13);
}

// basis rows for npts points, row-major out[(i*K + k)*2 + {0,1}] = Re, Im.  params only supplies floating shapes.
void orc_basis(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res, const double* params,
               int64_t npts, const double* s12, const double* s13, double* out)
{
    const Model m = make_model(kin, n, knots, R, res);
    const Unpacked u = unpack(m, params);
    const std::vector<double> Mx = cardinal_second_derivs(m);
    const int K = n + R;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < npts; ++i) {
        std::vector<cplx> B(K);
        basis_row(m, u.res, Mx, s12[i], s13[i], B.data());
        for (int k = 0; k < K; ++k) { out[((size_t)i * K + k) * 2] = B[k].real(); out[((size_t)i * K + k) * 2 + 1] = B[k].imag(); }
    }
}

// Gram matrix G_kl = sum_j w_j conj(B_jk) B_jl (row-major K x K complex, interleaved Re, Im); I = c^H G c.
void orc_gram(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res, const double* params,
              int64_t n_norm, const double* g12, const double* g13, const double* w, double* out)
{
    const Model m = make_model(kin, n, knots, R, res);
    const Unpacked u = unpack(m, params);
    const std::vector<double> Mx = cardinal_second_derivs(m);
    const int K = n + R;
    std::vector<Acc> G((size_t)K * K * 2);
    std::vector<cplx> B(K);
    for (int64_t j = 0; j < n_norm; ++j) {
        basis_row(m, u.res, Mx, g12[j], g13[j], B.data());
        const double wj = w ? w[j] : 1.0 / (double)n_norm;
        for (int k = 0; k < K; ++k)
            for (int l = 0; l < K; ++l) {
                const cplx v = wj * std::conj(B[k]) * B[l];
                G[((size_t)k * K + l) * 2].add(v.real());
                G[((size_t)k * K + l) * 2 + 1].add(v.imag());
            }
    }
    for (size_t t = 0; t < G.size(); ++t) out[t] = (double)G[t].value();
}

// ---- O9: NLL and its analytic gradient w.r.t. the 2N + 2R linear-coefficient parameters (reading P16) ----------
//   calG_k = dNLL/dRe c_k + i dNLL/dIm c_k = -2 sum_i conj(B_ik)/conj(A_i) + (2 n_ev/I) sum_j w_j A_j conj(B_jk)
//   c = rho e^{i theta}:  dNLL/drho = Re(calG e^{-i theta}),  dNLL/dtheta = Re(calG conj(i c)).
// grad layout = params layout: [d/da_k | d/dphi_k | (d/d|c_r|, d/d arg c_r)].
// The same sums also give the two pieces a sharded likelihood exchanges: with S = sum_i ln|A_i|^2,
//   grad_ev = d(-S)/dtheta  (calG_k = -2 sum_i conj(B_ik)/conj(A_i)),   grad_nm = dI/dtheta  (calG_k = 2 sum_j w_j A_j conj(B_jk)),
// so that grad = grad_ev + (n_ev / I) grad_nm.  Optional outputs; the arithmetic of nll and grad does not depend on them.
static void nll_grad_linear(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res, const double* params,
                            int64_t n_ev, const double* e12, const double* e13,
                            int64_t n_norm, const double* g12, const double* g13, const double* w,
                            double* nll, double* grad, double* sum_log, double* integral, double* grad_ev, double* grad_nm)
{
    const Model m = make_model(kin, n, knots, R, res);
    const Unpacked u = unpack(m, params);
    const std::vector<double> Mx = cardinal_second_derivs(m);
    const int K = n + R;
    const int T = orc_num_threads();
    std::vector<std::vector<Acc>> ev(T, std::vector<Acc>(2 * K)), nm(T, std::vector<Acc>(2 * K));
    std::vector<Acc> accS(T), accI(T);
#pragma omp parallel num_threads(T)
    {
#ifdef _OPENMP
        const int t = omp_get_thread_num();
#else
        const int t = 0;
#endif
        std::vector<cplx> B(K);
#pragma omp for schedule(static) nowait
        for (int64_t i = 0; i < n_ev; ++i) {
            basis_row(m, u.res, Mx, e12[i], e13[i], B.data());
            const cplx A = amplitude(m, u, e12[i], e13[i]);
            accS[t].add(std::log(std::norm(A)));
            for (int k = 0; k < K; ++k) {
                const cplx v = std::conj(B[k]) / std::conj(A);
                ev[t][2 * k].add(v.real()); ev[t][2 * k + 1].add(v.imag());
            }
        }
#pragma omp for schedule(static)
        for (int64_t j = 0; j < n_norm; ++j) {
            basis_row(m, u.res, Mx, g12[j], g13[j], B.data());
            const cplx A = amplitude(m, u, g12[j], g13[j]);
            const double wj = w ? w[j] : 1.0 / (double)n_norm;
            accI[t].add((long double)wj * std::norm(A));
            for (int k = 0; k < K; ++k) {
                const cplx v = wj * A * std::conj(B[k]);
                nm[t][2 * k].add(v.real()); nm[t][2 * k + 1].add(v.imag());
            }
        }
    }
    Acc S, I;
    for (int t = 0; t < T; ++t) { S.add(accS[t].value()); I.add(accI[t].value()); }
    const long double Iv = I.value(), Sv = S.value();
    *nll = (double)(-Sv + (long double)n_ev * logl(Iv));
    for (int k = 0; k < K; ++k) {
        Acc er, ei, nr, ni;
        for (int t = 0; t < T; ++t) {
            er.add(ev[t][2 * k].value()); ei.add(ev[t][2 * k + 1].value());
            nr.add(nm[t][2 * k].value()); ni.add(nm[t][2 * k + 1].value());
        }
        const long double f = 2.0L * (long double)n_ev / Iv;
        const cplx G((double)(-2.0L * er.value() + f * nr.value()), (double)(-2.0L * ei.value() + f * ni.value()));
        const cplx Ge((double)(-2.0L * er.value()), (double)(-2.0L * ei.value()));
        const cplx Gn((double)(2.0L * nr.value()), (double)(2.0L * ni.value()));
        const cplx calG[3] = { G, Ge, Gn };
        double* out[3] = { grad, grad_ev, grad_nm };
        for (int q = 0; q < 3; ++q) {
            if (!out[q]) continue;
            if (k < n) {
                const double phi = params[n + k];
                out[q][k] = (calG[q] * cplx(std::cos(phi), -std::sin(phi))).real();
                out[q][n + k] = (calG[q] * std::conj(cplx(0.0, 1.0) * u.y[k])).real();
            } else {
                const int r = k - n;
                const double th = params[2 * n + 2 * r + 1];
                out[q][2 * n + 2 * r] = (calG[q] * cplx(std::cos(th), -std::sin(th))).real();
                out[q][2 * n + 2 * r + 1] = (calG[q] * std::conj(cplx(0.0, 1.0) * u.c[r])).real();
            }
        }
    }
    if (sum_log) *sum_log = (double)Sv;
    if (integral) *integral = (double)Iv;
}

void orc_nll_grad(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res, const double* params,
                  int64_t n_ev, const double* e12, const double* e13,
                  int64_t n_norm, const double* g12, const double* g13, const double* w,
                  double* nll, double* grad)
{
    nll_grad_linear(kin, n, knots, R, res, params, n_ev, e12, e13, n_norm, g12, g13, w, nll, grad, nullptr, nullptr,
                    nullptr, nullptr);
}

// ---- O10: test access to the shape derivatives of one resonance term: out = (Re, Im dT/dm0, Re, Im dT/dGamma0) ----
void orc_resonance_term_dshape(const orc_kin* k, const orc_res* r, double x, double y, double* out)
{
    cplx dm, dg;
    resonance_term_dshape(*k, *r, x, y, &dm, &dg);
    out[0] = dm.real(); out[1] = dm.imag(); out[2] = dg.real(); out[3] = dg.imag();
}

// ---- O10: derivatives of the NLL w.r.t. (mass, width) of every shape_floats resonance, in list order ---------------
//   dA/dtheta = c_r [dT_r(s12,s13)/dtheta + dT_r(s13,s12)/dtheta]
//   dNLL/dtheta = -2 sum_i Re(conj(A_i) dA_i) / |A_i|^2 + (2 n_ev / I) sum_j w_j Re(conj(A_j) dA_j)
// grad_shape has 2F entries: (d/dmass, d/dwidth) per floating resonance.
// Optional pieces as in O9b: shape_ev = d(-S)/dtheta, shape_nm = dI/dtheta (2F entries each).
static void nll_grad_shape_impl(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res,
                                const double* params, int64_t n_ev, const double* e12, const double* e13,
                                int64_t n_norm, const double* g12, const double* g13, const double* w,
                                double* nll, double* grad_shape, double* shape_ev, double* shape_nm)
{
    const Model m = make_model(kin, n, knots, R, res);
    const Unpacked u = unpack(m, params);
    std::vector<int> fl;
    for (int r = 0; r < R; ++r) if (m.res[r].shape_floats) fl.push_back(r);
    const int F = (int)fl.size();
    std::vector<Acc> ev(2 * F), nm(2 * F);
    Acc S, I;
    for (int64_t i = 0; i < n_ev; ++i) {
        const cplx A = amplitude(m, u, e12[i], e13[i]);
        S.add(std::log(std::norm(A)));
        for (int f = 0; f < F; ++f) {
            cplx am, ag, bm, bg;
            resonance_term_dshape(m.kin, u.res[fl[f]], e12[i], e13[i], &am, &ag);
            resonance_term_dshape(m.kin, u.res[fl[f]], e13[i], e12[i], &bm, &bg);
            ev[2 * f].add((std::conj(A) * (u.c[fl[f]] * (am + bm))).real() / std::norm(A));
            ev[2 * f + 1].add((std::conj(A) * (u.c[fl[f]] * (ag + bg))).real() / std::norm(A));
        }
    }
    for (int64_t j = 0; j < n_norm; ++j) {
        const cplx A = amplitude(m, u, g12[j], g13[j]);
        const double wj = w ? w[j] : 1.0 / (double)n_norm;
        I.add((long double)wj * std::norm(A));
        for (int f = 0; f < F; ++f) {
            cplx am, ag, bm, bg;
            resonance_term_dshape(m.kin, u.res[fl[f]], g12[j], g13[j], &am, &ag);
            resonance_term_dshape(m.kin, u.res[fl[f]], g13[j], g12[j], &bm, &bg);
            nm[2 * f].add(wj * (std::conj(A) * (u.c[fl[f]] * (am + bm))).real());
            nm[2 * f + 1].add(wj * (std::conj(A) * (u.c[fl[f]] * (ag + bg))).real());
        }
    }
    const long double Iv = I.value();
    *nll = (double)(-S.value() + (long double)n_ev * logl(Iv));
    for (int t = 0; t < 2 * F; ++t) {
        if (grad_shape) grad_shape[t] = (double)(-2.0L * ev[t].value() + 2.0L * (long double)n_ev / Iv * nm[t].value());
        if (shape_ev) shape_ev[t] = (double)(-2.0L * ev[t].value());
        if (shape_nm) shape_nm[t] = (double)(2.0L * nm[t].value());
    }
}

void orc_nll_grad_shape(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res,
                        const double* params, int64_t n_ev, const double* e12, const double* e13,
                        int64_t n_norm, const double* g12, const double* g13, const double* w,
                        double* nll, double* grad_shape)
{
    nll_grad_shape_impl(kin, n, knots, R, res, params, n_ev, e12, e13, n_norm, g12, g13, w, nll, grad_shape, nullptr,
                        nullptr);
}

// ---- O9b: the pieces one rank of a sharded likelihood contributes: S = sum_i ln|A_i|^2, I, and
// grad_ev = d(-S)/dtheta, grad_nm = dI/dtheta over ALL parameters (2N + 2R linear ones, then (mass, width) of every
// floating resonance), so that NLL = -sum_r S_r + n ln(sum_r I_r) and grad = sum_r grad_ev_r + (n / I) sum_r grad_nm_r.
void orc_nll_grad_parts(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res, const double* params,
                        int64_t n_ev, const double* e12, const double* e13,
                        int64_t n_norm, const double* g12, const double* g13, const double* w,
                        double* sum_log, double* integral, double* grad_ev, double* grad_nm)
{
    double nll;
    nll_grad_linear(kin, n, knots, R, res, params, n_ev, e12, e13, n_norm, g12, g13, w, &nll, nullptr, sum_log, integral,
                    grad_ev, grad_nm);
    nll_grad_shape_impl(kin, n, knots, R, res, params, n_ev, e12, e13, n_norm, g12, g13, w, &nll, nullptr,
                        grad_ev + 2 * n + 2 * R, grad_nm + 2 * n + 2 * R);
}

// ---- O11 (not in the paper): Hessian of the NLL in the 2N + 2R linear-coefficient parameters, for
// fixed resonance shapes.  With c = [y_0..y_{N-1}, c_0..c_{R-1}], A_i = sum_k c_k B_ik, I = c^H G c,
// G_kl = sum_j w_j conj(B_jk) B_jl, and Wirtinger derivatives d/dc_k = (d/dRe c_k - i d/dIm c_k)/2:
//     g_k       = dNLL/dc_k          = -sum_i B_ik/A_i + n_ev (c^H G)_k / I
//     Hcc_kl    = d2NLL/dc_k dc_l    =  sum_i B_ik B_il / A_i^2 - n_ev (c^H G)_k (c^H G)_l / I^2
//     Hcb_kl    = d2NLL/dc_k dconj(c_l) = n_ev G_lk / I - n_ev (c^H G)_k (G c)_l / I^2      (ln|A|^2 has no mixed part)
// and for real parameters t_a, t_b with c = c(t):
//     d2NLL/dt_a dt_b = 2 Re sum_kl [ Hcc_kl dc_k/dt_a dc_l/dt_b + Hcb_kl dc_k/dt_a conj(dc_l/dt_b) ]
//                     + 2 Re sum_k g_k d2c_k/dt_a dt_b.
// Polar form c = rho e^{i phi}: dc/drho = e^{i phi}, dc/dphi = i c, d2c/drho dphi = i e^{i phi}, d2c/dphi2 = -c.
// hess: P x P row-major, P = 2N + 2R, same order as params / grad.  shape_floats entries of params are ignored.
void orc_nll_hessian(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res, const double* params,
                     int64_t n_ev, const double* e12, const double* e13,
                     int64_t n_norm, const double* g12, const double* g13, const double* w, double* hess)
{
    const Model m = make_model(kin, n, knots, R, res);
    const Unpacked u = unpack(m, params);
    const std::vector<double> Mx = cardinal_second_derivs(m);
    const int K = n + R, P = 2 * n + 2 * R;
    std::vector<cplx> c(K), B(K);
    for (int k = 0; k < n; ++k) c[k] = u.y[k];
    for (int r = 0; r < R; ++r) c[n + r] = u.c[r];
    std::vector<Acc> Mr((size_t)K * K), Mi((size_t)K * K), Gr((size_t)K * K), Gi((size_t)K * K), vr(K), vi(K);
    for (int64_t i = 0; i < n_ev; ++i) {
        basis_row(m, u.res, Mx, e12[i], e13[i], B.data());
        cplx A = 0.0;
        for (int k = 0; k < K; ++k) A += c[k] * B[k];
        for (int k = 0; k < K; ++k) {
            const cplx bk = B[k] / A;
            vr[k].add(bk.real()); vi[k].add(bk.imag());
            for (int l = 0; l < K; ++l) {
                const cplx t = bk * (B[l] / A);
                Mr[(size_t)k * K + l].add(t.real()); Mi[(size_t)k * K + l].add(t.imag());
            }
        }
    }
    for (int64_t j = 0; j < n_norm; ++j) {
        basis_row(m, u.res, Mx, g12[j], g13[j], B.data());
        const double wj = w ? w[j] : 1.0 / (double)n_norm;
        for (int k = 0; k < K; ++k)
            for (int l = 0; l < K; ++l) {
                const cplx t = wj * std::conj(B[k]) * B[l];
                Gr[(size_t)k * K + l].add(t.real()); Gi[(size_t)k * K + l].add(t.imag());
            }
    }
    auto G = [&](int k, int l) { return cplx((double)Gr[(size_t)k * K + l].value(), (double)Gi[(size_t)k * K + l].value()); };
    std::vector<cplx> cG(K), Gc(K);                       // (c^H G)_k and (G c)_k
    cplx I = 0.0;
    for (int k = 0; k < K; ++k) {
        cplx a = 0.0, b = 0.0;
        for (int l = 0; l < K; ++l) { a += std::conj(c[l]) * G(l, k); b += G(k, l) * c[l]; }
        cG[k] = a; Gc[k] = b;
    }
    for (int k = 0; k < K; ++k) I += std::conj(c[k]) * Gc[k];
    const double Iv = I.real(), nev = (double)n_ev;
    std::vector<cplx> g(K), Hcc((size_t)K * K), Hcb((size_t)K * K);
    for (int k = 0; k < K; ++k) {
        g[k] = -cplx((double)vr[k].value(), (double)vi[k].value()) + nev * cG[k] / Iv;
        for (int l = 0; l < K; ++l) {
            Hcc[(size_t)k * K + l] = cplx((double)Mr[(size_t)k * K + l].value(), (double)Mi[(size_t)k * K + l].value())
                                     - nev * cG[k] * cG[l] / (Iv * Iv);
            Hcb[(size_t)k * K + l] = nev * G(l, k) / Iv - nev * cG[k] * Gc[l] / (Iv * Iv);
        }
    }
    // polar Jacobians: column index of (rho_k, phi_k) in the parameter vector
    std::vector<int> ir(K), ip(K);
    std::vector<cplx> dr(K), dp(K);
    for (int k = 0; k < K; ++k) {
        ir[k] = k < n ? k : 2 * n + 2 * (k - n);
        ip[k] = k < n ? n + k : 2 * n + 2 * (k - n) + 1;
        const double phi = params[ip[k]];
        dr[k] = cplx(std::cos(phi), std::sin(phi));
        dp[k] = cplx(0.0, 1.0) * c[k];
    }
    for (int t = 0; t < P * P; ++t) hess[t] = 0.0;
    for (int k = 0; k < K; ++k)
        for (int l = 0; l < K; ++l) {
            const cplx hcc = Hcc[(size_t)k * K + l], hcb = Hcb[(size_t)k * K + l];
            const cplx dk[2] = { dr[k], dp[k] }, dl[2] = { dr[l], dp[l] };
            const int ik[2] = { ir[k], ip[k] }, il[2] = { ir[l], ip[l] };
            for (int a = 0; a < 2; ++a)
                for (int b = 0; b < 2; ++b)
                    hess[(size_t)ik[a] * P + il[b]] += 2.0 * (hcc * dk[a] * dl[b] + hcb * dk[a] * std::conj(dl[b])).real();
        }
    for (int k = 0; k < K; ++k) {
        const cplx d2rp = cplx(0.0, 1.0) * dr[k], d2pp = -c[k];
        hess[(size_t)ir[k] * P + ip[k]] += 2.0 * (g[k] * d2rp).real();
        hess[(size_t)ip[k] * P + ir[k]] += 2.0 * (g[k] * d2rp).real();
        hess[(size_t)ip[k] * P + ip[k]] += 2.0 * (g[k] * d2pp).real();
    }
}

// ---- O12 ("signal purity 90 %"): likelihood of a signal + background mixture.  Per event
// the PDF is f_s |A_i|^2 / I + (1 - f_s) b_i with b_i the (normalised) background density at the event, supplied by
// the caller, and f_s the signal fraction:
//     NLL = - sum_i ln( f_s |A_i|^2 / I + (1 - f_s) b_i ),      I = sum_j w_j |A_j|^2.
// Gradient with respect to the 2N + 2R linear-coefficient parameters through calG_k = dNLL/dRe c_k + i dNLL/dIm c_k:
//     p_i = f_s |A_i|^2 / I + (1 - f_s) b_i
//     calG_k = -(2 f_s / I) sum_i A_i conj(B_ik) / p_i + (2 f_s / I^2) [sum_i |A_i|^2 / p_i] sum_j w_j A_j conj(B_jk)
// and dNLL/df_s = - sum_i ( |A_i|^2 / I - b_i ) / p_i.      grad: 2N + 2R entries (polar chain rule as O9).
void orc_nll_mix(const orc_kin* kin, int n, const double* knots, int R, const orc_res* res, const double* params,
                 int64_t n_ev, const double* e12, const double* e13, const double* bkg, double f_sig,
                 int64_t n_norm, const double* g12, const double* g13, const double* w,
                 double* nll, double* grad, double* dnll_dfsig)
{
    const Model m = make_model(kin, n, knots, R, res);
    const Unpacked u = unpack(m, params);
    const std::vector<double> Mx = cardinal_second_derivs(m);
    const int K = n + R;
    std::vector<cplx> B(K);
    Acc I;
    std::vector<Acc> nr(K), ni(K);
    for (int64_t j = 0; j < n_norm; ++j) {
        const cplx A = amplitude(m, u, g12[j], g13[j]);
        const double wj = w ? w[j] : 1.0 / (double)n_norm;
        I.add((long double)wj * std::norm(A));
        if (grad) {
            basis_row(m, u.res, Mx, g12[j], g13[j], B.data());
            for (int k = 0; k < K; ++k) {
                const cplx v = wj * A * std::conj(B[k]);
                nr[k].add(v.real()); ni[k].add(v.imag());
            }
        }
    }
    const double Iv = (double)I.value();
    Acc S, Q, Fs;
    std::vector<Acc> er(K), ei(K);
    for (int64_t i = 0; i < n_ev; ++i) {
        const cplx A = amplitude(m, u, e12[i], e13[i]);
        const double a2 = std::norm(A);
        const double p = f_sig * a2 / Iv + (1.0 - f_sig) * bkg[i];
        S.add(std::log(p));
        Q.add(a2 / p);
        Fs.add((a2 / Iv - bkg[i]) / p);
        if (grad) {
            basis_row(m, u.res, Mx, e12[i], e13[i], B.data());
            for (int k = 0; k < K; ++k) {
                const cplx v = A * std::conj(B[k]) / p;
                er[k].add(v.real()); ei[k].add(v.imag());
            }
        }
    }
    *nll = (double)(-S.value());
    if (dnll_dfsig) *dnll_dfsig = (double)(-Fs.value());
    if (!grad) return;
    const double c1 = -2.0 * f_sig / Iv, c2 = 2.0 * f_sig / (Iv * Iv) * (double)Q.value();
    for (int k = 0; k < K; ++k) {
        const cplx G(c1 * (double)er[k].value() + c2 * (double)nr[k].value(),
                     c1 * (double)ei[k].value() + c2 * (double)ni[k].value());
        if (k < n) {
            const double phi = params[n + k];
            grad[k] = (G * cplx(std::cos(phi), -std::sin(phi))).real();
            grad[n + k] = (G * std::conj(cplx(0.0, 1.0) * u.y[k])).real();
        } else {
            const int r = k - n;
            const double th = params[2 * n + 2 * r + 1];
            grad[2 * n + 2 * r] = (G * cplx(std::cos(th), -std::sin(th))).real();
            grad[2 * n + 2 * r + 1] = (G * std::conj(cplx(0.0, 1.0) * u.c[r])).real();
        }
    }
}

}  // extern "C"
