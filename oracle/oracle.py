"""ctypes loader for the CPU oracle (oracle/mipwa_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It never imports the CUDA package and the CUDA package never imports it.  All arithmetic lives in
the C++ file; this module only marshals numpy arrays (argument checking and dtype/contiguity conversion).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mipwa_oracle.cpp")
_LIB = os.path.join(_HERE, "libmipwa_oracle.so")


def build(force=False):
    """Compile the oracle: plain g++, -O2, no FMA contraction, no fast-math."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
           "-o", _LIB, _SRC]
    subprocess.run(cmd, check=True)
    return _LIB


class Kin(C.Structure):
    _fields_ = [("M", C.c_double), ("m1", C.c_double), ("m2", C.c_double), ("m3", C.c_double)]


class Res(C.Structure):
    _fields_ = [("mass", C.c_double), ("width", C.c_double), ("spin", C.c_int32), ("shape_floats", C.c_int32),
                ("r_res", C.c_double), ("r_parent", C.c_double)]


_dp = C.POINTER(C.c_double)
_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        kp, rp, i32, i64, d = C.POINTER(Kin), C.POINTER(Res), C.c_int, C.c_int64, C.c_double
        model = [kp, i32, _dp, i32, rp]
        L.orc_num_threads.restype = i32
        L.orc_kallen.restype = d; L.orc_kallen.argtypes = [d, d, d]
        L.orc_inside.restype = i32; L.orc_inside.argtypes = [kp, d, d]
        L.orc_s13_limits.restype = None; L.orc_s13_limits.argtypes = [kp, d, _dp, _dp]
        L.orc_q2.restype = d; L.orc_q2.argtypes = [kp, d]
        L.orc_pstar2.restype = d; L.orc_pstar2.argtypes = [kp, d]
        L.orc_barrier.restype = d; L.orc_barrier.argtypes = [i32, d, d]
        L.orc_running_width.restype = d; L.orc_running_width.argtypes = [kp, rp, d]
        L.orc_breit_wigner.restype = None; L.orc_breit_wigner.argtypes = [kp, rp, d, _dp, _dp]
        L.orc_zemach.restype = d; L.orc_zemach.argtypes = [kp, i32, d, d]
        L.orc_resonance_term.restype = None; L.orc_resonance_term.argtypes = [kp, rp, d, d, _dp, _dp]
        L.orc_spline_second_derivs.restype = None; L.orc_spline_second_derivs.argtypes = [i32, _dp, _dp, _dp]
        L.orc_spline_eval.restype = None
        L.orc_spline_eval.argtypes = [i32, _dp, _dp, _dp, i64, _dp, _dp, _dp]
        L.orc_n_params.restype = i32; L.orc_n_params.argtypes = model
        L.orc_amplitude.restype = None; L.orc_amplitude.argtypes = model + [_dp, i64, _dp, _dp, _dp, _dp]
        L.orc_abs2.restype = None; L.orc_abs2.argtypes = model + [_dp, i64, _dp, _dp, _dp]
        L.orc_nll.restype = None
        L.orc_nll.argtypes = model + [_dp, i64, _dp, _dp, i64, _dp, _dp, _dp, _dp, _dp, _dp]
        L.orc_basis.restype = None; L.orc_basis.argtypes = model + [_dp, i64, _dp, _dp, _dp]
        L.orc_gram.restype = None; L.orc_gram.argtypes = model + [_dp, i64, _dp, _dp, _dp, _dp]
        L.orc_nll_grad.restype = None
        L.orc_nll_grad.argtypes = model + [_dp, i64, _dp, _dp, i64, _dp, _dp, _dp, _dp, _dp]
        L.orc_nll_mix.restype = None
        L.orc_nll_mix.argtypes = model + [_dp, i64, _dp, _dp, _dp, d, i64, _dp, _dp, _dp, _dp, _dp, _dp]
        L.orc_nll_hessian.restype = None
        L.orc_nll_hessian.argtypes = model + [_dp, i64, _dp, _dp, i64, _dp, _dp, _dp, _dp]
        L.orc_nll_grad_shape.restype = None
        L.orc_nll_grad_shape.argtypes = model + [_dp, i64, _dp, _dp, i64, _dp, _dp, _dp, _dp, _dp]
        L.orc_resonance_term_dshape.restype = None; L.orc_resonance_term_dshape.argtypes = [kp, rp, d, d, _dp]
        L.orc_nll_grad_parts.restype = None
        L.orc_nll_grad_parts.argtypes = model + [_dp, i64, _dp, _dp, i64, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
        _lib = L
    return _lib


def _a(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def kin_of(kin):
    """kin = (M, m1, m2, m3) or dict with those keys."""
    if isinstance(kin, dict):
        kin = (kin["M"], kin["m1"], kin["m2"], kin["m3"])
    return Kin(*[float(v) for v in kin])


def res_array(resonances):
    """resonances = sequence of dicts {mass, width, spin, r_res, r_parent, shape_floats(optional)}."""
    arr = (Res * max(len(resonances), 1))()
    for i, r in enumerate(resonances):
        arr[i] = Res(float(r["mass"]), float(r["width"]), int(r["spin"]), int(r.get("shape_floats", 0)),
                     float(r["r_res"]), float(r["r_parent"]))
    return arr


class Oracle:
    """The oracle bound to one model (kinematics, knots, resonance list)."""

    def __init__(self, kin, knots, resonances):
        self.L = lib()
        self.kin = kin_of(kin)
        self.knots = _a(knots)
        self.n = int(self.knots.size)
        self.R = len(resonances)
        self.resonances = list(resonances)
        self.res = res_array(resonances)
        self._model = (C.byref(self.kin), self.n, _p(self.knots), self.R, self.res)
        self.n_params = self.L.orc_n_params(*self._model)
        self.K = self.n + self.R

    def _params(self, params):
        p = _a(params)
        if p.size != self.n_params:
            raise ValueError(f"expected {self.n_params} parameters, got {p.size}")
        return p

    def amplitude(self, params, s12, s13):
        p, a, b = self._params(params), _a(s12), _a(s13)
        re, im = np.empty_like(a), np.empty_like(a)
        self.L.orc_amplitude(*self._model, _p(p), a.size, _p(a), _p(b), _p(re), _p(im))
        return re + 1j * im

    def abs2(self, params, s12, s13):
        p, a, b = self._params(params), _a(s12), _a(s13)
        out = np.empty_like(a)
        self.L.orc_abs2(*self._model, _p(p), a.size, _p(a), _p(b), _p(out))
        return out

    def nll(self, params, e12, e13, g12, g13, w=None, parts=False):
        p, e12, e13, g12, g13 = self._params(params), _a(e12), _a(e13), _a(g12), _a(g13)
        w = None if w is None else _a(w)
        nll, sl, integ = C.c_double(), C.c_double(), C.c_double()
        self.L.orc_nll(*self._model, _p(p), e12.size, _p(e12), _p(e13), g12.size, _p(g12), _p(g13), _p(w),
                       C.byref(nll), C.byref(sl), C.byref(integ))
        return (nll.value, sl.value, integ.value) if parts else nll.value

    def nll_grad(self, params, e12, e13, g12, g13, w=None):
        p, e12, e13, g12, g13 = self._params(params), _a(e12), _a(e13), _a(g12), _a(g13)
        w = None if w is None else _a(w)
        nll = C.c_double()
        grad = np.empty(2 * self.n + 2 * self.R)
        self.L.orc_nll_grad(*self._model, _p(p), e12.size, _p(e12), _p(e13), g12.size, _p(g12), _p(g13), _p(w),
                            C.byref(nll), _p(grad))
        return nll.value, grad

    def nll_mix(self, params, e12, e13, bkg, f_sig, g12, g13, w=None, grad=False):
        """signal + background mixture (O12): NLL, or (NLL, gradient over 2N + 2R, dNLL/df_sig) if grad"""
        p, e12, e13, bkg, g12, g13 = self._params(params), _a(e12), _a(e13), _a(bkg), _a(g12), _a(g13)
        w = None if w is None else _a(w)
        nll, dfs = C.c_double(), C.c_double()
        g = np.zeros(2 * self.n + 2 * self.R) if grad else None
        self.L.orc_nll_mix(*self._model, _p(p), e12.size, _p(e12), _p(e13), _p(bkg), float(f_sig), g12.size, _p(g12),
                           _p(g13), _p(w), C.byref(nll), _p(g), C.byref(dfs))
        return (nll.value, g, dfs.value) if grad else nll.value

    def nll_hessian(self, params, e12, e13, g12, g13, w=None):
        """P x P Hessian of the NLL in the 2N + 2R linear-coefficient parameters (fixed shapes)  -- O11"""
        p, e12, e13, g12, g13 = self._params(params), _a(e12), _a(e13), _a(g12), _a(g13)
        w = None if w is None else _a(w)
        P = 2 * self.n + 2 * self.R
        H = np.zeros((P, P))
        self.L.orc_nll_hessian(*self._model, _p(p), e12.size, _p(e12), _p(e13), g12.size, _p(g12), _p(g13), _p(w), _p(H))
        return H

    def nll_grad_shape(self, params, e12, e13, g12, g13, w=None):
        """(NLL, [d/dmass, d/dwidth of every shape_floats resonance in list order])  -- O10"""
        p, e12, e13, g12, g13 = self._params(params), _a(e12), _a(e13), _a(g12), _a(g13)
        w = None if w is None else _a(w)
        nll = C.c_double()
        F = sum(1 for r in self.resonances if r.get("shape_floats"))
        grad = np.zeros(max(2 * F, 1))
        self.L.orc_nll_grad_shape(*self._model, _p(p), e12.size, _p(e12), _p(e13), g12.size, _p(g12), _p(g13), _p(w),
                                  C.byref(nll), _p(grad))
        return nll.value, grad[:2 * F]

    def nll_grad_parts(self, params, e12, e13, g12, g13, w=None):
        """(S = sum ln|A|^2, I, d(-S)/dtheta, dI/dtheta) over all parameters, floating shapes last  -- O9b"""
        p, e12, e13, g12, g13 = self._params(params), _a(e12), _a(e13), _a(g12), _a(g13)
        w = None if w is None else _a(w)
        S, Iv = C.c_double(), C.c_double()
        F = sum(1 for r in self.resonances if r.get("shape_floats"))
        P = 2 * self.n + 2 * self.R + 2 * F
        gev, gnm = np.zeros(P + 1), np.zeros(P + 1)
        self.L.orc_nll_grad_parts(*self._model, _p(p), e12.size, _p(e12), _p(e13), g12.size, _p(g12), _p(g13), _p(w),
                                  C.byref(S), C.byref(Iv), _p(gev), _p(gnm))
        return S.value, Iv.value, gev[:P], gnm[:P]

    def resonance_term_dshape(self, r, x, y):
        """(dT/dm0, dT/dGamma0) of one resonance dict r at (x, y)  -- O10"""
        out = np.zeros(4)
        ra = res_array([r])
        self.L.orc_resonance_term_dshape(C.byref(self.kin), ra, float(x), float(y), _p(out))
        return complex(out[0], out[1]), complex(out[2], out[3])

    def basis(self, params, s12, s13):
        p, a, b = self._params(params), _a(s12), _a(s13)
        out = np.empty((a.size, self.K, 2))
        self.L.orc_basis(*self._model, _p(p), a.size, _p(a), _p(b), _p(out))
        return out[..., 0] + 1j * out[..., 1]

    def gram(self, params, g12, g13, w=None):
        p, a, b = self._params(params), _a(g12), _a(g13)
        w = None if w is None else _a(w)
        out = np.empty((self.K, self.K, 2))
        self.L.orc_gram(*self._model, _p(p), a.size, _p(a), _p(b), _p(w), _p(out))
        return out[..., 0] + 1j * out[..., 1]

    # ---- pieces ----
    def inside(self, s12, s13):
        a, b = np.atleast_1d(_a(s12)), np.atleast_1d(_a(s13))
        return np.array([self.L.orc_inside(C.byref(self.kin), float(x), float(y)) for x, y in zip(a, b)], dtype=bool)

    def s13_limits(self, s12):
        lo, hi = C.c_double(), C.c_double()
        self.L.orc_s13_limits(C.byref(self.kin), float(s12), C.byref(lo), C.byref(hi))
        return lo.value, hi.value

    def q2(self, x):
        return self.L.orc_q2(C.byref(self.kin), float(x))

    def pstar2(self, x):
        return self.L.orc_pstar2(C.byref(self.kin), float(x))

    def running_width(self, r, x):
        return self.L.orc_running_width(C.byref(self.kin), C.byref(self.res[r]), float(x))

    def breit_wigner(self, r, x):
        re, im = C.c_double(), C.c_double()
        self.L.orc_breit_wigner(C.byref(self.kin), C.byref(self.res[r]), float(x), C.byref(re), C.byref(im))
        return complex(re.value, im.value)

    def zemach(self, L, x, y):
        return self.L.orc_zemach(C.byref(self.kin), int(L), float(x), float(y))

    def resonance_term(self, r, x, y):
        re, im = C.c_double(), C.c_double()
        self.L.orc_resonance_term(C.byref(self.kin), C.byref(self.res[r]), float(x), float(y),
                                  C.byref(re), C.byref(im))
        return complex(re.value, im.value)


def barrier(L, z, z0):
    return lib().orc_barrier(int(L), float(z), float(z0))


def kallen(a, b, c):
    return lib().orc_kallen(float(a), float(b), float(c))


def spline_second_derivs(x, y):
    x, y = _a(x), _a(y)
    out = np.empty_like(x)
    lib().orc_spline_second_derivs(x.size, _p(x), _p(y), _p(out))
    return out


def spline_eval(x, y, s):
    """Complex natural spline through (x_k, y_k) evaluated at s (any shape 1-D)."""
    x = _a(x)
    y = np.asarray(y, dtype=np.complex128)
    yre, yim = _a(y.real), _a(y.imag)
    s = np.atleast_1d(_a(s))
    re, im = np.empty_like(s), np.empty_like(s)
    lib().orc_spline_eval(x.size, _p(x), _p(yre), _p(yim), s.size, _p(s), _p(re), _p(im))
    return re + 1j * im


def num_threads():
    return lib().orc_num_threads()
