"""Thin ctypes binding of libmipwa.so (include/mipwa.h).  Argument marshalling only: every step of the hot path
runs in the CUDA kernels behind the C ABI.  There is no CPU fallback: if the library is missing or no B200 is
present, construction raises.

Method names mirror the C entry points: Mipwa.set_events -> mipwa_set_events, Mipwa.nll -> mipwa_nll, ...
Device arrays are passed as torch CUDA tensors (float64, contiguous) and are BORROWED by the library; host arrays
are numpy float64 and are copied by the library.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmipwa.so")

OK, ERR_ARG, ERR_DOMAIN, ERR_STATE, ERR_CUDA, ERR_NOMEM = 0, -1, -2, -3, -4, -5
MEM_HOST, MEM_DEVICE = 0, 1
PATH_AUTO, PATH_RECOMPUTE, PATH_CACHED, PATH_CACHED_COMPACT, PATH_HYBRID, PATH_CACHED_REAL, PATH_CACHED_F32 = 0, 1, 2, 3, 4, 5, 6
STATIC_MAX_BLOCKS = 512           # MIPWA_STATIC_MAX_BLOCKS of include/mipwa.h
_ERR_NAMES = {ERR_ARG: "MIPWA_ERR_ARG", ERR_DOMAIN: "MIPWA_ERR_DOMAIN", ERR_STATE: "MIPWA_ERR_STATE",
              ERR_CUDA: "MIPWA_ERR_CUDA", ERR_NOMEM: "MIPWA_ERR_NOMEM"}

# every symbol include/mipwa.h declares
SYMBOLS = ["mipwa_create", "mipwa_destroy", "mipwa_set_stream", "mipwa_set_events", "mipwa_set_norm_points",
           "mipwa_prepare", "mipwa_n_params", "mipwa_set_path", "mipwa_basis_bytes", "mipwa_set_basis_buffer", "mipwa_nll",
           "mipwa_nll_parts", "mipwa_nll_grad", "mipwa_nll_grad_full", "mipwa_nll_grad_parts", "mipwa_nll_hessian", "mipwa_set_event_background", "mipwa_nll_mix",
           "mipwa_nll_mix_grad", "mipwa_generate", "mipwa_eval_abs2", "mipwa_eval_basis", "mipwa_enable_timing",
           "mipwa_last_kernel_ms", "mipwa_launch_count", "mipwa_measure_fp64_peak", "mipwa_last_error",
           "mipwa_version", "mipwa_nll_parts_device", "mipwa_combine_parts_device", "mipwa_combine_parts",
           "mipwa_combine_grad_parts", "mipwa_norm_parts", "mipwa_nll_mix_parts", "mipwa_combine_mix_parts",
           "mipwa_hessian_parts_len", "mipwa_hessian_parts", "mipwa_hessian_assemble", "mipwa_nll_hessian_full",
           "mipwa_nll_parts_static", "mipwa_nll_batch", "mipwa_combine_parts_batch"]


class MipwaError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"{_ERR_NAMES.get(code, code)}: {text}")
        self.code = code


class Kinematics(C.Structure):
    _fields_ = [("m_parent", C.c_double), ("m1", C.c_double), ("m2", C.c_double), ("m3", C.c_double)]


class Resonance(C.Structure):
    _fields_ = [("mass", C.c_double), ("width", C.c_double), ("spin", C.c_int32), ("shape_floats", C.c_int32),
                ("r_res", C.c_double), ("r_parent", C.c_double)]


_dp = C.POINTER(C.c_double)
_lib = None


def load_library():
    """dlopen libmipwa.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1703_03284_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, d = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    L.mipwa_create.restype = i32
    L.mipwa_create.argtypes = [C.POINTER(Kinematics), _dp, i32, C.POINTER(Resonance), i32, i32, C.POINTER(vp)]
    L.mipwa_destroy.restype = None; L.mipwa_destroy.argtypes = [vp]
    L.mipwa_set_stream.restype = i32; L.mipwa_set_stream.argtypes = [vp, vp]
    L.mipwa_set_events.restype = i32; L.mipwa_set_events.argtypes = [vp, vp, vp, i64, i32]
    L.mipwa_set_norm_points.restype = i32; L.mipwa_set_norm_points.argtypes = [vp, vp, vp, vp, i64, i32]
    L.mipwa_prepare.restype = i32; L.mipwa_prepare.argtypes = [vp]
    L.mipwa_n_params.restype = i32; L.mipwa_n_params.argtypes = [vp, C.POINTER(i64)]
    L.mipwa_set_path.restype = i32; L.mipwa_set_path.argtypes = [vp, i32]
    L.mipwa_basis_bytes.restype = i64; L.mipwa_basis_bytes.argtypes = [vp]
    L.mipwa_set_basis_buffer.restype = i32; L.mipwa_set_basis_buffer.argtypes = [vp, vp, i64]
    L.mipwa_nll.restype = i32; L.mipwa_nll.argtypes = [vp, _dp, i64, _dp]
    L.mipwa_nll_parts.restype = i32; L.mipwa_nll_parts.argtypes = [vp, _dp, i64, _dp, _dp, _dp]
    L.mipwa_nll_grad.restype = i32; L.mipwa_nll_grad.argtypes = [vp, _dp, i64, _dp, _dp]
    L.mipwa_nll_grad_full.restype = i32; L.mipwa_nll_grad_full.argtypes = [vp, _dp, i64, _dp, _dp]
    L.mipwa_nll_grad_parts.restype = i32; L.mipwa_nll_grad_parts.argtypes = [vp, _dp, i64, _dp, _dp, _dp, _dp]
    L.mipwa_nll_hessian.restype = i32; L.mipwa_nll_hessian.argtypes = [vp, _dp, i64, _dp, _dp, _dp]
    L.mipwa_set_event_background.restype = i32; L.mipwa_set_event_background.argtypes = [vp, vp, i32]
    L.mipwa_nll_mix.restype = i32; L.mipwa_nll_mix.argtypes = [vp, _dp, i64, C.c_double, _dp]
    L.mipwa_nll_mix_grad.restype = i32; L.mipwa_nll_mix_grad.argtypes = [vp, _dp, i64, C.c_double, _dp, _dp, _dp]
    L.mipwa_generate.restype = i32
    L.mipwa_generate.argtypes = [vp, _dp, i64, C.c_uint64, i64, i32, i32, vp, vp, i32, C.POINTER(i64)]
    L.mipwa_eval_abs2.restype = i32; L.mipwa_eval_abs2.argtypes = [vp, _dp, i64, i32, _dp, i64]
    L.mipwa_eval_basis.restype = i32; L.mipwa_eval_basis.argtypes = [vp, _dp, i64, i32, i64, i64, _dp]
    L.mipwa_enable_timing.restype = i32; L.mipwa_enable_timing.argtypes = [vp, i32]
    L.mipwa_last_kernel_ms.restype = i32; L.mipwa_last_kernel_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.mipwa_launch_count.restype = i64; L.mipwa_launch_count.argtypes = [vp]
    L.mipwa_measure_fp64_peak.restype = i32; L.mipwa_measure_fp64_peak.argtypes = [i32, d, _dp, _dp]
    L.mipwa_last_error.restype = C.c_char_p; L.mipwa_last_error.argtypes = [vp]
    L.mipwa_version.restype = C.c_char_p; L.mipwa_version.argtypes = []
    pi64 = C.POINTER(i64)
    L.mipwa_nll_parts_device.restype = i32; L.mipwa_nll_parts_device.argtypes = [vp, _dp, i64, vp]
    L.mipwa_nll_parts_static.restype = i32; L.mipwa_nll_parts_static.argtypes = [vp, _dp, i64, i32, vp]
    L.mipwa_combine_parts_batch.restype = i32; L.mipwa_combine_parts_batch.argtypes = [i32, i32, _dp, _dp]
    L.mipwa_nll_batch.restype = i32; L.mipwa_nll_batch.argtypes = [vp, _dp, i64, i32, _dp, _dp, _dp]
    L.mipwa_combine_parts_device.restype = i32; L.mipwa_combine_parts_device.argtypes = [vp, vp, i32, _dp, _dp, _dp, pi64]
    L.mipwa_combine_parts.restype = i32; L.mipwa_combine_parts.argtypes = [i32, _dp, _dp, _dp, _dp, pi64]
    L.mipwa_combine_grad_parts.restype = i32; L.mipwa_combine_grad_parts.argtypes = [i32, i64, _dp, _dp, _dp, _dp, _dp, pi64]
    L.mipwa_norm_parts.restype = i32; L.mipwa_norm_parts.argtypes = [vp, _dp, i64, _dp, _dp]
    L.mipwa_nll_mix_parts.restype = i32; L.mipwa_nll_mix_parts.argtypes = [vp, _dp, i64, d, d, _dp, _dp, _dp]
    L.mipwa_combine_mix_parts.restype = i32; L.mipwa_combine_mix_parts.argtypes = [i32, i64, d, _dp, _dp, _dp, _dp, _dp]
    L.mipwa_nll_hessian_full.restype = i32; L.mipwa_nll_hessian_full.argtypes = [vp, _dp, i64, _dp, _dp, _dp]
    L.mipwa_hessian_parts_len.restype = i64; L.mipwa_hessian_parts_len.argtypes = [vp]
    L.mipwa_hessian_parts.restype = i32; L.mipwa_hessian_parts.argtypes = [vp, _dp, i64, _dp, _dp]
    L.mipwa_hessian_assemble.restype = i32; L.mipwa_hessian_assemble.argtypes = [vp, _dp, i64, i64, _dp, _dp, _dp, _dp]
    _lib = L
    return L


def _host(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _is_torch(x):
    return type(x).__module__.startswith("torch")


def _dev_ptr(t, n=None):
    import torch
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError("device arrays must be contiguous float64 CUDA tensors")
    if n is not None and t.numel() != n:
        raise ValueError("array lengths differ")
    return C.c_void_p(t.data_ptr())


class Mipwa:
    """One model context (mipwa_create ... mipwa_destroy)."""

    def __init__(self, kin, knots, resonances, device=0):
        self.L = load_library()
        if isinstance(kin, dict):
            kin = (kin["M"], kin["m1"], kin["m2"], kin["m3"])
        self._kin = Kinematics(*[float(v) for v in kin])
        knots = _host(knots)
        res = (Resonance * max(len(resonances), 1))()
        for i, r in enumerate(resonances):
            res[i] = Resonance(float(r["mass"]), float(r["width"]), int(r["spin"]), int(r.get("shape_floats", 0)),
                               float(r["r_res"]), float(r["r_parent"]))
        self.N, self.R = int(knots.size), len(resonances)
        self.K = self.N + self.R
        self._h = C.c_void_p()
        rc = self.L.mipwa_create(C.byref(self._kin), knots.ctypes.data_as(_dp), self.N, res, self.R, int(device),
                                 C.byref(self._h))
        if rc != OK:
            self._h = None
            raise MipwaError(rc, "mipwa_create failed (bad model, or no sm_100 CUDA device: there is no CPU path)")
        self.device = int(device)
        self._keep = {}                     # borrowed tensors kept alive
        n = C.c_int64()
        self._check(self.L.mipwa_n_params(self._h, C.byref(n)))
        self.n_params = n.value
        self.n_events = self.n_norm = -1

    def _check(self, rc):
        if rc != OK:
            raise MipwaError(rc, self.L.mipwa_last_error(self._h).decode())

    def close(self):
        h = getattr(self, "_h", None)
        if h is not None and h.value:
            self._h = None
            self.L.mipwa_destroy(h)
            self._keep = {}

    def __del__(self):
        try:
            self.close()
        except Exception:           # interpreter shutdown: module globals may be gone
            pass

    def set_stream(self, stream):
        """stream: a torch.cuda.Stream, a raw cudaStream_t integer, or None (default stream)."""
        ptr = getattr(stream, "cuda_stream", stream)
        self._check(self.L.mipwa_set_stream(self._h, C.c_void_p(ptr or 0)))

    def _set(self, fn, name, arrays, n_extra_ok):
        s12 = arrays[0]
        if _is_torch(s12):
            n = s12.numel()
            ptrs = [_dev_ptr(a, n) for a in arrays]
            self._keep[name] = arrays
            self._check(fn(self._h, *ptrs, n, MEM_DEVICE))
        else:
            host = [None if a is None else _host(a) for a in arrays]
            n = host[0].size
            if any(h is not None and h.size != n for h in host):
                raise ValueError("array lengths differ")
            ptrs = [None if h is None else C.c_void_p(h.ctypes.data) for h in host]
            self._keep.pop(name, None)
            self._check(fn(self._h, *ptrs, n, MEM_HOST))
        return n

    def set_events(self, s12, s13):
        self.n_events = -1
        self.n_events = self._set(self.L.mipwa_set_events, "ev", [s12, s13], False)

    def set_norm_points(self, s12, s13, w=None):
        self.n_norm = -1
        self.n_norm = self._set(self.L.mipwa_set_norm_points, "nm", [s12, s13, w], True)

    def prepare(self):
        self._check(self.L.mipwa_prepare(self._h))

    def set_path(self, path):
        self._check(self.L.mipwa_set_path(self._h, int(path)))

    def basis_bytes(self):
        n = self.L.mipwa_basis_bytes(self._h)
        if n < 0:
            self._check(int(n))
        return int(n)

    def set_basis_buffer(self, tensor):
        import torch
        if not (tensor.is_cuda and tensor.is_contiguous()):
            raise TypeError("basis buffer must be a contiguous CUDA tensor")
        self._keep["basis"] = tensor
        self._check(self.L.mipwa_set_basis_buffer(self._h, C.c_void_p(tensor.data_ptr()),
                                                  tensor.numel() * tensor.element_size()))

    def _params(self, params):
        p = _host(params)
        return p, p.ctypes.data_as(_dp), p.size

    def nll(self, params):
        p, pp, n = self._params(params)
        out = C.c_double()
        self._check(self.L.mipwa_nll(self._h, pp, n, C.byref(out)))
        return out.value

    def nll_batch(self, params, parts=False):
        """NLL at every row of params (n_batch x n_params), kernels pipelined, one wait; parts: also (S, I) per row"""
        p = np.ascontiguousarray(params, dtype=np.float64)
        if p.ndim != 2:
            raise ValueError("params must be n_batch x n_params")
        nb, n = p.shape
        out = np.empty(nb)
        sl, integ = (np.empty(nb), np.empty(nb)) if parts else (None, None)
        self._check(self.L.mipwa_nll_batch(self._h, p.ctypes.data_as(_dp), n, nb, out.ctypes.data_as(_dp),
                                           sl.ctypes.data_as(_dp) if parts else None,
                                           integ.ctypes.data_as(_dp) if parts else None))
        return (out, sl, integ) if parts else out

    def nll_parts(self, params):
        p, pp, n = self._params(params)
        out, sl, integ = C.c_double(), C.c_double(), C.c_double()
        self._check(self.L.mipwa_nll_parts(self._h, pp, n, C.byref(out), C.byref(sl), C.byref(integ)))
        return out.value, sl.value, integ.value

    def nll_grad(self, params):
        p, pp, n = self._params(params)
        out = C.c_double()
        grad = np.empty(2 * self.N + 2 * self.R)
        self._check(self.L.mipwa_nll_grad(self._h, pp, n, C.byref(out), grad.ctypes.data_as(_dp)))
        return out.value, grad

    def nll_grad_full(self, params):
        """(NLL, gradient over all n_params parameters incl. floating masses and widths)"""
        p, pp, n = self._params(params)
        out = C.c_double()
        grad = np.empty(p.size)
        self._check(self.L.mipwa_nll_grad_full(self._h, pp, n, C.byref(out), grad.ctypes.data_as(_dp)))
        return out.value, grad

    def nll_grad_parts(self, params):
        """one rank's pieces of a sharded likelihood: (sum ln|A|^2, I, d(-sum ln|A|^2)/dtheta, dI/dtheta)"""
        p, pp, n = self._params(params)
        S, Iv = C.c_double(), C.c_double()
        gev, gnm = np.empty(p.size), np.empty(p.size)
        self._check(self.L.mipwa_nll_grad_parts(self._h, pp, n, C.byref(S), C.byref(Iv), gev.ctypes.data_as(_dp),
                                                gnm.ctypes.data_as(_dp)))
        return S.value, Iv.value, gev, gnm

    def set_event_background(self, b):
        """background density per event (numpy: copied; CUDA torch tensor: borrowed), in the order of set_events"""
        if b is None:
            self._check(self.L.mipwa_set_event_background(self._h, None, MEM_HOST))
            self._bkg = None
            return
        if hasattr(b, "data_ptr"):
            self._bkg = b                                  # keep the borrowed tensor alive
            self._check(self.L.mipwa_set_event_background(self._h, C.c_void_p(b.data_ptr()), MEM_DEVICE))
        else:
            a = np.ascontiguousarray(b, dtype=np.float64)
            self._check(self.L.mipwa_set_event_background(self._h, C.c_void_p(a.ctypes.data), MEM_HOST))

    def nll_mix(self, params, f_sig):
        p, pp, n = self._params(params)
        out = C.c_double()
        self._check(self.L.mipwa_nll_mix(self._h, pp, n, float(f_sig), C.byref(out)))
        return out.value

    def nll_mix_grad(self, params, f_sig):
        """(NLL, gradient over 2N + 2R, dNLL/df_sig) of the signal + background mixture"""
        p, pp, n = self._params(params)
        out, dfs = C.c_double(), C.c_double()
        grad = np.empty(2 * self.N + 2 * self.R)
        self._check(self.L.mipwa_nll_mix_grad(self._h, pp, n, float(f_sig), C.byref(out), grad.ctypes.data_as(_dp),
                                              C.byref(dfs)))
        return out.value, grad, dfs.value

    def nll_hessian(self, params):
        """(NLL, gradient, Hessian) in the 2N + 2R linear-coefficient parameters; fixed shapes only."""
        p, pp, n = self._params(params)
        P = 2 * self.N + 2 * self.R
        out, grad, H = C.c_double(), np.empty(P), np.empty((P, P))
        self._check(self.L.mipwa_nll_hessian(self._h, pp, n, C.byref(out), grad.ctypes.data_as(_dp), H.ctypes.data_as(_dp)))
        return out.value, grad, H

    def nll_hessian_full(self, params):
        """(NLL, gradient, Hessian) over all n_params parameters, floating masses and widths included"""
        p, pp, n = self._params(params)
        out, grad, H = C.c_double(), np.empty(p.size), np.empty((p.size, p.size))
        self._check(self.L.mipwa_nll_hessian_full(self._h, pp, n, C.byref(out), grad.ctypes.data_as(_dp), H.ctypes.data_as(_dp)))
        return out.value, grad, H

    def nll_parts_device(self, params, dev_parts):
        """launch this rank's likelihood kernel; (S, I, n_ev) stay in the CUDA tensor dev_parts (3 float64); no wait"""
        p, pp, n = self._params(params)
        self._check(self.L.mipwa_nll_parts_device(self._h, pp, n, _dev_ptr(dev_parts, 3)))

    def nll_parts_static(self, params, dev_parts, blocks=0):
        """nll_parts_device on the recompute path with the kernel's scratch in the library's static device array: no
        device allocation in the call (include/mipwa.h); blocks > STATIC_MAX_BLOCKS is refused"""
        p, pp, n = self._params(params)
        self._check(self.L.mipwa_nll_parts_static(self._h, pp, n, int(blocks), _dev_ptr(dev_parts, 3)))

    def combine_parts_device(self, dev_parts_all, n_ranks):
        """(NLL, S, I, n_ev) of the whole sample from the gathered pieces (CUDA tensor, 3 n_ranks float64)"""
        out, S, Iv, nn = C.c_double(), C.c_double(), C.c_double(), C.c_int64()
        self._check(self.L.mipwa_combine_parts_device(self._h, _dev_ptr(dev_parts_all, 3 * n_ranks), int(n_ranks),
                                                      C.byref(out), C.byref(S), C.byref(Iv), C.byref(nn)))
        return out.value, S.value, Iv.value, nn.value

    def norm_parts(self, params, grad=True):
        """phase 1 of the sharded mixture likelihood: (I_r, dI_r/dtheta or None)"""
        p, pp, n = self._params(params)
        Iv = C.c_double()
        g = np.empty(2 * self.N + 2 * self.R) if grad else None
        self._check(self.L.mipwa_norm_parts(self._h, pp, n, C.byref(Iv), g.ctypes.data_as(_dp) if grad else None))
        return Iv.value, g

    def nll_mix_parts(self, params, f_sig, integral_total, grad=True):
        """phase 2: (S_r, Q_r, d(-S_r)/dtheta or None) with the integral of the whole sample"""
        p, pp, n = self._params(params)
        S, Q = C.c_double(), C.c_double()
        g = np.empty(2 * self.N + 2 * self.R) if grad else None
        self._check(self.L.mipwa_nll_mix_parts(self._h, pp, n, float(f_sig), float(integral_total), C.byref(S), C.byref(Q),
                                               g.ctypes.data_as(_dp) if grad else None))
        return S.value, Q.value, g

    def hessian_parts(self, params):
        """this rank's (M, G): K x K complex arrays of the event sum and the Gram matrix (mipwa_hessian_parts)"""
        p, pp, n = self._params(params)
        ln = int(self.L.mipwa_hessian_parts_len(self._h))
        M, G = np.empty(ln), np.empty(ln)
        self._check(self.L.mipwa_hessian_parts(self._h, pp, n, M.ctypes.data_as(_dp), G.ctypes.data_as(_dp)))
        return M, G

    def hessian_assemble(self, params, n_ev_total, M, G, grad):
        p, pp, n = self._params(params)
        P = 2 * self.N + 2 * self.R
        M, G, grad = _host(M), _host(G), _host(grad)
        H = np.empty((P, P))
        self._check(self.L.mipwa_hessian_assemble(self._h, pp, n, int(n_ev_total), M.ctypes.data_as(_dp),
                                                  G.ctypes.data_as(_dp), grad.ctypes.data_as(_dp), H.ctypes.data_as(_dp)))
        return H

    def generate(self, params, key, n, n_side=1024, n_coarse=64, device=False):
        """n toy events with density |A(params)|^2 (accept-reject on the GPU, counter-based stream `key`).
        Returns (s12, s13, candidates drawn); numpy arrays, or CUDA torch tensors if device=True."""
        p, pp, npar = self._params(params)
        tried = C.c_int64(0)
        if device:
            import torch
            a = torch.empty(int(n), dtype=torch.float64, device=f"cuda:{self.device}")
            b = torch.empty_like(a)
            pa, pb, mem = C.c_void_p(a.data_ptr()), C.c_void_p(b.data_ptr()), MEM_DEVICE
        else:
            a, b = np.empty(int(n)), np.empty(int(n))
            pa, pb, mem = C.c_void_p(a.ctypes.data), C.c_void_p(b.ctypes.data), MEM_HOST
        self._check(self.L.mipwa_generate(self._h, pp, npar, C.c_uint64(int(key)), int(n), int(n_side), int(n_coarse),
                                          pa, pb, mem, C.byref(tried)))
        return a, b, tried.value

    def eval_abs2(self, params, which=0):
        p, pp, n = self._params(params)
        size = self.n_events if which == 0 else self.n_norm
        out = np.empty(max(size, 0))
        self._check(self.L.mipwa_eval_abs2(self._h, pp, n, int(which), out.ctypes.data_as(_dp), size))
        return out

    def eval_basis(self, params, which=0, first=0, count=None):
        p, pp, n = self._params(params)
        size = self.n_events if which == 0 else self.n_norm
        count = size - first if count is None else count
        out = np.empty((count, self.K, 2))
        self._check(self.L.mipwa_eval_basis(self._h, pp, n, int(which), int(first), int(count),
                                            out.ctypes.data_as(_dp)))
        return out[..., 0] + 1j * out[..., 1]

    def enable_timing(self, on=True):
        self._check(self.L.mipwa_enable_timing(self._h, int(bool(on))))

    def last_kernel_ms(self):
        ms = C.c_float()
        self._check(self.L.mipwa_last_kernel_ms(self._h, C.byref(ms)))
        return ms.value

    def launch_count(self):
        return int(self.L.mipwa_launch_count(self._h))


def measure_fp64_peak(device=0, seconds=2.0):
    """(TFLOP/s of the FP64 pipe on 2-register + immediate DFMAs, TFLOP/s on 3-register DFMAs)"""
    L = load_library()
    out, out3 = C.c_double(), C.c_double()
    rc = L.mipwa_measure_fp64_peak(int(device), float(seconds), C.byref(out), C.byref(out3))
    if rc != OK:
        raise MipwaError(rc, "mipwa_measure_fp64_peak failed")
    return out.value, out3.value


def combine_parts(parts):
    """A7 over gathered (S_r, I_r, n_r) rows in rank order (C library, host only): (nll, S, I, n_ev)"""
    L = load_library()
    a = np.ascontiguousarray(parts, dtype=np.float64).reshape(-1, 3)
    out, S, Iv, nn = C.c_double(), C.c_double(), C.c_double(), C.c_int64()
    rc = L.mipwa_combine_parts(a.shape[0], a.ctypes.data_as(_dp), C.byref(out), C.byref(S), C.byref(Iv), C.byref(nn))
    if rc != OK:
        raise MipwaError(rc, "mipwa_combine_parts failed")
    return out.value, S.value, Iv.value, nn.value


def combine_parts_batch(parts, n_batch):
    """A7 at every vector of a batch over gathered rows (S_r[0..B), I_r[0..B), n_r), rank order (C library): B values"""
    L = load_library()
    a = np.ascontiguousarray(parts, dtype=np.float64).reshape(-1, 2 * n_batch + 1)
    out = np.empty(n_batch)
    rc = L.mipwa_combine_parts_batch(a.shape[0], int(n_batch), a.ctypes.data_as(_dp), out.ctypes.data_as(_dp))
    if rc != OK:
        raise MipwaError(rc, "mipwa_combine_parts_batch failed")
    return out


def combine_grad_parts(parts, n_params):
    """whole-sample (nll, grad, S, I, n_ev) from gathered rows (S_r, I_r, n_r, grad_ev_r, grad_nm_r), rank order"""
    L = load_library()
    a = np.ascontiguousarray(parts, dtype=np.float64).reshape(-1, 3 + 2 * n_params)
    out, S, Iv, nn = C.c_double(), C.c_double(), C.c_double(), C.c_int64()
    g = np.zeros(max(n_params, 1))
    rc = L.mipwa_combine_grad_parts(a.shape[0], int(n_params), a.ctypes.data_as(_dp), C.byref(out), g.ctypes.data_as(_dp),
                                    C.byref(S), C.byref(Iv), C.byref(nn))
    if rc != OK:
        raise MipwaError(rc, "mipwa_combine_grad_parts failed")
    return out.value, g[:n_params], S.value, Iv.value, nn.value


def combine_mix_parts(norm_parts, ev_parts, n_lin, f_sig):
    """whole-sample mixture (nll, grad, dnll/df_sig) from gathered rows (I_r, grad_nm_r) and (S_r, Q_r, n_r, grad_ev_r)"""
    L = load_library()
    a = np.ascontiguousarray(norm_parts, dtype=np.float64).reshape(-1, 1 + n_lin)
    b = np.ascontiguousarray(ev_parts, dtype=np.float64).reshape(-1, 3 + n_lin)
    out, dfs = C.c_double(), C.c_double()
    g = np.zeros(max(n_lin, 1))
    rc = L.mipwa_combine_mix_parts(a.shape[0], int(n_lin), float(f_sig), a.ctypes.data_as(_dp), b.ctypes.data_as(_dp),
                                   C.byref(out), g.ctypes.data_as(_dp), C.byref(dfs))
    if rc != OK:
        raise MipwaError(rc, "mipwa_combine_mix_parts failed")
    return out.value, g[:n_lin], dfs.value


def version():
    return load_library().mipwa_version().decode()
