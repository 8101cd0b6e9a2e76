"""Seeded synthetic inputs for the MIPWA hot path (BASELINE.json configs 0-4 made concrete).

This module serves BOTH the oracle-side tests and the CUDA-side bench/tests and therefore holds none of the
method's arithmetic: no spline, no Breit-Wigner, no barrier, no angular factor, no likelihood.  It contains only
  * a counter-based random generator (splitmix64 finaliser over seed/stream/counter; uniforms (x>>11) 2^-53,
    normals by Box-Muller) so that any chunking of the draws gives identical numbers,
  * the three-body phase-space boundary needed to place points (its own implementation; the oracle and the CUDA
    library each carry theirs),
  * the model descriptions (knot positions, resonance lists, truth parameters) of the five configs,
  * accept-reject on a density supplied by the CALLER as a callback `abs2_fn(s12, s13) -> |A|^2`
    (tests pass the oracle; bench.py passes the CUDA library's per-point hook).

The paper measures on an LHCb D+ -> K+K+K- sample and on a 100 K-event toy whose inputs are not printed
(PAPER.md:45-47); these configs stand in for both (same structure: Dalitz-distributed (s12,s13) pairs drawn
from |A|^2, 10-50 knots bracketing the paper's 40, 1e4-1e8 events bracketing its 1e5).  Recipe: DESIGN.md 4.
"""
import math

import numpy as np

M_D = 1.86966          # GeV  (BASELINE.json configs[0])
M_PI = 0.13957         # GeV
KIN = {"M": M_D, "m1": M_PI, "m2": M_PI, "m3": M_PI}
M_K = 0.493677         # GeV; the paper's own decay D+ -> K+ K+ K- 
KIN_KKK = {"M": M_D, "m1": M_K, "m2": M_K, "m3": M_K}
KNOT_LO, KNOT_HI = 0.0779, 2.9929          # GeV^2 (BASELINE.json configs[0])
R_RES, R_PARENT = 1.5, 5.0                 # GeV^-1 (configs[0]; reading P11: the same for every resonance)

_MASK = np.uint64(0xFFFFFFFFFFFFFFFF)


# ----------------------------------------------------------------------------------------------------------------
# counter-based RNG
# ----------------------------------------------------------------------------------------------------------------
def _mix(z):
    """splitmix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def stream_key(seed, config, stream):
    """One 64-bit key per (seed, config, stream-id)."""
    with np.errstate(over="ignore"):
        k = _mix(np.uint64(seed) * np.uint64(0x9E3779B97F4A7C15) + np.uint64(0x1234567))
        k = _mix(k ^ (np.uint64(config + 1) * np.uint64(0xD1B54A32D192ED03)))
        k = _mix(k ^ (np.uint64(stream + 1) * np.uint64(0x8CB92BA72F3D8DD7)))
    return np.uint64(k)


def uniforms(key, start, count):
    """count uniforms in [0,1) for counters start .. start+count-1 of the stream `key`."""
    ctr = np.arange(start, start + count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x = _mix(_mix(ctr * np.uint64(0x9E3779B97F4A7C15) + np.uint64(key)) ^ np.uint64(key))
    return (x >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normals(key, start, count):
    """count standard normals (Box-Muller on uniform pairs 2i, 2i+1 of the stream)."""
    u = uniforms(key, 2 * start, 2 * count)
    u1, u2 = 1.0 - u[0::2], u[1::2]                       # u1 in (0,1]
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)


# stream ids (draw order of reading P21)
S_KNOT_MAG, S_KNOT_PHASE, S_COEF, S_EVENTS, S_NORM, S_PERTURB = 0, 1, 2, 3, 4, 5


# ----------------------------------------------------------------------------------------------------------------
# phase space (placement of points only)
# ----------------------------------------------------------------------------------------------------------------
def _lam(a, b, c):
    return a * a + b * b + c * c - 2.0 * (a * b + a * c + b * c)


def s_limits(kin=KIN):
    return (kin["m1"] + kin["m2"]) ** 2, (kin["M"] - kin["m3"]) ** 2


def s13_band(s12, kin=KIN):
    """centre and half-width of the allowed s13 interval at s12 (arrays)."""
    M2, a, b, c = kin["M"] ** 2, kin["m1"] ** 2, kin["m2"] ** 2, kin["m3"] ** 2
    s12 = np.asarray(s12, dtype=np.float64)
    centre = a + c + (s12 + a - b) * (M2 - s12 - c) / (2.0 * s12)
    prod = _lam(s12, a, b) * _lam(M2, s12, c)
    half = np.sqrt(np.maximum(prod, 0.0)) / (2.0 * s12)
    return centre, half


def inside(s12, s13, kin=KIN):
    lo, hi = s_limits(kin)
    s12 = np.asarray(s12, dtype=np.float64)
    s13 = np.asarray(s13, dtype=np.float64)
    ok = (s12 >= lo) & (s12 <= hi)
    centre, half = s13_band(np.where(ok, s12, lo), kin)
    return ok & (np.abs(s13 - centre) <= half)


def dalitz_area(kin=KIN, order=256):
    """Area = int 2 h(s) ds, Gauss-Legendre after s = lo + (hi-lo) sin^2 t (removes the sqrt end points)."""
    lo, hi = s_limits(kin)
    t, w = np.polynomial.legendre.leggauss(order)
    t = 0.25 * math.pi * (t + 1.0)
    w = 0.25 * math.pi * w
    s = lo + (hi - lo) * np.sin(t) ** 2
    M2, a, b, c = kin["M"] ** 2, kin["m1"] ** 2, kin["m2"] ** 2, kin["m3"] ** 2
    # lambda(s,a,b) = (s-lo)(s-(m1-m2)^2), lambda(M2,s,c) = (hi-s)((M+m3)^2-s); sqrt((s-lo)(hi-s)) = (hi-lo) sin t cos t
    r1 = s - (kin["m1"] - kin["m2"]) ** 2
    r2 = (kin["M"] + kin["m3"]) ** 2 - s
    two_h = (hi - lo) * np.sin(t) * np.cos(t) * np.sqrt(r1 * r2) / s
    ds = 2.0 * (hi - lo) * np.sin(t) * np.cos(t)
    return float(np.sum(w * two_h * ds))


def grid_points(n_side, kin=KIN):
    """n_side x n_side cells over the bounding square, points at cell centres, kept iff the centre is inside;
    w = cell area (reading P12; "evenly distributed grid points in the Dalitz plot plane")."""
    lo, hi = s_limits(kin)
    h = (hi - lo) / n_side
    c = lo + (np.arange(n_side, dtype=np.float64) + 0.5) * h
    g12, g13 = np.meshgrid(c, c, indexing="ij")
    g12, g13 = g12.ravel(), g13.ravel()
    keep = inside(g12, g13, kin)
    g12, g13 = g12[keep].copy(), g13[keep].copy()
    return g12, g13, np.full(g12.size, h * h)


def phase_space_points(n, key, kin=KIN, chunk=1 << 21):
    """n points uniform inside the Dalitz boundary: candidate i = (u_{2i}, u_{2i+1}) scaled to the bounding
    square, kept iff inside, in counter order."""
    lo, hi = s_limits(kin)
    out12, out13, have, ctr = [], [], 0, 0
    while have < n:
        u = uniforms(key, 2 * ctr, 2 * chunk)
        a = lo + (hi - lo) * u[0::2]
        b = lo + (hi - lo) * u[1::2]
        keep = inside(a, b, kin)
        out12.append(a[keep]); out13.append(b[keep])
        have += int(keep.sum()); ctr += chunk
    return np.concatenate(out12)[:n].copy(), np.concatenate(out13)[:n].copy()


class Envelope:
    """Piecewise-constant envelope of |A|^2 over an n_coarse x n_coarse partition of the bounding square.

    env[cx, cy] = 1.2 x max |A|^2 over the cell centres of the n_side^2 fine grid that fall inside the Dalitz
    boundary and inside coarse cell (cx, cy) (reading P22 applied per coarse cell; n_coarse = 1 is the single
    global envelope).  A coarse cell without any fine point but next to one that has some takes the largest
    neighbouring value, so thin slivers along the boundary stay covered.  Accept-reject against it samples
    exactly the density |A|^2 / integral wherever the envelope bounds |A|^2; larger values clamp."""

    def __init__(self, abs2_fn, kin=KIN, n_side=1024, n_coarse=64):
        lo, hi = s_limits(kin)
        self.lo, self.hi, self.nc = lo, hi, int(n_coarse)
        self.H = (hi - lo) / self.nc
        g12, g13, _ = grid_points(n_side, kin)
        a2 = np.asarray(abs2_fn(g12, g13), dtype=np.float64)
        cx = np.minimum(((g12 - lo) / self.H).astype(np.int64), self.nc - 1)
        cy = np.minimum(((g13 - lo) / self.H).astype(np.int64), self.nc - 1)
        own = np.zeros((self.nc, self.nc))
        np.maximum.at(own, (cx, cy), a2)
        pad = np.pad(own, 1)
        neigh = np.max([pad[1 + dx:1 + dx + self.nc, 1 + dy:1 + dy + self.nc]
                        for dx in (-1, 0, 1) for dy in (-1, 0, 1)], axis=0)
        self.env = 1.2 * np.where(own > 0, own, neigh)
        self.global_max = float(a2.max())
        cum = np.cumsum(self.env.ravel())
        self.cum = cum / cum[-1]

    def draw(self, u_cell, u_x, u_y):
        """coarse cell from u_cell (inverse CDF over cells weighted by env), then a uniform point in it."""
        cell = np.minimum(np.searchsorted(self.cum, u_cell, side="right"), self.nc * self.nc - 1)
        cx, cy = cell // self.nc, cell % self.nc
        return self.lo + (cx + u_x) * self.H, self.lo + (cy + u_y) * self.H, self.env.ravel()[cell]


def accept_reject(n, key, abs2_fn, envelope, kin=KIN, chunk=1 << 21):
    """n events with density proportional to abs2_fn inside the boundary.  Candidate i uses uniforms 4i .. 4i+3 of
    the stream: coarse cell, position in the cell, and the accept threshold u * env(cell) < |A|^2.  Events are the
    first n accepted candidates in counter order, so the result does not depend on `chunk`."""
    out12, out13, have, ctr = [], [], 0, 0
    while have < n:
        u = uniforms(key, 4 * ctr, 4 * chunk)
        a, b, env = envelope.draw(u[0::4], u[1::4], u[2::4])
        thr = u[3::4] * env
        keep = inside(a, b, kin)
        a, b, thr = a[keep], b[keep], thr[keep]
        acc = thr < np.asarray(abs2_fn(a, b))
        out12.append(a[acc]); out13.append(b[acc])
        have += int(acc.sum()); ctr += chunk
    return np.concatenate(out12)[:n].copy(), np.concatenate(out13)[:n].copy()


def envelope_of(abs2_fn, kin=KIN, n_side=1024, n_coarse=64):
    return Envelope(abs2_fn, kin, n_side, n_coarse)


# ----------------------------------------------------------------------------------------------------------------
# the five configs of BASELINE.json
# ----------------------------------------------------------------------------------------------------------------
def _res(mass, width, spin, shape_floats=0):
    return {"mass": mass, "width": width, "spin": spin, "r_res": R_RES, "r_parent": R_PARENT,
            "shape_floats": shape_floats}


RHO770 = (0.775, 0.149, 1)
F2_1270 = (1.2755, 0.1867, 2)
RHO1450 = (1.465, 0.4, 1)
# reading P19: three synthetic entries completing config 4's "6 fixed-shape resonances"
SYN_A, SYN_B, SYN_C = (1.720, 0.250, 1), (1.5174, 0.086, 2), (0.78266, 0.00868, 1)


def knots_uniform(n):
    return np.linspace(KNOT_LO, KNOT_HI, n)


def knots_config2():
    """40 knots, half of them in [0.8, 1.2] (reading P17)."""
    a = np.linspace(KNOT_LO, 0.8, 7)[:-1]          # 6 knots KNOT_LO + i (0.8 - KNOT_LO)/6
    b = np.linspace(0.8, 1.2, 20)                  # 20 knots 0.8 + i 0.4/19, end points exact
    c = np.linspace(1.2, KNOT_HI, 15)[1:]          # 14 knots 1.2 + (i+1)(KNOT_HI - 1.2)/14
    return np.concatenate([a, b, c]).astype(np.float64)


_SPECS = {
    0: dict(knots=lambda: knots_uniform(10), res=[_res(*RHO770)], n_ev=10_000, norm=("grid", 100), calls=1),
    1: dict(knots=lambda: knots_uniform(30), res=[_res(*RHO770), _res(*F2_1270)], n_ev=100_000,
            norm=("mc", 200_000), calls=100),
    2: dict(knots=knots_config2, res=[_res(*RHO770), _res(*RHO1450), _res(*F2_1270)], n_ev=1_000_000,
            norm=("mc", 1_000_000), calls=1000),
    3: dict(knots=lambda: knots_uniform(50), res=[_res(*RHO770, shape_floats=1), _res(*RHO1450), _res(*F2_1270)],
            n_ev=10_000_000, norm=("mc", 10_000_000), calls=1000),
    # 5: not in BASELINE.json - the paper's own toy: D+ -> K+K+K-, 100 K events, 40 knots (39 slices)
    # across the whole m^2(K+K-) range + phi(1020), normalisation grid of spacing 0.001 GeV^2 (918 x 918 cells).
    # The paper prints no parameter values; the knot values follow the same recipe as configs 0-4, phi(1020) takes
    # its PDG mass and width and the radii of reading P11.
    5: dict(kin=KIN_KKK, knots=lambda: np.linspace(4 * M_K ** 2, (M_D - M_K) ** 2, 40), res=[_res(1.019461, 0.004249, 1)],
            n_ev=100_000, norm=("grid", 918), calls=100),
    4: dict(knots=lambda: knots_uniform(50),
            res=[_res(*RHO770), _res(*RHO1450), _res(*F2_1270), _res(*SYN_A), _res(*SYN_B), _res(*SYN_C)],
            n_ev=1_000_000, norm=("mc", 10_000_000), calls=20),
}


class Config:
    """Model description + truth parameter vector of BASELINE.json configs[idx] (seed 1 by default).

    Parameter layout (include/mipwa.h): [a_0..a_{N-1} | phi_0..phi_{N-1} | (|c_r|, arg c_r)... | (mass, width)
    of every shape_floats resonance in list order].
    """

    def __init__(self, idx, seed=1, n_ev=None, n_norm=None):
        spec = _SPECS[idx]
        self.idx, self.seed = idx, seed
        self.kin = dict(spec.get("kin", KIN))
        self.knots = spec["knots"]()
        self.resonances = [dict(r) for r in spec["res"]]
        self.N, self.R = self.knots.size, len(self.resonances)
        self.n_ev = spec["n_ev"] if n_ev is None else int(n_ev)
        kind, size = spec["norm"]
        self.norm_kind = kind
        self.norm_size = size if n_norm is None else int(n_norm)
        self.calls = spec["calls"]
        self.truth = self._truth()
        self.n_params = self.truth.size

    def key(self, stream):
        return stream_key(self.seed, self.idx, stream)

    def _truth(self):
        N, R = self.N, self.R
        mag = 0.5 + 1.5 * uniforms(self.key(S_KNOT_MAG), 0, N)                        # a_k ~ U[0.5, 2]
        phase = math.pi * np.arange(N) / (N - 1) + 0.2 * normals(self.key(S_KNOT_PHASE), 0, N)
        coef = []
        if self.idx == 0:
            coef = [1.0, 0.0]                                                          # rho(770) with c = 1
        else:
            u = uniforms(self.key(S_COEF), 0, 2 * R)
            for r in range(R):
                cm = 0.1 + 1.9 * u[2 * r]
                if self.idx == 4 and r == 5:
                    cm *= 0.01                                                         # reading P19 (narrow peak)
                if self.idx == 5:
                    cm *= 0.1          # |T| = 1/(m0 Gamma0) = 231 at the phi(1020) pole: this scale gives the phi a
                                       # fit fraction of 29 % beside the S-wave instead of > 99 %
                coef += [cm, 2.0 * math.pi * u[2 * r + 1]]
        shapes = []
        for r in self.resonances:
            if r["shape_floats"]:
                shapes += [r["mass"], r["width"]]
        return np.concatenate([mag, phase, np.array(coef), np.array(shapes)]).astype(np.float64)

    def perturbed(self, t):
        """Parameters of call t: truth + 1e-3 z_t, z iid standard normal, independent around truth (P20)."""
        z = normals(self.key(S_PERTURB), t * self.n_params, self.n_params)
        return self.truth + 1e-3 * z

    def norm_points(self, stream=0):
        """(s12, s13, w): config 0 = cell-centre grid with w = cell area; others = uniform phase-space sample with
        w = Area / n (reading P12)."""
        if self.norm_kind == "grid":
            return grid_points(self.norm_size, self.kin)
        g12, g13 = phase_space_points(self.norm_size, self.key(S_NORM + 16 * stream), self.kin)
        return g12, g13, np.full(g12.size, dalitz_area(self.kin) / g12.size)

    def events(self, abs2_fn, envelope=None, n=None, stream=0, chunk=1 << 21):
        """accept-reject events from the truth model; abs2_fn(s12, s13) must evaluate |A|^2 at self.truth."""
        if envelope is None:
            envelope = envelope_of(abs2_fn, self.kin)
        return accept_reject(self.n_ev if n is None else n, self.key(S_EVENTS + 16 * stream), abs2_fn, envelope,
                             self.kin, chunk=chunk)
