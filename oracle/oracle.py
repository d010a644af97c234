"""ctypes front-end of the fp64 CPU oracle (oracle/u1u1_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It shares nothing with
paper_2208_01525_b200 and never imports it.

The C file holds the per-site formulas; this module holds only argument marshalling, the lattice-wide
sums written as plain numpy reductions, and the derived scalars of PAPER.md Eq. 31-37
(:185-221).  State arrays are float64 numpy arrays of shape (20, nz, ny, nx) (canonical layout, see
the C header comment).

Pins of the diagnostic combinations (tests/test_oracle_pins_diag.py): the Lagrangian density and its a-weights by
the variational principle against the pinned kicks (c != 1), virial theorems on the normal modes, the
Euler-Lagrange damping ratio omega/delta = 1 - beta; xi_L and mu = 2 pi sigma^2 on the Bogomolny vortex; V_int on
hand-computed sites; f_total / f_p on hand-built lines; the near-cut mask on hand-built links.  Nothing is left
"parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "u1u1_oracle.c")
_LIB = os.path.join(_HERE, "libu1u1_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP over z-planes of the two kick loops only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
             "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Lattice(ctypes.Structure):
    _fields_ = [("nx", ctypes.c_int), ("ny", ctypes.c_int), ("nz", ctypes.c_int),
                ("dx", ctypes.c_double)]


class _Couplings(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in
                ("lambda1", "lambda2", "e1", "e2", "eta1", "eta2", "kappa")]


@dataclass
class Couplings:
    """lambda_p0, lambda_q0, e_p0, e_q0, sigma_p, sigma_q, kappa_0 (PAPER.md:52 Eq. 4, :268-270)."""
    lambda1: float = 2.0
    lambda2: float = 2.0
    e1: float = 1.0
    e2: float = 1.0
    eta1: float = 1.0
    eta2: float = 1.0
    kappa: float = 0.9

    def c(self) -> _Couplings:
        return _Couplings(self.lambda1, self.lambda2, self.e1, self.e2, self.eta1, self.eta2,
                          self.kappa)


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        d = ctypes.c_double
        LP, KP = ctypes.POINTER(_Lattice), ctypes.POINTER(_Couplings)
        L.orc_scalars.argtypes = [d, d, d, d, d, dp]
        L.orc_kick_scalars.argtypes = [LP, KP, dp, d, d, d]
        L.orc_kick_gauge.argtypes = [LP, KP, dp, d, d, d]
        L.orc_friction.argtypes = [LP, dp, d]
        L.orc_drift.argtypes = [LP, dp, d]
        L.orc_step.argtypes = [LP, KP, dp, d, d, d, d, d, d]
        L.orc_cool_step.argtypes = [LP, KP, dp, d, dp]
        L.orc_gauss_field.argtypes = [LP, KP, dp, ctypes.c_int, d, dp, dp, dp]
        L.orc_windings.argtypes = [LP, dp, ctypes.c_int, d, ctypes.POINTER(ctypes.c_int32),
                                   ctypes.POINTER(ctypes.c_uint8)]
        L.orc_cells.argtypes = [LP, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32)]
        L.orc_densities.argtypes = [LP, KP, dp] + [dp] * 6
        L.orc_philox4x32_10.argtypes = [ctypes.POINTER(ctypes.c_uint32)] * 3
        L.orc_init_random_phase.argtypes = [LP, KP, ctypes.c_uint64, dp]
        L.orc_init_smoothed.argtypes = [LP, KP, ctypes.c_uint64, d, ctypes.c_int, dp]
        for f in ("orc_scalars", "orc_kick_scalars", "orc_kick_gauge", "orc_friction", "orc_drift",
                  "orc_step", "orc_cool_step", "orc_gauss_field", "orc_windings", "orc_cells", "orc_densities",
                  "orc_philox4x32_10", "orc_init_random_phase", "orc_init_smoothed"):
            getattr(L, f).restype = None
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _lat(state: np.ndarray, dx: float) -> _Lattice:
    assert state.ndim == 4 and state.shape[0] == 20, state.shape
    _, nz, ny, nx = state.shape
    return _Lattice(nx, ny, nz, dx)


# ------------------------------------------------------------------------------------------------
def scalars(tau, m, beta, dtau, tau_norm=1.0):
    """(a, c=a^{2 beta}, delta, omega) at conformal time tau.  PAPER.md:133 Eq. 19, :147 Eq. 22."""
    out = np.zeros(4)
    lib().orc_scalars(tau, m, beta, dtau, tau_norm, _dp(out))
    return tuple(out)


def philox(ctr, key):
    c = (ctypes.c_uint32 * 4)(*ctr)
    k = (ctypes.c_uint32 * 2)(*key)
    o = (ctypes.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


def init_random_phase(n, seed, K: Couplings = Couplings(), dims=None) -> np.ndarray:
    nz, ny, nx = dims if dims else (n, n, n)
    state = np.zeros((20, nz, ny, nx))
    kc = K.c()
    lat = _Lattice(nx, ny, nz, 1.0)
    lib().orc_init_random_phase(ctypes.byref(lat), ctypes.byref(kc), seed, _dp(state))
    return state


def init_smoothed(n, seed, width=5.0, trunc=20, K: Couplings = Couplings()) -> np.ndarray:
    state = np.zeros((20, n, n, n))
    kc = K.c()
    lat = _Lattice(n, n, n, 1.0)
    lib().orc_init_smoothed(ctypes.byref(lat), ctypes.byref(kc), seed, width, trunc, _dp(state))
    return state


def kick_scalars(state, dx, K, c, delta, dtau):
    lat, kc = _lat(state, dx), K.c()
    lib().orc_kick_scalars(ctypes.byref(lat), ctypes.byref(kc), _dp(state), c, delta, dtau)


def kick_gauge(state, dx, K, c, omega, dtau):
    lat, kc = _lat(state, dx), K.c()
    lib().orc_kick_gauge(ctypes.byref(lat), ctypes.byref(kc), _dp(state), c, omega, dtau)


def friction(state, dx, f):
    lat = _lat(state, dx)
    lib().orc_friction(ctypes.byref(lat), _dp(state), f)


def drift(state, dx, dtau):
    lat = _lat(state, dx)
    lib().orc_drift(ctypes.byref(lat), _dp(state), dtau)


def step(state, dx, K, tau, m, beta, dtau, tau_norm=1.0, friction=1.0, n=1):
    """n leapfrog steps in place; step k uses tau_k = tau + k*dtau.  Returns the final time."""
    lat, kc = _lat(state, dx), K.c()
    for k in range(n):
        lib().orc_step(ctypes.byref(lat), ctypes.byref(kc), _dp(state), tau + k * dtau, m, beta,
                       dtau, tau_norm, friction)
    return tau + n * dtau


def cool(state, dx, K, dcool, n=1):
    """n explicit Euler steps of the diffusive cooling equations, Eq. 27-30 (reading R-20):
    first-order flow of phi, psi (no kappa term) and of the links; momenta are zero on exit."""
    lat, kc = _lat(state, dx), K.c()
    scratch = np.zeros(10 * state[0].size)
    for _ in range(n):
        lib().orc_cool_step(ctypes.byref(lat), ctypes.byref(kc), _dp(state), dcool, _dp(scratch))


def gauss_coefficient(tau_last, m, beta, dtau, tau_norm=1.0):
    """c_G = c(tau_last)(1+delta)/(1+omega) of the step just completed (reading R-5)."""
    _, c, delta, omega = scalars(tau_last, m, beta, dtau, tau_norm)
    return c * (1.0 + delta) / (1.0 + omega)


def gauss_field(state, dx, K, sector, cG):
    lat, kc = _lat(state, dx), K.c()
    shp = state.shape[1:]
    g, rho, div = np.zeros(shp), np.zeros(shp), np.zeros(shp)
    lib().orc_gauss_field(ctypes.byref(lat), ctypes.byref(kc), _dp(state), sector, cG, _dp(g),
                          _dp(rho), _dp(div))
    return g, rho, div


def gauss_violation(state, dx, K, cG):
    """8 doubles: per sector ||g||_2, ||rho||_2, max|g|, ||g||_2 / max(||rho||_2, ||divE||_2, tiny)."""
    out = []
    for sec in (0, 1):
        g, rho, div = gauss_field(state, dx, K, sec, cG)
        l2g, l2r, l2d = (float(np.sqrt(np.sum(a * a))) for a in (g, rho, div))
        out += [l2g, l2r, float(np.max(np.abs(g))), l2g / max(l2r, l2d, 1e-300)]
    return np.array(out)


def windings(state, dx, sector, cut_tol=1e-5):
    """W[3, nz, ny, nx] (xy, yz, zx) int32 and the near-branch-cut mask (same shape, uint8)."""
    lat = _lat(state, dx)
    shp = (3,) + state.shape[1:]
    W = np.zeros(shp, dtype=np.int32)
    near = np.zeros(shp, dtype=np.uint8)
    lib().orc_windings(ctypes.byref(lat), _dp(state), sector, cut_tol,
                       W.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                       near.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)))
    return W, near


def cells(W, dx=1.0):
    _, nz, ny, nx = W.shape
    lat = _Lattice(nx, ny, nz, dx)
    C = np.zeros((nz, ny, nx), dtype=np.int32)
    Wc = np.ascontiguousarray(W, dtype=np.int32)
    lib().orc_cells(ctypes.byref(lat), Wc.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                    C.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)))
    return C


def cells_pq_tolerant(Cp, Cq):
    """Fast method with one cell of tolerance, PAPER.md:234 ("non-zero at the same location, or displaced by one
    cell in any direction"), reading R-13b: (number of pierced p cells with a pierced q cell in their periodic
    3x3x3 neighbourhood, number of pierced q cells with a pierced p cell in theirs)."""
    def dilate(mask):
        out = np.zeros_like(mask)
        for dz in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dx_ in (-1, 0, 1):
                    out |= np.roll(mask, (dz, dy, dx_), axis=(0, 1, 2))
        return out
    p, q = Cp > 0, Cq > 0
    return int(np.sum(p & dilate(q))), int(np.sum(q & dilate(p)))


def pq_mask(Cp, Cq, tolerant=False):
    """Cells counted as pierced by a pq string: exact overlap, or with one cell of tolerance (R-13b):
    a pierced cell of either type with a pierced cell of the other type in its periodic 3x3x3 neighbourhood."""
    p, q = Cp > 0, Cq > 0
    if not tolerant:
        return p & q
    def dilate(mask):
        out = np.zeros_like(mask)
        for dz in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dx_ in (-1, 0, 1):
                    out |= np.roll(mask, (dz, dy, dx_), axis=(0, 1, 2))
        return out
    return (p & dilate(q)) | (q & dilate(p))


def pq_segments(Cp, Cq, dx, min_cells=1, tolerant=False):
    """The robust method's numbers (reading R-21) by plain flood fill: connected regions
    of pq cells over the periodic 26-neighbourhood.  A region's cell count is N = (its cells pierced by p + its cells
    pierced by q) / 2 (reading R-21b): the number of its cells for exact overlap, and for one cell of tolerance the
    SAME length for a coincident and for a one-cell-displaced pair of lines (as L_pq^tol of R-13b; the plain cell count
    of the union mask would double for the displaced pair).  N_pq = regions with N >= min_cells, L_pq = dx sum (N - 1)
    over them (:248), l_pq = L_pq / N_pq (Eq. 38).  `cells_mask` is the plain cell count of the union mask, the reading
    R-21b replaced.  Returns (dict, sorted list of all region counts N)."""
    mask = pq_mask(Cp, Cq, tolerant)
    nz, ny, nx = mask.shape
    seen = np.zeros(mask.shape, dtype=bool)
    sizes = []
    for start in zip(*np.nonzero(mask)):
        if seen[start]:
            continue
        seen[start] = True
        stack, n2 = [start], 0
        while stack:
            z, y, x = stack.pop()
            n2 += int(Cp[z, y, x] > 0) + int(Cq[z, y, x] > 0)
            for dz in (-1, 0, 1):
                for dy in (-1, 0, 1):
                    for dx_ in (-1, 0, 1):
                        c = ((z + dz) % nz, (y + dy) % ny, (x + dx_) % nx)
                        if mask[c] and not seen[c]:
                            seen[c] = True
                            stack.append(c)
        sizes.append(n2 / 2 if n2 % 2 else n2 // 2)
    kept = [n for n in sizes if n >= min_cells]
    L = dx * sum(n - 1 for n in kept)
    out = {"N_pq": len(kept), "L_pq": L, "l_pq": L / len(kept) if kept else 0.0, "cells_kept": sum(kept),
           "segments_all": len(sizes), "cells_all": sum(sizes), "largest": max(sizes) if sizes else 0,
           # the OTHER reading of a tolerant region's size, for comparison with the paper's Fig. 1: the plain number of cells
           # of the union mask (equal to cells_all for exact overlap, about twice it for displaced pairs)
           "cells_mask": int(np.sum(mask))}
    return out, sorted(sizes)


def densities(state, dx, K):
    """dict of per-site arrays kin, grad, elec, mag, pot, vint (no scale-factor weights)."""
    lat, kc = _lat(state, dx), K.c()
    shp = state.shape[1:]
    names = ("kin", "grad", "elec", "mag", "pot", "vint")
    arrs = [np.zeros(shp) for _ in names]
    lib().orc_densities(ctypes.byref(lat), ctypes.byref(kc), _dp(state), *[_dp(a) for a in arrs])
    return dict(zip(names, arrs))


def energy(state, dx, K):
    """Flat-space (c = 1) lattice Hamiltonian, O-11."""
    d = densities(state, dx, K)
    return dx ** 3 * float(np.sum(d["kin"] + d["grad"] + d["elec"] + d["mag"] + d["pot"]))


def lagrangian(state, dx, K, c):
    """Per-site Lagrangian density L_x of PAPER.md:198 Eq. 33 (reading R-14): Eq. 1 (:43) in the comoving variables of
    the discretisation, divided by a^2, with the couplings of Eq. 12 (:89) -- kin - grad + (elec - mag)/c - c pot,
    c = a^{2 beta}.  Returns (L_x, the dict of unweighted densities it was formed from)."""
    d = densities(state, dx, K)
    return d["kin"] - d["grad"] + (d["elec"] - d["mag"]) / c - c * d["pot"], d


def diagnostics(state, dx, K, c, cut_tol=1e-5):
    """All in-loop diagnostics of PAPER.md Eq. 31-37 from one snapshot, as a dict."""
    out = {}
    Ws, Cs = [], []
    for sec, tag in ((0, "p"), (1, "q")):
        W, near = windings(state, dx, sec, cut_tol)
        C = cells(W)
        Ws.append(W)
        Cs.append(C)
        out[f"sumW_{tag}"] = int(np.sum(np.abs(W)))
        out[f"near_{tag}"] = int(np.sum(near))
        out[f"cells_{tag}"] = int(np.sum(C > 0))
        out[f"maxW_{tag}"] = int(np.max(np.abs(W)))
    out["cells_pq"] = int(np.sum((Cs[0] > 0) & (Cs[1] > 0)))
    out["cells_pq_tol_p"], out["cells_pq_tol_q"] = cells_pq_tolerant(Cs[0], Cs[1])
    out["L_pq_tol"] = 0.5 * dx * (out["cells_pq_tol_p"] + out["cells_pq_tol_q"])
    lag, d = lagrangian(state, dx, K, c)
    out["sum_L"] = float(np.sum(lag))
    out["sum_kin_L"] = float(np.sum(d["kin"] * lag))
    out["sum_grad_L"] = float(np.sum(d["grad"] * lag))
    out["sum_kin_V"] = float(np.sum(d["kin"] * d["vint"]))
    out["sum_grad_V"] = float(np.sum(d["grad"] * d["vint"]))
    out["sum_vint"] = float(np.sum(d["vint"]))
    for k in ("kin", "grad", "elec", "mag", "pot"):
        out[f"sum_{k}"] = float(np.sum(d[k]))
    out.update(derived(out, state.shape[1:], dx, K))
    return out


def derived(s, shape, dx, K):
    """Eq. 31-37 from the lattice sums.  L_pq = dx N_pq; L_p = dx sum|W^p| - L_pq."""
    nz, ny, nx = shape
    vol = nx * ny * nz * dx ** 3
    L_pq = dx * s["cells_pq"]
    L_p = dx * s["sumW_p"] - L_pq
    L_q = dx * s["sumW_q"] - L_pq
    inf = float("inf")
    xi = lambda L: float(np.sqrt(vol / L)) if L > 0 else inf
    mu = 2.0 * np.pi * K.eta1 ** 2
    denom = dx ** 3 * s["sum_L"]
    R_L = s["sum_kin_L"] / s["sum_grad_L"] if s["sum_grad_L"] != 0 else float("nan")
    R_V = s["sum_kin_V"] / s["sum_grad_V"] if s["sum_grad_V"] != 0 else float("nan")
    tot = L_pq + L_p + L_q
    return {
        "L_p": L_p, "L_q": L_q, "L_pq": L_pq,
        "xi_p": xi(L_p), "xi_q": xi(L_q), "xi_pq": xi(L_pq), "xi_W": xi(tot),
        "xi_L": float(np.sqrt(-mu * vol / denom)) if denom < 0 else float("nan"),
        "f_total": L_pq / tot if tot > 0 else 0.0,
        "f_p": L_pq / L_p if L_p > 0 else 0.0,
        "v2_L": 2 * R_L / (1 + R_L), "v2_pq": 2 * R_V / (1 + R_V),
        # Eq. 36 is a velocity only for 0 <= R <= 1 (0 <= <v^2> <= 1): bit 0 for W = L, bit 1 for W = V_int
        "v2_valid": (1 if 0.0 <= R_L <= 1.0 else 0) + (2 if 0.0 <= R_V <= 1.0 else 0),
    }
