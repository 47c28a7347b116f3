"""ctypes/numpy front end of the fp64 CPU ORACLE (oracle/orc.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It shares no code with the CUDA path.

Everything here is argument marshalling; the arithmetic is in orc.c, which cites the paper.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# ORC_LIBORC: load a prebuilt copy instead (tests/oracle_mutants.py points the pin tests at deliberately broken builds)
_LIB_PATH = os.environ.get("ORC_LIBORC") or os.path.join(_HERE, "liborc.so")

CART, SPH, QSPH = 0, 1, 2
PERIODIC, ABSORB, AXIS = 0, 1, 2
NGHOST = 2


def build(force: bool = False) -> str:
    """Compile oracle/orc.c -> oracle/liborc.so with gcc (no fast-math: the oracle must stay IEEE)."""
    if os.environ.get("ORC_LIBORC"):
        return _LIB_PATH
    src = os.path.join(_HERE, "orc.c")
    hdr = os.path.join(_HERE, "orc.h")
    if (not force and os.path.exists(_LIB_PATH)
            and os.path.getmtime(_LIB_PATH) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _LIB_PATH
    cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB_PATH, src, "-lm"]
    subprocess.check_call(cmd)
    return _LIB_PATH


class _Grid(C.Structure):
    _fields_ = [("D", C.c_int32), ("N", C.c_int32 * 3), ("bc", C.c_int32 * 3), ("kind", C.c_int32),
                ("xmin", C.c_double * 3), ("xmax", C.c_double * 3), ("r0", C.c_double), ("vartheta", C.c_double)]


class _Particles(C.Structure):
    _fields_ = [("n", C.c_int64), ("i", C.c_void_p * 3), ("d", C.c_void_p * 3), ("phi", C.c_void_p),
                ("u", C.c_void_p * 3), ("w", C.c_void_p), ("tag", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB_PATH)
        dp = C.POINTER(C.c_double)
        L.orc_metric_h.argtypes = [C.POINTER(_Grid), dp, dp]
        L.orc_metric_h_many.argtypes = [C.POINTER(_Grid), C.c_int64, dp, dp, dp]
        L.orc_theta_of_T.restype = C.c_double; L.orc_theta_of_T.argtypes = [C.c_double, C.c_double]
        L.orc_dtheta_dT.restype = C.c_double; L.orc_dtheta_dT.argtypes = [C.c_double, C.c_double]
        L.orc_T_of_theta.restype = C.c_double; L.orc_T_of_theta.argtypes = [C.c_double, C.c_double]
        L.orc_T_of_theta_printed_B3.restype = C.c_double; L.orc_T_of_theta_printed_B3.argtypes = [C.c_double, C.c_double]
        L.orc_dx_min.restype = C.c_double; L.orc_dx_min.argtypes = [C.POINTER(_Grid)]
        L.orc_code_to_cart.argtypes = [C.POINTER(_Grid), dp, dp]
        L.orc_cart_to_code.argtypes = [C.POINTER(_Grid), dp, dp]
        L.orc_gather.argtypes = [C.POINTER(_Grid), C.POINTER(C.c_void_p), C.POINTER(C.c_int32), dp, dp]
        L.orc_to_cartesian_basis.argtypes = [C.POINTER(_Grid), dp, dp, dp]
        L.orc_boris.argtypes = [dp, dp, dp, C.c_double, C.c_double]
        L.orc_vay.argtypes = [dp, dp, dp, C.c_double, C.c_double]
        L.orc_set_pusher.restype = C.c_int; L.orc_set_pusher.argtypes = [C.c_int]
        L.orc_set_gca.argtypes = [C.c_double, C.c_double]
        L.orc_gca_project.restype = C.c_int; L.orc_gca_project.argtypes = [dp, dp, dp, dp, C.c_double]
        L.orc_gather_push.restype = C.c_int
        L.orc_gather_push.argtypes = [C.POINTER(_Grid), C.POINTER(C.c_void_p), C.POINTER(_Particles), C.POINTER(_Particles),
                                      C.c_double, C.c_double]
        L.orc_deposit.restype = C.c_int
        L.orc_deposit.argtypes = [C.POINTER(_Grid), C.POINTER(_Particles), C.POINTER(_Particles), C.POINTER(C.c_void_p),
                                  C.c_double, C.c_double]
        L.orc_fold_current.argtypes = [C.POINTER(_Grid), C.POINTER(C.c_void_p)]
        L.orc_fold_scalar.argtypes = [C.POINTER(_Grid), C.c_void_p]
        L.orc_filter_current.argtypes = [C.POINTER(_Grid), C.POINTER(C.c_void_p), C.c_int, C.c_int]
        L.orc_faraday.argtypes = [C.POINTER(_Grid), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.c_double]
        L.orc_ampere.argtypes = [C.POINTER(_Grid), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.c_void_p, C.c_double, C.c_double]
        L.orc_axis_area.restype = C.c_double; L.orc_axis_area.argtypes = [C.POINTER(_Grid), C.c_double]
        L.orc_fill_field_ghosts.argtypes = [C.POINTER(_Grid), C.POINTER(C.c_void_p)]
        L.orc_step.restype = C.c_int
        L.orc_step.argtypes = [C.POINTER(_Grid), C.POINTER(C.c_void_p), C.POINTER(_Particles), C.POINTER(C.c_void_p),
                               C.c_double, C.c_double, C.c_double]
        L.orc_charge_density.argtypes = [C.POINTER(_Grid), C.POINTER(_Particles), C.c_void_p, C.c_double, C.c_void_p]
        L.orc_continuity_residual.restype = C.c_double
        L.orc_continuity_residual.argtypes = [C.POINTER(_Grid), C.POINTER(C.c_void_p), C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        L.orc_compact.restype = C.c_int64
        L.orc_compact.argtypes = [C.c_int, C.c_int, C.POINTER(_Particles), C.POINTER(_Particles)]
        L.orc_sort_check.restype = C.c_int
        L.orc_sort_check.argtypes = [C.c_int64, C.c_void_p, C.c_int64, C.c_void_p]
        L.orc_padded_size.restype = C.c_int64; L.orc_padded_size.argtypes = [C.POINTER(_Grid)]
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.restype = C.c_int; L.orc_set_num_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


@dataclass
class Grid:
    """Grid + metric parameters: D, N, boundary kinds, metric kind and its parameters."""
    D: int
    N: tuple
    bc: tuple
    kind: int = CART
    xmin: tuple = (0.0, 0.0, 0.0)
    xmax: tuple = (1.0, 1.0, 1.0)
    r0: float = 0.0
    vartheta: float = 0.0

    def c(self) -> _Grid:
        g = _Grid()
        g.D = self.D
        N = list(self.N) + [1] * (3 - len(self.N))
        bc = list(self.bc) + [PERIODIC] * (3 - len(self.bc))
        xmin = list(self.xmin) + [0.0] * (3 - len(self.xmin))
        xmax = list(self.xmax) + [1.0] * (3 - len(self.xmax))
        for a in range(3):
            g.N[a] = int(N[a]) if a < self.D else 1
            g.bc[a] = int(bc[a])
            g.xmin[a] = float(xmin[a])
            g.xmax[a] = float(xmax[a])
        g.kind = self.kind
        g.r0 = self.r0
        g.vartheta = self.vartheta
        return g

    @property
    def axisym(self) -> bool:
        return self.kind != CART

    @property
    def padded_shape(self) -> tuple:
        """numpy shape (slowest..fastest) of a planar padded array: x1 is the fastest index."""
        ext = [int(self.N[a]) + 2 * NGHOST for a in range(self.D)]
        return tuple(reversed(ext))


@dataclass
class Particles:
    """Oracle particle block: int32 cell indices per dimension, float64 everything else."""
    i: list                    # D arrays int32
    d: list                    # D arrays float64
    u: list                    # 3 arrays float64
    w: np.ndarray
    phi: np.ndarray | None = None
    tag: np.ndarray | None = None      # int8, 1 alive / 0 dead
    _keep: list = field(default_factory=list, repr=False)

    @property
    def n(self) -> int:
        return int(self.w.shape[0])

    def copy(self) -> "Particles":
        return Particles(i=[a.copy() for a in self.i], d=[a.copy() for a in self.d], u=[a.copy() for a in self.u],
                         w=self.w.copy(), phi=None if self.phi is None else self.phi.copy(),
                         tag=None if self.tag is None else self.tag.copy())

    def c(self) -> _Particles:
        p = _Particles()
        p.n = self.n
        for a in range(3):
            if a < len(self.i):
                assert self.i[a].dtype == np.int32 and self.i[a].flags.c_contiguous
                assert self.d[a].dtype == np.float64 and self.d[a].flags.c_contiguous
                p.i[a] = self.i[a].ctypes.data
                p.d[a] = self.d[a].ctypes.data
            else:
                p.i[a] = None
                p.d[a] = None
            assert self.u[a].dtype == np.float64 and self.u[a].flags.c_contiguous
            p.u[a] = self.u[a].ctypes.data
        assert self.w.dtype == np.float64
        p.w = self.w.ctypes.data
        p.phi = None if self.phi is None else self.phi.ctypes.data
        if self.tag is not None:
            assert self.tag.dtype == np.int8
        p.tag = None if self.tag is None else self.tag.ctypes.data
        return p


def _vec(x):
    a = np.ascontiguousarray(x, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _fieldptrs(F):
    assert len(F) == 6
    arr = (C.c_void_p * 6)()
    for c in range(6):
        assert F[c].dtype == np.float32 and F[c].flags.c_contiguous
        arr[c] = F[c].ctypes.data
    return arr


def _jptrs(J):
    arr = (C.c_void_p * 3)()
    for c in range(3):
        assert J[c].dtype == np.float64 and J[c].flags.c_contiguous
        arr[c] = J[c].ctypes.data
    return arr


# ---- thin wrappers (argument marshalling only) ----
def metric_h(g: Grid, x) -> np.ndarray:
    xa, xp = _vec(x); h = np.zeros(3); lib().orc_metric_h(C.byref(g.c()), xp, h.ctypes.data_as(C.POINTER(C.c_double)))
    return h


def metric_h_many(g: Grid, x1, x2) -> np.ndarray:
    """h_11, h_22, h_33 at many code positions (x1[k], x2[k]): orc_metric_h called in a loop; returns shape (n, 3)."""
    a1, p1 = _vec(x1); a2, p2 = _vec(x2)
    h = np.zeros((a1.shape[0], 3))
    lib().orc_metric_h_many(C.byref(g.c()), a1.shape[0], p1, p2, h.ctypes.data_as(C.POINTER(C.c_double)))
    return h


def theta_of_T(vt, T): return lib().orc_theta_of_T(vt, T)
def dtheta_dT(vt, T): return lib().orc_dtheta_dT(vt, T)
def T_of_theta(vt, th): return lib().orc_T_of_theta(vt, th)
def T_of_theta_printed_B3(vt_signed, th): return lib().orc_T_of_theta_printed_B3(vt_signed, th)
def dx_min(g: Grid): return lib().orc_dx_min(C.byref(g.c()))


def code_to_cart(g: Grid, x) -> np.ndarray:
    xa, xp = _vec(x); X = np.zeros(3); lib().orc_code_to_cart(C.byref(g.c()), xp, X.ctypes.data_as(C.POINTER(C.c_double)))
    return X


def cart_to_code(g: Grid, X) -> np.ndarray:
    Xa, Xp = _vec(X); x = np.zeros(3); lib().orc_cart_to_code(C.byref(g.c()), Xp, x.ctypes.data_as(C.POINTER(C.c_double)))
    return x


def gather(g: Grid, F, i, d) -> np.ndarray:
    ia = np.zeros(3, dtype=np.int32); ia[:len(i)] = i
    da = np.zeros(3); da[:len(d)] = d
    out = np.zeros(6)
    lib().orc_gather(C.byref(g.c()), _fieldptrs(F), ia.ctypes.data_as(C.POINTER(C.c_int32)),
                     da.ctypes.data_as(C.POINTER(C.c_double)), out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def to_cartesian_basis(g: Grid, x, A) -> np.ndarray:
    xa, xp = _vec(x); Aa, Ap = _vec(A); out = np.zeros(3)
    lib().orc_to_cartesian_basis(C.byref(g.c()), xp, Ap, out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def boris(u, E, B, q_over_m, dt) -> np.ndarray:
    ua = np.array(u, dtype=np.float64); Ea, Ep = _vec(E); Ba, Bp = _vec(B)
    lib().orc_boris(ua.ctypes.data_as(C.POINTER(C.c_double)), Ep, Bp, q_over_m, dt)
    return ua


def vay(u, E, B, q_over_m, dt) -> np.ndarray:
    ua = np.array(u, dtype=np.float64); Ea, Ep = _vec(E); Ba, Bp = _vec(B)
    lib().orc_vay(ua.ctypes.data_as(C.POINTER(C.c_double)), Ep, Bp, q_over_m, dt)
    return ua


def set_gca(rho_crit: float, eovb: float) -> None:
    """thresholds of the hybrid pusher: critical Larmor radius and the largest |E|/|B| of the guiding-centre regime"""
    lib().orc_set_gca(float(rho_crit), float(eovb))


def gca_project(u, u_before, E, B, q_over_m):
    """returns (u after the guiding-centre step, applied?)"""
    a, pa = _vec(u); _, pb = _vec(u_before); _, pe = _vec(E); _, pB = _vec(B)
    a = a.copy(); pa = a.ctypes.data_as(C.POINTER(C.c_double))
    r = lib().orc_gca_project(pa, pb, pe, pB, float(q_over_m))
    return a, bool(r)


def set_pusher(kind: int) -> int:
    """0 = Boris (default), 1 = Vay: the pusher orc.gather_push / orc.step use; returns the previous kind"""
    return lib().orc_set_pusher(int(kind))


def gather_push(g: Grid, F, p: Particles, q_over_m: float, dt: float) -> Particles:
    """Steps 3-7 (+ crossing bookkeeping); returns a new block, input untouched."""
    out = p.copy()
    if out.tag is None:
        out.tag = np.ones(p.n, dtype=np.int8)
    rc = lib().orc_gather_push(C.byref(g.c()), _fieldptrs(F), C.byref(p.c()), C.byref(out.c()), q_over_m, dt)
    if rc != 0:
        raise RuntimeError(f"orc_gather_push failed rc={rc}")
    return out


def zeros_current(g: Grid):
    return [np.zeros(g.padded_shape, dtype=np.float64) for _ in range(3)]


def deposit(g: Grid, pold: Particles, pnew: Particles, J, q: float, dt: float) -> None:
    rc = lib().orc_deposit(C.byref(g.c()), C.byref(pold.c()), C.byref(pnew.c()), _jptrs(J), q, dt)
    if rc != 0:
        raise RuntimeError(f"orc_deposit failed rc={rc} (|delta i| > 1?)")


def fold_current(g: Grid, J) -> None:
    lib().orc_fold_current(C.byref(g.c()), _jptrs(J))


def fold_scalar(g: Grid, rho) -> None:
    lib().orc_fold_scalar(C.byref(g.c()), rho.ctypes.data)


def filter_current(g: Grid, J, npasses: int, divide: bool = False) -> None:
    """step 9: digital filter passes (Eqs. 9-11) in place, then optionally J = conformal J / sqrt(h)"""
    lib().orc_filter_current(C.byref(g.c()), _jptrs(J), int(npasses), 1 if divide else 0)


def _dptrs(A, n):
    arr = (C.c_void_p * n)()
    for c in range(n):
        assert A[c].dtype == np.float64 and A[c].flags.c_contiguous
        arr[c] = A[c].ctypes.data
    return arr


def faraday(g: Grid, E, B, dt: float) -> None:
    """Eq. A1: B -= dt curl(h E) / sqrt(h), in place on the three float64 arrays of B; Eq. 12 on the axis"""
    lib().orc_faraday(C.byref(g.c()), _dptrs(E, 3), _dptrs(B, 3), float(dt))


def ampere(g: Grid, E, B, J, dt: float, jc: float) -> None:
    """Eq. A2: E += dt (curl(h B) - jc conformal J) / sqrt(h), in place on E; Eqs. 12-13 on the axis; J may be None"""
    lib().orc_ampere(C.byref(g.c()), _dptrs(E, 3), _dptrs(B, 3), None if J is None else _dptrs(J, 3), float(dt), float(jc))


def axis_area(g: Grid, x1: float) -> float:
    return lib().orc_axis_area(C.byref(g.c()), float(x1))


def fill_field_ghosts(g: Grid, F) -> None:
    lib().orc_fill_field_ghosts(C.byref(g.c()), _dptrs(F, 6))


def step(g: Grid, F, p: Particles, J, q: float, m: float, dt: float) -> None:
    """Fused steps 3-8, in place on p, accumulating into J (no fold)."""
    if p.tag is None:
        p.tag = np.ones(p.n, dtype=np.int8)
    rc = lib().orc_step(C.byref(g.c()), _fieldptrs(F), C.byref(p.c()), _jptrs(J), q, m, dt)
    if rc != 0:
        raise RuntimeError(f"orc_step failed rc={rc}")


def charge_density(g: Grid, p: Particles, q: float, mask=None, rho=None) -> np.ndarray:
    if rho is None:
        rho = np.zeros(g.padded_shape, dtype=np.float64)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.int8)
    lib().orc_charge_density(C.byref(g.c()), C.byref(p.c()), None if m is None else m.ctypes.data, q, rho.ctypes.data)
    return rho


def continuity_residual(g: Grid, J, rho_old, rho_new, dt, want_field=False):
    R = np.zeros(g.padded_shape, dtype=np.float64) if want_field else None
    worst = lib().orc_continuity_residual(C.byref(g.c()), _jptrs(J), rho_old.ctypes.data, rho_new.ctypes.data, dt,
                                          None if R is None else R.ctypes.data)
    return (worst, R) if want_field else worst


def compact(p: Particles):
    """tag sort: returns (new block with the alive particles first, number alive)"""
    out = p.copy()
    if out.tag is None:
        out.tag = np.ones(p.n, dtype=np.int8)
    na = lib().orc_compact(len(p.i), 0 if p.phi is None else 1, C.byref(p.c()), C.byref(out.c()))
    return out, int(na)


def sort_check(keys_sorted, ncell, offsets=None) -> int:
    k = np.ascontiguousarray(keys_sorted, dtype=np.int32)
    o = None if offsets is None else np.ascontiguousarray(offsets, dtype=np.int32)
    return lib().orc_sort_check(k.shape[0], k.ctypes.data, int(ncell), None if o is None else o.ctypes.data)


def num_threads() -> int:
    return lib().orc_num_threads()


def set_num_threads(n: int) -> int:
    """OpenMP thread count of the following oracle calls; returns the previous one (bench.py's single-thread figure)"""
    return lib().orc_set_num_threads(int(n))
