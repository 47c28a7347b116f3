"""ctypes binding of libent.so (include/ent.h).  Same names as the C ABI; argument marshalling only.

torch is used for device memory and streams: every tensor handed in must already live on the ctx's CUDA device
(except for ent_step_host, which takes host tensors).  No arithmetic of the method happens in this file.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass, field

import torch

from . import build as _build

CART, SPH, QSPH = 0, 1, 2
PERIODIC, ABSORB, AXIS = 0, 1, 2
NGHOST = 2
OK, EINVAL, EUNSUPPORTED, ECUDA, ENOMEM = 0, -1, -2, -3, -4
OPT_STEP_IMPL, OPT_TILE_1, OPT_TILE_2, OPT_TILE_3, OPT_SORT_MODE, OPT_CURV_FP64, OPT_PUSHER, OPT_SORT_STAGING = 1, 2, 3, 4, 5, 6, 7, 8
(STAT_TILE_1, STAT_TILE_2, STAT_TILE_3, STAT_NKEYS, STAT_NTILES, STAT_LAUNCHES, STAT_BAD_MOVES, STAT_STRAYS,
 STAT_SCRATCH_BYTES, STAT_LAST_STEP_TILED, STAT_LAST_SORT_REBIN, STAT_SLOT_ERRORS, STAT_CARRIES, STAT_GLOBAL_ADDS) = range(1, 15)

SYMBOLS = ["ent_create", "ent_destroy", "ent_last_error", "ent_set_grid", "ent_gather_push", "ent_deposit", "ent_sort",
           "ent_step", "ent_step_pair", "ent_step_sorted", "ent_workspace_bytes", "ent_reserve", "ent_forget", "ent_tile_offsets", "ent_zero_current", "ent_fold_current", "ent_filter_current", "ent_faraday", "ent_ampere", "ent_fill_field_ghosts", "ent_compact", "ent_compact_static", "ent_step_host", "ent_step_host_pair", "ent_set_option", "ent_set_gca", "ent_get_stat", "ent_version"]


class EntError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"ent error {code}: {msg}")
        self.code = code


class _Grid(C.Structure):
    _fields_ = [("D", C.c_int32), ("N", C.c_int32 * 3), ("bc", C.c_int32 * 3), ("kind", C.c_int32),
                ("xmin", C.c_double * 3), ("xmax", C.c_double * 3), ("r0", C.c_double), ("vartheta", C.c_double)]


class _Fields(C.Structure):
    _fields_ = [("comp", C.c_void_p * 6)]


class _Current(C.Structure):
    _fields_ = [("comp", C.c_void_p * 3)]


class _Particles(C.Structure):
    _fields_ = [("n", C.c_int64), ("cell", C.c_void_p), ("d", C.c_void_p * 3), ("phi", C.c_void_p), ("u", C.c_void_p * 3),
                ("w", C.c_void_p), ("tag", C.c_void_p), ("q", C.c_float), ("m", C.c_float)]


_lib = None


def lib():
    """Loads libent.so (building it if the sources are newer).  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.build()
        if not os.path.exists(path):
            raise RuntimeError("libent.so is missing: the CUDA library is the product, there is no fallback")
        L = C.CDLL(path)
        vp = C.c_void_p
        L.ent_version.restype = C.c_char_p
        L.ent_last_error.restype = C.c_char_p; L.ent_last_error.argtypes = [vp]
        L.ent_create.argtypes = [C.POINTER(vp), C.c_int, vp]
        L.ent_destroy.argtypes = [vp]
        L.ent_set_grid.argtypes = [vp, C.POINTER(_Grid)]
        L.ent_gather_push.argtypes = [vp, C.POINTER(_Fields), C.POINTER(_Particles), C.POINTER(_Particles), C.c_float]
        L.ent_deposit.argtypes = [vp, C.POINTER(_Particles), C.POINTER(_Particles), C.POINTER(_Current), C.c_float]
        L.ent_sort.argtypes = [vp, C.POINTER(_Particles), C.POINTER(_Particles), vp]
        L.ent_tile_offsets.argtypes = [vp, C.POINTER(_Particles), vp]
        L.ent_step_sorted.argtypes = [vp, C.POINTER(_Fields), C.POINTER(_Particles), C.POINTER(_Particles), C.POINTER(_Current), C.c_float]
        L.ent_workspace_bytes.argtypes = [vp, C.c_int64, C.POINTER(C.c_size_t)]
        L.ent_reserve.argtypes = [vp, C.c_int64]
        L.ent_forget.argtypes = [vp, C.POINTER(_Particles)]
        L.ent_step.argtypes = [vp, C.POINTER(_Fields), C.POINTER(_Particles), C.POINTER(_Current), C.c_float]
        L.ent_step_pair.argtypes = [vp, C.POINTER(_Fields), C.POINTER(_Particles), C.POINTER(_Particles), C.POINTER(_Current), C.c_float]
        L.ent_zero_current.argtypes = [vp, C.POINTER(_Current)]
        L.ent_fold_current.argtypes = [vp, C.POINTER(_Current)]
        L.ent_filter_current.argtypes = [vp, C.POINTER(_Current), C.c_int, C.c_int]
        L.ent_faraday.argtypes = [vp, C.POINTER(_Fields), C.c_float]
        L.ent_ampere.argtypes = [vp, C.POINTER(_Fields), C.POINTER(_Current), C.c_float, C.c_float]
        L.ent_fill_field_ghosts.argtypes = [vp, C.POINTER(_Fields)]
        L.ent_compact.argtypes = [vp, C.POINTER(_Particles), C.POINTER(_Particles), vp]
        L.ent_compact_static.argtypes = [vp, C.POINTER(_Particles), C.POINTER(_Particles), vp]
        L.ent_step_host.argtypes = [vp, C.POINTER(_Fields), C.POINTER(_Particles), C.POINTER(_Current), C.c_float, C.c_int,
                                    C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.ent_step_host_pair.argtypes = [vp, C.POINTER(_Fields), C.POINTER(_Particles), C.POINTER(_Particles), C.POINTER(_Current), C.c_float, C.c_int,
                                         C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.ent_set_option.argtypes = [vp, C.c_int, C.c_int64]
        L.ent_set_gca.argtypes = [vp, C.c_double, C.c_double]
        L.ent_get_stat.argtypes = [vp, C.c_int, C.POINTER(C.c_int64)]
        for s in SYMBOLS:
            if s not in ("ent_version", "ent_last_error"):
                getattr(L, s).restype = C.c_int
        _lib = L
    return _lib


@dataclass
class Grid:
    """ent_grid: D, N, boundary kinds, metric kind and parameters."""
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
        pad = lambda t, fill: list(t) + [fill] * (3 - len(t))
        N, bc, xmin, xmax = pad(self.N, 1), pad(self.bc, PERIODIC), pad(self.xmin, 0.0), pad(self.xmax, 1.0)
        for a in range(3):
            g.N[a], g.bc[a], g.xmin[a], g.xmax[a] = int(N[a]), int(bc[a]), float(xmin[a]), float(xmax[a])
        g.kind, g.r0, g.vartheta = self.kind, self.r0, self.vartheta
        return g

    @property
    def axisym(self) -> bool:
        return self.kind != CART

    @property
    def padded_shape(self) -> tuple:
        """torch/numpy shape (slowest..fastest) of a padded planar array; x1 is the fastest index."""
        return tuple(reversed([int(self.N[a]) + 2 * NGHOST for a in range(self.D)]))

    @property
    def ncells(self) -> int:
        n = 1
        for a in range(self.D):
            n *= int(self.N[a])
        return n


def _ptr(t, dtype, name, cuda=True):
    if t is None:
        return None
    if t.dtype != dtype or not t.is_contiguous() or (cuda and not t.is_cuda) or (not cuda and t.is_cuda):
        raise TypeError(f"{name}: need a contiguous {'CUDA' if cuda else 'host'} tensor of {dtype}, got {t.dtype} on {t.device}")
    return t.data_ptr()


@dataclass
class Particles:
    """ent_particles: SoA block of one species held in torch tensors."""
    cell: torch.Tensor
    d: list
    u: list
    w: torch.Tensor
    phi: torch.Tensor | None = None
    tag: torch.Tensor | None = None
    q: float = 1.0
    m: float = 1.0

    @property
    def n(self) -> int:
        return int(self.cell.shape[0])

    def c(self, cuda=True) -> _Particles:
        p = _Particles()
        p.n = self.n
        p.cell = _ptr(self.cell, torch.int32, "cell", cuda)
        for a in range(3):
            p.d[a] = _ptr(self.d[a], torch.float32, f"d[{a}]", cuda) if a < len(self.d) else None
            p.u[a] = _ptr(self.u[a], torch.float32, f"u[{a}]", cuda)
        p.phi = _ptr(self.phi, torch.float32, "phi", cuda)
        p.w = _ptr(self.w, torch.float32, "w", cuda)
        p.tag = _ptr(self.tag, torch.uint8, "tag", cuda)
        p.q, p.m = float(self.q), float(self.m)
        return p

    def clone(self) -> "Particles":
        cl = lambda t: None if t is None else t.clone()
        return Particles(cell=self.cell.clone(), d=[cl(t) for t in self.d], u=[cl(t) for t in self.u], w=self.w.clone(),
                         phi=cl(self.phi), tag=cl(self.tag), q=self.q, m=self.m)

    def empty_like(self) -> "Particles":
        e = lambda t: None if t is None else torch.empty_like(t)
        return Particles(cell=e(self.cell), d=[e(t) for t in self.d], u=[e(t) for t in self.u], w=e(self.w),
                         phi=e(self.phi), tag=e(self.tag), q=self.q, m=self.m)

    def to(self, device, pin=False) -> "Particles":
        def mv(t):
            if t is None:
                return None
            r = t.to(device)
            return r.pin_memory() if pin and not r.is_cuda else r
        return Particles(cell=mv(self.cell), d=[mv(t) for t in self.d], u=[mv(t) for t in self.u], w=mv(self.w),
                         phi=mv(self.phi), tag=mv(self.tag), q=self.q, m=self.m)


def _fields(F, cuda=True) -> _Fields:
    s = _Fields()
    assert len(F) == 6
    for c in range(6):
        s.comp[c] = _ptr(F[c], torch.float32, f"field[{c}]", cuda)
    return s


def _current(J, cuda=True) -> _Current:
    s = _Current()
    assert len(J) == 3
    for c in range(3):
        s.comp[c] = _ptr(J[c], torch.float32, f"J[{c}]", cuda)
    return s


class Ctx:
    """ent_ctx handle.  Creating one without a CUDA device raises (no CPU fallback)."""

    def __init__(self, device: int = 0, stream: "torch.cuda.Stream | None" = None):
        self._h = C.c_void_p()
        self.device = device
        self._stream = stream
        sp = None if stream is None else stream.cuda_stream
        rc = lib().ent_create(C.byref(self._h), device, sp)
        if rc != OK:
            self._h = C.c_void_p()
            raise EntError(rc, "ent_create failed (no usable CUDA device? there is no CPU fallback)")
        self.grid = None

    def _ck(self, rc):
        if rc != OK:
            raise EntError(rc, lib().ent_last_error(self._h).decode())

    def close(self):
        if self._h:
            lib().ent_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def ent_create(device: int = 0, stream=None) -> Ctx:
    return Ctx(device, stream)


def ent_destroy(ctx: Ctx) -> None:
    ctx.close()


def ent_version() -> str:
    return lib().ent_version().decode()


def ent_set_grid(ctx: Ctx, grid: Grid) -> None:
    ctx._ck(lib().ent_set_grid(ctx._h, C.byref(grid.c())))
    ctx.grid = grid


def ent_gather_push(ctx: Ctx, EB, pin: Particles, pout: Particles, dt: float) -> None:
    ctx._ck(lib().ent_gather_push(ctx._h, C.byref(_fields(EB)), C.byref(pin.c()), C.byref(pout.c()), dt))


def ent_deposit(ctx: Ctx, pold: Particles, pnew: Particles, J, dt: float) -> None:
    ctx._ck(lib().ent_deposit(ctx._h, C.byref(pold.c()), C.byref(pnew.c()), C.byref(_current(J)), dt))


def ent_sort(ctx: Ctx, pin: Particles, pout: Particles, key_offsets: torch.Tensor | None = None) -> None:
    ko = _ptr(key_offsets, torch.int32, "key_offsets")
    ctx._ck(lib().ent_sort(ctx._h, C.byref(pin.c()), C.byref(pout.c()), ko))


def ent_tile_offsets(ctx: Ctx, block: Particles) -> torch.Tensor:
    """int32[ntiles + 1] device tensor: the tile offsets the ctx keeps for a sorted block"""
    out = torch.empty(ent_get_stat(ctx, STAT_NTILES) + 1, dtype=torch.int32, device=block.cell.device)
    ctx._ck(lib().ent_tile_offsets(ctx._h, C.byref(block.c()), out.data_ptr()))
    return out


def ent_step(ctx: Ctx, EB, p: Particles, J, dt: float) -> None:
    ctx._ck(lib().ent_step(ctx._h, C.byref(_fields(EB)), C.byref(p.c()), C.byref(_current(J)), dt))


def ent_step_pair(ctx: Ctx, EB, p1: Particles, p2: Particles, J, dt: float) -> None:
    ctx._ck(lib().ent_step_pair(ctx._h, C.byref(_fields(EB)), C.byref(p1.c()), C.byref(p2.c()), C.byref(_current(J)), dt))


def ent_step_sorted(ctx: Ctx, EB, pin: Particles, pout: Particles, J, dt: float) -> None:
    ctx._ck(lib().ent_step_sorted(ctx._h, C.byref(_fields(EB)), C.byref(pin.c()), C.byref(pout.c()), C.byref(_current(J)), dt))


def ent_workspace_bytes(ctx: Ctx, npart: int) -> int:
    b = C.c_size_t(0)
    ctx._ck(lib().ent_workspace_bytes(ctx._h, npart, C.byref(b)))
    return b.value


def ent_reserve(ctx: Ctx, npart: int) -> None:
    ctx._ck(lib().ent_reserve(ctx._h, npart))


def ent_forget(ctx: Ctx, block: Particles) -> None:
    ctx._ck(lib().ent_forget(ctx._h, C.byref(block.c())))


def ent_zero_current(ctx: Ctx, J) -> None:
    ctx._ck(lib().ent_zero_current(ctx._h, C.byref(_current(J))))


def ent_fold_current(ctx: Ctx, J) -> None:
    ctx._ck(lib().ent_fold_current(ctx._h, C.byref(_current(J))))


def ent_compact(ctx: Ctx, pin: Particles, pout: Particles) -> torch.Tensor:
    """tag sort; returns a one-element int64 device tensor holding the number of alive particles"""
    na = torch.zeros(1, dtype=torch.int64, device=pin.cell.device)
    ctx._ck(lib().ent_compact(ctx._h, C.byref(pin.c()), C.byref(pout.c()), na.data_ptr()))
    return na


COMPACT_STATIC_MAX_N = 1 << 20


def ent_compact_static(ctx: Ctx, pin: Particles, pout: Particles, n_alive: torch.Tensor) -> None:
    """ent_compact with the library's static scratch: no device allocation by the call (n <= COMPACT_STATIC_MAX_N); n_alive is the
    caller's one-element int64 device tensor"""
    ctx._ck(lib().ent_compact_static(ctx._h, C.byref(pin.c()), C.byref(pout.c()), n_alive.data_ptr()))


def ent_filter_current(ctx: Ctx, J, npasses: int, divide_by_sqrt_h: bool = False) -> None:
    ctx._ck(lib().ent_filter_current(ctx._h, C.byref(_current(J)), int(npasses), 1 if divide_by_sqrt_h else 0))


def ent_faraday(ctx: Ctx, EB, dt: float) -> None:
    ctx._ck(lib().ent_faraday(ctx._h, C.byref(_fields(EB)), dt))


def ent_ampere(ctx: Ctx, EB, J, dt: float, j_coeff: float) -> None:
    ctx._ck(lib().ent_ampere(ctx._h, C.byref(_fields(EB)), None if J is None else C.byref(_current(J)), dt, j_coeff))


def ent_fill_field_ghosts(ctx: Ctx, EB) -> None:
    ctx._ck(lib().ent_fill_field_ghosts(ctx._h, C.byref(_fields(EB))))


def ent_step_host(ctx: Ctx, EB, p: Particles, J, dt: float, nsteps: int = 1):
    """Host tensors in, host tensors out; returns (h2d_bytes, d2h_bytes)."""
    up, down = C.c_int64(0), C.c_int64(0)
    ctx._ck(lib().ent_step_host(ctx._h, C.byref(_fields(EB, cuda=False)), C.byref(p.c(cuda=False)),
                                C.byref(_current(J, cuda=False)), dt, nsteps, C.byref(up), C.byref(down)))
    return up.value, down.value


def ent_step_host_pair(ctx: Ctx, EB, p1: Particles, p2: Particles, J, dt: float, nsteps: int = 1):
    """Host tensors in, host tensors out, both species pipelined; returns (h2d_bytes, d2h_bytes)."""
    up, down = C.c_int64(0), C.c_int64(0)
    ctx._ck(lib().ent_step_host_pair(ctx._h, C.byref(_fields(EB, cuda=False)), C.byref(p1.c(cuda=False)), C.byref(p2.c(cuda=False)),
                                     C.byref(_current(J, cuda=False)), dt, nsteps, C.byref(up), C.byref(down)))
    return up.value, down.value


def ent_set_gca(ctx: Ctx, rho_crit: float, e_over_b_max: float) -> None:
    ctx._ck(lib().ent_set_gca(ctx._h, float(rho_crit), float(e_over_b_max)))


def ent_set_option(ctx: Ctx, key: int, value: int) -> None:
    ctx._ck(lib().ent_set_option(ctx._h, key, value))


def ent_get_stat(ctx: Ctx, key: int) -> int:
    v = C.c_int64(0)
    ctx._ck(lib().ent_get_stat(ctx._h, key, C.byref(v)))
    return v.value


def zeros_current(grid: Grid, device) -> list:
    return [torch.zeros(grid.padded_shape, dtype=torch.float32, device=device) for _ in range(3)]
