"""Small helpers shared by the tests (no method arithmetic: only array packing)."""
import numpy as np


def make_particles(orc, i, d, u, w=None, phi=None, tag=None):
    """i: (n,D) ints, d: (n,D) floats, u: (n,3)."""
    i = np.atleast_2d(np.asarray(i, dtype=np.int32))
    d = np.atleast_2d(np.asarray(d, dtype=np.float64))
    u = np.atleast_2d(np.asarray(u, dtype=np.float64))
    n, D = i.shape
    w = np.ones(n) if w is None else np.ascontiguousarray(np.broadcast_to(np.asarray(w, dtype=np.float64), (n,)))
    return orc.Particles(i=[np.ascontiguousarray(i[:, a]) for a in range(D)],
                         d=[np.ascontiguousarray(d[:, a]) for a in range(D)],
                         u=[np.ascontiguousarray(u[:, a]) for a in range(3)],
                         w=w.copy(),
                         phi=None if phi is None else np.ascontiguousarray(np.broadcast_to(np.asarray(phi, dtype=np.float64), (n,))).copy(),
                         tag=None if tag is None else np.ascontiguousarray(tag, dtype=np.int8))


def uniform_fields(orc, g, E=(0, 0, 0), B=(0, 0, 0)):
    """Six padded planar fp32 arrays holding constant contravariant components."""
    vals = list(E) + list(B)
    return [np.full(g.padded_shape, v, dtype=np.float32) for v in vals]


def cart_grid(orc, D, N, L, bc=None):
    bc = bc or (orc.PERIODIC,) * D
    N = tuple(N) if hasattr(N, "__len__") else (N,) * D
    L = tuple(L) if hasattr(L, "__len__") else (L,) * D
    return orc.Grid(D=D, N=N, bc=bc, kind=orc.CART, xmin=(0.0,) * D, xmax=L)


def sph_grid(orc, N=(32, 32), rmin=1.0, rmax=10.0):
    return orc.Grid(D=2, N=N, bc=(orc.ABSORB, orc.AXIS), kind=orc.SPH, xmin=(rmin, 0.0), xmax=(rmax, np.pi))


def qsph_grid(orc, N=(32, 32), rmin=1.0, rmax=20.0, r0=0.0, vartheta=0.0):
    return orc.Grid(D=2, N=N, bc=(orc.ABSORB, orc.AXIS), kind=orc.QSPH, xmin=(rmin, 0.0), xmax=(rmax, np.pi),
                    r0=r0, vartheta=vartheta)
