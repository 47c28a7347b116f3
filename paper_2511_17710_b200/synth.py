"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the CUDA path and the CPU oracle (tests hand the same arrays to each).  It holds none of
the method's arithmetic (no gather, push, map or deposit): only a counter-based random generator, analytic field
profiles evaluated on the Yee lattice, particle loading, and index packing.  torch only (CPU or CUDA device).
The paper uses no dataset: every experiment is a simulation set up by a problem generator, and these
recipes stand in for those set-ups.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import torch

CART, SPH, QSPH = 0, 1, 2
PERIODIC, ABSORB, AXIS = 0, 1, 2
NGHOST = 2
_M64 = (1 << 64) - 1


def _i64(x: int) -> int:
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    """logical right shift of int64 bit patterns"""
    return (z >> k) & ((1 << (64 - k)) - 1)


def rand_bits(seed: int, stream: int, n: int, device, start: int = 0) -> torch.Tensor:
    """SplitMix64 finaliser of the counter seed*GOLDEN + stream*2^40 + index (int64 bit patterns)."""
    base = _i64(seed * 0x9E3779B97F4A7C15 + (stream << 40) + start)
    z = torch.arange(n, dtype=torch.int64, device=device) + base
    z = (z ^ _lsr(z, 30)) * _i64(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _i64(0x94D049BB133111EB)
    return z ^ _lsr(z, 31)


def uniform(seed: int, stream: int, n: int, device, start: int = 0, dtype=torch.float32) -> torch.Tensor:
    """U in [0,1): 24 random bits for float32, 53 for float64."""
    z = rand_bits(seed, stream, n, device, start)
    if dtype == torch.float64:
        return _lsr(z, 11).to(torch.float64) * (2.0 ** -53)
    return _lsr(z, 40).to(torch.float32) * (2.0 ** -24)


@dataclass
class GridSpec:
    D: int
    N: tuple
    bc: tuple
    kind: int = CART
    xmin: tuple = (0.0, 0.0, 0.0)
    xmax: tuple = (1.0, 1.0, 1.0)
    r0: float = 0.0
    vartheta: float = 0.0

    @property
    def padded_shape(self):
        return tuple(reversed([int(self.N[a]) + 2 * NGHOST for a in range(self.D)]))

    @property
    def ncells(self):
        return math.prod(int(self.N[a]) for a in range(self.D))


@dataclass
class Species:
    """one species: unpacked cell indices (int32), offsets, momenta, weights as torch tensors"""
    q: float
    m: float
    i: list
    d: list
    u: list
    w: torch.Tensor
    phi: torch.Tensor | None = None

    @property
    def n(self):
        return int(self.w.shape[0])


@dataclass
class Workload:
    name: str
    grid: GridSpec
    dt: float
    steps: int
    fields: list            # 6 padded planar float32 tensors (contravariant components on the Yee lattice)
    species: list           # list[Species]
    seed: int = 0
    note: str = ""

    @property
    def nparticles(self):
        return sum(s.n for s in self.species)


def pack_cell(grid: GridSpec, i: list) -> torch.Tensor:
    """linear active-cell index i1 + N1*(i2 + N2*i3) (ent.h)"""
    c = i[0].to(torch.int64)
    if grid.D >= 2:
        c = c + int(grid.N[0]) * i[1].to(torch.int64)
    if grid.D == 3:
        c = c + int(grid.N[0]) * int(grid.N[1]) * i[2].to(torch.int64)
    return c.to(torch.int32)


def unpack_cell(grid: GridSpec, cell: torch.Tensor) -> list:
    c = cell.to(torch.int64)
    N0, N1 = int(grid.N[0]), int(grid.N[1])
    if grid.D == 2:
        return [(c % N0).to(torch.int32), (c // N0).to(torch.int32)]
    return [(c % N0).to(torch.int32), ((c // N0) % N1).to(torch.int32), (c // (N0 * N1)).to(torch.int32)]


def sort_key(grid: GridSpec, i: list, T: tuple) -> torch.Tensor:
    """tile-major sort key documented in ent.h (ent_sort); pure index arithmetic"""
    D = grid.D
    nt = [(int(grid.N[a]) + T[a] - 1) // T[a] for a in range(D)]
    t = [i[a].to(torch.int64) // T[a] for a in range(D)]
    l = [i[a].to(torch.int64) % T[a] for a in range(D)]
    tile, local, ts, ls = 0, 0, 1, 1
    for a in range(D):
        tile = tile + ts * t[a]; ts *= nt[a]
        local = local + ls * l[a]; ls *= T[a]
    return tile * ls + local


# ------------------------------------------------------------------------------------------------------------
# Maxwell-Juettner momenta: f(u) ~ u^2 exp(-sqrt(1+u^2)/theta), tabulated inverse CDF, isotropic directions
# ------------------------------------------------------------------------------------------------------------
def _mj_table(theta: float, device, npts: int = 1 << 16):
    gmax = 1.0 + 40.0 * theta
    umax = math.sqrt(gmax * gmax - 1.0)
    u = torch.linspace(0.0, umax, npts, dtype=torch.float64, device=device)
    f = u * u * torch.exp(-(torch.sqrt(1.0 + u * u) - 1.0) / theta)
    cdf = torch.cumsum(0.5 * (f[1:] + f[:-1]), 0)
    cdf = torch.cat([torch.zeros(1, dtype=torch.float64, device=device), cdf])
    return u, cdf / cdf[-1]


def maxwell_juettner(seed: int, streams: tuple, n: int, theta: float, device, beta_x=None):
    """returns [ux, uy, uz] float32.  beta_x: optional per-particle drift speed along x (tensor), applied with the
    flipping rule (flip u'_x if -beta u'_x/gamma' > U) and a Lorentz boost."""
    u_tab, cdf = _mj_table(theta, device)
    U = uniform(seed, streams[0], n, device, dtype=torch.float64)
    k = torch.searchsorted(cdf, U, right=True).clamp(1, cdf.numel() - 1)
    c0, c1 = cdf[k - 1], cdf[k]
    umag = u_tab[k - 1] + (u_tab[k] - u_tab[k - 1]) * ((U - c0) / (c1 - c0).clamp_min(1e-300))
    mu = 2.0 * uniform(seed, streams[1], n, device, dtype=torch.float64) - 1.0
    az = 2.0 * math.pi * uniform(seed, streams[2], n, device, dtype=torch.float64)
    st = torch.sqrt((1.0 - mu * mu).clamp_min(0.0))
    ux, uy, uz = umag * mu, umag * st * torch.cos(az), umag * st * torch.sin(az)
    if beta_x is not None:
        b = beta_x.to(torch.float64)
        g = torch.sqrt(1.0 + umag * umag)
        flip = (-b * ux / g) > uniform(seed, streams[0] + 100, n, device, dtype=torch.float64)
        ux = torch.where(flip, -ux, ux)
        G = 1.0 / torch.sqrt(1.0 - b * b)
        ux = G * (ux + b * g)
    return [ux.to(torch.float32), uy.to(torch.float32), uz.to(torch.float32)]


# ------------------------------------------------------------------------------------------------------------
# Yee lattice positions and metric factors for turning orthonormal profiles into the
# contravariant components the library expects (A^i = A^hat{i} / sqrt(h_ii)).  Closed forms of P:227-267.
# ------------------------------------------------------------------------------------------------------------
STAGGER = [(0.5, 0, 0), (0, 0.5, 0), (0, 0, 0.5), (0, 0.5, 0.5), (0.5, 0, 0.5), (0.5, 0.5, 0)]


def yee_axes(grid: GridSpec, comp: int, device):
    """1-D code-coordinate axes (incl. ghosts) of component comp: list of D float64 tensors"""
    return [torch.arange(int(grid.N[a]) + 2 * NGHOST, dtype=torch.float64, device=device) - NGHOST + STAGGER[comp][a]
            for a in range(grid.D)]


def _qs_params(grid: GridSpec):
    Rmin = math.log(grid.xmin[0] - grid.r0)
    dR = (math.log(grid.xmax[0] - grid.r0) - Rmin) / grid.N[0]
    dT = math.pi / grid.N[1]
    return Rmin, dR, dT


def sph_geometry(grid: GridSpec, x1: torch.Tensor, x2: torch.Tensor):
    """(r, theta, sqrt h11, sqrt h22, sqrt h33) at code positions; float64 tensors (broadcastable)"""
    if grid.kind == SPH:
        dr = (grid.xmax[0] - grid.xmin[0]) / grid.N[0]
        dth = math.pi / grid.N[1]
        r = grid.xmin[0] + x1 * dr
        th = x2 * dth
        return r, th, torch.full_like(r, dr), r * dth, r * torch.sin(th)
    Rmin, dR, dT = _qs_params(grid)
    eR = torch.exp(Rmin + x1 * dR)
    T = x2 * dT
    vt = grid.vartheta
    r = grid.r0 + eR
    th = T + 2.0 * vt * T * (1.0 - 2.0 * T / math.pi) * (1.0 - T / math.pi)
    dthdT = 1.0 + 2.0 * vt + 12.0 * vt * (T / math.pi) * (T / math.pi - 1.0)
    return r, th, dR * eR, dT * dthdT * r, r * torch.sin(th)


def cfl_dx_min(grid: GridSpec) -> float:
    """Eq. 8: min over cell centres of (sum_{d<D} 1/h_dd)^(-1/2)"""
    if grid.kind == CART:
        return 1.0 / math.sqrt(sum((grid.N[a] / (grid.xmax[a] - grid.xmin[a])) ** 2 for a in range(grid.D)))
    x1 = torch.arange(grid.N[0], dtype=torch.float64)[None, :] + 0.5
    x2 = torch.arange(grid.N[1], dtype=torch.float64)[:, None] + 0.5
    _, _, h1, h2, _ = sph_geometry(grid, x1, x2)
    return float((1.0 / torch.sqrt(1.0 / (h1 * h1) + 1.0 / (h2 * h2))).min())


def axisym_fields(grid: GridSpec, profile, device) -> list:
    """profile(r, theta) -> dict of orthonormal (Er, Eth, Eph, Br, Bth, Bph).  Ghosts in theta are filled by rotation
    symmetry (r-component even, theta- and phi-components odd about the axis, G10); on-axis E^3 = B^2 = 0;
    radial ghosts are the analytic profile."""
    out = []
    Nth = grid.N[1]
    for c in range(6):
        a1, a2 = yee_axes(grid, c, device)
        x2r = torch.where(a2 < 0, -a2, torch.where(a2 > Nth, 2.0 * Nth - a2, a2))       # reflect about the axis
        sign = torch.where((a2 < 0) | (a2 > Nth), -1.0, 1.0) if (c % 3) != 0 else torch.ones_like(a2)
        X1, X2 = a1[None, :], x2r[:, None]
        r, th, h1, h2, h3 = sph_geometry(grid, X1, X2)
        hat = profile(r + 0 * th, th + 0 * r)[c]
        h = (h1, h2, h3)[c % 3] + 0 * r + 0 * th
        on_axis = (h3 + 0 * r + 0 * th).abs() < 1e-12 * r.abs().max()
        if c % 3 == 2:
            val = torch.where(on_axis, torch.zeros_like(hat), hat / torch.where(on_axis, torch.ones_like(h), h))
        else:
            val = hat / h
        if c == 4:                                                                        # B^2 on the axis
            axis_rows = ((x2r == 0) | (x2r == Nth))[:, None]
            val = torch.where(axis_rows, torch.zeros_like(val), val)
        out.append((val * sign[:, None]).to(torch.float32).contiguous())
    return out


# ------------------------------------------------------------------------------------------------------------
# particle loading
# ------------------------------------------------------------------------------------------------------------
def _cells_from_counts(counts: torch.Tensor) -> torch.Tensor:
    return torch.repeat_interleave(torch.arange(counts.numel(), device=counts.device, dtype=torch.int64), counts)


def load_pairs(grid: GridSpec, seed: int, counts: torch.Tensor, theta: float, q: float, m: float, device,
               beta_fn=None, weight_fn=None) -> list:
    """e- / e+ pairs created on top of each other with independent momenta: `counts[c]` pairs in linear cell c,
    in cell order (so the block is cell-sorted), uniform in-cell offsets.  Returns [electrons, positrons]."""
    cell = _cells_from_counts(counts.to(device))
    n = int(cell.numel())
    i = unpack_cell(grid, cell)
    d = [uniform(seed, a, n, device) for a in range(grid.D)]
    phi = (2.0 * math.pi * uniform(seed, 6, n, device, dtype=torch.float64)).to(torch.float32) if grid.kind != CART else None
    if phi is not None:
        phi = phi.clamp_max(6.2831850)
    w = weight_fn(i, d) if weight_fn is not None else torch.ones(n, dtype=torch.float32, device=device)
    out = []
    for s, (qs, base) in enumerate(((-q, 10), (q, 20))):
        beta = beta_fn(n, device) if beta_fn is not None else None
        u = maxwell_juettner(seed, (base, base + 1, base + 2), n, theta, device, beta_x=beta)
        out.append(Species(q=qs, m=m, i=[t.clone() for t in i], d=[t.clone() for t in d], u=u, w=w.clone(),
                           phi=None if phi is None else phi.clone()))
    return out


# ------------------------------------------------------------------------------------------------------------
# the five configurations of BASELINE.json.  `shrink` divides every grid extent (per-cell
# statistics unchanged) so that the CPU oracle can follow; shrink = 1 is the full size.
# ------------------------------------------------------------------------------------------------------------
def _cart_fields_from_modes(grid: GridSpec, comps_modes, const, device) -> list:
    """comps_modes[c] = list of (amp, (m1,m2,m3), psi): sum of amp*cos(2 pi m.x/L + psi) in ORTHONORMAL components,
    evaluated at each component's Yee points (ghosts included: the profile is periodic), then / cell size."""
    D = grid.D
    dx = [(grid.xmax[a] - grid.xmin[a]) / grid.N[a] for a in range(D)]
    out = []
    for c in range(6):
        ax = yee_axes(grid, c, device)
        shape = grid.padded_shape
        val = torch.full(shape, float(const[c]), dtype=torch.float64, device=device)
        for amp, mvec, psi in comps_modes[c]:
            ph = torch.full(shape, float(psi), dtype=torch.float64, device=device)
            for a in range(D):
                view = [1] * D
                view[D - 1 - a] = -1
                ph = ph + (2.0 * math.pi * mvec[a] / grid.N[a]) * ax[a].view(view)      # x/L = code coordinate / N
            val = val + amp * torch.cos(ph)
        scale = dx[c % 3] if (c % 3) < D else 1.0                                       # h33 = 1 in 2D
        out.append((val / scale).to(torch.float32).contiguous())
    return out


def config1(shrink: int = 1, device="cpu") -> Workload:
    """C1: 2D Cartesian 64x64 periodic, pair plasma 16 ppc, MJ theta = 0.1, B0 = z + random E,B modes (k <= 4)."""
    seed, N = 0, max(8, 64 // shrink)
    grid = GridSpec(D=2, N=(N, N), bc=(PERIODIC, PERIODIC), kind=CART, xmin=(0.0, 0.0), xmax=(0.5 * N, 0.5 * N))
    Um = uniform(seed, 8, 6 * 8 * 8, "cpu", dtype=torch.float64).view(6, 8, 8)
    modes = []
    for c in range(6):
        lst = []
        for k in range(8):
            m1 = m2 = 0
            j = 0
            while m1 == 0 and m2 == 0:
                m1, m2 = int(Um[c, k, j] * 9) - 4, int(Um[c, k, j + 1] * 9) - 4
                j += 2
            lst.append((0.1 / math.sqrt(8.0) * math.sqrt(2.0), (m1, m2, 0), 2.0 * math.pi * float(Um[c, k, 7])))
        modes.append(lst)
    fields = _cart_fields_from_modes(grid, modes, (0, 0, 0, 0, 0, 1.0), device)
    counts = torch.full((grid.ncells,), 8, dtype=torch.int64)
    sp = load_pairs(grid, seed, counts, 0.1, 1.0, 1.0, device)
    return Workload("C1", grid, 0.45 * 0.5, 10, fields, sp, seed, "2D Cartesian, generic periodic tests of sect. 5.1")


def _alfven_modes(seed: int, nmodes: int, amp: float, vA: float):
    U = uniform(seed, 8, 16 * nmodes * 5, "cpu", dtype=torch.float64).view(-1, 5)
    bx, by, ex, ey = [], [], [], []
    for row in U:
        m = [int(row[a] * 17) - 8 for a in range(3)]
        if m[0] == 0 and m[1] == 0 or m[0] ** 2 + m[1] ** 2 + m[2] ** 2 > 64:
            continue
        kp = math.hypot(m[0], m[1])
        e = (m[1] / kp, -m[0] / kp)                       # (k x z)/|k x z|
        psi = 2.0 * math.pi * float(row[3])
        sg = 1.0 if row[4] < 0.5 else -1.0
        bx.append((amp * e[0], tuple(m), psi)); by.append((amp * e[1], tuple(m), psi))
        ex.append((sg * vA * amp * e[1], tuple(m), psi)); ey.append((-sg * vA * amp * e[0], tuple(m), psi))   # dB x z
        if len(bx) == nmodes:
            break
    assert len(bx) == nmodes
    return [ex, ey, [], bx, by, []]


def config3(shrink: int = 1, device="cpu") -> Workload:
    """C3: 3D Cartesian 256^3 periodic, pair plasma 8 ppc, MJ theta = 1, B0 = z + 64 Alfvenic modes (dB/B0 = 0.5)."""
    seed, N = 2, max(8, 256 // shrink)
    grid = GridSpec(D=3, N=(N, N, N), bc=(PERIODIC,) * 3, kind=CART, xmin=(0.0,) * 3, xmax=(0.5 * N,) * 3)
    modes = _alfven_modes(seed, 64, math.sqrt(2.0 * 0.25 / 64.0), math.sqrt(0.5))
    fields = _cart_fields_from_modes(grid, modes, (0, 0, 0, 0, 0, 1.0), device)
    counts = torch.full((grid.ncells,), 4, dtype=torch.int64)
    sp = load_pairs(grid, seed, counts, 1.0, 1.0, 1.0, device)
    return Workload("C3", grid, 0.45 * 0.5, 10, fields, sp, seed, "3D driven-turbulence shape (sect. 5.1.4)")


def config4(shrink: int = 1, device="cpu", shuffled: bool = False) -> Workload:
    """C4: 3D Cartesian 512^3 periodic, pair plasma 4 ppc, theta = 0.3, beams drifting at +-0.5c along x, B0 = 0.1 z."""
    seed, N = 3, max(8, 512 // shrink)
    grid = GridSpec(D=3, N=(N, N, N), bc=(PERIODIC,) * 3, kind=CART, xmin=(0.0,) * 3, xmax=(0.5 * N,) * 3)
    fields = _cart_fields_from_modes(grid, [[] for _ in range(6)], (0, 0, 0, 0, 0, 0.1), device)
    counts = torch.full((grid.ncells,), 2, dtype=torch.int64)
    beta = lambda n, dev: torch.where(torch.arange(n, device=dev) % 2 == 0, 0.5, -0.5).to(torch.float64)
    sp = load_pairs(grid, seed, counts, 0.3, 1.0, 1.0, device, beta_fn=beta)
    if shuffled:
        for s in sp:
            perm = torch.argsort(rand_bits(seed, 30, s.n, device))
            s.i = [t[perm].contiguous() for t in s.i]; s.d = [t[perm].contiguous() for t in s.d]
            s.u = [t[perm].contiguous() for t in s.u]; s.w = s.w[perm].contiguous()
    return Workload("C4" + ("-shuffled" if shuffled else ""), grid, 0.45 * 0.5, 10, fields, sp, seed,
                    "the paper's own performance workload: 3D counter-streaming / Weibel (P:801)")


# ------------------------------------------------------------------------------------------------------------
# axisymmetric configurations (magnetosphere shape, sect. 5.2)
# ------------------------------------------------------------------------------------------------------------
def _dipole_corotation(Omega: float):
    """static dipole B ~ r^-3 plus corotation E = -(Omega x r) x B (Eq. 23 form); orthonormal components"""
    def profile(r, th):
        Br, Bth = 2.0 * torch.cos(th) / r ** 3, torch.sin(th) / r ** 3
        Er, Eth = Omega * r * Bth * torch.sin(th), -Omega * r * Br * torch.sin(th)
        z = torch.zeros_like(r)
        return (Er, Eth, z, Br, Bth, z)
    return profile


def _magnetosphere(Omega: float, sheet_width: float = 0.05):
    """rotating dipole inside the light cylinder R_LC = 1/Omega blended into a split monopole with a Harris-type
    equatorial reversal outside (Michel solution, Eq. 24); E = -(Omega r sin(theta) phi-hat) x B"""
    RLC = 1.0 / Omega
    BL = 2.0 / RLC ** 3

    def profile(r, th):
        s = 0.5 * (1.0 + torch.tanh((r - RLC) / (0.1 * RLC)))
        Br_d, Bth_d = 2.0 * torch.cos(th) / r ** 3, torch.sin(th) / r ** 3
        Br_o = BL * (RLC / r) ** 2 * torch.tanh((0.5 * math.pi - th) / sheet_width)
        Bph_o = -(r * torch.sin(th) / RLC) * Br_o
        Br, Bth, Bph = (1 - s) * Br_d + s * Br_o, (1 - s) * Bth_d, s * Bph_o
        vph = Omega * r * torch.sin(th)                     # corotation speed (phi-hat)
        Er, Eth = vph * Bth, -vph * Br                      # -(v_phi phi-hat) x B
        return (Er, Eth, torch.zeros_like(r), Br, Bth, Bph)
    return profile


def _axisym_workload(name, seed, N, rmax, vartheta, mean_pairs, theta_T, qm, profile, steps, device, note) -> Workload:
    grid = GridSpec(D=2, N=(N, N), bc=(ABSORB, AXIS), kind=QSPH, xmin=(1.0, 0.0), xmax=(rmax, math.pi), r0=0.0,
                    vartheta=vartheta)
    fields = axisym_fields(grid, profile, device)
    # pairs per cell ~ r_c^-2 (the non-uniform injector pattern), stochastic rounding with stream 7
    x1c = torch.arange(N, dtype=torch.float64, device=device) + 0.5
    rc, _, _, _, _ = sph_geometry(grid, x1c, torch.zeros_like(x1c))
    dens = rc ** -2
    dens = dens * (mean_pairs / float(dens.mean()))
    want = dens[None, :].expand(N, N).reshape(-1)                                       # linear cell = i1 + N*i2
    counts = torch.floor(want + uniform(seed, 7, N * N, device, dtype=torch.float64)).to(torch.int64)
    # weights w = sqrt(h)(x_p) / V0, V0 = sqrt(h) at the centre of cell (0,0)  (reading G14)
    h0 = sph_geometry(grid, torch.tensor(0.5, dtype=torch.float64), torch.tensor(0.5, dtype=torch.float64))
    V0 = float(h0[2] * h0[3] * h0[4])

    def weight_fn(i, d):
        _, _, h1, h2, h3 = sph_geometry(grid, i[0].to(torch.float64) + d[0].to(torch.float64),
                                        i[1].to(torch.float64) + d[1].to(torch.float64))
        return (h1 * h2 * h3 / V0).to(torch.float32)

    sp = load_pairs(grid, seed, counts, theta_T, 1.0, 1.0 / qm, device, weight_fn=weight_fn)
    dt = 0.5 * cfl_dx_min(grid)                                                          # Eq. 8 with CFL = 0.5 (G13)
    return Workload(name, grid, dt, steps, fields, sp, seed, note)


def config2(shrink: int = 1, device="cpu") -> Workload:
    """C2: axisymmetric log-spherical (QSPH r0 = 0, vartheta = 0; reading G15) 256x256, r in [1,20], static dipole plus
    corotation E (Omega = 0.1), pair plasma 32 ppc ~ r^-2, theta_T = 0.05, |q/m| = 100, 20 steps."""
    N = max(16, 256 // shrink)
    # |q/m| = 100 at full size puts omega_c dt = |q/m| B dt at ~0.8 at the pole of the stellar surface (B = 2); dt grows with the
    # cell size, so the shrunk variants scale |q/m| by N/256 to keep that number (and with it the conditioning of the push)
    return _axisym_workload("C2", 1, N, 20.0, 0.0, 16.0, 0.05, 100.0 * N / 256.0, _dipole_corotation(0.1), 20, device,
                            "magnetosphere shape (sect. 5.2), log-r uniform-theta grid (P:993)")


def config5(shrink: int = 1, device="cpu") -> Workload:
    """C5: quasi-spherical 2048x2048 (r0 = 0, vartheta = 0.4; reading G16), r in [1,50], rotating-dipole magnetosphere with
    an equatorial Harris-type current sheet (Omega = 0.2), pair plasma 64 ppc ~ r^-2, theta_T = 0.1, |q/m| = 1000, 20 steps."""
    N = max(16, 2048 // shrink)
    return _axisym_workload("C5", 4, N, 50.0, 0.4, 32.0, 0.1, 1000.0 * N / 2048.0, _magnetosphere(0.2), 20, device,
                            "pulsar-magnetosphere shape (sect. 5.2, P:993), theta stretched toward the equator")


def sph_small(N: int = 64, device="cpu") -> Workload:
    """parity-only variant with the linear-r SPH metric so that all three metrics are exercised (G15)"""
    seed = 5
    grid = GridSpec(D=2, N=(N, N), bc=(ABSORB, AXIS), kind=SPH, xmin=(1.0, 0.0), xmax=(10.0, math.pi))
    fields = axisym_fields(grid, _dipole_corotation(0.1), device)
    counts = torch.full((N * N,), 4, dtype=torch.int64)
    sp = load_pairs(grid, seed, counts, 0.05, 1.0, 1.0 / 12.0, device)       # omega_c dt ~ 0.8 at the pole
    return Workload("SPH-small", grid, 0.5 * cfl_dx_min(grid), 20, fields, sp, seed, "linear-r spherical metric")


def cart_absorb_small(D: int = 3, device="cpu") -> Workload:
    """parity-only edge case: Cartesian box with ABSORB sides in x1 (and x3), periodic in x2, extents that are not multiples
    of the tile (partial tiles), a particle count that is not a multiple of 4, hot plasma so that particles do leave"""
    seed = 6
    N = (20, 16, 12) if D == 3 else (36, 24)
    bc = (ABSORB, PERIODIC, ABSORB) if D == 3 else (ABSORB, PERIODIC)
    grid = GridSpec(D=D, N=N, bc=bc, kind=CART, xmin=(0.0,) * D, xmax=tuple(0.5 * n for n in N))
    Um = uniform(seed, 8, 6 * 4 * 4, "cpu", dtype=torch.float64).view(6, 4, 4)
    modes = [[(0.2, (int(Um[c, k, 0] * 3) + 1, int(Um[c, k, 1] * 3), int(Um[c, k, 2] * 3) if D == 3 else 0),
               2.0 * math.pi * float(Um[c, k, 3])) for k in range(4)] for c in range(6)]
    fields = _cart_fields_from_modes(grid, modes, (0, 0, 0, 0, 0, 1.0), device)
    counts = torch.full((grid.ncells,), 3, dtype=torch.int64)
    sp = load_pairs(grid, seed, counts, 0.5, 1.0, 1.0, device)
    for s_ in sp:                                            # ragged tail: n % 4 == 1
        keep = s_.n - 3
        s_.i = [t[:keep].contiguous() for t in s_.i]; s_.d = [t[:keep].contiguous() for t in s_.d]
        s_.u = [t[:keep].contiguous() for t in s_.u]; s_.w = s_.w[:keep].contiguous()
    return Workload(f"CART-absorb-{D}D", grid, 0.45 * 0.5, 12, fields, sp, seed, "absorbing Cartesian box, partial tiles, ragged n")


def cart_periodic_odd(device="cpu") -> Workload:
    """parity-only edge case: fully periodic 3D box whose extents are not multiples of the tile (20 x 12 x 9 with 8^3 tiles: the last
    tiles are 4, 4 and 1 cells thick and wrap onto the first), two tiles per periodic axis, hot plasma"""
    seed = 9
    N = (20, 12, 9)
    grid = GridSpec(D=3, N=N, bc=(PERIODIC,) * 3, kind=CART, xmin=(0.0,) * 3, xmax=tuple(0.5 * n for n in N))
    Um = uniform(seed, 8, 6 * 4 * 4, "cpu", dtype=torch.float64).view(6, 4, 4)
    modes = [[(0.2, (int(Um[c, k, 0] * 3) + 1, int(Um[c, k, 1] * 3), int(Um[c, k, 2] * 3)), 2.0 * math.pi * float(Um[c, k, 3]))
              for k in range(4)] for c in range(6)]
    fields = _cart_fields_from_modes(grid, modes, (0, 0, 0, 0, 0, 1.0), device)
    counts = torch.full((grid.ncells,), 5, dtype=torch.int64)
    sp = load_pairs(grid, seed, counts, 0.5, 1.0, 1.0, device)
    return Workload("CART-periodic-odd", grid, 0.45 * 0.5, 12, fields, sp, seed, "periodic Cartesian box, partial tiles that wrap")


CONFIGS = {"C1": config1, "C2": config2, "C3": config3, "C4": config4, "C5": config5}
