"""GPU parity of the COLD paths of the tiled kernels: code that the five BASELINE.json configurations never or hardly ever reach,
forced here by construction and checked against the fp64 oracle at the bars of tests/parity.py:
  * a signed wrap of a fixed-point J-tile accumulator (`carry_fix`): > 128 coherent contributions on one node;
  * weights changed after the sort (`wguard` -> deposit through global atomics);
  * strays (no re-sort for many steps), the stray list and its overflow fallback;
  * contributions too large for the tile's fixed-point range next to the polar axis (`global_add`);
  * the re-bin's "far" class (destination more than one tile away), its unordered branch (more stayers than staging room),
    a tile shared by several CTAs (TILE_CHUNK) and the same for ent_step_sorted.
"""
import numpy as np
import pytest
import torch

import parity as P
from test_gpu_parity import _match_perm, _host_keys

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env(orc):
    from paper_2511_17710_b200 import binding as bind, synth
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback for the product path")
    ctx = bind.ent_create(0, None)
    yield bind, synth, ctx, orc
    bind.ent_destroy(ctx)


def _species(synth, g, i, d, u, w, q=-1.0, m=1.0, phi=None):
    t32 = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float32)
    return synth.Species(q=q, m=m, i=[torch.as_tensor(np.ascontiguousarray(i[:, a]), dtype=torch.int32) for a in range(g.D)],
                         d=[t32(d[:, a]) for a in range(g.D)], u=[t32(u[:, a]) for a in range(3)], w=t32(w),
                         phi=None if phi is None else t32(phi))


class Runner:
    """one species on the GPU (through the C ABI) and in the oracle, step by step; follows the permutations of ent_sort"""

    def __init__(self, env, g, fields, sp, dt):
        self.bind, self.synth, self.ctx, self.orc = env
        bind, orc = self.bind, self.orc
        self.g, self.dt, self.sp = g, dt, sp
        self.eg, self.og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
        bind.ent_set_option(self.ctx, bind.OPT_STEP_IMPL, 0)
        bind.ent_set_option(self.ctx, bind.OPT_SORT_MODE, 0)
        bind.ent_set_grid(self.ctx, self.eg)
        self.F_dev, self.F_orc = [f.cuda() for f in fields], P.fields_to_orc(fields)
        self.pe = P.species_to_ent(bind, self.synth, g, sp, "cuda")
        self.po = P.species_to_orc(orc, sp)
        self.order = np.arange(sp.n)
        self.Jg = bind.zeros_current(self.eg, "cuda")
        self.steps = 0

    def sort(self, full=False):
        bind = self.bind
        ps = self.pe.empty_like()
        if full:
            bind.ent_set_option(self.ctx, bind.OPT_SORT_MODE, 1)
        bind.ent_sort(self.ctx, self.pe, ps, None)
        bind.ent_set_option(self.ctx, bind.OPT_SORT_MODE, 0)
        perm = _match_perm(self.g, self.pe, ps)
        self.order = self.order[perm]
        self.pe = ps
        return bind.ent_get_stat(self.ctx, bind.STAT_LAST_SORT_REBIN)

    def step(self, check=True):
        bind, orc = self.bind, self.orc
        before = P.ent_to_orc(orc, self.g, self.pe) if check else None
        bind.ent_zero_current(self.ctx, self.Jg)
        bind.ent_step(self.ctx, self.F_dev, self.pe, self.Jg, self.dt)
        bind.ent_fold_current(self.ctx, self.Jg)
        torch.cuda.synchronize()
        Jo = orc.zeros_current(self.og)
        po_before = self.po.copy() if check else None
        orc.step(self.og, self.F_orc, self.po, Jo, self.sp.q, self.sp.m, self.dt)
        orc.fold_current(self.og, Jo)
        self.steps += 1
        res = {}
        if check:
            after = P.ent_to_orc(orc, self.g, self.pe)
            res["zigzag_straddlers"], corr = P.straddler_correction(orc, self.g, self.og, po_before, self.po, before, after, self.sp.q, self.dt, self.order)
            if corr is not None:
                Jo = [a + b for a, b in zip(Jo, corr)]
            res["J"] = P.compare_current(self.Jg, Jo, P.offset_format_bound(orc, self.g, self.og, before, self.sp.q, self.dt) if self.eg.axisym else None)
            res["Jraw"] = P.compare_current.last_raw
            res["Jstrict"] = P.compare_current(self.Jg, P.deposit_of_gpu_positions(orc, self.og, before, after, self.sp.q, self.dt))
            res["cont"] = P.continuity_of_gpu_step(orc, self.og, before, after, self.Jg, self.sp.q, self.dt)
            assert res["cont"] <= P.CONT_TOL, res
        return res

    def check_particles(self):
        return P.compare_particles(self.g, self.pe, self.po, self.order, steps=self.steps, orc_metric=(self.orc, self.og))

    def stat(self, key):
        return self.bind.ent_get_stat(self.ctx, key)


def _cart_box(synth, N=(16, 16, 16)):
    return synth.GridSpec(D=3, N=N, bc=(0, 0, 0), kind=synth.CART, xmin=(0.0, 0.0, 0.0), xmax=tuple(0.5 * n for n in N))


def _fields_uniform(g, B=(0.0, 0.0, 0.2)):
    F = [torch.zeros(g.padded_shape, dtype=torch.float32) for _ in range(6)]
    for c in range(3):
        F[3 + c] += B[c]
    return F


def test_carry_of_the_fixed_point_tile(env):
    """3000 identical-momentum particles in ONE cell: ~3000 coherent contributions of nearly the largest size on the same nodes wrap
    the 32-bit fixed-point accumulators (128 suffice); the carries go to the global array and the current still matches the oracle."""
    bind, synth, ctx, orc = env
    g = _cart_box(synth)
    rng = np.random.default_rng(1)
    n = 3000
    i = np.tile(np.array([[5, 6, 7]]), (n, 1))
    d = rng.uniform(0.2, 0.8, (n, 3))
    u = np.tile(np.array([[3.0, 0.2, -0.1]]), (n, 1)) + 0.01 * rng.standard_normal((n, 3))
    r = Runner(env, g, _fields_uniform(g), _species(synth, g, i, d, u, np.ones(n)), 0.225)
    c0 = r.stat(bind.STAT_CARRIES)
    r.sort(full=True)
    for _ in range(3):
        res = r.step()
        assert r.stat(bind.STAT_LAST_STEP_TILED) == 1 and r.stat(bind.STAT_STRAYS) == 0
    assert r.stat(bind.STAT_CARRIES) > c0, "no accumulator wrapped: the carry path was not exercised"
    print("carry:", res, r.check_particles(), "carries", r.stat(bind.STAT_CARRIES) - c0)


def test_weights_changed_after_the_sort_take_the_global_path(env):
    """The fixed-point scale of a tile comes from the max |w| recorded by ent_sort.  Weights multiplied by 100 afterwards (in place,
    same block) exceed the guard (60 x) and must deposit through the global path; the rest of the tile keeps the tile's scale."""
    bind, synth, ctx, orc = env
    wl = synth.config3(16)
    sp = wl.species[0]
    r = Runner(env, wl.grid, wl.fields, sp, wl.dt)
    r.sort(full=True)
    heavy = torch.arange(r.pe.n, device="cuda") % 7 == 0
    r.pe.w[heavy] *= 100.0
    r.po.w[r.order[heavy.cpu().numpy()]] *= 100.0
    for _ in range(2):
        res = r.step()
        assert r.stat(bind.STAT_LAST_STEP_TILED) == 1
    print("wguard:", res, r.check_particles())


def test_strays_stray_list_and_its_overflow(env):
    """14 steps without a re-sort: particles drift out of their tile's halo (strays), first fewer than the stray list holds, in the
    end more (the tile kernel then advances them in line).  Every step is compared with the oracle."""
    bind, synth, ctx, orc = env
    wl = synth.config3(8)
    sp = wl.species[0]
    r = Runner(env, wl.grid, wl.fields, sp, wl.dt)
    r.sort(full=True)
    cap = sp.n // 16 + 4096
    seen_some = seen_overflow = False
    for s in range(14):
        r.step(check=(s % 3 == 1 or s >= 12))
        k = r.stat(bind.STAT_STRAYS)
        seen_some |= 0 < k <= cap
        seen_overflow |= k > cap
    assert seen_some and seen_overflow, f"strays at the end {k}, list capacity {cap}"
    print("strays:", k, "capacity", cap, r.check_particles())
    # the re-bin of such a block meets particles more than one tile away ("far" class) -- only if a tile is small enough
    assert r.sort() == 1
    T = [r.stat(k_) for k_ in (bind.STAT_TILE_1, bind.STAT_TILE_2, bind.STAT_TILE_3)]
    keys, _ = _host_keys(synth, bind, ctx, wl.grid, r.pe.cell)
    toff = bind.ent_tile_offsets(ctx, r.pe).cpu().numpy()
    assert orc.sort_check((keys // int(np.prod(T))).astype(np.int32), r.stat(bind.STAT_NTILES), toff) == 0
    r.step()
    assert r.stat(bind.STAT_STRAYS) == 0
    r.check_particles()


def test_rebin_far_class_with_thin_tiles(env):
    """tile 8 x 8 x 4: after 12 steps without a sort fast particles sit two tiles away along z; the incremental ent_sort must send them
    through its 'far' class.  Checked: permutation, tile contiguity + offsets (oracle's sort checker), parity after more steps."""
    bind, synth, ctx, orc = env
    wl = synth.config3(8)
    sp = wl.species[0]
    bind.ent_set_option(ctx, bind.OPT_TILE_3, 4)
    try:
        r = Runner(env, wl.grid, wl.fields, sp, wl.dt)
        assert r.stat(bind.STAT_TILE_3) == 4
        r.sort(full=True)
        cell0 = r.pe.cell.clone()
        for s in range(12):
            r.step(check=False)
        i0 = synth.unpack_cell(wl.grid, cell0.cpu())[2].numpy() // 4
        i1 = synth.unpack_cell(wl.grid, r.pe.cell.cpu())[2].numpy() // 4
        dz = np.abs(i1 - i0); dz = np.minimum(dz, wl.grid.N[2] // 4 - dz)
        assert (dz >= 2).sum() > 0, "no particle is two tiles away: the far class is not exercised"
        assert r.sort() == 1
        keys, T = _host_keys(synth, bind, ctx, wl.grid, r.pe.cell)
        toff = bind.ent_tile_offsets(ctx, r.pe).cpu().numpy()
        assert orc.sort_check((keys // int(np.prod(T))).astype(np.int32), r.stat(bind.STAT_NTILES), toff) == 0
        res = r.step()
        assert r.stat(bind.STAT_STRAYS) == 0 and r.stat(bind.STAT_LAST_STEP_TILED) == 1
        print("far class:", int((dz >= 2).sum()), "particles two tiles away;", res, r.check_particles())
    finally:
        bind.ent_set_option(ctx, bind.OPT_TILE_3, 0)


def test_clustered_density_heavy_tile_and_heavy_cell(env):
    """one tile with ~20 x the mean population (shared by several CTAs: TILE_CHUNK), one cell with 400 particles: the re-bin's
    unordered branch (more stayers than staging room), chunked tiles in ent_step and in ent_step_sorted."""
    bind, synth, ctx, orc = env
    wl = synth.config3(8)
    g = wl.grid
    base = wl.species[0]
    rng = np.random.default_rng(2)
    nx = 9000
    i = np.stack([rng.integers(8, 16, nx), rng.integers(8, 16, nx), rng.integers(16, 24, nx)], 1)
    i[:400] = [9, 10, 17]
    d = rng.uniform(0, 1, (nx, 3))
    u = rng.standard_normal((nx, 3))
    extra = _species(synth, g, i, d, u, np.ones(nx), q=base.q, m=base.m)
    cat = lambda a, b: torch.cat([a, b])
    sp = synth.Species(q=base.q, m=base.m, i=[cat(a, b) for a, b in zip(base.i, extra.i)], d=[cat(a, b) for a, b in zip(base.d, extra.d)],
                       u=[cat(a, b) for a, b in zip(base.u, extra.u)], w=cat(base.w, extra.w))
    r = Runner(env, g, wl.fields, sp, wl.dt)
    r.sort(full=True)
    toff = bind.ent_tile_offsets(ctx, r.pe).cpu().numpy()
    assert np.diff(toff).max() > 4096, "no tile is shared by several CTAs"
    for s in range(3):
        res = r.step()
        assert r.stat(bind.STAT_LAST_STEP_TILED) == 1 and r.stat(bind.STAT_STRAYS) == 0
    assert r.sort() == 1                                      # the heavy tile has more stayers than the staging area holds
    for s in range(2):
        res = r.step()
    print("clustered:", res, r.check_particles())
    # the same block through ent_step_sorted (chunked tile, global slot reservations of several CTAs into one range)
    a, b = r.pe, r.pe.empty_like()
    for s in range(3):
        Jo = orc.zeros_current(r.og)
        orc.step(r.og, r.F_orc, r.po, Jo, sp.q, sp.m, wl.dt)
        bind.ent_zero_current(ctx, r.Jg)
        bind.ent_step_sorted(ctx, r.F_dev, a, b, r.Jg, wl.dt)
        a, b = b, a
    bind.ent_fold_current(ctx, r.Jg); orc.fold_current(r.og, Jo)
    torch.cuda.synchronize()
    assert r.stat(bind.STAT_SLOT_ERRORS) == 0 and r.stat(bind.STAT_STRAYS) == 0
    P.compare_current(r.Jg, Jo)
    # ent_step_sorted permutes: compare as multisets through a sort of both sides by (cell, offsets, momentum)
    key = lambda cell, d0, u0: np.lexsort([u0, d0, cell])
    ig = a.cell.cpu().numpy(); ko = key(ig, a.d[0].cpu().numpy(), a.u[0].cpu().numpy())
    co = (r.po.i[0] + g.N[0] * (r.po.i[1] + g.N[1] * r.po.i[2])).astype(np.int64)
    oo = key(co, r.po.d[0], r.po.u[0])
    agree = (ig[ko] == co[oo]).mean()
    assert agree > 0.9999, agree                              # straddlers of a cell face may differ
    assert np.abs(np.sort(a.u[2].cpu().numpy().astype(np.float64)) - np.sort(r.po.u[2])).max() < 1e-4


def test_contributions_beyond_the_tile_range_next_to_the_axis(env):
    """SPH grid, particles a hair from the polar axis with azimuthal momentum.  J^3 = q w v^phihat / (r sin theta) at the midpoint of the
    move is bounded by ~2 q w / dt (the move itself carries the particle away from the axis), so it only leaves the tile's
    fixed-point range when the weight is also well above the tile's recorded maximum: the weights of those particles are
    multiplied by 50 after the sort (below the 60 x guard that would send them to the stray path).  Such contributions go to the
    global array directly (`global_add`)."""
    bind, synth, ctx, orc = env
    wl = synth.sph_small(48)
    g = wl.grid
    base = wl.species[0]
    rng = np.random.default_rng(3)
    nx = 600
    i = np.stack([rng.integers(4, 40, nx), np.where(rng.uniform(size=nx) < 0.5, 0, g.N[1] - 1)], 1)
    d = np.stack([rng.uniform(0, 1, nx), np.where(i[:, 1] == 0, rng.uniform(1e-5, 1e-3, nx), 1.0 - rng.uniform(1e-5, 1e-3, nx))], 1)
    phi = rng.uniform(0, 2 * np.pi, nx)
    vphi = rng.uniform(0.2, 0.6, nx) * rng.choice([-1.0, 1.0], nx)
    gam = 1.0 / np.sqrt(1.0 - vphi ** 2)
    u = np.stack([-gam * vphi * np.sin(phi), gam * vphi * np.cos(phi), 0.05 * rng.standard_normal(nx)], 1)
    w = np.full(nx, float(base.w.mean()))
    extra = _species(synth, g, i, d, u, w, q=base.q, m=base.m, phi=phi)
    cat = lambda a, b: torch.cat([a, b])
    sp = synth.Species(q=base.q, m=base.m, i=[cat(a, b) for a, b in zip(base.i, extra.i)], d=[cat(a, b) for a, b in zip(base.d, extra.d)],
                       u=[cat(a, b) for a, b in zip(base.u, extra.u)], w=cat(base.w, extra.w), phi=cat(base.phi, extra.phi))
    r = Runner(env, g, wl.fields, sp, wl.dt)
    g0 = r.stat(bind.STAT_GLOBAL_ADDS)
    r.sort(full=True)
    added = torch.as_tensor(r.order >= base.n, device="cuda")
    r.pe.w[added] *= 50.0
    r.po.w[base.n:] *= 50.0
    for s in range(3):
        res = r.step()
        assert r.stat(bind.STAT_LAST_STEP_TILED) == 1
    assert r.stat(bind.STAT_GLOBAL_ADDS) > g0, "no contribution left the tile's fixed-point range"
    print("axis:", res, "global adds", r.stat(bind.STAT_GLOBAL_ADDS) - g0)
