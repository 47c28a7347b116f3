"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the fp64 oracle, element by element, on
the same seeded synthetic inputs.  Sizes: the oracle finishes each case in seconds; every case spans several tiles and a
ragged tail.  Tolerances are BASELINE.json's (north_star), written in tests/parity.py.
"""
import numpy as np
import pytest
import torch

import parity as P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env(orc):
    from paper_2511_17710_b200 import binding as bind, synth
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback for the product path")
    ctx = bind.ent_create(0, None)
    yield bind, synth, ctx, orc
    bind.ent_destroy(ctx)


def _workloads(synth):
    return {
        "C1": lambda: synth.config1(1),                 # full size: 64x64, 65,536 particles
        "C2/4": lambda: synth.config2(4),               # 64x64 log-spherical, ~131k particles, density ~ r^-2
        "C3/8": lambda: synth.config3(8),               # 32^3, 262,144 particles
        "C4/16": lambda: synth.config4(16),             # 32^3, 131,072 particles, counter-streaming beams
        "C4/16-shuffled": lambda: synth.config4(16, shuffled=True),
        "C5/32": lambda: synth.config5(32),             # 64x64 quasi-spherical vartheta = 0.4, ~262k particles
        "SPH": lambda: synth.sph_small(48),             # linear-r spherical metric
        "ABS3": lambda: synth.cart_absorb_small(3),     # absorbing Cartesian box, partial tiles, n % 4 != 0
        "ABS2": lambda: synth.cart_absorb_small(2),
        "PER3": lambda: synth.cart_periodic_odd(),      # periodic box 20 x 12 x 9: partial tiles (one of them 1 cell thick) that wrap
    }


def _match_perm(g, p_from, p_to):
    """ent_sort permutes every array alike and leaves the order inside a cell (or, re-binning, inside a tile) unspecified
    (G18): the permutation is recovered by matching records -- (cell, offsets, momentum) is unique per particle in these
    workloads.  Returns perm with p_to[k] == p_from[perm[k]], and checks that every array was permuted alike."""
    def rank(p):
        cols = [p.u[0], p.d[1], p.d[0], p.cell] if g.D == 2 else [p.u[0], p.d[2], p.d[1], p.d[0], p.cell]
        return np.lexsort([c.detach().cpu().numpy() for c in cols])
    r_from, r_to = rank(p_from), rank(p_to)
    perm = np.empty(p_from.n, dtype=np.int64)
    perm[r_to] = r_from
    pt = torch.from_numpy(perm).to(p_from.cell.device)
    same = lambda a, b: (a is None and b is None) or torch.equal(b, a[pt])
    assert same(p_from.cell, p_to.cell) and same(p_from.w, p_to.w) and same(p_from.phi, p_to.phi) and same(p_from.tag, p_to.tag)
    assert all(same(a, b) for a, b in zip(p_from.d + p_from.u, p_to.d + p_to.u)), "ent_sort is not a permutation of the records"
    return perm


def _run_case(env, wl, impl, steps=None, sort_first=False, check_every_step=True, resort_every=0):
    bind, synth, ctx, orc = env
    g = wl.grid
    eg, og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, impl)
    bind.ent_set_grid(ctx, eg)
    F_dev = [f.cuda() for f in wl.fields]
    F_orc = P.fields_to_orc(wl.fields)
    steps = wl.steps if steps is None else steps
    out = {}
    for si, sp in enumerate(wl.species):                       # species loop is serial on the host
        pe = P.species_to_ent(bind, synth, g, sp, "cuda")
        po = P.species_to_orc(orc, sp)
        order = None
        if sort_first:
            ps = pe.empty_like()
            bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 1)       # full cell-level sort (a fresh tensor may reuse the address of
            bind.ent_sort(ctx, pe, ps, None)                      # a block sorted earlier, which would select the re-bin form)
            bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 0)
            assert bind.ent_get_stat(ctx, bind.STAT_LAST_SORT_REBIN) == 0
            order = _match_perm(g, pe, ps)
            pe = ps
        Jg = bind.zeros_current(eg, "cuda")
        worstJ = worstC = rawJ = strictJ = 0.0
        zz = 0
        for s in range(steps):
            if resort_every and s > 0 and s % resort_every == 0:
                # incremental ent_sort (re-bin) of the drifted block: tile contiguity only
                ps = pe.empty_like()
                bind.ent_sort(ctx, pe, ps, None)
                assert bind.ent_get_stat(ctx, bind.STAT_LAST_SORT_REBIN) == 1
                perm = _match_perm(g, pe, ps)
                order = order[perm]
                T = [bind.ent_get_stat(ctx, k) for k in (bind.STAT_TILE_1, bind.STAT_TILE_2, bind.STAT_TILE_3)][:g.D]
                tile = (synth.sort_key(g, synth.unpack_cell(g, ps.cell.cpu()), tuple(T)) // int(np.prod(T))).numpy()
                assert np.all(np.diff(tile) >= 0), "re-binned block is not tile-contiguous"
                pe = ps
            before = P.ent_to_orc(orc, g, pe) if check_every_step else None
            bind.ent_zero_current(ctx, Jg)
            bind.ent_step(ctx, F_dev, pe, Jg, wl.dt)
            bind.ent_fold_current(ctx, Jg)
            torch.cuda.synchronize()
            Jo = orc.zeros_current(og)
            po_before = po.copy()
            orc.step(og, F_orc, po, Jo, sp.q, sp.m, wl.dt)
            orc.fold_current(og, Jo)
            if check_every_step:
                after = P.ent_to_orc(orc, g, pe)
                nz, corr = P.straddler_correction(orc, g, og, po_before, po, before, after, sp.q, wl.dt, order)    # zig-zag relay of face straddlers (G12)
                zz += nz
                if corr is not None:
                    Jo = [a + b for a, b in zip(Jo, corr)]
            if check_every_step or s == steps - 1:
                bound = P.offset_format_bound(orc, g, og, before, sp.q, wl.dt) if (eg.axisym and before is not None) else None
                worstJ = max(worstJ, P.compare_current(Jg, Jo, bound))
                rawJ = max(rawJ, P.compare_current.last_raw)
            if check_every_step:
                # STRICT current check, no allowance: the oracle's deposit of the GPU's own stored move (isolates sub-step 8)
                strictJ = max(strictJ, P.compare_current(Jg, P.deposit_of_gpu_positions(orc, og, before, after, sp.q, wl.dt)))
                c = P.continuity_of_gpu_step(orc, og, before, after, Jg, sp.q, wl.dt)
                assert c <= P.CONT_TOL, f"continuity residual {c:.3e} at step {s}"
                worstC = max(worstC, c)
        stats = P.compare_particles(g, pe, po, order, steps=steps, orc_metric=(orc, og))
        assert bind.ent_get_stat(ctx, bind.STAT_BAD_MOVES) == 0
        stats["tiled"] = bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED)
        stats["strays"] = bind.ent_get_stat(ctx, bind.STAT_STRAYS)
        stats.update(worstJ=worstJ, rawJ=rawJ, strictJ=strictJ, worstC=worstC, zigzag_straddlers=zz)
        out[si] = stats
    return out


@pytest.mark.parametrize("name", ["C1", "C2/4", "C3/8", "C4/16", "C4/16-shuffled", "C5/32", "SPH", "ABS3", "ABS2"])
def test_fused_step_untiled_matches_oracle(env, name):
    wl = _workloads(env[1])[name]()
    stats = _run_case(env, wl, impl=1)
    print(name, stats)


@pytest.mark.parametrize("name", ["C1", "C3/8", "C5/32"])
def test_two_kernel_step_matches_oracle(env, name):
    """ent_gather_push + ent_deposit with the old block kept in memory (the paper's structure)"""
    wl = _workloads(env[1])[name]()
    stats = _run_case(env, wl, impl=2, steps=3)
    print(name, stats)


@pytest.mark.parametrize("name", ["C1", "C2/4", "C3/8", "C4/16-shuffled", "C5/32", "SPH"])
def test_sorted_step_auto_path_matches_oracle(env, name):
    """ent_sort, then ent_step on the sorted block (auto: the tiled kernel where it is supported)"""
    wl = _workloads(env[1])[name]()
    stats = _run_case(env, wl, impl=0, sort_first=True)
    print(name, stats)
    assert all(st["tiled"] == 1 for st in stats.values()), "the tiled kernel did not run on a sorted block"


@pytest.mark.parametrize("name", ["C1", "C2/4", "C3/8", "C4/16-shuffled", "C5/32", "SPH", "ABS3", "ABS2", "PER3"])
def test_rebinned_block_matches_oracle(env, name):
    """ent_sort, steps, incremental ent_sort (re-bin) every 3 steps, steps: the tiled kernel on re-binned blocks"""
    wl = _workloads(env[1])[name]()
    stats = _run_case(env, wl, impl=0, sort_first=True, resort_every=3)
    print(name, stats)
    assert all(st["tiled"] == 1 and st["strays"] == 0 for st in stats.values())


def _ids(p):
    """particle identity carried by the weights of _with_id_weights"""
    return torch.round((p.w.double() - 1.0) * 2.0 ** 20).long().cpu().numpy()


def _with_id_weights(sp):
    """w_k = 1 + k 2^-20 (exact in fp32): the weight doubles as a particle id, so that the permutation ent_step_sorted applies can
    be followed without assuming anything about it.  Changes the recipe's uniform weights by < 26 %; both sides get the same w."""
    assert sp.n < (1 << 18)
    sp.w = (1.0 + torch.arange(sp.n, dtype=torch.float64) * 2.0 ** -20).to(torch.float32)
    return sp


def _take(orc, p, idx):
    f = lambda a: None if a is None else np.ascontiguousarray(a[idx])
    return orc.Particles(i=[f(a) for a in p.i], d=[f(a) for a in p.d], u=[f(a) for a in p.u], w=f(p.w), phi=f(p.phi), tag=f(p.tag))


@pytest.mark.parametrize("name", ["C1", "C3/8", "C4/16", "C4/16-shuffled", "ABS3", "ABS2"])
def test_step_sorted_matches_oracle(env, name):
    """ent_step_sorted (fused step + re-bin, ping-pong between two blocks, no ent_sort after the first): every step is compared
    with the oracle -- positions, momenta, current (end to end and the strict deposit check), continuity -- and the layout of
    the output block is checked: tile offsets = exclusive scan of the histogram of the tiles of the INPUT positions (oracle's
    sort checker), every particle in the range of the tile it started the step in, no strays, no slot errors."""
    bind, synth, ctx, orc = env
    wl = _workloads(synth)[name]()
    g = wl.grid
    eg, og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, 0)
    bind.ent_set_grid(ctx, eg)
    ntiles = bind.ent_get_stat(ctx, bind.STAT_NTILES)
    F_dev, F_orc = [f.cuda() for f in wl.fields], P.fields_to_orc(wl.fields)
    for sp in wl.species:
        sp = _with_id_weights(sp)
        pe0 = P.species_to_ent(bind, synth, g, sp, "cuda")
        po = P.species_to_orc(orc, sp)
        a, b = pe0.empty_like(), pe0.empty_like()
        bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 1)
        bind.ent_sort(ctx, pe0, a, None)
        bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 0)
        Jg = bind.zeros_current(eg, "cuda")
        worstJ = worstC = strictJ = 0.0
        for s in range(wl.steps):
            ida = _ids(a)
            before = P.ent_to_orc(orc, g, a)
            keys, T = _host_keys(synth, bind, ctx, g, a.cell)
            tile_before = keys // int(np.prod(T))
            bind.ent_zero_current(ctx, Jg)
            bind.ent_step_sorted(ctx, F_dev, a, b, Jg, wl.dt)
            bind.ent_fold_current(ctx, Jg)
            torch.cuda.synchronize()
            assert bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED) == 1
            assert bind.ent_get_stat(ctx, bind.STAT_SLOT_ERRORS) == 0 and bind.ent_get_stat(ctx, bind.STAT_STRAYS) == 0
            assert bind.ent_get_stat(ctx, bind.STAT_BAD_MOVES) == 0
            idb = _ids(b)
            assert np.array_equal(np.sort(idb), np.arange(sp.n)), "ent_step_sorted lost or duplicated particles"
            # layout of the output block
            toff = bind.ent_tile_offsets(ctx, b).cpu().numpy()
            inv = np.empty(sp.n, dtype=np.int64); inv[ida] = np.arange(sp.n)          # slot in a of particle id
            tile_of_slot_b = tile_before[inv[idb]].astype(np.int32)                   # tile each output slot's particle started in
            assert orc.sort_check(tile_of_slot_b, ntiles, toff) == 0, "output block is not contiguous by the tiles of the input positions"
            # oracle step, same particles in the oracle's own (original) order
            Jo = orc.zeros_current(og)
            po_before = po.copy()
            orc.step(og, F_orc, po, Jo, sp.q, sp.m, wl.dt)
            orc.fold_current(og, Jo)
            after_slots = P.ent_to_orc(orc, g, b)
            after = _take(orc, after_slots, np.argsort(idb)[ida])                     # the output in the order of `before`
            nz, corr = P.straddler_correction(orc, g, og, po_before, po, before, after, sp.q, wl.dt, ida)
            if corr is not None:
                Jo = [x + y for x, y in zip(Jo, corr)]
            worstJ = max(worstJ, P.compare_current(Jg, Jo))
            strictJ = max(strictJ, P.compare_current(Jg, P.deposit_of_gpu_positions(orc, og, before, after, sp.q, wl.dt)))
            c = P.continuity_of_gpu_step(orc, og, before, after, Jg, sp.q, wl.dt)
            assert c <= P.CONT_TOL, f"continuity residual {c:.3e} at step {s}"
            worstC = max(worstC, c)
            st = P.compare_particles(g, b, po, idb, steps=s + 1)
            a, b = b, a
        print(name, sp.q, st, dict(worstJ=worstJ, strictJ=strictJ, worstC=worstC))


def test_step_sorted_after_in_place_steps_and_error_paths(env):
    """mixing calls: ent_step (in place, tiled) moves the particles inside their ranges, so ent_step_sorted must recount the tile
    populations before it lays out its output; an unsorted input, overlapping blocks and axisymmetric grids are refused."""
    bind, synth, ctx, orc = env
    wl = synth.config3(8)
    g = wl.grid
    eg, og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, 0)
    bind.ent_set_grid(ctx, eg)
    F_dev, F_orc = [f.cuda() for f in wl.fields], P.fields_to_orc(wl.fields)
    sp = _with_id_weights(wl.species[0])
    pe0 = P.species_to_ent(bind, synth, g, sp, "cuda")
    po = P.species_to_orc(orc, sp)
    a, b = pe0.empty_like(), pe0.empty_like()
    Jg = bind.zeros_current(eg, "cuda")
    with pytest.raises(bind.EntError) as ei:
        bind.ent_step_sorted(ctx, F_dev, pe0, b, Jg, wl.dt)                           # not a sorted block
    assert ei.value.code == bind.EINVAL
    bind.ent_sort(ctx, pe0, a, None)
    with pytest.raises(bind.EntError):
        bind.ent_step_sorted(ctx, F_dev, a, a, Jg, wl.dt)                             # overlap
    for s in range(4):
        Jo = orc.zeros_current(og)
        orc.step(og, F_orc, po, Jo, sp.q, sp.m, wl.dt)
        bind.ent_zero_current(ctx, Jg)
        if s % 2 == 0:
            bind.ent_step(ctx, F_dev, a, Jg, wl.dt)                                   # in place, tiled
        else:
            bind.ent_step_sorted(ctx, F_dev, a, b, Jg, wl.dt)
            a, b = b, a
        assert bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED) == 1
    bind.ent_fold_current(ctx, Jg); orc.fold_current(og, Jo)
    torch.cuda.synchronize()
    assert bind.ent_get_stat(ctx, bind.STAT_SLOT_ERRORS) == 0
    P.compare_current(Jg, Jo)
    P.compare_particles(g, a, po, _ids(a), steps=4)
    bind.ent_forget(ctx, a)
    with pytest.raises(bind.EntError):
        bind.ent_step_sorted(ctx, F_dev, a, b, Jg, wl.dt)                             # forgotten
    wl5 = synth.config5(32)
    bind.ent_set_grid(ctx, P.grid_to_ent(bind, wl5.grid))
    p5 = P.species_to_ent(bind, synth, wl5.grid, wl5.species[0], "cuda")
    q5, r5 = p5.empty_like(), p5.empty_like()
    bind.ent_sort(ctx, p5, q5, None)
    with pytest.raises(bind.EntError) as ei:
        bind.ent_step_sorted(ctx, [f.cuda() for f in wl5.fields], q5, r5, bind.zeros_current(P.grid_to_ent(bind, wl5.grid), "cuda"), wl5.dt)
    assert ei.value.code == bind.EUNSUPPORTED


def _host_keys(synth, bind, ctx, g, cell):
    """sort keys recomputed on the host from the cell indices with the formula of include/ent.h (ent_sort)"""
    T = tuple(bind.ent_get_stat(ctx, k) for k in (bind.STAT_TILE_1, bind.STAT_TILE_2, bind.STAT_TILE_3))[:g.D]
    return synth.sort_key(g, synth.unpack_cell(g, cell.cpu()), T).numpy().astype(np.int32), T


@pytest.mark.parametrize("staging", [0, 1])
@pytest.mark.parametrize("name", ["C1", "C3/8", "C4/16-shuffled", "C5/32", "ABS3", "ABS2"])
def test_full_sort_passes_the_oracle_checker(env, name, staging):
    """S10: ent_sort (full form) with a key_offsets output.  Keys are recomputed on the host from out.cell; the ORACLE's checker
    (orc_sort_check: non-decreasing keys, offsets = exclusive scan of the key histogram) must accept them, and the records must
    be a permutation of the input (every array permuted alike)."""
    bind, synth, ctx, orc = env
    wl = _workloads(synth)[name]()
    g = wl.grid
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, 0)
    bind.ent_set_grid(ctx, P.grid_to_ent(bind, g))
    nkeys = bind.ent_get_stat(ctx, bind.STAT_NKEYS)
    for sp in wl.species:
        pe = P.species_to_ent(bind, synth, g, sp, "cuda")
        ps = pe.empty_like()
        ko = torch.full((nkeys + 1,), -7, dtype=torch.int32, device="cuda")
        bind.ent_set_option(ctx, bind.OPT_SORT_STAGING, staging)      # 1: records staged through the 32-byte side buffer
        try:
            bind.ent_sort(ctx, pe, ps, ko)
        finally:
            bind.ent_set_option(ctx, bind.OPT_SORT_STAGING, 0)
        torch.cuda.synchronize()
        assert bind.ent_get_stat(ctx, bind.STAT_LAST_SORT_REBIN) == 0
        _match_perm(g, pe, ps)
        keys, T = _host_keys(synth, bind, ctx, g, ps.cell)
        assert orc.sort_check(keys, nkeys, ko.cpu().numpy()) == 0, "ent_sort output rejected by orc_sort_check"
        tcells = int(np.prod(T))
        toff = bind.ent_tile_offsets(ctx, ps).cpu().numpy()
        assert np.array_equal(toff, ko.cpu().numpy()[::tcells]), "tile offsets != key offsets at the tile boundaries"


@pytest.mark.parametrize("name", ["C1", "C3/8", "C4/16-shuffled", "C5/32", "ABS3", "PER3"])
def test_rebin_tile_offsets_are_the_scan_of_the_tile_histogram(env, name):
    """S10, incremental form: after steps + re-bin, the block is tile-contiguous and the ctx's tile offsets equal the exclusive scan
    of the histogram of tile(key) recomputed on the host (checked with the oracle's checker on the TILE keys)."""
    bind, synth, ctx, orc = env
    wl = _workloads(synth)[name]()
    g = wl.grid
    eg = P.grid_to_ent(bind, g)
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, 0)
    bind.ent_set_grid(ctx, eg)
    ntiles = bind.ent_get_stat(ctx, bind.STAT_NTILES)
    F = [f.cuda() for f in wl.fields]
    J = bind.zeros_current(eg, "cuda")
    sp = wl.species[0]
    pe = P.species_to_ent(bind, synth, g, sp, "cuda")
    ps = pe.empty_like()
    bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 1)
    bind.ent_sort(ctx, pe, ps, None)
    bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 0)
    pe, ps = ps, pe
    for _ in range(3):
        bind.ent_step(ctx, F, pe, J, wl.dt)
    bind.ent_sort(ctx, pe, ps, None)
    torch.cuda.synchronize()
    assert bind.ent_get_stat(ctx, bind.STAT_LAST_SORT_REBIN) == 1
    _match_perm(g, pe, ps)
    keys, T = _host_keys(synth, bind, ctx, g, ps.cell)
    tile_keys = (keys // int(np.prod(T))).astype(np.int32)
    toff = bind.ent_tile_offsets(ctx, ps).cpu().numpy()
    assert toff.shape[0] == ntiles + 1
    assert orc.sort_check(tile_keys, ntiles, toff) == 0, "re-binned block / tile offsets rejected by orc_sort_check"


def test_sort_into_a_block_with_tags_from_one_without_marks_every_particle_alive(env):
    """ent.h (ent_sort): `in` without a tag array and `out` with one -> every particle of `out` is alive.  Both forms of the sort: the
    full counting sort and, from the sorted block after a few steps, the incremental re-bin."""
    bind, synth, ctx, orc = env
    wl = _workloads(synth)["C3/8"]()
    g = wl.grid
    eg = P.grid_to_ent(bind, g)
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, 0)
    bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 0)
    bind.ent_set_grid(ctx, eg)
    F = [f.cuda() for f in wl.fields]
    J = bind.zeros_current(eg, "cuda")
    src = P.species_to_ent(bind, synth, g, wl.species[0], "cuda", with_tag=False)
    mk = lambda: bind.Particles(cell=torch.empty_like(src.cell), d=[torch.empty_like(t) for t in src.d], u=[torch.empty_like(t) for t in src.u],
                                w=torch.empty_like(src.w), phi=None, tag=torch.full((src.n,), 7, dtype=torch.uint8, device="cuda"), q=src.q, m=src.m)
    a = mk()
    bind.ent_sort(ctx, src, a, None)                      # full sort
    torch.cuda.synchronize()
    assert bind.ent_get_stat(ctx, bind.STAT_LAST_SORT_REBIN) == 0 and bool((a.tag == 1).all())
    notag = bind.Particles(cell=a.cell, d=a.d, u=a.u, w=a.w, phi=None, tag=None, q=a.q, m=a.m)      # the same sorted block, seen without tags
    for _ in range(3):
        bind.ent_step(ctx, F, notag, J, wl.dt)
    b = mk()
    bind.ent_sort(ctx, notag, b, None)                    # re-bin
    torch.cuda.synchronize()
    assert bind.ent_get_stat(ctx, bind.STAT_LAST_SORT_REBIN) == 1 and bool((b.tag == 1).all())
    _match_perm(g, bind.Particles(cell=a.cell, d=a.d, u=a.u, w=a.w, phi=None, tag=b.tag, q=a.q, m=a.m), b)


def test_empty_block_is_accepted(env):
    """n = 0: every call returns ENT_OK and touches nothing (ent.h: n may be any value >= 0)"""
    bind, synth, ctx, orc = env
    wl = synth.config3(16)
    eg = P.grid_to_ent(bind, wl.grid)
    bind.ent_set_grid(ctx, eg)
    F = [f.cuda() for f in wl.fields]
    e = lambda dt: torch.empty(0, dtype=dt, device="cuda")
    mk = lambda: bind.Particles(cell=e(torch.int32), d=[e(torch.float32) for _ in range(3)], u=[e(torch.float32) for _ in range(3)],
                                w=e(torch.float32), q=-1.0, m=1.0)
    p, p2 = mk(), mk()
    J = bind.zeros_current(eg, "cuda")
    bind.ent_step(ctx, F, p, J, wl.dt)
    bind.ent_gather_push(ctx, F, p, p2, wl.dt)
    bind.ent_deposit(ctx, p, p2, J, wl.dt)
    torch.cuda.synchronize()
    assert all(float(j.abs().max()) == 0.0 for j in J)


def test_error_paths_on_device(env):
    """misaligned / missing arrays and mismatched sizes are refused with ENT_EINVAL, nothing is launched"""
    bind, synth, ctx, orc = env
    wl = synth.config3(16)
    g = wl.grid
    eg = P.grid_to_ent(bind, g)
    bind.ent_set_grid(ctx, eg)
    F = [f.cuda() for f in wl.fields]
    pe = P.species_to_ent(bind, synth, g, wl.species[0], "cuda", with_tag=False)
    J = bind.zeros_current(eg, "cuda")
    before = bind.ent_get_stat(ctx, bind.STAT_LAUNCHES)
    bad = pe.clone(); bad.d[1] = torch.zeros(pe.n + 1, dtype=torch.float32, device="cuda")[1:]          # 4-byte aligned only
    with pytest.raises(bind.EntError) as ei:
        bind.ent_step(ctx, F, bad, J, wl.dt)
    assert ei.value.code == bind.EINVAL
    out = pe.empty_like(); out.cell = out.cell[:-1]
    with pytest.raises(bind.EntError):
        bind.ent_sort(ctx, pe, out, None)                                                               # in->n != out->n
    with pytest.raises(bind.EntError):
        bind.ent_sort(ctx, pe, pe, None)                                                                # not out of place
    with pytest.raises(bind.EntError):
        bind.ent_step(ctx, F, pe, J, -1.0)                                                              # dt <= 0
    assert bind.ent_get_stat(ctx, bind.STAT_LAUNCHES) == before


@pytest.mark.parametrize("name,impl,sort_first", [("C1", 0, True), ("C3/8", 0, True), ("C3/8", 1, False), ("C5/32", 0, True), ("ABS3", 0, True)])
def test_vay_pusher_matches_oracle(env, name, impl, sort_first):
    """ENT_OPT_PUSHER = 1 (Vay 2008) against the oracle's orc_vay through the whole step, tiled and untiled kernels"""
    bind, synth, ctx, orc = env
    wl = _workloads(synth)[name]()
    bind.ent_set_option(ctx, bind.OPT_PUSHER, 1)
    orc.set_pusher(1)
    try:
        stats = _run_case(env, wl, impl=impl, sort_first=sort_first, steps=min(wl.steps, 6), resort_every=3 if sort_first else 0)
    finally:
        bind.ent_set_option(ctx, bind.OPT_PUSHER, 0)
        orc.set_pusher(0)
    print(name, "vay", stats)
    assert all(st["max_u_rel"] <= P.MOM_TOL for st in stats.values())


@pytest.mark.parametrize("name,pusher,rho_crit,eovb,sort_first", [("C3/8", 2, 2.0, 0.5, True), ("C3/8", 3, 2.0, 0.5, False),
                                                                   ("C2/4", 2, 0.05, 0.9, True), ("C1", 2, 0.4, 0.3, True)])
def test_hybrid_gca_pusher_matches_oracle(env, name, pusher, rho_crit, eovb, sort_first):
    """ENT_OPT_PUSHER = 2 / 3 ("Boris,GCA" / "Vay,GCA", reading G26) against the oracle with the same thresholds, tiled
    and untiled kernels, Cartesian and quasi-spherical grids.  Both sides start every step from the SAME state (the GPU's): a particle
    whose |E|/|B| or gyroradius sits within fp32 rounding of a threshold takes the other branch on the GPU, which is a different but
    equally valid trajectory, so a handful of such particles per step are allowed to differ and everything else must meet the bars;
    the currents are checked against the oracle's deposit of the GPU's own moves (strict) and by continuity."""
    bind, synth, ctx, orc = env
    wl = _workloads(synth)[name]()
    g = wl.grid
    eg, og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, 0)
    bind.ent_set_grid(ctx, eg)
    bind.ent_set_option(ctx, bind.OPT_PUSHER, pusher)
    bind.ent_set_gca(ctx, rho_crit, eovb)
    orc.set_gca(rho_crit, eovb)
    F_dev, F_orc = [f.cuda() for f in wl.fields], P.fields_to_orc(wl.fields)
    try:
        for sp in wl.species[:1]:
            pe = P.species_to_ent(bind, synth, g, sp, "cuda")
            if sort_first:
                ps = pe.empty_like()
                bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 1)
                bind.ent_sort(ctx, pe, ps, None)
                bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 0)
                pe = ps
            Jg = bind.zeros_current(eg, "cuda")
            fracs = []
            for s in range(3):
                before = P.ent_to_orc(orc, g, pe)
                bind.ent_zero_current(ctx, Jg)
                bind.ent_step(ctx, F_dev, pe, Jg, wl.dt)
                bind.ent_fold_current(ctx, Jg)
                torch.cuda.synchronize()
                assert bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED) == (1 if sort_first else 0)
                after = P.ent_to_orc(orc, g, pe)
                orc.set_pusher(pusher)
                want = orc.gather_push(og, F_orc, before, sp.q / sp.m, wl.dt)
                orc.set_pusher(pusher & 1)
                conv = orc.gather_push(og, F_orc, before, sp.q / sp.m, wl.dt)          # the conventional pusher alone: who was in the regime?
                ug, uo, uc = np.stack(after.u), np.stack(want.u), np.stack(conv.u)
                alive = (want.tag != 0) & (after.tag != 0) if want.tag is not None else np.ones(ug.shape[1], bool)
                fracs.append(float((np.abs(uo - uc).max(axis=0) > 1e-9)[alive].mean()))
                umag = np.sqrt((uo * uo).sum(axis=0))
                floor = P.U_FLOOR_FRAC * np.sqrt((umag * umag).mean())
                bad_u = np.abs(ug - uo).max(axis=0) / np.maximum(umag, floor) > P.MOM_TOL
                bad_x = np.zeros_like(bad_u)
                for a in range(g.D):
                    diff = (after.i[a] + after.d[a]) - (want.i[a] + want.d[a])
                    if g.bc[a] == synth.PERIODIC:
                        diff = diff - g.N[a] * np.round(diff / g.N[a])
                    bad_x |= np.abs(diff) > P.POS_TOL
                nbad = int(((bad_u | bad_x) & alive).sum())
                allowed = 10 + int(1e-4 * pe.n)
                print(name, "pusher", pusher, "step", s, "in the guiding-centre regime:", fracs[-1], " threshold straddlers:", nbad, "of", pe.n)
                assert nbad <= allowed
                if want.tag is not None:
                    assert int((want.tag != after.tag).sum()) <= allowed
                strict = P.compare_current(Jg, P.deposit_of_gpu_positions(orc, og, before, after, sp.q, wl.dt))
                c = P.continuity_of_gpu_step(orc, og, before, after, Jg, sp.q, wl.dt)
                assert c <= P.CONT_TOL
            assert 0.02 < np.mean(fracs) < 0.98, "the case must exercise both regimes"
    finally:
        bind.ent_set_option(ctx, bind.OPT_PUSHER, 0)
        bind.ent_set_gca(ctx, 0.0, 0.0)
        orc.set_pusher(0); orc.set_gca(0.0, 0.0)


@pytest.mark.parametrize("name", ["ABS3", "C5/32", "C1"])
def test_compact_matches_oracle(env, name):
    """ent_compact (tag sort) after a few steps on grids that lose particles (and one that does not): bit-exact against the
    oracle's stable partition of the same block -- every array, the tags and the count"""
    bind, synth, ctx, orc = env
    wl = _workloads(synth)[name]()
    g = wl.grid
    eg = P.grid_to_ent(bind, g)
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, 0)
    bind.ent_set_grid(ctx, eg)
    F = [f.cuda() for f in wl.fields]
    J = bind.zeros_current(eg, "cuda")
    pe = P.species_to_ent(bind, synth, g, wl.species[0], "cuda")
    for _ in range(5):
        bind.ent_step(ctx, F, pe, J, wl.dt)
    out = pe.empty_like()
    na = bind.ent_compact(ctx, pe, out)
    torch.cuda.synchronize()
    want, na_o = orc.compact(P.ent_to_orc(orc, g, pe))
    assert int(na.item()) == na_o
    if name != "C1":
        assert 0 < na_o < pe.n
    got = P.ent_to_orc(orc, g, out)
    for a, b in zip(got.i + got.d + got.u + [got.w, got.tag] + ([got.phi] if got.phi is not None else []),
                    want.i + want.d + want.u + [want.w, want.tag] + ([want.phi] if want.phi is not None else [])):
        assert np.array_equal(a, b)
    # the alive head of the compacted block is a block of its own: sort it and step it (n = number alive)
    head = bind.Particles(cell=out.cell[:na_o], d=[t[:na_o] for t in out.d], u=[t[:na_o] for t in out.u], w=out.w[:na_o],
                          phi=None if out.phi is None else out.phi[:na_o], tag=out.tag[:na_o], q=out.q, m=out.m)
    srt = head.clone()
    bind.ent_sort(ctx, head, srt, None)
    bind.ent_step(ctx, F, srt, J, wl.dt)
    torch.cuda.synchronize()
    assert bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED) == 1


@pytest.mark.parametrize("forced", [True, False])
@pytest.mark.parametrize("name", ["C1", "C3/8", "C3/8-uneven", "C4/16-shuffled", "ABS3", "ABS2", "PER3"])
def test_step_pair_matches_oracle(env, name, forced):
    """ent_step_pair: both species of the pair plasma through one launch of the tiled kernel (one E,B box, one J tile per tile).
    Same bars as the single-species tests: the summed current of the two species against the oracle's, particles per species,
    continuity of the GPU's own output; blocks re-binned every 3 steps."""
    bind, synth, ctx, orc = env
    uneven = name.endswith("-uneven")
    wl = _workloads(synth)[name.replace("-uneven", "")]()
    if uneven:         # species of different size, charge-to-mass ratio and weight scale: one fixed-point scale serves both
        sp = wl.species[1]
        keep = torch.arange(sp.n) % 3 != 0
        wl.species[1] = synth.Species(q=2.0 * sp.q, m=3.0 * sp.m, i=[t[keep] for t in sp.i], d=[t[keep] for t in sp.d],
                                      u=[t[keep] for t in sp.u], w=7.3 * sp.w[keep])
    g = wl.grid
    eg, og = P.grid_to_ent(bind, g), P.grid_to_orc(orc, g)
    # these grids have fewer than 444 tiles: ENT_OPT_STEP_IMPL = 3 asks for the one-launch form, 0 takes two work-list launches
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, 3 if forced else 0)
    bind.ent_set_grid(ctx, eg)
    F_dev, F_orc = [f.cuda() for f in wl.fields], P.fields_to_orc(wl.fields)
    assert len(wl.species) == 2
    pes, pos, orders = [], [], []
    bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 1)
    for sp in wl.species:
        pe = P.species_to_ent(bind, synth, g, sp, "cuda")
        ps = pe.empty_like()
        bind.ent_sort(ctx, pe, ps, None)
        orders.append(_match_perm(g, pe, ps)); pes.append(ps); pos.append(P.species_to_orc(orc, sp))
    bind.ent_set_option(ctx, bind.OPT_SORT_MODE, 0)
    Jg = bind.zeros_current(eg, "cuda")
    steps = min(wl.steps, 8)
    worstJ = worstC = 0.0
    for s in range(steps):
        if s > 0 and s % 3 == 0:
            for k in range(2):
                ps = pes[k].empty_like()
                bind.ent_sort(ctx, pes[k], ps, None)
                assert bind.ent_get_stat(ctx, bind.STAT_LAST_SORT_REBIN) == 1
                orders[k] = orders[k][_match_perm(g, pes[k], ps)]
                pes[k] = ps
        before = [P.ent_to_orc(orc, g, pe) for pe in pes]
        bind.ent_zero_current(ctx, Jg)
        bind.ent_step_pair(ctx, F_dev, pes[0], pes[1], Jg, wl.dt)
        bind.ent_fold_current(ctx, Jg)
        torch.cuda.synchronize()
        assert bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED) == 1
        after = [P.ent_to_orc(orc, g, pe) for pe in pes]
        Jo = orc.zeros_current(og)
        Jown = orc.zeros_current(og)                       # the oracle's deposit of the GPU's own stored moves (strict, no allowance)
        for k, sp in enumerate(wl.species):
            po_before = pos[k].copy()
            orc.step(og, F_orc, pos[k], Jo, sp.q, sp.m, wl.dt)
            _, corr = P.straddler_correction(orc, g, og, po_before, pos[k], before[k], after[k], sp.q, wl.dt, orders[k])
            if corr is not None:
                Jo = [a + b for a, b in zip(Jo, corr)]
            own = P.deposit_of_gpu_positions(orc, og, before[k], after[k], sp.q, wl.dt, fold=False)
            Jown = [a + b for a, b in zip(Jown, own)]
        orc.fold_current(og, Jo)
        orc.fold_current(og, Jown)
        worstJ = max(worstJ, P.compare_current(Jg, Jo), P.compare_current(Jg, Jown))
        c = P.continuity_of_gpu_steps(orc, og, before, after, Jg, [sp.q for sp in wl.species], wl.dt)
        assert c <= P.CONT_TOL, f"continuity residual {c:.3e} at step {s}"
        worstC = max(worstC, c)
    for k in range(2):
        st = P.compare_particles(g, pes[k], pos[k], orders[k], steps=steps)
        assert st["tag_mismatch"] == 0
    assert bind.ent_get_stat(ctx, bind.STAT_BAD_MOVES) == 0
    print(name, "pair: max|dJ|/max|J| =", worstJ, " continuity", worstC)
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, 0)
    assert worstJ <= P.J_TOL
