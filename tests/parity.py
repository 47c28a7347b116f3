"""Parity plumbing shared by the GPU tests, smoke() and nothing else: packs one seeded synthetic workload for the CUDA
library (binding.Particles, fp32 on the device) and for the fp64 oracle (orc.Particles, numpy), and compares results
with the rules of DESIGN.md "parity definition".  No arithmetic of the method lives here.
"""
from __future__ import annotations

import numpy as np
import torch

POS_TOL = 1e-5          # |delta(i + d)| in cells (BASELINE.json: positions within 1e-5)
MOM_TOL = 1e-5          # |delta u|_inf / max(|u|_2, U_FLOOR_FRAC * rms|u|)  (BASELINE.json: momenta within a relative error of 1e-5)
U_FLOOR_FRAC = 0.1      # a gyrating / drifting particle swings through |u| ~ 0 while its rounding errors scale with the swing
J_TOL = 1e-5            # max|J_gpu - J_orc| / max|J_orc|
CONT_TOL = 1e-6         # continuity residual / normaliser
FACE_EPS = 1e-5         # oracle offsets closer than this to a face are "straddlers" (G12)
PHI_ULP = 2.0 ** -22    # half an ulp of an fp32 azimuth in [4, 2 pi): what storing phi in fp32 (real_t phi) costs per step
OFFSET_ULP = 2.0 ** -23  # ulp of an fp32 in-cell offset in [0.5, 1) (prtldx_t = float)


def species_to_ent(bind, synth, grid, sp, device, with_tag=True):
    """synth.Species -> binding.Particles on `device` (packed linear cell index, fp32)"""
    dev = torch.device(device)
    mv = lambda t: t.to(dev).contiguous()
    return bind.Particles(cell=mv(synth.pack_cell(grid, sp.i)), d=[mv(t) for t in sp.d], u=[mv(t) for t in sp.u], w=mv(sp.w),
                          phi=None if sp.phi is None else mv(sp.phi),
                          tag=torch.ones(sp.n, dtype=torch.uint8, device=dev) if with_tag else None, q=sp.q, m=sp.m)


def species_to_orc(orc, sp):
    """synth.Species -> orc.Particles (int32 indices per dimension, float64 copies of the SAME fp32 values)"""
    f64 = lambda t: np.ascontiguousarray(t.detach().cpu().numpy().astype(np.float64))
    return orc.Particles(i=[np.ascontiguousarray(t.detach().cpu().numpy().astype(np.int32)) for t in sp.i],
                         d=[f64(t) for t in sp.d], u=[f64(t) for t in sp.u], w=f64(sp.w),
                         phi=None if sp.phi is None else f64(sp.phi), tag=np.ones(sp.n, dtype=np.int8))


def grid_to_ent(bind, g):
    return bind.Grid(D=g.D, N=tuple(g.N), bc=tuple(g.bc), kind=g.kind, xmin=tuple(g.xmin), xmax=tuple(g.xmax), r0=g.r0,
                     vartheta=g.vartheta)


def grid_to_orc(orc, g):
    return orc.Grid(D=g.D, N=tuple(g.N), bc=tuple(g.bc), kind=g.kind, xmin=tuple(g.xmin), xmax=tuple(g.xmax), r0=g.r0,
                    vartheta=g.vartheta)


def fields_to_orc(fields):
    return [np.ascontiguousarray(f.detach().cpu().numpy()) for f in fields]


def unpack_cell_np(grid, cell):
    c = cell.astype(np.int64)
    N0, N1 = int(grid.N[0]), int(grid.N[1])
    if grid.D == 2:
        return [c % N0, c // N0]
    return [c % N0, (c // N0) % N1, c // (N0 * N1)]


def compare_particles(grid, pe, po, order=None, steps=1, orc_metric=None):
    """pe: binding.Particles (any device), po: orc.Particles.  `order`: optional index array such that GPU particle k is
    oracle particle order[k] (after a sort).  `steps`: steps taken since the two states were equal (enters only the
    fp32-storage allowance of phi).  `orc_metric`: (orc module, orc grid), needed on the axisymmetric grids (the azimuth error is
    measured as an arc with the ORACLE's metric).  Returns a dict of maxima and counts; raises AssertionError on a violation."""
    cell = pe.cell.detach().cpu().numpy()
    ig = unpack_cell_np(grid, cell)
    sel = (lambda a: a) if order is None else (lambda a: a[order])
    tag_g = np.ones(cell.shape[0], dtype=bool) if pe.tag is None else pe.tag.detach().cpu().numpy() != 0
    tag_o = np.ones(cell.shape[0], dtype=bool) if po.tag is None else sel(po.tag) != 0
    both = tag_g & tag_o
    stats = {"n": int(cell.shape[0]), "alive": int(both.sum()), "tag_mismatch": int((tag_g != tag_o).sum()), "straddlers": 0,
             "max_pos_err": 0.0, "max_u_rel": 0.0, "max_phi_err": 0.0}
    strad_any = np.zeros(cell.shape[0], dtype=bool)
    PERIODIC = 0
    for a in range(grid.D):
        dg = pe.d[a].detach().cpu().numpy().astype(np.float64)
        io, do = sel(po.i[a]).astype(np.int64), sel(po.d[a])
        assert np.all((dg >= 0.0) & (dg < 1.0)), f"GPU offset outside [0,1) in dimension {a}"
        strad = np.minimum(do, 1.0 - do) <= FACE_EPS
        strad_any |= strad & both
        ok = both & ~strad
        assert np.array_equal(ig[a][ok], io[ok]), (
            f"cell index mismatch in dimension {a} for {int((ig[a][ok] != io[ok]).sum())} non-straddling particles")
        diff = (ig[a] + dg) - (io + do)
        if grid.bc[a] == PERIODIC:
            N = int(grid.N[a])
            diff = diff - N * np.round(diff / N)
        err = np.abs(diff[both])
        if err.size:
            stats["max_pos_err"] = max(stats["max_pos_err"], float(err.max()))
    stats["straddlers"] = int(strad_any.sum())
    ug = np.stack([t.detach().cpu().numpy().astype(np.float64) for t in pe.u])
    uo = np.stack([sel(t) for t in po.u])
    umag = np.sqrt((uo * uo).sum(axis=0))
    rel = np.abs(ug - uo).max(axis=0) / np.maximum(umag, U_FLOOR_FRAC * np.sqrt((umag * umag).mean()) + 1e-300)
    rel = rel[both]
    if rel.size:
        stats["max_u_rel"] = float(rel.max())
    if pe.phi is not None:
        # azimuth: phi is ill-conditioned near the axis (d phi = d x / (r sin theta)), so its
        # error is measured as the ARC it spans in units of the theta-cell, sqrt(h33) |d phi| / sqrt(h22) <= POS_TOL like the
        # other two coordinates, on top of what storing phi as an fp32 in [0, 2 pi) costs (half an ulp per step).
        assert orc_metric is not None, "compare_particles on an axisymmetric grid needs orc_metric=(orc, og)"
        dphi = pe.phi.detach().cpu().numpy().astype(np.float64) - sel(po.phi)
        dphi = dphi - 2.0 * np.pi * np.round(dphi / (2.0 * np.pi))
        h = orc_metric[0].metric_h_many(orc_metric[1], sel(po.i[0]).astype(np.float64) + sel(po.d[0]),
                                        sel(po.i[1]).astype(np.float64) + sel(po.d[1]))
        arc = (np.abs(dphi) - steps * PHI_ULP).clip(min=0.0) * np.sqrt(h[:, 2] / h[:, 1])
        if both.any():
            stats["max_phi_err"] = float(np.abs(dphi[both]).max())
            stats["max_phi_arc_cells"] = float(arc[both].max())
        assert stats.get("max_phi_arc_cells", 0.0) <= POS_TOL, stats
    assert stats["max_pos_err"] <= POS_TOL, stats
    assert stats["max_u_rel"] <= MOM_TOL, stats
    # a tag can only differ for a particle that straddles an absorbing face
    assert stats["tag_mismatch"] <= stats["straddlers"], stats
    return stats


def compare_current(Jg, Jo, fmt_bound=None):
    """Jg: list of 3 torch tensors (after fold), Jo: list of 3 float64 numpy arrays (after fold).
    BASELINE.json's bar: |J_gpu - J_orc| <= 1e-5 max|J| at every element.  fmt_bound (optional, 3 padded arrays): what the
    fp32 particle FORMAT itself allows at each element (see offset_format_bound); an element may exceed the bar by that.
    Returns max over elements of (error - allowance) / max|J|, asserted <= J_TOL; compare_current.last_raw holds the RAW
    max|J_gpu - J_orc| / max|J_orc| of the same call (no allowance subtracted), which the tests print beside it."""
    scale = max(float(np.abs(j).max()) for j in Jo)
    worst = raw = 0.0
    for c, (g, o) in enumerate(zip(Jg, Jo)):
        e = np.abs((g.detach().cpu().numpy().astype(np.float64) if torch.is_tensor(g) else g) - o)
        raw = max(raw, float(e.max()))
        if fmt_bound is not None:
            e = (e - fmt_bound[c]).clip(min=0.0)
        worst = max(worst, float(e.max()))
    rel = worst / scale if scale > 0 else worst
    compare_current.last_raw = raw / scale if scale > 0 else raw
    assert rel <= J_TOL, f"max|J_gpu - J_orc| / max|J_orc| = {rel:.3e} (raw {compare_current.last_raw:.3e}, scale {scale:.3e})"
    return rel


compare_current.last_raw = 0.0


def deposit_of_gpu_positions(orc, og, p_before, p_after, q, dt, fold=True):
    """The STRICT current check (no allowance): the oracle's deposit fed with the GPU's own stored positions before and after the
    step (fp32 values up-cast) and the GPU's new momenta.  Whatever the push did, the GPU's J must equal this to J_TOL * max|J|:
    it isolates sub-step 8 from the conditioning of sub-steps 3-7.  Returns 3 padded float64 arrays."""
    J = orc.zeros_current(og)
    orc.deposit(og, p_before, p_after, J, q, dt)
    if fold:
        orc.fold_current(og, J)
    return J


def straddler_correction(orc, grid, og, po_before, po_after, pe_before, pe_after, q, dt, order=None):
    """The zig-zag path of P:575 is DISCONTINUOUS in the crossing decision: a particle that starts or ends within rounding of a cell
    face is routed through the face (relay on the face) if it crossed and through the midpoint if it did not, and the two paths
    put a single-particle-sized amount of current on different nodes (both conserve charge).  fp32 and fp64 take that decision
    differently for a few particles per million per step (the straddlers of reading G12 / F3).  For exactly those particles --
    cell index before or after the step differing between the GPU and the oracle while the real positions agree (compare_particles
    checks that) -- the oracle's current is re-evaluated on the GPU's stored positions; returns (number of such particles,
    3 padded arrays to ADD to the oracle's folded current, or None).  pe_before / pe_after: orc.Particles built from the GPU arrays
    (ent_to_orc), in GPU slot order; order[k] = oracle index of GPU slot k."""
    n = po_before.n
    sel = np.arange(n) if order is None else np.asarray(order)
    inv = np.empty(n, dtype=np.int64); inv[sel] = np.arange(n)          # oracle particle j sits in GPU slot inv[j]
    mism = np.zeros(n, dtype=bool)
    for a in range(grid.D):
        mism |= (pe_after.i[a][inv] != po_after.i[a]) | (pe_before.i[a][inv] != po_before.i[a])
    alive = np.ones(n, dtype=bool)
    for p, g in ((po_after, False), (po_before, False), (pe_after, True), (pe_before, True)):
        if p.tag is not None:
            alive &= (p.tag[inv] if g else p.tag) != 0
    idx = np.nonzero(mism & alive)[0]
    if idx.size == 0:
        return 0, None
    take = lambda p, ii: orc.Particles(i=[np.ascontiguousarray(a[ii]) for a in p.i], d=[np.ascontiguousarray(a[ii]) for a in p.d],
                                       u=[np.ascontiguousarray(a[ii]) for a in p.u], w=np.ascontiguousarray(p.w[ii]),
                                       phi=None if p.phi is None else np.ascontiguousarray(p.phi[ii]), tag=None)
    Jp, Jm = orc.zeros_current(og), orc.zeros_current(og)
    orc.deposit(og, take(pe_before, inv[idx]), take(pe_after, inv[idx]), Jp, q, dt)
    orc.deposit(og, take(po_before, idx), take(po_after, idx), Jm, q, dt)
    orc.fold_current(og, Jp); orc.fold_current(og, Jm)
    return int(idx.size), [a - b for a, b in zip(Jp, Jm)]


def _box3(a):
    b = np.zeros_like(a)
    for s2 in (-1, 0, 1):
        for s1 in (-1, 0, 1):
            b += np.roll(np.roll(a, s2, axis=0), s1, axis=1)
    return b


def offset_format_bound(orc, grid, og, p_before, q, dt):
    """Per-element allowance for J on the curvilinear grids; returns 3 padded arrays.
    The new in-cell offset is stored as fp32, i.e. rounded by up to OFFSET_ULP/2.  The GPU deposits the move between
    STORED positions (which is what keeps Eq. 6 exact), the fp64 oracle the unrounded one, so however well the move itself
    was computed
      * one particle's in-plane current differs by up to |q| w / dt * OFFSET_ULP: where the move per step is ~1e-3 cells
        (outer radii of the log-r grids) that alone is 1e-5..1e-4 of the particle's current;
      * its out-of-plane current q w v^3 ~ 1/sqrt(h33) = 1/(r sin theta) (reading G8) differs by the relative amount
        |d ln sin(theta) / d x2| * OFFSET_ULP = |cos theta| sqrt(h22)/sqrt(h33) * OFFSET_ULP, unbounded toward the axis.
    The allowance at an element is that figure summed over the particles within one cell of it (3x3 box sum of a nodal
    deposit; the in-plane one is the oracle's charge_density of |q| w)."""
    inplane = _box3(orc.charge_density(og, p_before, abs(q))) * (OFFSET_ULP / dt)
    x1 = p_before.i[0].astype(np.float64) + p_before.d[0]
    x2 = p_before.i[1].astype(np.float64) + p_before.d[1]
    h = orc.metric_h_many(og, x1, x2)                                    # the ORACLE's metric
    # d sqrt(h33) / d x2 by a centred difference of the oracle's own h33: no second statement of the metric in the tests
    eps = 1e-4
    dh3 = (np.sqrt(orc.metric_h_many(og, x1, x2 + eps)[:, 2]) - np.sqrt(orc.metric_h_many(og, x1, x2 - eps)[:, 2])) / (2 * eps)
    h3 = np.maximum(np.sqrt(h[:, 2]), 1e-300)
    per = abs(q) * p_before.w / h3 * (np.abs(dh3) / h3) * OFFSET_ULP     # |v^phi-hat| <= 1; |d ln sqrt(h33) / d x2| per offset ulp
    if p_before.tag is not None:
        per = per * (p_before.tag != 0)
    out3 = np.zeros(inplane.shape, dtype=np.float64)
    np.add.at(out3, (p_before.i[1].astype(np.int64) + 2, p_before.i[0].astype(np.int64) + 2), per)
    out3 = _box3(_box3(out3))
    return [inplane, inplane, out3]


def continuity_of_gpu_step(orc, og, p_before, p_after, Jg_folded, q, dt):
    """Eq. 6 on the GPU's own output: the oracle's CHECKER is applied to the GPU positions and currents.
    p_before / p_after: orc.Particles built from the GPU arrays (fp32 values up-cast).  Returns residual / normaliser."""
    alive = np.ones(p_before.n, dtype=np.int8)
    if p_before.tag is not None:
        alive &= (p_before.tag != 0).astype(np.int8)
    if p_after.tag is not None:
        alive &= (p_after.tag != 0).astype(np.int8)
    rho0 = orc.charge_density(og, p_before, q, mask=alive)
    rho1 = orc.charge_density(og, p_after, q, mask=alive)
    norm = orc.charge_density(og, p_before, abs(q), mask=alive)
    J = [np.ascontiguousarray(j.detach().cpu().numpy().astype(np.float64)) for j in Jg_folded]
    orc.fold_scalar(og, rho0); orc.fold_scalar(og, rho1); orc.fold_scalar(og, norm)
    res = orc.continuity_residual(og, J, rho0, rho1, dt)
    scale = float(np.abs(norm).max()) / dt
    return res / scale if scale > 0 else res


def continuity_of_gpu_steps(orc, og, befores, afters, Jg_folded, qs, dt):
    """continuity_of_gpu_step for several species that deposited into the same J (ent_step_pair): the charge arrays are summed"""
    rho0 = rho1 = norm = None
    for pb, pa, q in zip(befores, afters, qs):
        alive = np.ones(pb.n, dtype=np.int8)
        if pb.tag is not None:
            alive &= (pb.tag != 0).astype(np.int8)
        if pa.tag is not None:
            alive &= (pa.tag != 0).astype(np.int8)
        rho0 = orc.charge_density(og, pb, q, mask=alive, rho=rho0)
        rho1 = orc.charge_density(og, pa, q, mask=alive, rho=rho1)
        norm = orc.charge_density(og, pb, abs(q), mask=alive, rho=norm)
    J = [np.ascontiguousarray(j.detach().cpu().numpy().astype(np.float64)) for j in Jg_folded]
    orc.fold_scalar(og, rho0); orc.fold_scalar(og, rho1); orc.fold_scalar(og, norm)
    res = orc.continuity_residual(og, J, rho0, rho1, dt)
    scale = float(np.abs(norm).max()) / dt
    return res / scale if scale > 0 else res


def ent_to_orc(orc, grid, pe):
    """binding.Particles (GPU result) -> orc.Particles holding the same values (for the continuity checker)"""
    cell = pe.cell.detach().cpu().numpy()
    i = [np.ascontiguousarray(a.astype(np.int32)) for a in unpack_cell_np(grid, cell)]
    f64 = lambda t: np.ascontiguousarray(t.detach().cpu().numpy().astype(np.float64))
    return orc.Particles(i=i, d=[f64(t) for t in pe.d], u=[f64(t) for t in pe.u], w=f64(pe.w),
                         phi=None if pe.phi is None else f64(pe.phi),
                         tag=None if pe.tag is None else np.ascontiguousarray(pe.tag.detach().cpu().numpy().astype(np.int8)))
