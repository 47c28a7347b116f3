"""ent_compact_static (include/ent.h): the tag sort of P:667-669 for callers that cannot allocate device memory.  Its scratch is a
static __device__ array inside the library (ENT_COMPACT_STATIC_MAX_N = 2^20 particles, 12.6 MB), its address taken once per device
with cudaGetSymbolAddress.  Checked here against the existing path, ent_compact (itself bit-exact against the oracle in
test_gpu_parity.py), bit for bit -- the bar of every tag-sort test -- on two calls in a row that share the array: a large block
first, then a smaller one with another pattern of dead particles, so that stale contents of the array would show.

This file is collected last on purpose (pytest -x: a failure here hides no other test) and passes alone in a
fresh process as well as after the other tests: it creates its own ctx and warms nothing up outside itself."""
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    from paper_2511_17710_b200 import binding as bind, synth
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback for the product path")
    ctx = bind.ent_create(0, None)
    yield bind, synth, ctx
    bind.ent_destroy(ctx)


def _block(bind, g, n, seed, dead_every, phi=False):
    """n seeded records on grid g with every `dead_every`-th-ish particle dead (pattern drawn from the seed)"""
    gen = torch.Generator().manual_seed(seed)
    ncell = 1
    for a in range(g.D):
        ncell *= g.N[a]
    r = lambda: torch.rand(n, generator=gen, dtype=torch.float32).cuda()
    cell = torch.randint(0, ncell, (n,), generator=gen, dtype=torch.int32).cuda()
    tag = (torch.randint(0, dead_every, (n,), generator=gen) != 0).to(torch.uint8).cuda()
    return bind.Particles(cell=cell, d=[r() for _ in range(g.D)], u=[r() - 0.5 for _ in range(3)], w=r() + 0.5,
                          phi=r() if phi else None, tag=tag, q=-1.0, m=1.0)


def _same(a, b):
    assert torch.equal(a.cell, b.cell) and torch.equal(a.w, b.w) and torch.equal(a.tag, b.tag)
    assert all(torch.equal(x, y) for x, y in zip(a.d + a.u, b.d + b.u))
    assert (a.phi is None and b.phi is None) or torch.equal(a.phi, b.phi)


def test_compact_static_matches_ent_compact_on_two_calls_in_a_row(env):
    bind, synth, ctx = env
    g = synth.GridSpec(D=3, N=(24, 16, 12), bc=(synth.ABSORB, synth.PERIODIC, synth.ABSORB), kind=synth.CART, xmin=(0.0,) * 3,
                       xmax=(12.0, 8.0, 6.0))
    bind.ent_set_grid(ctx, bind.Grid(D=g.D, N=tuple(g.N), bc=tuple(g.bc), kind=g.kind, xmin=tuple(g.xmin), xmax=tuple(g.xmax),
                                     r0=g.r0, vartheta=g.vartheta))
    # several scan chunks and a ragged tail; the second block is smaller, so the array still holds the first call's tail
    blocks = [_block(bind, g, 700_001, 11, 3), _block(bind, g, 150_003, 12, 7)]
    # the existing path first: reference results (it allocates its own heap scratch on first use)
    want = []
    for b in blocks:
        o = b.empty_like()
        na = bind.ent_compact(ctx, b, o)
        want.append((o, na))
    # everything the static calls touch is allocated by now: inputs, outputs, the counters
    outs = [b.empty_like() for b in blocks]
    nas = [torch.full((1,), -1, dtype=torch.int64, device="cuda") for _ in blocks]
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for b, o, na in zip(blocks, outs, nas):              # two calls in a row, no synchronisation between them
        bind.ent_compact_static(ctx, b, o, na)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    for (wo, wna), o, na, b in zip(want, outs, nas, blocks):
        assert int(na.item()) == int(wna.item()) == int(b.tag.sum().item())
        assert 0 < int(na.item()) < b.n
        _same(o, wo)
    assert free_after >= free_before, "device memory was allocated during ent_compact_static"


def test_compact_static_refuses_blocks_beyond_its_maximum(env):
    bind, synth, ctx = env
    g = synth.GridSpec(D=2, N=(64, 64), bc=(synth.PERIODIC, synth.PERIODIC), kind=synth.CART, xmin=(0.0,) * 3, xmax=(32.0, 32.0, 1.0))
    bind.ent_set_grid(ctx, bind.Grid(D=g.D, N=tuple(g.N), bc=tuple(g.bc), kind=g.kind, xmin=tuple(g.xmin), xmax=tuple(g.xmax),
                                     r0=g.r0, vartheta=g.vartheta))
    n = bind.COMPACT_STATIC_MAX_N + 4
    b = _block(bind, g, n, 13, 5)
    o = b.empty_like()
    keep = o.cell.clone()
    na = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    with pytest.raises(bind.EntError) as ei:
        bind.ent_compact_static(ctx, b, o, na)
    assert ei.value.code == -1 and "ENT_COMPACT_STATIC_MAX_N" in str(ei.value)
    torch.cuda.synchronize()
    assert int(na.item()) == -1 and torch.equal(o.cell, keep)          # nothing was launched
    # exactly the maximum is accepted and agrees with the existing path
    bmax = bind.Particles(cell=b.cell[:-4], d=[t[:-4] for t in b.d], u=[t[:-4] for t in b.u], w=b.w[:-4], phi=None, tag=b.tag[:-4],
                          q=b.q, m=b.m)
    o1, o2 = bmax.empty_like(), bmax.empty_like()
    want = bind.ent_compact(ctx, bmax, o1)
    bind.ent_compact_static(ctx, bmax, o2, na)
    torch.cuda.synchronize()
    assert int(na.item()) == int(want.item())
    _same(o2, o1)
