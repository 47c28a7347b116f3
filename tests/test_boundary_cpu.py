"""CPU-side checks of the boundary: libent.so builds (nvcc cross-compiles sm_100a without a GPU), loads, exports every
symbol include/ent.h declares, and refuses to work without a CUDA device (no CPU fallback).  Plus the seeded input
generator (counter-based RNG) against a pure-Python restatement, and the host index helpers."""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    txt = open(os.path.join(ROOT, "include", "ent.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(ent_[a-z_]+)\s*\(", txt)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2511_17710_b200 import build, binding
    path = build.build()
    lib = ctypes.CDLL(path)
    syms = _declared_symbols()
    assert len(syms) >= 14
    for s in syms:
        assert hasattr(lib, s), f"{s} is declared in include/ent.h but not exported by libent.so"
    assert set(binding.SYMBOLS) == set(syms), "binding.py and ent.h disagree on the entry points"
    assert binding.ent_version().count(".") == 1


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback_without_a_device():
    from paper_2511_17710_b200 import binding
    with pytest.raises(binding.EntError):
        binding.ent_create(0, None)


def test_sm100a_code_is_in_the_library():
    from paper_2511_17710_b200 import build
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def _splitmix_ref(seed, stream, index):
    M = (1 << 64) - 1
    z = (seed * 0x9E3779B97F4A7C15 + (stream << 40) + index) & M
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
    return z ^ (z >> 31)


def test_counter_rng_matches_python_integers():
    from paper_2511_17710_b200 import synth
    for seed, stream in [(0, 0), (3, 7), (4, 21)]:
        bits = synth.rand_bits(seed, stream, 1000, "cpu", start=123456789)
        u32 = synth.uniform(seed, stream, 1000, "cpu", start=123456789)
        u64 = synth.uniform(seed, stream, 1000, "cpu", start=123456789, dtype=torch.float64)
        for k in (0, 1, 17, 999):
            ref = _splitmix_ref(seed, stream, 123456789 + k)
            assert (int(bits[k]) & ((1 << 64) - 1)) == ref
            assert float(u32[k]) == (ref >> 40) * 2.0 ** -24
            assert float(u64[k]) == (ref >> 11) * 2.0 ** -53
    u = synth.uniform(1, 2, 200000, "cpu", dtype=torch.float64)
    assert abs(float(u.mean()) - 0.5) < 5e-3 and 0.0 <= float(u.min()) and float(u.max()) < 1.0


def test_pack_unpack_and_sort_key_are_consistent():
    from paper_2511_17710_b200 import synth
    g = synth.GridSpec(D=3, N=(10, 7, 5), bc=(0, 0, 0))
    cell = torch.arange(g.ncells, dtype=torch.int32)
    i = synth.unpack_cell(g, cell)
    assert torch.equal(synth.pack_cell(g, i), cell)
    key = synth.sort_key(g, i, (4, 4, 2))
    assert len(torch.unique(key)) == g.ncells                       # injective
    nt = (3, 2, 3)
    assert int(key.max()) < nt[0] * nt[1] * nt[2] * 32


def test_workload_recipes_have_the_stated_shape():
    from paper_2511_17710_b200 import synth
    w = synth.config1()
    assert w.grid.N == (64, 64) and w.nparticles == 65536 and abs(w.dt - 0.225) < 1e-15
    assert [s.q for s in w.species] == [-1.0, 1.0]
    assert torch.equal(w.species[0].d[0], w.species[1].d[0])          # pairs created on top of each other
    w = synth.config2(4)
    assert w.grid.kind == synth.QSPH and w.grid.vartheta == 0.0 and w.grid.bc == (synth.ABSORB, synth.AXIS)
    n_in = sum(int((s.i[0] < 8).sum()) for s in w.species)
    n_out = sum(int((s.i[0] >= 56).sum()) for s in w.species)
    assert n_in > 20 * n_out                                          # density ~ r^-2 on a log-r grid
    w = synth.config4(32)
    ux = w.species[0].u[0]
    assert float(ux[0::2].mean()) > 0.3 and float(ux[1::2].mean()) < -0.3   # two counter-streaming beams
    for f in synth.config5(64).fields:
        assert torch.isfinite(f).all()


def _build_abi_check(tmp_path):
    """tests/c/abi_check.c compiled with gcc against include/ent.h and linked with libent.so: the ABI is usable from plain C"""
    import subprocess
    from paper_2511_17710_b200 import build
    lib = build.build()
    exe = str(tmp_path / "abi_check")
    subprocess.check_call(["gcc", "-std=c11", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), os.path.join(ROOT, "tests", "c", "abi_check.c"),
                           "-o", exe, lib, "-Wl,-rpath," + os.path.dirname(lib)])
    return exe


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_c_program_against_the_abi_without_a_device(tmp_path):
    import subprocess
    r = subprocess.run([_build_abi_check(tmp_path)], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and "no device" in r.stdout, (r.stdout, r.stderr)


@pytest.mark.gpu
def test_c_program_against_the_abi_on_the_gpu(tmp_path):
    import subprocess
    r = subprocess.run([_build_abi_check(tmp_path)], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "abi ok" in r.stdout, (r.stdout, r.stderr)
