"""paper_2511_17710_b200 -- B200-native particle hot path of arXiv 2511.17710 (Entity, special-relativistic PIC).

The product is the CUDA library `libent.so` (csrc/, C ABI in include/ent.h).  This package holds only
  build    -- the nvcc command that builds it in-tree for sm_100a,
  binding  -- a thin ctypes binding with the C ABI's names (argument marshalling only),
  synth    -- seeded synthetic inputs shaped like the paper's workloads (no method arithmetic).
There is no CPU fallback: importing `binding` without a built library, or creating a context without a CUDA
device, raises.
"""
__all__ = ["build", "binding", "synth"]
