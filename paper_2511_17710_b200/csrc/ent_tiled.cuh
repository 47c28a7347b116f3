// ent_tiled.cuh -- tiled fused step (placeholder until the tiled kernel lands: reports "unsupported" so that
// ent_step takes the untiled kernel).
#pragma once
#include "ent_kernels.cuh"

namespace ent {

struct TiledState { size_t scratch = 0; };

inline void tiled_release(TiledState &) {}
inline size_t tiled_scratch_bytes(const TiledState &t) { return t.scratch; }
inline int tiled_set_grid(TiledState &, const GridDev &, char *, size_t) { return ENT_OK; }
inline bool tiled_supported(const TiledState &, const GridDev &) { return false; }
inline int tiled_step(TiledState &, const GridDev &, cudaStream_t, FieldPtrs, PartPtrs, CurrentPtrs, long long, const int32_t *,
                      float, float, float, float, unsigned long long *, long long *, char *, size_t) { return ENT_EUNSUPPORTED; }

}  // namespace ent
