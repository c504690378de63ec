// placeholder until the tile kernel lands
#pragma once
#include "pgg_common.cuh"
namespace pgg {
struct TilePlan { int dummy; };
inline bool tile_supported(int, uint32_t) { return false; }
inline int tile_plan(int, uint32_t, uint32_t, TilePlan*) { return 0; }
inline void tile_launch(const TilePlan&, int, const PhaseArgs&, uint32_t, uint32_t, cudaStream_t) {}
}
