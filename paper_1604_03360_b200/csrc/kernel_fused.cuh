// kernel_fused.cuh -- placeholder until the fused stage kernel lands (next commit).
#pragma once
#include "grid.cuh"
#include "kernel_generic.cuh"
namespace hydro {
struct FusedPlan { char err[256] = {0}; };
inline bool fused_supported(const Geom&, int, int) { return false; }
inline int build_fused_plan(FusedPlan&, const Geom&, int, int) { return -1; }
template <class T>
int launch_fused(FusedPlan&, const Geom&, int, const StageArgs&, const T*, const T*, const T*, T*, Ctl*, cudaStream_t) { return -1; }
}
