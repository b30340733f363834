// islbm_tiled.cuh — shared-memory tiled, fused stream+interpolate+collide step.
// (placeholder plan: filled in after the generic kernel is parity-green)
#pragma once

#include <cuda_runtime.h>

#include <string>

#include "islbm_kernels.cuh"

namespace islbmk {

struct TiledPlan {
  bool available = false;
  const char *name = "tiled";
  int launches_per_step = 1;
};

inline int tiled_plan_create(TiledPlan &p, int, const int *, int, void *, void *, std::string &) {
  p.available = false;
  return 0;
}

inline int tiled_step(TiledPlan &, const DevMesh &, const NodeParams &, int, cudaStream_t, std::string &err) {
  err = "tiled kernel not available";
  return -6;
}

}  // namespace islbmk
