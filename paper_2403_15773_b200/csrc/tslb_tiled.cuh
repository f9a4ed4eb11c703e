// tslb_tiled.cuh -- TMA-staged tiled kernel (placeholder until the first GPU parity run of the
// generic path; replaced by the real kernel).
#pragma once
#include <cuda_runtime.h>
#include <string>
#include "tslb_math.cuh"

namespace tslb {

struct TiledPlan {
  std::string name;
};

inline bool tiled_supported(int precision, int nx, int ny, int nz) { return false; }
inline bool tiled_plan_create(TiledPlan &, int, const Layout &, void *[2][NF_MAX], int, int, std::string &why) {
  why = "not built";
  return false;
}
inline void tiled_plan_destroy(TiledPlan &) {}
template <typename T>
cudaError_t launch_tiled(TiledPlan &, const StepParams<T> &, int, int, bool, cudaStream_t) {
  return cudaErrorNotSupported;
}

}  // namespace tslb
