// K8 / K9: reverse-scan adjoint d(sum w * cube) / d n_H2 (placeholder until the kernels land).
#pragma once
#include "cell_kernels.cuh"
#include "transfer_common.cuh"

namespace iris {

struct AdjointConsts {
  float c_e, c_a, c_d, gr;
  int upper, lower;
  float T_inf;
  float scale;      // d(out) / d(D in Kelvin)
  int subtract;
};

inline cudaError_t launch_adjoint(const MarchConsts&, const AdjointConsts&, const LevelConsts&, int, const float*, int64_t,
                                  int, int, int, bool, const float*, const float*, const float*, float*, cudaStream_t,
                                  uint64_t*) {
  return cudaErrorNotSupported;
}

}  // namespace iris
