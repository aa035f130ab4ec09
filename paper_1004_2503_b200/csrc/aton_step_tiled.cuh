// placeholder: tiled streaming kernel (variant 1) -- not built yet
#pragma once
#include "aton_step_ref.cuh"
namespace aton {
inline bool tiled_shape_ok(const Grid &, int, int) { return false; }
template <int FLAGS>
cudaError_t launch_step_tiled(const FieldsIO &, const Grid &, const StepConst &, int, int, cudaStream_t) {
    return cudaErrorNotSupported;
}
}  // namespace aton
