// em_fused.cuh -- fused H+E+source+Joule sweep (EM_KERNEL_FUSED).  Placeholder until the sweep lands.
#pragma once
#include "em_aux.cuh"
#include "em_common.cuh"

namespace em {

struct FusedPlan { int n_tiles; };

inline FusedPlan make_fused_plan(int, int, int, int) { return FusedPlan{1}; }
inline int tile_of(const FusedPlan &, int, int, int) { return 0; }

template <typename R>
cudaError_t launch_fused(const FusedPlan &, const DevParams<R> &, const DevSources<R> &, const int *, int, bool,
                         long long, cudaStream_t) {
    return cudaErrorNotSupported;
}

}  // namespace em
