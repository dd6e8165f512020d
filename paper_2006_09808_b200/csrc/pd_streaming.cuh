// pd_streaming.cuh -- helpers shared by the streaming kernels (pd_streaming_fd.cuh).
//
// The first streaming path of this library (four launches per iteration over fp32 planes, in-place updates) lived
// here; it ran at about 1.2 TB/s and was replaced by the kernels of pd_streaming_fd.cuh, which also cover the
// literal W != I iteration.
#pragma once
#include "fft_regs.cuh"

namespace pdk {

// sum over the T threads of one line (T a power of two <= 32, the group is aligned inside its warp)
template <int T>
__device__ __forceinline__ float group_sum(float v) {
#pragma unroll
    for (int o = T / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace pdk
