// attend_mma.cuh -- rows a5 (GQA decode) and a7 (chunk prefill): tensor-core tile kernel.  STUB.
#pragma once
#include "attend_common.cuh"

namespace metronome {
inline void configure_attend_mma_kernels() {}
inline bool attend_mma_supported(int32_t, int32_t) { return false; }
inline int launch_attend_mma(const AttendParams&, int32_t, int32_t, int32_t, int32_t, cudaStream_t) { return 1; }
}  // namespace metronome
