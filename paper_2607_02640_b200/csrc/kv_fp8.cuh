// kv_fp8.cuh -- NEXT row f4: K / V rows stored as fp8 (E4M3) codes, composed with the window
// (sec. 4.1: "Orthogonal to KV compression, which shrinks each token ...: we bound which tokens stay
// resident, and the two compose").  The paper names no format: DESIGN.md reading R18.
#pragma once
#include <cuda_fp16.h>

#include "layout.cuh"

namespace metronome {

// The fp8 KV quantiser (reading R18; the oracle states it in oracle/kv_fp8.py): a row of D bf16 values of
// one (token, KV head) -> D E4M3 codes + one float32 scale = max |x| / 448 (1 for an all-zero row); code = x / scale
// (IEEE float32 division) rounded to nearest even, saturating.  Each of the row's D / 8 lanes (consecutive lanes of a
// warp, `lanes` of them, a power of two) holds 8 values; the lane given `scale_out` stores the scale.
__device__ __forceinline__ uint2 quantize_chunk_e4m3(uint4 x, int32_t lanes, float* scale_out) {
    const uint32_t w[4] = {x.x, x.y, x.z, x.w};
    float f[8];
    float amax = 0.f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        f[2 * k] = __uint_as_float(w[k] << 16);
        f[2 * k + 1] = __uint_as_float(w[k] & 0xFFFF0000u);
        amax = fmaxf(amax, fmaxf(fabsf(f[2 * k]), fabsf(f[2 * k + 1])));
    }
    // (only the row's own lanes take part: the other rows of the warp may belong to threads that have left)
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t gmask = lanes >= 32 ? 0xffffffffu : ((1u << lanes) - 1u) << (lane & ~(uint32_t)(lanes - 1));
    for (int32_t o = lanes >> 1; o >= 1; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(gmask, amax, o));
    const float scale = amax > 0.f ? __fdiv_rn(amax, 448.f) : 1.f;
    if (scale_out) *scale_out = scale;
    uint32_t out[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        uint16_t lo, hi;
        asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(lo) : "f"(__fdiv_rn(f[4 * k + 1], scale)), "f"(__fdiv_rn(f[4 * k], scale)));
        asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(hi) : "f"(__fdiv_rn(f[4 * k + 3], scale)), "f"(__fdiv_rn(f[4 * k + 2], scale)));
        out[k] = (uint32_t)lo | ((uint32_t)hi << 16);
    }
    return make_uint2(out[0], out[1]);
}
// value(code) * scale, in float32: what a stored element decodes to
__device__ __forceinline__ void dequant8_e4m3(uint2 q, float scale, float (&f)[8]) {
    const uint32_t w[2] = {q.x, q.y};
#pragma unroll
    for (int k = 0; k < 2; ++k) {
#pragma unroll
        for (int hpart = 0; hpart < 2; ++hpart) {
            uint32_t h2;
            asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"((uint16_t)(w[k] >> (16 * hpart))));
            const __half2 hv = *reinterpret_cast<const __half2*>(&h2);
            f[4 * k + 2 * hpart] = __low2float(hv) * scale;
            f[4 * k + 2 * hpart + 1] = __high2float(hv) * scale;
        }
    }
}

}  // namespace metronome
