// layout.cuh -- how the bounded KV cache is laid out in HBM.
//
// The pool owns the layout, so it is chosen for the kernels that stream it, not for the writer:
//
//   kv[layer][block][kv_head][K|V][half = d/64][row = token%16][64 bf16, 16-byte chunks XOR-swizzled]
//
// * One (block, kv_head) = K tile + V tile = 2 * 16 * D * 2 bytes, CONTIGUOUS (8 KiB at D=128): the
//   unit a decode CTA streams; one bulk async copy (UBLKCP) or 512 coalesced 16-byte loads.
// * Inside a tile, a "half" is 16 rows x 128 bytes.  The 16-byte chunk c (0..7) of row r is stored at
//   chunk position c ^ (r & 7).  That is exactly the 128-byte-swizzle, K-major shared-memory layout
//   of sm_100 UMMA descriptors and what makes `ldmatrix` conflict-free, so a LINEAR copy
//   HBM -> shared memory lands a tile already swizzled: no tensor map, no re-layout pass.
// * A token row is two 128-byte segments (one per half); the append kernel writes 16-byte chunks.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace metronome {

constexpr int kBlockTokens = 16;   // PAPER.md:L149 "S=16 -- one KV block"
constexpr int kHalfDim = 64;       // 128-byte rows: the swizzle span

struct KvLayout {
    int32_t head_dim;       // D
    int32_t n_kv_heads;     // Hkv
    int32_t fp8;            // METRONOME_FLAG_KV_FP8: rows are E4M3 codes + one float32 scale per (token, KV head)
    int64_t tile_bytes;     // 16 * D * 2          (K or V of one block-head; 16 * D in the fp8 layout)
    int64_t head_bytes;     // 2 * tile_bytes      (K then V; + 128 in the fp8 layout: 16 K scales, 16 V scales)
    int64_t block_bytes;    // Hkv * head_bytes
    int64_t layer_bytes;    // n_blocks * block_bytes
};

// fp8 layout of one (block, kv head):  [K codes 16 x D bytes][V codes 16 x D][K scales 16 f32][V scales 16 f32]
// (NEXT row f4, "the two compose"; quantiser: DESIGN.md reading R18).  The 16-byte chunks of a code tile
// are XOR-swizzled inside 128-byte lines (fp8_chunk_offset) so that `ldmatrix` and the 16-byte V-row loads of the GQA
// decode kernel are conflict-free after a LINEAR copy HBM -> shared memory, as for the bf16 tiles.
__host__ __device__ inline KvLayout make_layout(int32_t D, int32_t Hkv, int64_t n_blocks, bool fp8 = false) {
    KvLayout L;
    L.head_dim = D;
    L.n_kv_heads = Hkv;
    L.fp8 = fp8 ? 1 : 0;
    L.tile_bytes = (int64_t)kBlockTokens * D * (fp8 ? 1 : 2);
    L.head_bytes = 2 * L.tile_bytes + (fp8 ? 2 * kBlockTokens * 4 : 0);
    L.block_bytes = (int64_t)Hkv * L.head_bytes;
    L.layer_bytes = n_blocks * L.block_bytes;
    return L;
}

// Byte offset, inside a K or V tile, of 16-byte chunk `c` (0 .. D/8-1) of token row `r` (0..15).
__host__ __device__ __forceinline__ int32_t tile_chunk_offset(int32_t r, int32_t c) {
    return ((c >> 3) * (kBlockTokens * 128)) + r * 128 + (((c & 7) ^ (r & 7)) << 4);
}

// fp8 KV: byte offset, inside a K or V code tile (16 rows x D bytes), of 16-byte chunk `c` (0 .. D/16-1) of token row
// `r`.  The tile is a sequence of 128-byte lines (one row at D = 128, two rows at D = 64); chunk position p of line l is
// stored at p ^ (l & 7).
__host__ __device__ __forceinline__ int32_t fp8_chunk_offset(int32_t D, int32_t r, int32_t c) {
    const int32_t q = r * (D >> 4) + c;
    const int32_t line = q >> 3;
    return line * 128 + (((q & 7) ^ (line & 7)) << 4);
}
// ... of the 8-byte unit `u` (8 codes, 0 .. D/8-1) of token row `r`
__host__ __device__ __forceinline__ int32_t fp8_unit_offset(int32_t D, int32_t r, int32_t u) {
    return fp8_chunk_offset(D, r, u >> 1) + ((u & 1) << 3);
}

// Slot of logical block `b` in a session's block table: the first n_sink entries are the pinned
// sink blocks, the rest is a ring over the window blocks (pinned head, freed middle).
__host__ __device__ __forceinline__ int32_t table_slot(int32_t b, int32_t n_sink, int32_t ring) {
    return b < n_sink ? b : n_sink + (b - n_sink) % ring;
}

// Programmatic dependent launch (PDL): a kernel launched with the programmatic-serialization
// attribute may start while its predecessor on the stream is still running; it must not touch
// anything the predecessor reads or writes before pdl_wait() (= full completion + flush of the
// predecessor).  Both are no-ops for a plain launch.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// One thread: wait until the 32-bit flag (written in stream order by a copy engine or by another grid) has reached
// `seq` (wrap-safe), with acquire semantics at system scope: what was written before the flag is visible afterwards.
__device__ __forceinline__ void spin_until_reached_sys(const int32_t* flag, int32_t seq) {
    int32_t seen;
    do {
        asm volatile("ld.acquire.sys.global.s32 %0, [%1];" : "=r"(seen) : "l"(flag) : "memory");
        if (seen - seq < 0) __nanosleep(64);
    } while (seen - seq < 0);
}

template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl,
                                 Args... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

}  // namespace metronome
