// Shared declarations of the CUDA path: device-side graph layout and small helpers.
//
// Device layout of a loaded graph ("SELL-16 with row splitting"):
//   * vertices are relabelled by (colour asc, degree desc, caller id asc); `perm` maps the
//     internal row back to the caller's vertex id (which is what enters the Philox counter);
//   * a SLICE is the work of one warp: 16 sub-rows x G groups x 4 edges.  A row of
//     degree d is split into SPR in {1,2,4,8,16} sub-rows (group q of the row goes to
//     sub-row q % SPR), so a slice holds 16/SPR rows; hub rows (SPR = 16) own a whole
//     warp and are finished by a warp-level segmented reduction;
//   * col4[off + g*16 + sr] is an int4 with the four (relabelled) neighbour rows of group g
//     of sub-row sr, w4[...] the four int8 weights packed in one word (w4w[...]: int4 of
//     int32 weights for graphs whose weights do not fit int8).  Padding slots carry
//     weight 0 and point at a valid row, so they contribute nothing;
//   * spins are replica-interleaved: state[tile][row][32] int8 (+1/-1), one 32-byte
//     sector per spin per tile of 32 replicas, so a neighbour gather is one sector and a
//     thread pair reads it with two 16-byte loads.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "philox.cuh"

namespace ising {

constexpr int kTile = 32;            // replicas per tile == bytes per spin per tile
constexpr int kSubRows = 16;         // sub-rows per slice (lane pairs per warp)
constexpr int kWarpsPerCta = 8;
constexpr int kSweepThreads = kWarpsPerCta * 32;
constexpr int kSubRowEdges = 32;     // a row is split until a sub-row has <= this many edges

struct SliceDesc {
    uint32_t off;    // first (group, sub-row) cell of this slice in col4 / w4
    uint32_t row0;   // first internal row
    uint32_t G;      // groups (of 4 edges) per sub-row
    uint32_t meta;   // log2(SPR) | (valid rows << 8)
};

enum SweepKind : int { kKindGS = 0, kKindJacobi = 1, kKindEval = 2 };

struct SweepParams {
    const int4* col4;
    const uint32_t* w4;
    const int4* w4w;            // wide weights, or nullptr
    const SliceDesc* slices;
    const int32_t* perm;
    const uint8_t* src;         // state read
    uint8_t* dst;               // state written (== src for in-place Gauss-Seidel)
    long long* accum;           // [tiles * 32] energy bookkeeping, atomically added
    unsigned long long tile_stride;   // bytes between tiles = n * 32
    uint32_t slice_begin, slice_end;
    uint32_t thr;               // flip threshold of this sweep
    uint32_t T;                 // absolute sweep index (Philox counter word 1)
    uint32_t rep0;              // global id of replica 0 of this call
    int32_t tie_rule;
    uint32_t flush_rows;        // rows a lane may accumulate in int32 before flushing
    PhiloxKeys keys;
};

// Streaming, read-only data (graph arrays): read-only path, do not keep in L1.
__device__ __forceinline__ int4 ld_stream(const int4* p) {
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ uint32_t ld_stream(const uint32_t* p) {
    uint32_t r;
    asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(r) : "l"(p));
    return r;
}
// Spin sectors: coherent loads.  Every phase is its own launch and a colour class is an
// independent set, so no spin read in a phase is written in the same phase (except a row's
// own spin, read and written by the same thread).
__device__ __forceinline__ uint4 ld_spin(const uint8_t* p) {
    return *reinterpret_cast<const uint4*>(p);
}

__device__ __forceinline__ uint32_t warp_bcast(uint32_t v, int src) { return __shfl_sync(0xffffffffu, v, src); }

}  // namespace ising
