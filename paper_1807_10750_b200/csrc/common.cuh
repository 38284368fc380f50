// Shared declarations of the CUDA path: device-side graph layout and small helpers.
//
// Device layout of a loaded graph ("SELL-16 with row splitting + CTA hubs"):
//   * vertices are relabelled by (colour asc, degree desc, caller id asc); `perm` maps the
//     internal row back to the caller's vertex id (which is what enters the Philox counter);
//   * a SLICE is the work of one warp: 16 sub-rows x G groups x 4 edges.  A row of up to
//     16 x kSubRowEdges edges is split into SPR in {1,2,4,8,16} sub-rows (group q of the row goes
//     to sub-row q % SPR), so a slice holds 16/SPR rows; the sub-rows of one row are
//     finished by a warp-level segmented (butterfly) reduction;
//   * a HUB is a row with more edges than one slice holds; it is cut into P balanced PARTS, one
//     slice each (SPR = 16), scheduled like any other slice.  A part adds its partial local fields
//     to hub_acc[hub][tile][32] (integer atomics, order-free) and counts itself in hub_cnt; the part
//     that arrives last reads the sums, finishes the row and clears hub_acc for the next sweep;
//   * a CELL is one int4 of four (relabelled) neighbour rows plus one word of four int8
//     weights (w4w: an int4 of int32 weights for graphs whose weights do not fit int8).
//     Padding entries carry weight 0 and point at the sub-row's own row (a sector that is read
//     anyway), so gathers need no predicate.
//     Cell arrays: groups 0 and 1 of slice s sit at HEAD cells (s*2 + g)*16 + sub-row, so that
//     everything a warp needs to start a slice (descriptor, first cells, caller ids) is addressed
//     by the slice index alone and can be prefetched with independent loads, also across the grid
//     barrier that separates colour phases; groups g >= 2 sit at desc.off + (g-2)*16 + sub-row;
//   * spins are replica-interleaved: state[tile][row][32] int8 (+1/-1), one 32-byte
//     sector per spin per tile of 32 replicas, so a neighbour gather is one sector and a
//     thread pair reads it with two 16-byte loads;
//   * ranges[phase][cta] is the static, cost-balanced split of every colour phase over the
//     CTAs of the grid (launch-per-phase kernels); the persistent kernel deals the slices
//     phase_slices[phase] .. phase_slices[phase + 1] out itself (strided over all warps of the grid).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "philox.cuh"

namespace ising {

constexpr int kTile = 32;            // replicas per tile == bytes per spin per tile
constexpr int kSubRows = 16;         // sub-rows per slice (lane pairs per warp)
constexpr int kWarpsPerCta = 16;
constexpr int kSweepThreads = kWarpsPerCta * 32;
constexpr int kHeadGroups = 2;       // groups of every slice stored at slice-indexed (prefetchable) positions
constexpr int kSubRowEdges = 16;                      // a row is split until a sub-row has <= this many edges ...
                                                       // ... up to 16 sub-rows; rows above that are hubs (cut into parts)
constexpr int kMaxPersistReplicas = 512;               // replicas per persistent launch

struct SliceDesc {
    uint32_t off;    // first tail cell (groups >= kHeadGroups) of this slice
    uint32_t row0;   // first internal row
    uint32_t G;      // groups (of 4 edges) per sub-row, >= 1
    uint32_t meta;   // log2(SPR) | (valid rows << 8) | (parts P of the hub this slice is a part of, else 0) << 16
};

struct PhaseRange {  // work of one CTA in one colour phase of the launch-per-phase kernels (absolute slice indices)
    uint32_t s0, s1;
};

enum SweepKind : int { kKindGS = 0, kKindJacobi = 1, kKindEval = 2 };

struct GraphView {
    const int4* col4;
    const uint32_t* w4;
    const int4* w4w;            // wide weights, or nullptr
    const SliceDesc* slices;
    const uint32_t* sorig;      // [n_slices * 16] caller id of each sub-row's row (0xffffffff: none); hub part:
                                //   {caller id, hub id, part index, 0xffffffff ...}
    unsigned long long* hub_acc;   // [n_hubs][tiles_max][32] partial local fields of hub rows (zero between sweeps)
    unsigned int* hub_cnt;      // [n_hubs][tiles_max] parts arrived so far (monotone)
    uint32_t tiles_max;
    const PhaseRange* ranges;   // [n_phases][n_cta]
    const uint32_t* phase_slices;   // [n_phases + 1] first slice of every phase
    uint32_t n_cta;             // CTAs the ranges were built for (== gridDim.x)
    uint32_t n_phases;
};

struct SweepParams {
    GraphView g;
    const uint8_t* src;         // state read
    uint8_t* dst;               // state written (== src for in-place Gauss-Seidel)
    long long* accum;           // [tiles * 32] energy bookkeeping, atomically added
    unsigned long long tile_stride;   // bytes between tiles = n * 32
    uint32_t phase_begin, phase_end;  // colour phases processed by this launch
    uint32_t tiles;
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
// Spin sectors: L2-coherent loads (ld.global.cg).  Inside the persistent kernel a spin
// written in colour phase c by another SM is read in phase c+1 after the grid barrier, so
// the (incoherent) L1 must never serve it.
__device__ __forceinline__ uint4 ld_spin(const uint8_t* p) {
    return __ldcg(reinterpret_cast<const uint4*>(p));
}
// Neighbour gather.  Padding entries point at the sub-row's own row with weight 0: all paddings of
// a sub-row hit one sector (which the row's owner reads anyway), so they need no predicate.
__device__ __forceinline__ uint4 ld_nbr(const uint8_t* base, int c) {
    return __ldcg(reinterpret_cast<const uint4*>(base + (size_t)(uint32_t)c * kTile));
}

}  // namespace ising
