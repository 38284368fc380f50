// Sparse annealing sweep and its bookkeeping kernels.
//
// One warp owns one slice (common.cuh): lane = 2*sub_row + half, every lane keeps the
// int32 local fields h_i = sum_j w_ij s_j (eq. (2)) of 16 replicas.  Four
// neighbour sectors are gathered per step (16-byte L2 loads), byte-transposed with PRMT so
// that one dp4a multiplies the four edge weights into one replica's field.  Rows split
// over several sub-rows are finished by a warp-level segmented (butterfly) reduction; hub
// rows are cut into parts (one slice each) whose partial fields meet in global memory.
// The epilogue takes the energy-minimising value (L47-49 with the sign reading Q1:
// s_i <- +1 if h_i < 0 else -1), applies the scheduled flip of Algorithm 2 (L177) with the
// stateless Philox word, writes the spin sector and accumulates the energy bookkeeping
// (a7): Gauss-Seidel  dE_i = (a_i - s_i) h_i  (exact because a colour class is an
// independent set), Jacobi / evaluation  s_i h_i  (sum_i s_i h_i = 2 E).
//
// Two drivers share these passes:
//   k_sweep      one launch = colour phases [phase_begin, phase_end) of one sweep (Jacobi,
//                evaluation, racy mode, wide weights);
//   k_anneal_gs  the persistent cooperative kernel of the Gauss-Seidel hot path: all sweeps x
//                colour phases of one ising_anneal call in ONE launch, a grid barrier between
//                phases, static graph data of the next phase prefetched across the barrier,
//                the cut reduction, trace and best-state capture fused in (a7, a9).
#pragma once
#include "common.cuh"
#include "primitives.cuh"
#include "chain.cuh"

namespace ising {

__device__ __forceinline__ void field_cell(int (&h)[16], const uint4& e0, const uint4& e1, const uint4& e2,
                                           const uint4& e3, uint32_t w) {
    field_word(h, 0, e0.x, e1.x, e2.x, e3.x, w);
    field_word(h, 1, e0.y, e1.y, e2.y, e3.y, w);
    field_word(h, 2, e0.z, e1.z, e2.z, e3.z, w);
    field_word(h, 3, e0.w, e1.w, e2.w, e3.w, w);
}

__device__ __forceinline__ void field_cell_wide(int (&h)[16], const uint4& e0, const uint4& e1, const uint4& e2,
                                                const uint4& e3, const int4& w) {
    field_word_wide(h, 0, e0.x, w.x); field_word_wide(h, 1, e0.y, w.x);
    field_word_wide(h, 2, e0.z, w.x); field_word_wide(h, 3, e0.w, w.x);
    field_word_wide(h, 0, e1.x, w.y); field_word_wide(h, 1, e1.y, w.y);
    field_word_wide(h, 2, e1.z, w.y); field_word_wide(h, 3, e1.w, w.y);
    field_word_wide(h, 0, e2.x, w.z); field_word_wide(h, 1, e2.y, w.z);
    field_word_wide(h, 2, e2.z, w.z); field_word_wide(h, 3, e2.w, w.z);
    field_word_wide(h, 0, e3.x, w.w); field_word_wide(h, 1, e3.y, w.w);
    field_word_wide(h, 2, e3.z, w.w); field_word_wide(h, 3, e3.w, w.w);
}

// Flip decisions of Algorithm 2 (L177) for the 16 replicas rep_lane0 .. rep_lane0+15 of spin
// `orig` in sweep T: bit j set <=> philox(seed; ctr=(orig, T, r>>2, FLIP))[r&3] < thr, r = rep_lane0 + j.
// The 16 replicas span 4 Philox calls (5 when first_replica is not a multiple of 4).  The `spr`
// lanes that share a row split the calls among themselves: lane part q takes calls q, q+spr, ...;
// the partial masks are OR-ed by the caller's segmented reduction (finish_flip_mask after it).
__device__ __forceinline__ uint32_t flip_mask_part(uint32_t orig, uint32_t T, uint32_t rep_lane0, uint32_t thr,
                                                   uint32_t q, uint32_t spr, const PhiloxKeys& keys) {
    if (thr == 0) return 0u;
    const uint32_t cw = rep_lane0 >> 2;
    const uint32_t ncalls = (rep_lane0 & 3u) ? 5u : 4u;
    uint32_t m = 0;
    if (ncalls == 5) {   // rare: generic strided loop
        for (uint32_t k = q; k < ncalls; k += spr)
            m |= lt4(philox4x32_10(orig, T, cw + k, kDomainFlip, keys), thr) << (4 * k);
    } else if (spr == 1) {
#pragma unroll
        for (int k = 0; k < 4; ++k) m |= lt4(philox4x32_10(orig, T, cw + k, kDomainFlip, keys), thr) << (4 * k);
    } else if (spr == 2) {   // two independent calls per lane, straight-line so that they interleave
        const uint4 u0 = philox4x32_10(orig, T, cw + q, kDomainFlip, keys);
        const uint4 u1 = philox4x32_10(orig, T, cw + q + 2, kDomainFlip, keys);
        m = (lt4(u0, thr) << (4 * q)) | (lt4(u1, thr) << (4 * q + 8));
    } else if (q < 4) {      // one call per lane (parts 0..3 of the row)
        m = lt4(philox4x32_10(orig, T, cw + q, kDomainFlip, keys), thr) << (4 * q);
    }
    return m;
}
__device__ __forceinline__ uint32_t finish_flip_mask(uint32_t m, uint32_t rep_lane0) {
    return (m >> (rep_lane0 & 3u)) & 0xffffu;
}

// Where a lane keeps its 16 per-replica energy increments: registers (launch-per-sweep kernels), or a private
// column of shared memory (persistent kernel: the increments are touched only where a spin changed, which is rare
// at low temperature, and 16 registers per thread are worth more there).
template <typename T>
struct RegAcc {
    using value_type = T;
    T (&a)[16];
    __device__ __forceinline__ void add(int i, T v) const { a[i] += v; }
};
struct SmemAcc {
    using value_type = int;
    int* p;   // &s_dE[0][thread]; element i at p[i * kSweepThreads]
    __device__ __forceinline__ void add(int i, int v) const { atomicAdd(p + i * kSweepThreads, v); }   // one ATOMS instead of LDS + IADD + STS (the slot is this thread's own)
};

// Sum (or OR) over the 16 lanes of the same half (lane parity) with one REDUX per value: the even and the
// odd lanes run their own redux.sync with their own member mask.
__device__ __forceinline__ void half_reduce16(int (&v)[16], uint32_t& bits, int half) {
    if (half) {
#pragma unroll
        for (int k = 0; k < 16; ++k) asm volatile("redux.sync.add.s32 %0, %0, 0xaaaaaaaa;" : "+r"(v[k]));
        asm volatile("redux.sync.or.b32 %0, %0, 0xaaaaaaaa;" : "+r"(bits));
    } else {
#pragma unroll
        for (int k = 0; k < 16; ++k) asm volatile("redux.sync.add.s32 %0, %0, 0x55555555;" : "+r"(v[k]));
        asm volatile("redux.sync.or.b32 %0, %0, 0x55555555;" : "+r"(bits));
    }
}

template <typename AccT>
__device__ __forceinline__ void flush_acc(AccT (&acc)[16], long long* s_acc, int lane) {
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        AccT v = acc[k];
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        v += __shfl_xor_sync(0xffffffffu, v, 4);
        v += __shfl_xor_sync(0xffffffffu, v, 8);
        v += __shfl_xor_sync(0xffffffffu, v, 16);
        if (lane < 2 && v != 0)
            atomicAdd(reinterpret_cast<unsigned long long*>(s_acc + lane * 16 + k), (unsigned long long)(long long)v);
        acc[k] = 0;
    }
}

// Persistent kernel: a warp first reduces its lanes' increments into its own 32 shared slots
// (plain adds by lanes 0 and 1, no atomics); the slots are folded per CTA at the end of the sweep.
__device__ __forceinline__ void flush_warp(int (&acc)[16], long long* wacc, int lane) {
    uint32_t none = 0;
    half_reduce16(acc, none, lane & 1);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        if (lane < 2) wacc[lane * 16 + k] += (long long)acc[k];
        acc[k] = 0;
    }
}
__device__ __forceinline__ void flush_warp(const SmemAcc& acc, long long* wacc, int lane) {
    int v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) { v[k] = acc.p[k * kSweepThreads]; acc.p[k * kSweepThreads] = 0; }
    flush_warp(v, wacc, lane);
}
// The warp moves on to another replica tile: hand its slots over to the CTA accumulator of the old tile.
__device__ __forceinline__ void fold_warp(long long* wacc, long long* s_acc_tile, int lane) {
    __syncwarp();
    const long long v = wacc[lane];
    if (v != 0) {
        atomicAdd(reinterpret_cast<unsigned long long*>(s_acc_tile + lane), (unsigned long long)v);
        wacc[lane] = 0;
    }
    __syncwarp();
}

// Per-unit context of a lane (tile-adjusted pointers already include the lane's half).
struct PassCtx {
    const uint8_t* src;
    uint8_t* dst;
    uint8_t* best;         // best-state capture target of the fused path, or nullptr
    uint32_t cap16;        // capture mask: bit j set = replica j of this lane improved in the last sweep
    uint32_t rep_lane0;    // global id of this lane's replica 0
    uint32_t thr, T;
    int32_t tie_rule;
    uint32_t tile;         // replica tile of this unit (index into hub_acc / hub_cnt / h0)
};

// a4-a7 for one row and this lane's 16 replicas, four replicas (one word of spin bytes) at a time.
template <int KIND, typename Acc>
__device__ __forceinline__ void row_update(const PassCtx& x, const int (&h)[16], const uint4& so4, uint4 bold,
                                           uint32_t flip16, size_t row_off, const Acc& acc) {
    using AccT = typename Acc::value_type;
    const uint32_t so[4] = {so4.x, so4.y, so4.z, so4.w};
    if (KIND == kKindEval) {
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int b = 0; b < 4; ++b) acc.add(4 * k + b, (AccT)sbyte(so[k], b) * (AccT)h[4 * k + b]);
        return;
    }
    uint32_t nv[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        // a4 (L47-49, reading Q1/Q3): +1 (0x01) where h < 0, else -1 (0xff)
        uint32_t a = ~sign_bytes(h[4 * k], h[4 * k + 1], h[4 * k + 2], h[4 * k + 3]) | 0x01010101u;
        if (x.tie_rule == 1) {   // KEEP: h == 0 leaves the spin as it is
            uint32_t z = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) z |= h[4 * k + b] == 0 ? (0xffu << (8 * b)) : 0u;
            a = (a & ~z) | (so[k] & z);
        }
        // a5 (Alg. 2): negate the bytes whose flip bit is set (+1 <-> -1 is xor 0xfe)
        const uint32_t f4 = (flip16 >> (4 * k)) & 15u;
        a ^= ((f4 * 0x00204081u) & 0x01010101u) * 0xfeu;
        nv[k] = a;
        if (KIND == kKindGS) {
            // a7: dE = (a - s) h; a - s is +-2 exactly where the byte changed (a ^ s == 0xfe)
            const uint32_t d2 = (a << 1) & (a ^ so[k]);
            if (d2 != 0u) {   // at low temperature most words do not change
#pragma unroll
                for (int b = 0; b < 4; ++b) acc.add(4 * k + b, (AccT)sbyte(d2, b) * (AccT)h[4 * k + b]);
            }
        } else {
#pragma unroll
            for (int b = 0; b < 4; ++b) acc.add(4 * k + b, (AccT)sbyte(so[k], b) * (AccT)h[4 * k + b]);
        }
    }
    *reinterpret_cast<uint4*>(x.dst + row_off) = make_uint4(nv[0], nv[1], nv[2], nv[3]);
    if (KIND == kKindGS && x.cap16 != 0u) {
        // fused best-state capture: the value this row held after the previous sweep
        // (bold = the captured row as loaded by the caller when the mask is partial)
        uint4* bp = reinterpret_cast<uint4*>(x.best + row_off);
        if (x.cap16 == 0xffffu) {
            *bp = so4;
        } else {
            const uint32_t k0 = nibble_to_bytemask(x.cap16 & 15u), k1 = nibble_to_bytemask((x.cap16 >> 4) & 15u);
            const uint32_t k2 = nibble_to_bytemask((x.cap16 >> 8) & 15u), k3 = nibble_to_bytemask((x.cap16 >> 12) & 15u);
            bold.x = (so4.x & k0) | (bold.x & ~k0);
            bold.y = (so4.y & k1) | (bold.y & ~k1);
            bold.z = (so4.z & k2) | (bold.z & ~k2);
            bold.w = (so4.w & k3) | (bold.w & ~k3);
            *bp = bold;
        }
    }
}

// Early load of the captured row for a partial capture mask (row_update merges into it).
template <int KIND>
__device__ __forceinline__ uint4 ld_best_early(const PassCtx& x, bool owner, size_t row_off) {
    uint4 b = make_uint4(0u, 0u, 0u, 0u);
    if (KIND == kKindGS && owner && x.cap16 != 0u && x.cap16 != 0xffffu)
        b = __ldcg(reinterpret_cast<const uint4*>(x.best + row_off));
    return b;
}

// Hub part (common.cuh): this warp holds, spread over its 16 sub-rows, the partial local fields of one part of
// a hub row.  The partial sums of all parts meet in hub_acc by integer atomics (the result does not depend on
// their order); the part that arrives last reads the totals, clears them for the next sweep and finishes the
// row (a4-a7) like the owner lanes of an ordinary slice.
//   PACKED (int8 weights: a part's sum fits 16 bits): one 64-bit atomic per lane adds (1 << 32) + sum + 2^16 to
//   the replica's slot and returns what the slot held: arrivals in the high word, biased sum in the low one.
//   The warp whose lane 0 arrives last finishes the row; a lane whose own slot is not complete yet polls it
//   (the missing atomics are in flight: they were issued together with the ones lane 0 has seen).
//   Otherwise (int32 weights): 32-bit RED per lane, then an acq_rel arrival counter (hub_cnt).
constexpr int kPartBias = 1 << 16;

template <int KIND, bool PACKED, typename Acc>
__device__ __forceinline__ void part_finish(const GraphView& g, const PassCtx& x, uint32_t row0, uint32_t parts,
                                            uint32_t orig, uint32_t hub, int (&h)[16], const uint4& so4,
                                            const Acc& acc, const PhiloxKeys& keys) {
    const int lane = threadIdx.x & 31, sr = lane >> 1, half = lane & 1;
    uint32_t none = 0;
    half_reduce16(h, none, half);   // every lane: the part's sums of its half's 16 replicas
    int v = h[0];
#pragma unroll
    for (int k = 1; k < 16; ++k) v = sr == k ? h[k] : v;   // lane (sr, half) contributes replica half * 16 + sr
    const size_t slot = (size_t)hub * g.tiles_max + x.tile;
    const size_t row_off = (size_t)row0 * kTile;
    int total = 0;
    uint4 bold = make_uint4(0u, 0u, 0u, 0u);
    uint32_t flip = 0;
    // what only the finishing part needs (captured row, Philox flips) is computed by every part while its atomic
    // is in flight: it shortens the chain of the part that turns out to be last
    auto speculate = [&]() {
        bold = ld_best_early<KIND>(x, sr == 0, row_off);
        if (KIND != kKindEval) {
            flip = flip_mask_part(orig, x.T, x.rep_lane0, x.thr, (uint32_t)sr, (uint32_t)kSubRows, keys);
            if (half) asm volatile("redux.sync.or.b32 %0, %0, 0xaaaaaaaa;" : "+r"(flip));
            else asm volatile("redux.sync.or.b32 %0, %0, 0x55555555;" : "+r"(flip));
        }
    };
    if (PACKED) {
        unsigned long long* sp = g.hub_acc + slot * kTile + half * 16 + sr;
        const unsigned long long mine = (1ull << 32) + (unsigned long long)(uint32_t)(v + kPartBias);
        unsigned long long now;
        asm volatile("atom.relaxed.gpu.global.add.u64 %0, [%1], %2;" : "=l"(now) : "l"(sp), "l"(mine) : "memory");
        speculate();
        now += mine;
        if ((uint32_t)(__shfl_sync(0xffffffffu, now, 0) >> 32) != parts) return;
        while ((uint32_t)(now >> 32) != parts)
            asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(now) : "l"(sp) : "memory");
        asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(sp), "l"(0ull) : "memory");
        total = (int)((uint32_t)now - parts * (uint32_t)kPartBias);
    } else {
        int* accp = reinterpret_cast<int*>(g.hub_acc + slot * kTile) + half * 16 + sr;
        asm volatile("red.relaxed.gpu.global.add.s32 [%0], %1;" ::"l"(accp), "r"(v) : "memory");
        // arrival: the warp barrier orders the lanes' REDs before lane 0's release (cumulative), the last
        // part's acquire orders its reads of the sums after every part's REDs
        __syncwarp();
        unsigned int old = 0;
        if (lane == 0)
            asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(old) : "l"(g.hub_cnt + slot) : "memory");
        speculate();
        old = __shfl_sync(0xffffffffu, old, 0);
        if ((old + 1u) % parts != 0u) return;
        __syncwarp();
        total = __ldcg(accp);
        __stcg(accp, 0);
    }
#pragma unroll
    for (int k = 0; k < 16; ++k) h[k] = __shfl_sync(0xffffffffu, total, 2 * k + half);   // replica half * 16 + k
    if (sr == 0) {
        row_update<KIND>(x, h, so4, bold, finish_flip_mask(flip, x.rep_lane0), row_off, acc);
    }
}

// Everything a warp needs to start a slice; addressed by the slice index alone.
struct SliceHead {
    SliceDesc d;
    int4 c0, c1;       // head cells (groups 0 and 1)
    uint32_t w0, w1;
    uint32_t orig;
};

template <bool WIDE>
__device__ __forceinline__ SliceHead fetch_head(const GraphView& g, uint32_t s, int sr) {
    SliceHead h;
    const int4 dd = ld_stream(reinterpret_cast<const int4*>(g.slices + s));
    h.d.off = (uint32_t)dd.x; h.d.row0 = (uint32_t)dd.y; h.d.G = (uint32_t)dd.z; h.d.meta = (uint32_t)dd.w;
    const size_t at = (size_t)s * (kHeadGroups * kSubRows) + sr;
    h.c0 = ld_stream(g.col4 + at);
    h.c1 = ld_stream(g.col4 + at + kSubRows);
    h.w0 = WIDE ? 0u : ld_stream(g.w4 + at);
    h.w1 = WIDE ? 0u : ld_stream(g.w4 + at + kSubRows);
    h.orig = ld_stream(g.sorig + (size_t)s * kSubRows + sr);
    return h;
}

// One (slice, tile) unit, whole warp.
template <int KIND, bool WIDE, typename Acc>
__device__ __forceinline__ void slice_pass(const GraphView& g, const PassCtx& x, const SliceHead& hd, uint32_t s,
                                           int sr, const Acc& acc, const PhiloxKeys& keys) {
    const SliceDesc d = hd.d;
    const int log_spr = (int)(d.meta & 0xffu);
    const int nrows = (int)((d.meta >> 8) & 0xffu);
    const uint32_t spr = 1u << log_spr;
    const int rloc = sr >> log_spr;
    const bool owner = ((sr & (int)(spr - 1)) == 0) && rloc < nrows;
    const size_t row_off = (size_t)(d.row0 + (uint32_t)rloc) * kTile;
    const size_t head_at = (size_t)s * (kHeadGroups * kSubRows) + sr;

    // both head groups' gathers go out at once; everything else below overlaps their latency
    uint4 e0 = ld_nbr(x.src, hd.c0.x), e1 = ld_nbr(x.src, hd.c0.y), e2 = ld_nbr(x.src, hd.c0.z), e3 = ld_nbr(x.src, hd.c0.w);
    uint4 f0 = ld_nbr(x.src, hd.c1.x), f1 = ld_nbr(x.src, hd.c1.y), f2 = ld_nbr(x.src, hd.c1.z), f3 = ld_nbr(x.src, hd.c1.w);
    uint4 so4 = make_uint4(0u, 0u, 0u, 0u);
    if (owner) so4 = ld_spin(x.src + row_off);
    const uint4 bold = ld_best_early<KIND>(x, owner, row_off);
    int4 ww0 = make_int4(0, 0, 0, 0), ww1 = ww0;
    if (WIDE) { ww0 = ld_stream(g.w4w + head_at); ww1 = ld_stream(g.w4w + head_at + kSubRows); }
    // tail cells: groups 2 and 3 (a sub-row never holds more than 16 edges, so G <= 4); their indices are
    // requested right away so that both tail gathers can follow the head groups back to back
    const size_t tail_at = (size_t)d.off + sr;
    int4 c2 = make_int4(0, 0, 0, 0), c3 = c2, ww2 = c2, ww3 = c2;
    uint32_t w2 = 0, w3 = 0;
    if (d.G > 2) {
        c2 = ld_stream(g.col4 + tail_at);
        if (WIDE) ww2 = ld_stream(g.w4w + tail_at); else w2 = ld_stream(g.w4 + tail_at);
        if (d.G > 3) {
            c3 = ld_stream(g.col4 + tail_at + kSubRows);
            if (WIDE) ww3 = ld_stream(g.w4w + tail_at + kSubRows); else w3 = ld_stream(g.w4 + tail_at + kSubRows);
        }
    }
    uint32_t flip = 0;
    if (KIND != kKindEval && hd.orig != 0xffffffffu && (d.meta >> 16) == 0u)
        flip = flip_mask_part(hd.orig, x.T, x.rep_lane0, x.thr, (uint32_t)sr & (spr - 1), spr, keys);

    int h[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) h[k] = 0;
    if (WIDE) field_cell_wide(h, e0, e1, e2, e3, ww0); else field_cell(h, e0, e1, e2, e3, hd.w0);
    if (d.G > 2) { e0 = ld_nbr(x.src, c2.x); e1 = ld_nbr(x.src, c2.y); e2 = ld_nbr(x.src, c2.z); e3 = ld_nbr(x.src, c2.w); }
    if (d.G > 1) {
        if (WIDE) field_cell_wide(h, f0, f1, f2, f3, ww1); else field_cell(h, f0, f1, f2, f3, hd.w1);
    }
    if (d.G > 2) {
        if (d.G > 3) { f0 = ld_nbr(x.src, c3.x); f1 = ld_nbr(x.src, c3.y); f2 = ld_nbr(x.src, c3.z); f3 = ld_nbr(x.src, c3.w); }
        if (WIDE) field_cell_wide(h, e0, e1, e2, e3, ww2); else field_cell(h, e0, e1, e2, e3, w2);
        if (d.G > 3) {
            if (WIDE) field_cell_wide(h, f0, f1, f2, f3, ww3); else field_cell(h, f0, f1, f2, f3, w3);
        }
    }

    if (d.meta >> 16) {   // hub part: sorig = {caller id, hub id, part index, ...}
        const uint32_t orig = __shfl_sync(0xffffffffu, hd.orig, 0), hub = __shfl_sync(0xffffffffu, hd.orig, 2);
        part_finish<KIND, !WIDE>(g, x, d.row0, d.meta >> 16, orig, hub, h, so4, acc, keys);
        return;
    }
    // warp-level segmented reduction over the sub-rows of one row (fields add, flip bits OR)
    if (log_spr == 4) {
        half_reduce16(h, flip, (int)(threadIdx.x & 1));
    } else {
        for (int lvl = 0; lvl < log_spr; ++lvl) {
#pragma unroll
            for (int k = 0; k < 16; ++k) h[k] += __shfl_xor_sync(0xffffffffu, h[k], 2 << lvl);
            flip |= __shfl_xor_sync(0xffffffffu, flip, 2 << lvl);
        }
    }
    if (owner) row_update<KIND>(x, h, so4, bold, finish_flip_mask(flip, x.rep_lane0), row_off, acc);
}

// ---------------------------------------------------------------------------------------------
// Persistent kernel: the gathers of a slice land in shared memory (cp.async, 16 bytes per lane and
// neighbour, thread-private slots), so that the gathers of unit k+1 fly while unit k is computed and no
// register waits for them.  Slots 0-3: head group 0, 4-7: head group 1, 8: the row's own sector.
// ---------------------------------------------------------------------------------------------
constexpr int kGatherSlots = 2 * 4 + 1;
constexpr uint32_t kSlotBytes = kSweepThreads * 16;                    // one slot of every thread of the CTA
constexpr uint32_t kGatherBufBytes = kGatherSlots * kSlotBytes;

// Static data of a unit on its way to the compute stage.  Only the eight neighbour indices of the head groups
// travel through registers (they form the gather addresses); weights, caller ids and the descriptor go straight
// from global to shared memory (cp.async): meta slot m of this thread = {w0, w1, orig}, descriptor slot of the
// warp = {SliceDesc, tile}.  Three rotating slots: computing / gathers in flight / head in flight.
constexpr uint32_t kMetaSlots = 3;
constexpr uint32_t kMetaBytes = kMetaSlots * 3 * kSweepThreads * 4;
constexpr uint32_t kDescStride = 32;
constexpr uint32_t kDescBytes = kMetaSlots * kWarpsPerCta * kDescStride;

struct PipeAddr {      // shared-memory addresses of this thread
    uint32_t meta0;    // meta slot 0, word 0 (word k at + k * kSweepThreads * 4, slot m at + m * 3 * kSweepThreads * 4)
    uint32_t desc0;    // descriptor slot 0 of this warp (slot m at + m * kWarpsPerCta * kDescStride)
    __device__ __forceinline__ uint32_t meta(uint32_t m, uint32_t k) const { return meta0 + (m * 3u + k) * (kSweepThreads * 4u); }
    __device__ __forceinline__ uint32_t desc(uint32_t m) const { return desc0 + m * (kWarpsPerCta * kDescStride); }
};

struct HeadIdx { int4 c0, c1; };

__device__ __forceinline__ HeadIdx request_head(const GraphView& g, const PipeAddr& pa, uint32_t m, uint32_t s,
                                                uint32_t tile, int sr, int lane) {
    const size_t at = (size_t)s * (kHeadGroups * kSubRows) + sr;
    HeadIdx h;
    h.c0 = ld_stream(g.col4 + at);
    h.c1 = ld_stream(g.col4 + at + kSubRows);
    cp_async4(pa.meta(m, 0), g.w4 + at);
    cp_async4(pa.meta(m, 1), g.w4 + at + kSubRows);
    cp_async4(pa.meta(m, 2), g.sorig + (size_t)s * kSubRows + sr);
    if (lane == 0) {
        cp_async16(pa.desc(m), g.slices + s);
        sts32(pa.desc(m) + 16, tile);
    }
    cp_async_commit();
    return h;
}

// src: the unit's tile, lane half included.  gb: shared address of slot 0 of this thread in the target buffer.
__device__ __forceinline__ void issue_slice_gathers(const uint8_t* src, const HeadIdx& hd, const SliceDesc& d, int sr,
                                                    uint32_t gb, bool own) {
    const int log_spr = (int)(d.meta & 0xffu);
    const int nrows = (int)((d.meta >> 8) & 0xffu);
    const int rloc = sr >> log_spr;
    const bool owner = ((sr & ((1 << log_spr) - 1)) == 0) && rloc < nrows;
    // padding entries (weight 0) point at the sub-row's own row: they are not fetched at all (zero-filled slot), which
    // saves their L1 wavefronts (15 % of the slots of config 5)
    const uint32_t pad = d.row0 + (rloc < nrows ? (uint32_t)rloc : 0u);
    cp_async16_if(gb + 0 * kSlotBytes, src + (size_t)(uint32_t)hd.c0.x * kTile, (uint32_t)hd.c0.x != pad);
    cp_async16_if(gb + 1 * kSlotBytes, src + (size_t)(uint32_t)hd.c0.y * kTile, (uint32_t)hd.c0.y != pad);
    cp_async16_if(gb + 2 * kSlotBytes, src + (size_t)(uint32_t)hd.c0.z * kTile, (uint32_t)hd.c0.z != pad);
    cp_async16_if(gb + 3 * kSlotBytes, src + (size_t)(uint32_t)hd.c0.w * kTile, (uint32_t)hd.c0.w != pad);
    if (d.G > 1) {
        cp_async16_if(gb + 4 * kSlotBytes, src + (size_t)(uint32_t)hd.c1.x * kTile, (uint32_t)hd.c1.x != pad);
        cp_async16_if(gb + 5 * kSlotBytes, src + (size_t)(uint32_t)hd.c1.y * kTile, (uint32_t)hd.c1.y != pad);
        cp_async16_if(gb + 6 * kSlotBytes, src + (size_t)(uint32_t)hd.c1.z * kTile, (uint32_t)hd.c1.z != pad);
        cp_async16_if(gb + 7 * kSlotBytes, src + (size_t)(uint32_t)hd.c1.w * kTile, (uint32_t)hd.c1.w != pad);
    }
    if (owner && own) cp_async16(gb + 8 * kSlotBytes, src + (size_t)(d.row0 + (uint32_t)rloc) * kTile);
    cp_async_commit();
}

__device__ __forceinline__ SliceDesc lds_desc(uint32_t addr) {
    const uint4 v = lds128(addr);
    SliceDesc d;
    d.off = v.x; d.row0 = v.y; d.G = v.z; d.meta = v.w;
    return d;
}

// BULK pseudo-phase of the persistent kernel (chain.cuh, DELTA): the slices of the chain rows' colour classes do not
// update their rows; they add the rows' local fields, computed from the values all spins hold before the chain, to
// h0[tile][replica >> 2][row - row_lo][replica & 3] (fire-and-forget integer REDs; the chain clears them).
struct BulkDst {
    int* h0;
    uint32_t row_lo, n_t_pad;
};
__device__ __forceinline__ void bulk_red(int* p, int v) {
    asm volatile("red.relaxed.gpu.global.add.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void bulk_deposit(const BulkDst& bd, uint32_t tile, const SliceDesc& d, int (&h)[16],
                                             int log_spr, bool owner, int rloc) {
    const int lane = threadIdx.x & 31, sr = lane >> 1, half = lane & 1;
    if ((d.meta >> 16) != 0u || log_spr == 4) {   // one row per slice: lane (sr, half) deposits replica half * 16 + sr
        uint32_t none = 0;
        half_reduce16(h, none, half);
        int v = h[0];
#pragma unroll
        for (int k = 1; k < 16; ++k) v = sr == k ? h[k] : v;
        const uint32_t rep = (uint32_t)(half * 16 + sr);
        bulk_red(bd.h0 + ((((size_t)tile * kChainGroups + (rep >> 2)) * bd.n_t_pad + (d.row0 - bd.row_lo)) << 2) + (rep & 3u), v);
    } else {
        for (int lvl = 0; lvl < log_spr; ++lvl) {
#pragma unroll
            for (int k = 0; k < 16; ++k) h[k] += __shfl_xor_sync(0xffffffffu, h[k], 2 << lvl);
        }
        if (owner) {
            const uint32_t lr = d.row0 + (uint32_t)rloc - bd.row_lo;
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const uint32_t rep = (uint32_t)(half * 16 + k);
                bulk_red(bd.h0 + ((((size_t)tile * kChainGroups + (rep >> 2)) * bd.n_t_pad + lr) << 2) + (rep & 3u), h[k]);
            }
        }
    }
}

// Compute stage of one (slice, tile) unit whose head gathers have landed in buffer gb (Gauss-Seidel, int8 weights).
template <typename Acc>
__device__ __forceinline__ void slice_compute(const GraphView& g, const PassCtx& x, const SliceDesc& d, uint32_t ma,
                                              int sr, const Acc& acc, const PhiloxKeys& keys, uint32_t gb, bool bulk,
                                              const BulkDst& bd) {
    // ma: this thread's meta slot of the unit (w0, w1, orig one word plane apart)
    const int log_spr = (int)(d.meta & 0xffu);
    const int nrows = (int)((d.meta >> 8) & 0xffu);
    const uint32_t spr = 1u << log_spr;
    const int rloc = sr >> log_spr;
    const bool owner = ((sr & (int)(spr - 1)) == 0) && rloc < nrows;
    const size_t row_off = (size_t)(d.row0 + (uint32_t)rloc) * kTile;
    const uint4 bold = ld_best_early<kKindGS>(x, owner && !bulk, row_off);
    // tail cells (rows of 129..256 edges only): through registers, requested right away
    const size_t tail_at = (size_t)d.off + sr;
    int4 c2 = make_int4(0, 0, 0, 0), c3 = c2;
    uint32_t w2 = 0, w3 = 0;
    if (d.G > 2) {
        c2 = ld_stream(g.col4 + tail_at);
        w2 = ld_stream(g.w4 + tail_at);
        if (d.G > 3) {
            c3 = ld_stream(g.col4 + tail_at + kSubRows);
            w3 = ld_stream(g.w4 + tail_at + kSubRows);
        }
    }
    uint32_t flip = 0;
    const uint32_t orig = lds32(ma + 2u * kSweepThreads * 4u);
    const uint32_t parts = d.meta >> 16;
    if (orig != 0xffffffffu && parts == 0u && !bulk)
        flip = flip_mask_part(orig, x.T, x.rep_lane0, x.thr, (uint32_t)sr & (spr - 1), spr, keys);

    int h[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) h[k] = 0;
    {
        const uint4 e0 = lds128(gb + 0 * kSlotBytes), e1 = lds128(gb + 1 * kSlotBytes);
        const uint4 e2 = lds128(gb + 2 * kSlotBytes), e3 = lds128(gb + 3 * kSlotBytes);
        field_cell(h, e0, e1, e2, e3, lds32(ma));
    }
    if (d.G > 1) {
        const uint4 f0 = lds128(gb + 4 * kSlotBytes), f1 = lds128(gb + 5 * kSlotBytes);
        const uint4 f2 = lds128(gb + 6 * kSlotBytes), f3 = lds128(gb + 7 * kSlotBytes);
        field_cell(h, f0, f1, f2, f3, lds32(ma + kSweepThreads * 4u));
    }
    if (d.G > 2) {
        uint4 e0 = ld_nbr(x.src, c2.x), e1 = ld_nbr(x.src, c2.y), e2 = ld_nbr(x.src, c2.z), e3 = ld_nbr(x.src, c2.w);
        if (d.G > 3) {
            const uint4 f0 = ld_nbr(x.src, c3.x), f1 = ld_nbr(x.src, c3.y), f2 = ld_nbr(x.src, c3.z), f3 = ld_nbr(x.src, c3.w);
            field_cell(h, e0, e1, e2, e3, w2);
            field_cell(h, f0, f1, f2, f3, w3);
        } else {
            field_cell(h, e0, e1, e2, e3, w2);
        }
    }
    if (bulk) {
        bulk_deposit(bd, x.tile, d, h, log_spr, owner, rloc);
        return;
    }
    uint4 so4 = make_uint4(0u, 0u, 0u, 0u);
    if (owner) so4 = lds128(gb + 8 * kSlotBytes);

    if (parts != 0u) {   // hub part: sorig = {caller id, hub id, part index, ...}
        const uint32_t orig0 = __shfl_sync(0xffffffffu, orig, 0), hub = __shfl_sync(0xffffffffu, orig, 2);
        part_finish<kKindGS, true>(g, x, d.row0, parts, orig0, hub, h, so4, acc, keys);
        return;
    }
    // warp-level segmented reduction over the sub-rows of one row (fields add, flip bits OR)
    if (log_spr == 4) {
        half_reduce16(h, flip, (int)(threadIdx.x & 1));
    } else {
        for (int lvl = 0; lvl < log_spr; ++lvl) {
#pragma unroll
            for (int k = 0; k < 16; ++k) h[k] += __shfl_xor_sync(0xffffffffu, h[k], 2 << lvl);
            flip |= __shfl_xor_sync(0xffffffffu, flip, 2 << lvl);
        }
    }
    if (owner) row_update<kKindGS>(x, h, so4, bold, finish_flip_mask(flip, x.rep_lane0), row_off, acc);
}

__device__ __forceinline__ PhaseRange ld_range(const PhaseRange* p) {
    const uint2 v = __ldg(reinterpret_cast<const uint2*>(p));
    PhaseRange r;
    r.s0 = v.x; r.s1 = v.y;
    return r;
}

__device__ __forceinline__ PassCtx make_ctx(const uint8_t* src, uint8_t* dst, uint8_t* best, uint32_t cap_mask,
                                            unsigned long long tile_stride, uint32_t tile, int half, uint32_t rep0,
                                            uint32_t thr, uint32_t T, int32_t tie_rule) {
    PassCtx x;
    const size_t o = (size_t)tile * tile_stride + (size_t)half * 16;
    x.src = src + o;
    x.dst = dst + o;
    x.best = best ? best + o : nullptr;
    x.cap16 = (cap_mask >> (half * 16)) & 0xffffu;
    x.rep_lane0 = rep0 + tile * kTile + (uint32_t)half * 16u;
    x.thr = thr;
    x.T = T;
    x.tie_rule = tie_rule;
    x.tile = tile;
    return x;
}

// ---------------------------------------------------------------------------------------------
// k_sweep: colour phases [phase_begin, phase_end) of one sweep in one launch.
// KIND: kKindGS (in place), kKindJacobi (src -> dst), kKindEval (no write).
// WIDE: int32 weights (w4w) and int64 bookkeeping; otherwise int8 weights, dp4a, int32 bookkeeping
// flushed every p.flush_rows rows.  Grid = g.n_cta CTAs of kSweepThreads threads.
// ---------------------------------------------------------------------------------------------
template <int KIND, bool WIDE>
__global__ void __launch_bounds__(kSweepThreads, 1) k_sweep(const SweepParams p) {
    using AccT = typename std::conditional<WIDE, long long, int>::type;
    __shared__ long long s_acc[kMaxPersistReplicas];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sr = lane >> 1, half = lane & 1;
    const uint32_t tiles = p.tiles;
    for (uint32_t i = threadIdx.x; i < tiles * kTile; i += blockDim.x) s_acc[i] = 0;
    __syncthreads();

    AccT acc[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) acc[k] = 0;
    uint32_t rows_acc = 0, acc_tile = 0;

    for (uint32_t ph = p.phase_begin; ph < p.phase_end; ++ph) {
        const PhaseRange pr = ld_range(p.g.ranges + (size_t)ph * p.g.n_cta + blockIdx.x);
        const uint32_t nu = (pr.s1 - pr.s0) * tiles;
        for (uint32_t u = warp; u < nu; u += kWarpsPerCta) {
            const uint32_t s = pr.s0 + u / tiles, tile = u % tiles;
            const SliceHead hd = fetch_head<WIDE>(p.g, s, sr);
            if (tile != acc_tile) {
                flush_acc(acc, s_acc + acc_tile * kTile, lane);
                rows_acc = 0;
                acc_tile = tile;
            }
            const PassCtx x = make_ctx(p.src, p.dst, nullptr, 0u, p.tile_stride, tile, half, p.rep0, p.thr, p.T,
                                       p.tie_rule);
            slice_pass<KIND, WIDE>(p.g, x, hd, s, sr, RegAcc<AccT>{acc}, p.keys);
            if (!WIDE && ++rows_acc >= p.flush_rows) {
                flush_acc(acc, s_acc + acc_tile * kTile, lane);
                rows_acc = 0;
            }
        }
    }
    flush_acc(acc, s_acc + acc_tile * kTile, lane);
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < tiles * kTile; i += blockDim.x) {
        const long long v = s_acc[i];
        if (v != 0) atomicAdd(reinterpret_cast<unsigned long long*>(p.accum + i), (unsigned long long)v);
    }
}

// ---------------------------------------------------------------------------------------------
// k_anneal_gs: the persistent Gauss-Seidel annealer (int8 weights).  Cooperative launch,
// grid = g.n_cta CTAs (one per SM at most), all co-resident.
// ---------------------------------------------------------------------------------------------
constexpr size_t kAnnealDynSmem = 16 * kSweepThreads * sizeof(int) + 2 * (size_t)kGatherBufBytes + kMetaBytes + kDescBytes;   // s_dE, two gather buffers, meta / descriptor slots
constexpr int kPhaseCache = 128;   // virtual phases whose slice ranges are kept in shared memory
constexpr uint32_t kChainSmemBytes = 2u * kGatherBufBytes;   // what the chain may use of the dynamic shared memory (the gather buffers)

struct AnnealParams {
    GraphView g;
    uint8_t* state;                 // [tiles][n][32], updated in place
    uint8_t* best;                  // captured best state, same layout
    unsigned long long tile_stride;
    unsigned long long n;           // rows
    uint32_t tiles;
    uint32_t n_replicas;            // live replicas of this batch (<= tiles * 32)
    uint32_t rep0;                  // global id of replica 0 of this batch
    int32_t tie_rule;
    uint32_t flush_rows;
    uint32_t n_sweeps, sweep_offset;
    const uint32_t* thr;            // DEVICE [n_sweeps]
    long long W;
    const long long* E0;            // [tiles*32] energy of the initial state
    long long* accum;               // [3][tiles*32], zero at launch
    long long* trace;               // [n_sweeps][trace_stride] (column 0 = replica 0 of this batch) or nullptr
    unsigned long long trace_stride;
    long long* E_out;               // [tiles*32]
    long long* best_out;            // [tiles*32]
    int32_t* best_sweep_out;        // [tiles*32]
    unsigned int* barrier;          // zero at launch
    int32_t resume;                 // 1: best_out / best_sweep_out hold the bests of the sweeps before this chunk
    // Virtual phases of a sweep: the colour phases 0 .. n_vphases-1 as slice ranges.  With a chain (chain_on), the
    // last virtual phase is the BULK pseudo-phase: every slice of the chain rows' colour classes, fields deposited in
    // chain.h0 instead of updating the rows; the chain (chain.cuh, DELTA) follows it on CTAs 0 .. 8 * tiles - 1.
    const uint32_t* vphase_slices;  // [n_vphases + 1]
    uint32_t n_vphases;
    uint32_t chain_on;
    ChainView chain;
    // Chain overlap (k_anneal_gs<false, true>, chain_on): virtual phase 0 holds the rows [0, ov_rows) of colour class 0
    // that have no neighbour among the chain's rows.  It runs on the CTAs that are not chain CTAs: for sweep 0 on its
    // own, for sweep t + 1 while the chain finishes sweep t.  The improved mask of sweep t is not known then, so these
    // rows park the value they held in `alt` (same layout as state); the capture into `best` follows once the mask is known.
    uint32_t ov_rows;
    uint8_t* alt;
    unsigned long long* timing;     // diagnostics: [n_vphases + 1][n_cta][8] SM-clock stamps of sweep timing_sweep (0 / 1: arrival at
                                    // / departure from the barrier that ends the virtual phase; row n_vphases: the chain), or nullptr
    uint32_t timing_sweep;
    PhiloxKeys keys;
};

// Grid barrier of the persistent kernel (all CTAs co-resident: cooperative launch).  One
// release-add per CTA on a monotone counter, acquire-polled by thread 0; bar.sync on both sides
// extends the ordering to the whole CTA (PTX memory model: causality order is cumulative).
// pause between two polls of the grid-barrier counter: 148 pollers on one line slow the arrivals down
// (measured on config 5: 0 ns 111.40 ms, 20 ns 110.86, 40 ns 110.82, 100 ns 110.95, 250 ns 111.32)
constexpr unsigned kBarrierBackoffNs = 40;
template <bool CLUSTER>
__device__ __forceinline__ void grid_barrier(unsigned int* counter, unsigned int& epoch, unsigned int n_cta,
                                             unsigned long long* stamp) {
    if (CLUSTER) {   // hardware barrier of the thread-block cluster; release / acquire at cluster scope covers global memory
        asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
        return;
    }
    __syncthreads();
    epoch += n_cta;
    if (stamp && threadIdx.x == 0) stamp[0] = (unsigned long long)clock64();
    if (threadIdx.x == 0 && n_cta > 1) {
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(counter) : "memory");
        unsigned int v;
        for (;;) {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(counter) : "memory");
            if ((int)(v - epoch) >= 0) break;
            __nanosleep(kBarrierBackoffNs);
        }
    }
    __syncthreads();
    if (stamp && threadIdx.x == 0) stamp[1] = (unsigned long long)clock64();
}

template <bool CLUSTER, bool OV>
__global__ void __launch_bounds__(kSweepThreads, 1) k_anneal_gs(const AnnealParams p) {
    static_assert(!(CLUSTER && OV), "the chain overlap belongs to the grid variant");
    __shared__ long long s_acc[kMaxPersistReplicas];
    __shared__ long long s_wacc[kWarpsPerCta][kTile];
    __shared__ uint32_t s_wtile[kWarpsPerCta];
    __shared__ uint32_t s_ps[kPhaseCache + 1];                // first slice of every virtual phase
    __shared__ ChainChunk s_chunks[CLUSTER ? 1 : kChainMaxChunks];
    __shared__ ChainSeg s_segs[CLUSTER ? 1 : kChainMaxSegs];
    __shared__ long long s_cdE[kWarpsPerCta][4];
    // 128-byte alignment matters: a warp's 512-byte row of 16-byte slots must not straddle a fifth 128-byte line
    // (measured: +18 % time when the static arrays happened to end 16 bytes past a line)
    extern __shared__ __align__(128) int s_dE_raw[];         // dynamic: [16][kSweepThreads] per-thread energy increments (SmemAcc)
    int (*s_dE)[kSweepThreads] = reinterpret_cast<int (*)[kSweepThreads]>(s_dE_raw);
    // two gather buffers behind s_dE; gbuf0 / gbuf0 ^ gbuf_flip: this thread's slot 0 in buffer 0 / 1
    const uint32_t gbuf_base = (uint32_t)__cvta_generic_to_shared(s_dE_raw) + 16u * kSweepThreads * (uint32_t)sizeof(int);
    const uint32_t gbuf0 = gbuf_base + threadIdx.x * 16u;
    const uint32_t gbuf_flip = gbuf0 ^ (gbuf0 + kGatherBufBytes);
    PipeAddr pa;
    pa.meta0 = gbuf_base + 2u * kGatherBufBytes + threadIdx.x * 4u;
    pa.desc0 = gbuf_base + 2u * kGatherBufBytes + kMetaBytes + (uint32_t)(threadIdx.x >> 5) * kDescStride;
    __shared__ long long s_E[kMaxPersistReplicas];
    __shared__ long long s_best[kMaxPersistReplicas];
    __shared__ int s_bsweep[kMaxPersistReplicas];
    __shared__ uint32_t s_mask[kMaxPersistReplicas / kTile];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sr = lane >> 1, half = lane & 1;
    // CLUSTER: one thread-block cluster per replica tile (graphs whose phases fit the warps of a few SMs but not one
    // CTA's shared memory): the CTAs of a cluster share nothing with the other clusters, and the barrier between
    // colour phases is the hardware cluster barrier (~0.2 us) instead of the grid barrier (~1 us).  Otherwise: one
    // cooperative grid for all tiles.
    uint32_t cta = blockIdx.x, n_cta = p.g.n_cta, tile0 = 0;
    if (CLUSTER) {
        asm("mov.u32 %0, %%cluster_ctarank;" : "=r"(cta));
        asm("mov.u32 %0, %%cluster_nctarank;" : "=r"(n_cta));
        asm("mov.u32 %0, %%clusterid.x;" : "=r"(tile0));
    }
    const uint32_t tiles = CLUSTER ? 1u : p.tiles, nR = tiles * kTile, VP = p.n_vphases;
    const bool chain_on = !CLUSTER && p.chain_on != 0u;
    const bool chain_cta = chain_on && cta < (uint32_t)kChainGroups * tiles;
    // per-tile views of the launch parameters (grid variant: the parameters themselves, read where they are used)
    auto state = [&]() { return CLUSTER ? p.state + (size_t)tile0 * p.tile_stride : p.state; };
    auto bestp = [&]() { return CLUSTER ? p.best + (size_t)tile0 * p.tile_stride : p.best; };
    auto E0 = [&]() { return CLUSTER ? p.E0 + tile0 * kTile : p.E0; };
    auto accum = [&]() { return CLUSTER ? p.accum + (size_t)tile0 * 3u * kTile : p.accum; };
    auto trace = [&]() { return (CLUSTER && p.trace) ? p.trace + tile0 * kTile : p.trace; };
    auto E_out = [&]() { return CLUSTER ? p.E_out + tile0 * kTile : p.E_out; };
    auto best_out = [&]() { return CLUSTER ? p.best_out + tile0 * kTile : p.best_out; };
    auto best_sweep_out = [&]() { return CLUSTER ? p.best_sweep_out + tile0 * kTile : p.best_sweep_out; };
    auto rep0 = [&]() { return CLUSTER ? p.rep0 + tile0 * kTile : p.rep0; };
    auto n_rep = [&]() { return CLUSTER ? (p.n_replicas > tile0 * kTile ? min(p.n_replicas - tile0 * kTile, nR) : 0u) : p.n_replicas; };
    for (uint32_t i = threadIdx.x; i < nR; i += blockDim.x) {
        s_acc[i] = 0;
        s_E[i] = E0()[i];
        s_best[i] = p.resume ? best_out()[i] : (long long)0x8000000000000000ull;
        s_bsweep[i] = p.resume ? best_sweep_out()[i] : 0;
    }
    if (threadIdx.x < kMaxPersistReplicas / kTile) s_mask[threadIdx.x] = 0u;
    s_wacc[threadIdx.x >> 5][threadIdx.x & 31] = 0;
    for (uint32_t i = threadIdx.x; i <= min(VP, (uint32_t)kPhaseCache); i += blockDim.x) s_ps[i] = __ldg(p.vphase_slices + i);
    // chain CTA (cta = 8 * tile + g owns the word of replicas 4 g .. 4 g + 3 of every chain row of its tile): tables
    // into shared memory, compact copy of the chain rows' current spin words
    const uint32_t ctile = cta / (uint32_t)kChainGroups, cgrp = cta % (uint32_t)kChainGroups;
    if constexpr (!CLUSTER) if (chain_cta) {
        const ChainView& v = p.chain;
        for (uint32_t i = threadIdx.x; i < v.n_chunks * (uint32_t)(sizeof(ChainChunk) / 4); i += blockDim.x)
            reinterpret_cast<uint32_t*>(s_chunks)[i] = __ldg(reinterpret_cast<const uint32_t*>(v.chunks) + i);
        for (uint32_t i = threadIdx.x; i < v.n_segs * (uint32_t)(sizeof(ChainSeg) / 4); i += blockDim.x)
            reinterpret_cast<uint32_t*>(s_segs)[i] = __ldg(reinterpret_cast<const uint32_t*>(v.segs) + i);
        const uint8_t* sp = p.state + (size_t)ctile * p.tile_stride + (size_t)v.row_lo * kTile + 4u * cgrp;
        for (uint32_t r = threadIdx.x; r < v.n_t; r += blockDim.x)
            v.old[(size_t)cta * v.n_t_pad + r] = __ldcg(reinterpret_cast<const uint32_t*>(sp + (size_t)r * kTile));
    }
    __syncthreads();

    const SmemAcc acc{&s_dE[0][threadIdx.x]};
#pragma unroll
    for (int k = 0; k < 16; ++k) s_dE[k][threadIdx.x] = 0;
    uint32_t rows_acc = 0, acc_tile = 0;
    unsigned int epoch = 0;
    BulkDst bd{};
    if (!CLUSTER) { bd.h0 = p.chain.h0; bd.row_lo = p.chain.row_lo; bd.n_t_pad = p.chain.n_t_pad; }

    auto ps_of = [&](uint32_t vp_) { return vp_ <= (uint32_t)kPhaseCache ? s_ps[vp_] : __ldg(p.vphase_slices + vp_); };
    // Slice units of a phase (heaviest first) are dealt out statically: unit k of warp w of CTA b is
    // w * n_cta + b + k * (16 n_cta), so every warp gets the same mix of heavy and light units and the static data of
    // its first unit can be requested across the barrier that precedes the phase.
    const uint32_t n_static = n_cta * (uint32_t)kWarpsPerCta;
    const uint32_t u_static = (uint32_t)warp * n_cta + cta;
    // (OV: virtual phase 0 is dealt out over the CTAs that are not chain CTAs, like this)
    const uint32_t n_chain = OV ? (uint32_t)kChainGroups * tiles : 0u;
    const uint32_t n_static0 = OV ? (n_cta - n_chain) * (uint32_t)kWarpsPerCta : n_static;
    const uint32_t u_static0 = OV ? (chain_cta ? 0xffffffffu : (uint32_t)warp * (n_cta - n_chain) + (cta - n_chain)) : u_static;
    uint32_t ps0 = ps_of(0u);
    uint32_t nu = (ps_of(1u) - ps0) * tiles;
    // one-unit lookahead of the static data, kept across the barrier
    bool have = u_static0 < nu;
    HeadIdx nxt{};
    uint32_t mslot = 0;   // meta slot of the unit whose head is in flight (`nxt`)
    if (have) nxt = tiles == 1u ? request_head(p.g, pa, mslot, ps0 + u_static0, 0u, sr, lane)
                              : request_head(p.g, pa, mslot, ps0 + u_static0 / tiles, u_static0 % tiles, sr, lane);

    for (uint32_t t = 0; t < p.n_sweeps; ++t) {
        const uint32_t thr = __ldg(p.thr + t);
        const uint32_t T = p.sweep_offset + t;
        unsigned long long* const tsw = (!CLUSTER && p.timing && t == p.timing_sweep) ? p.timing + (size_t)cta * 8 : nullptr;
        const bool more_sweeps = t + 1 < p.n_sweeps;
        // OV: one (slice, tile) unit loop more, used beside the chain for virtual phase 0 of sweep t + 1 (same pipeline as
        // the loop of the ordinary phases below; the rows park their previous values in `alt`, see AnnealParams)
        auto run_phase0_parked = [&]() {
            if (!have) return;
            const uint32_t thr_u = __ldg(p.thr + t + 1), T_u = T + 1u;
            SliceDesc pend_d{};
            uint32_t pend_tile = 0;
            uint32_t u_pos = u_static0;
            auto stage_next = [&](uint32_t gb_) {
                pend_d = lds_desc(pa.desc(mslot));
                pend_tile = lds32(pa.desc(mslot) + 16);
                issue_slice_gathers(state() + (size_t)pend_tile * p.tile_stride + (size_t)half * 16, nxt, pend_d, sr, gb_, true);
                if (pend_d.G > (uint32_t)kHeadGroups) {
                    const size_t tail_at = (size_t)pend_d.off + sr;
                    if (half == 0) prefetch_l2(p.g.col4 + tail_at);
                    else if (pend_d.G > (uint32_t)kHeadGroups + 1u) prefetch_l2(p.g.col4 + tail_at + kSubRows);
                    if (lane == 0) prefetch_l2(p.g.w4 + tail_at);
                }
                u_pos += n_static0;
                have = u_pos < nu;
                if (have) {
                    mslot = mslot == kMetaSlots - 1u ? 0u : mslot + 1u;
                    nxt = tiles == 1u ? request_head(p.g, pa, mslot, ps0 + u_pos, 0u, sr, lane)
                                      : request_head(p.g, pa, mslot, ps0 + u_pos / tiles, u_pos % tiles, sr, lane);
                }
            };
            uint32_t gb = gbuf0;
            cp_async_wait<0>();
            __syncwarp();
            uint32_t cur_m = mslot;
            stage_next(gb);
            while (true) {
                const SliceDesc cur_d = pend_d;
                const uint32_t tile = pend_tile;
                const bool more = have;
                const uint32_t nxt_m = mslot;
                cp_async_wait<0>();
                if (more) {
                    __syncwarp();
                    stage_next(gb ^ gbuf_flip);
                }
                if (tile != acc_tile) {
                    flush_warp(acc, s_wacc[warp], lane);
                    fold_warp(s_wacc[warp], s_acc + acc_tile * kTile, lane);
                    rows_acc = 0;
                    acc_tile = tile;
                }
                const PassCtx x = make_ctx(state(), state(), p.alt, 0xffffffffu, p.tile_stride, tile, half, rep0(), thr_u, T_u, p.tie_rule);
                slice_compute(p.g, x, cur_d, pa.meta(cur_m, 0), sr, acc, p.keys, gb, false, bd);
                if (++rows_acc >= p.flush_rows) {
                    flush_warp(acc, s_wacc[warp], lane);
                    rows_acc = 0;
                }
                if (!more) break;
                gb ^= gbuf_flip;
                cur_m = nxt_m;
            }
        };
        for (uint32_t vp = (OV && t > 0u) ? 1u : 0u; vp < VP; ++vp) {
            const bool last_phase = vp + 1 == VP;
            const bool very_last = last_phase && t + 1 == p.n_sweeps;
            const bool bulk = chain_on && last_phase;
            const uint32_t vpn = last_phase ? 0u : vp + 1u;
            const uint32_t psn0 = ps_of(vpn), psn1 = ps_of(vpn + 1u);
            // (OV: virtual phase 0 has its own unit mapping)
            const uint32_t us = (OV && vp == 0u) ? u_static0 : u_static, ns = (OV && vp == 0u) ? n_static0 : n_static;
            const uint32_t usn = (OV && vpn == 0u) ? u_static0 : u_static, nsn = (OV && vpn == 0u) ? n_static0 : n_static;

            if (have) {
                // software pipeline: unit k is computed from gather buffer gb while the gathers of unit k+1 fly
                // into the other buffer and the head of unit k+2 is on its way (indices -> `nxt`, the rest -> its
                // meta slot)
                SliceDesc pend_d{};
                uint32_t pend_tile = 0;
                uint32_t u_pos = us;
                auto stage_next = [&](uint32_t gb_) {   // needs: head of `nxt` landed (cp.async.wait_group 0 + __syncwarp)
                    pend_d = lds_desc(pa.desc(mslot));
                    pend_tile = lds32(pa.desc(mslot) + 16);
                    issue_slice_gathers(state() + (size_t)pend_tile * p.tile_stride + (size_t)half * 16, nxt, pend_d, sr, gb_, !bulk);
                    if (pend_d.G > (uint32_t)kHeadGroups) {   // tail cells: towards L2 now, read when the unit is computed
                        const size_t tail_at = (size_t)pend_d.off + sr;
                        if (half == 0) prefetch_l2(p.g.col4 + tail_at);
                        else if (pend_d.G > (uint32_t)kHeadGroups + 1u) prefetch_l2(p.g.col4 + tail_at + kSubRows);
                        if (lane == 0) prefetch_l2(p.g.w4 + tail_at);
                    }
                    u_pos += ns;
                    have = u_pos < nu;
                    if (have) {
                        mslot = mslot == kMetaSlots - 1u ? 0u : mslot + 1u;
                        nxt = tiles == 1u ? request_head(p.g, pa, mslot, ps0 + u_pos, 0u, sr, lane)
                                          : request_head(p.g, pa, mslot, ps0 + u_pos / tiles, u_pos % tiles, sr, lane);
                    }
                };
                uint32_t gb = gbuf0;
                cp_async_wait<0>();
                __syncwarp();
                uint32_t cur_m = mslot;
                stage_next(gb);
                while (true) {
                    const SliceDesc cur_d = pend_d;
                    const uint32_t tile = pend_tile;
                    const bool more = have;
                    const uint32_t nxt_m = mslot;
                    cp_async_wait<0>();   // gathers of the current unit and, if any, the head of the next one
                    if (more) {
                        __syncwarp();
                        stage_next(gb ^ gbuf_flip);
                    }
                    if (tile != acc_tile) {
                        flush_warp(acc, s_wacc[warp], lane);
                        fold_warp(s_wacc[warp], s_acc + acc_tile * kTile, lane);
                        rows_acc = 0;
                        acc_tile = tile;
                    }
                    PassCtx x = tiles == 1u ? make_ctx(state(), state(), bestp(), s_mask[0], 0ull, 0u, half, rep0(), thr, T, p.tie_rule)
                                            : make_ctx(state(), state(), bestp(), s_mask[tile], p.tile_stride, tile, half, rep0(),
                                                       thr, T, p.tie_rule);
                    if (CLUSTER) x.tile += tile0;   // hub accumulators are indexed by the global tile
                    slice_compute(p.g, x, cur_d, pa.meta(cur_m, 0), sr, acc, p.keys, gb, bulk, bd);
                    if (++rows_acc >= p.flush_rows) {
                        flush_warp(acc, s_wacc[warp], lane);
                        rows_acc = 0;
                    }
                    if (!more) break;
                    gb ^= gbuf_flip;
                    cur_m = nxt_m;
                }
            }

            // static data of this warp's first slice of the next phase: issued before the barrier
            ps0 = psn0;
            nu = (psn1 - psn0) * tiles;
            have = !very_last && usn < nu;
            if (have && usn + nsn < nu) {   // this warp's second unit: head towards L2
                const uint32_t u2 = usn + nsn;
                const uint32_t s2 = ps0 + (tiles == 1u ? u2 : u2 / tiles);
                const size_t at2 = (size_t)s2 * (kHeadGroups * kSubRows) + sr;
                prefetch_l2(half == 0 ? p.g.col4 + at2 : p.g.col4 + at2 + kSubRows);
                if (lane == 0) { prefetch_l2(p.g.w4 + at2); prefetch_l2(p.g.sorig + (size_t)s2 * kSubRows); prefetch_l2(p.g.slices + s2); }
            }
            if (have) {
                mslot = mslot == kMetaSlots - 1u ? 0u : mslot + 1u;
                nxt = tiles == 1u ? request_head(p.g, pa, mslot, ps0 + usn, 0u, sr, lane)
                              : request_head(p.g, pa, mslot, ps0 + usn / tiles, usn % tiles, sr, lane);
            }

            if (last_phase) {   // a7: this sweep's energy increments -> accum slot t % 3
                flush_warp(acc, s_wacc[warp], lane);
                rows_acc = 0;
                if (lane == 0) s_wtile[warp] = acc_tile;
                __syncthreads();
                long long* slot = accum() + (size_t)(t % 3u) * nR;
                if (threadIdx.x < kTile) {   // one add per replica and run of warps on the same tile
                    long long run = 0;
                    uint32_t run_tile = s_wtile[0];
                    for (int wv = 0; wv < kWarpsPerCta; ++wv) {
                        const uint32_t wt = s_wtile[wv];
                        if (wt != run_tile) {
                            if (run != 0)
                                atomicAdd(reinterpret_cast<unsigned long long*>(slot + run_tile * kTile + threadIdx.x),
                                          (unsigned long long)run);
                            run = 0;
                            run_tile = wt;
                        }
                        run += s_wacc[wv][threadIdx.x];
                        s_wacc[wv][threadIdx.x] = 0;
                    }
                    if (run != 0)
                        atomicAdd(reinterpret_cast<unsigned long long*>(slot + run_tile * kTile + threadIdx.x),
                                  (unsigned long long)run);
                }
                for (uint32_t i = threadIdx.x; i < nR; i += blockDim.x) {   // tile hand-overs (several tiles per warp)
                    const long long v = s_acc[i];
                    if (v != 0) {
                        atomicAdd(reinterpret_cast<unsigned long long*>(slot + i), (unsigned long long)v);
                        s_acc[i] = 0;
                    }
                }
            }
            grid_barrier<CLUSTER>(p.barrier, epoch, n_cta, tsw ? tsw + (size_t)vp * n_cta * 8 : nullptr);
        }

        if constexpr (!CLUSTER) if (chain_on) {
            if constexpr (OV) {   // beside the chain: virtual phase 0 of sweep t + 1, then the head of this warp's first unit of phase 1
                if (more_sweeps) run_phase0_parked();
                ps0 = ps_of(1u);
                nu = (ps_of(2u) - ps0) * tiles;
                have = more_sweeps && u_static < nu;
                if (have) {
                    mslot = mslot == kMetaSlots - 1u ? 0u : mslot + 1u;
                    nxt = tiles == 1u ? request_head(p.g, pa, mslot, ps0 + u_static, 0u, sr, lane)
                                      : request_head(p.g, pa, mslot, ps0 + u_static / tiles, u_static % tiles, sr, lane);
                }
            }
            // the chain: the last colour classes level by level inside one CTA per word of four replicas
            if (chain_cta) {
                const ChainView& v = p.chain;
                ChainRt rt;
                rt.thr = thr; rt.T = T; rt.rl0 = p.rep0 + ctile * kTile + 4u * cgrp; rt.tie_rule = p.tie_rule;
                ChainGlobal cgl;

                const size_t o = (size_t)ctile * p.tile_stride + (size_t)v.row_lo * kTile + 4u * cgrp;
                cgl.state = p.state + o;
                cgl.best = p.best + o;
                cgl.old = v.old + (size_t)cta * v.n_t_pad;
                cgl.cap4 = (s_mask[ctile] >> (4u * cgrp)) & 15u;
                long long cdE[4] = {0, 0, 0, 0};
                const uint32_t cflip = gbuf_base + chain_align16(4u * v.n_t_pad);
                chain_pass_streamed<true, true>(v, s_chunks, s_segs, gbuf_base, cflip, cflip + chain_align16(v.n_t_pad), cta, rt,
                                          p.keys, cdE, cgl, threadIdx.x, (uint32_t)kSweepThreads, false,
                                          (tsw && cta == 0 && threadIdx.x == 0) ? p.timing : nullptr, n_cta * 8u);
                chain_reduce_dE(cdE, s_cdE, threadIdx.x, v.narrow != 0u);
                __syncthreads();
                if (threadIdx.x < 4) {
                    const long long v4 = chain_sum_dE(s_cdE, threadIdx.x, (uint32_t)kWarpsPerCta);
                    if (v4 != 0)
                        atomicAdd(reinterpret_cast<unsigned long long*>(p.accum + (size_t)(t % 3u) * nR + ctile * kTile +
                                                                         4u * cgrp + threadIdx.x), (unsigned long long)v4);
                }
            }
            // (diagnostics, OV: the chain step of the sweep before the recorded one is that sweep's virtual phase 0: row 0)
            grid_barrier<CLUSTER>(p.barrier, epoch, n_cta, tsw ? tsw + (size_t)VP * n_cta * 8
                                  : (OV && p.timing && t + 1u == p.timing_sweep) ? p.timing + (size_t)cta * 8 : nullptr);
        }

        // sweep end (every CTA redundantly): E, cut = (W - E)/2 (eq. 4), improved mask
        {
            const long long* slot = accum() + (size_t)(t % 3u) * nR;
            long long* zero_slot = accum() + (size_t)((t + 2u) % 3u) * nR;
            for (uint32_t i = threadIdx.x; i < nR; i += blockDim.x) {   // nR is a multiple of 32: warp-uniform
                const long long E = s_E[i] + __ldcg(slot + i);
                const long long cut = (p.W - E) / 2;
                const bool live = i < n_rep();
                const bool improved = live && cut > s_best[i];
                s_E[i] = E;
                if (improved) { s_best[i] = cut; s_bsweep[i] = (int)T; }
                const uint32_t m = __ballot_sync(0xffffffffu, improved);
                if (lane == 0) s_mask[i >> 5] = m;
                if (cta == 0) {
                    zero_slot[i] = 0;
                    if (live && trace()) trace()[(size_t)t * p.trace_stride + i] = cut;
                }
            }
            __syncthreads();
        }
        // chain overlap: the rows of virtual phase 0 were updated for sweep t + 1 before this sweep's improved mask
        // was known; the values they held (parked in `alt`) are captured now
        if constexpr (OV) if (more_sweeps) {
            for (uint32_t tile = 0; tile < tiles; ++tile) {
                const uint32_t mask = s_mask[tile];
                if (mask == 0u) continue;
                const uint4* alt = reinterpret_cast<const uint4*>(p.alt + (size_t)tile * p.tile_stride);
                uint4* best = reinterpret_cast<uint4*>(bestp() + (size_t)tile * p.tile_stride);
                const uint32_t m_lo = mask & 0xffffu, m_hi = mask >> 16;
                const uint32_t units = p.ov_rows * 2u;
                for (uint32_t uu = cta * blockDim.x + threadIdx.x; uu < units; uu += n_cta * blockDim.x) {
                    const uint32_t m = (uu & 1u) ? m_hi : m_lo;
                    if (m == 0u) continue;
                    const uint4 v = __ldcg(alt + uu);
                    if (m == 0xffffu) { best[uu] = v; continue; }
                    uint4 b = __ldcg(best + uu);
                    const uint32_t k0 = nibble_to_bytemask(m & 15u), k1 = nibble_to_bytemask((m >> 4) & 15u);
                    const uint32_t k2 = nibble_to_bytemask((m >> 8) & 15u), k3 = nibble_to_bytemask((m >> 12) & 15u);
                    b.x = (v.x & k0) | (b.x & ~k0);
                    b.y = (v.y & k1) | (b.y & ~k1);
                    b.z = (v.z & k2) | (b.z & ~k2);
                    b.w = (v.w & k3) | (b.w & ~k3);
                    best[uu] = b;
                }
            }
        }
    }

    // capture of the improvements of the final sweep (earlier ones were captured in flight)
    for (uint32_t tile = 0; tile < tiles; ++tile) {
        const uint32_t mask = s_mask[tile];
        if (mask == 0u) continue;
        const uint4* src = reinterpret_cast<const uint4*>(state() + (size_t)tile * p.tile_stride);
        uint4* best = reinterpret_cast<uint4*>(bestp() + (size_t)tile * p.tile_stride);
        const uint32_t m_lo = mask & 0xffffu, m_hi = mask >> 16;
        const unsigned long long units = p.n * 2ull;
        for (unsigned long long uu = (unsigned long long)cta * blockDim.x + threadIdx.x; uu < units;
             uu += (unsigned long long)n_cta * blockDim.x) {
            const uint32_t m = (uu & 1ull) ? m_hi : m_lo;
            if (m == 0u) continue;
            const uint4 s = __ldcg(src + uu);
            if (m == 0xffffu) { best[uu] = s; continue; }
            uint4 b = __ldcg(best + uu);
            const uint32_t k0 = nibble_to_bytemask(m & 15u), k1 = nibble_to_bytemask((m >> 4) & 15u);
            const uint32_t k2 = nibble_to_bytemask((m >> 8) & 15u), k3 = nibble_to_bytemask((m >> 12) & 15u);
            b.x = (s.x & k0) | (b.x & ~k0);
            b.y = (s.y & k1) | (b.y & ~k1);
            b.z = (s.z & k2) | (b.z & ~k2);
            b.w = (s.w & k3) | (b.w & ~k3);
            best[uu] = b;
        }
    }
    if (cta == 0) {
        for (uint32_t i = threadIdx.x; i < nR; i += blockDim.x) {
            E_out()[i] = s_E[i];
            best_out()[i] = s_best[i];
            best_sweep_out()[i] = s_bsweep[i];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Sweep end: per replica cut = (W - E)/2 (eq. 4), trace, best-state capture (a7).
// Every CTA recomputes the "improved" mask of its tile from the previous-parity
// bookkeeping arrays; CTA x == 0 of each tile writes the next-parity arrays, so no CTA reads
// what another writes.  energy_mode: 0  E_new = E_old + accum (Gauss-Seidel increments),
// 1  E_new = accum / 2 (Jacobi / evaluation: accum = sum_i s_i h_i), 2  as 1 but only
// records E (initial energy; no candidate, no trace).
// ---------------------------------------------------------------------------------------------
struct SweepEndParams {
    const uint8_t* src;            // state holding the candidate (after the sweep)
    uint8_t* best;                 // captured best state, same layout
    const long long* accum_in;     // parity p
    long long* accum_zero;         // parity p^1 (zeroed for the next sweep)
    const long long* E_in;         // parity p
    long long* E_out;              // parity p^1
    const long long* best_in;      // parity p
    long long* best_out;           // parity p^1
    int32_t* best_sweep;
    long long* trace_row;          // [n_replicas] or nullptr
    unsigned long long tile_stride;
    unsigned long long units;      // uint4 units per tile = n * 2
    long long W;
    int32_t n_replicas;
    int32_t energy_mode;
    int32_t first;                 // 1: no best recorded yet in this call
    int32_t T;
};

__global__ void __launch_bounds__(256) k_sweep_end(const SweepEndParams p) {
    __shared__ uint32_t s_mask;
    const uint32_t tile = blockIdx.y;
    if (threadIdx.x < 32) {
        const int r = (int)threadIdx.x;
        const size_t idx = (size_t)tile * kTile + r;
        const bool live = (int)(tile * kTile) + r < p.n_replicas;
        const long long a = p.accum_in[idx];
        const long long E = p.energy_mode == 0 ? p.E_in[idx] + a : a / 2;
        const long long cut = (p.W - E) / 2;
        const long long bprev = p.best_in[idx];
        const bool improved = live && p.energy_mode != 2 && (p.first || cut > bprev);
        const uint32_t mask = __ballot_sync(0xffffffffu, improved);
        if (r == 0) s_mask = mask;
        if (blockIdx.x == 0) {
            p.E_out[idx] = E;
            p.accum_zero[idx] = 0;
            p.best_out[idx] = improved ? cut : bprev;
            if (improved) p.best_sweep[idx] = p.T;
            if (live && p.trace_row && p.energy_mode != 2) p.trace_row[idx] = cut;
        }
    }
    __syncthreads();
    const uint32_t mask = s_mask;
    if (mask == 0) return;
    const uint4* src = reinterpret_cast<const uint4*>(p.src + (size_t)tile * p.tile_stride);
    uint4* best = reinterpret_cast<uint4*>(p.best + (size_t)tile * p.tile_stride);
    // unit u covers replicas (u & 1) * 16 .. +15 of row u >> 1
    const uint32_t m_lo = mask & 0xffffu, m_hi = mask >> 16;
    for (unsigned long long u = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; u < p.units;
         u += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t m = (u & 1ull) ? m_hi : m_lo;
        if (m == 0) continue;
        const uint4 s = src[u];
        if (m == 0xffffu) { best[u] = s; continue; }
        uint4 b = best[u];
        const uint32_t k0 = nibble_to_bytemask(m & 15u), k1 = nibble_to_bytemask((m >> 4) & 15u);
        const uint32_t k2 = nibble_to_bytemask((m >> 8) & 15u), k3 = nibble_to_bytemask((m >> 12) & 15u);
        b.x = (s.x & k0) | (b.x & ~k0);
        b.y = (s.y & k1) | (b.y & ~k1);
        b.z = (s.z & k2) | (b.z & ~k2);
        b.w = (s.w & k3) | (b.w & ~k3);
        best[u] = b;
    }
}

// ---------------------------------------------------------------------------------------------
// State initialisation / import / export
// ---------------------------------------------------------------------------------------------
// Philox INIT domain (Q4): s = (philox(seed; ctr=(i, 0, r>>2, 1))[r&3] & 1) ? +1 : -1.
__global__ void k_init_philox(uint8_t* state, const int32_t* perm, uint32_t n, unsigned long long tile_stride,
                              uint32_t rep0, const PhiloxKeys keys) {
    const uint32_t tile = blockIdx.y;
    const unsigned long long u = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;   // (row, half)
    if (u >= 2ull * n) return;
    const uint32_t row = (uint32_t)(u >> 1), half = (uint32_t)(u & 1);
    const uint32_t orig = (uint32_t)perm[row];
    const uint32_t rbase = rep0 + tile * kTile + half * 16;
    uint32_t out[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        uint32_t word = 0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const uint32_t rep = rbase + 4 * k + b;
            const uint4 v = philox4x32_10(orig, 0u, rep >> 2, kDomainInit, keys);   // CSE'd when aligned
            const uint32_t w = (rep & 3u) == 0 ? v.x : (rep & 3u) == 1 ? v.y : (rep & 3u) == 2 ? v.z : v.w;
            const uint32_t byte = (w & 1u) ? 0x01u : 0xffu;
            word |= byte << (8 * b);
        }
        out[k] = word;
    }
    *reinterpret_cast<uint4*>(state + (size_t)tile * tile_stride + (size_t)row * kTile + half * 16) =
        make_uint4(out[0], out[1], out[2], out[3]);
}

// caller layout [R][n] (caller ids) -> internal; replicas >= n_replicas are padded with -1.
__global__ void k_import(uint8_t* state, const int8_t* in, const int32_t* perm, uint32_t n,
                         unsigned long long tile_stride, int32_t n_replicas, int* bad_flag) {
    const uint32_t tile = blockIdx.y;
    const unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;   // (row, rr)
    if (t >= (unsigned long long)n * kTile) return;
    const uint32_t row = (uint32_t)(t >> 5), rr = (uint32_t)(t & 31);
    const int rep = (int)(tile * kTile + rr);
    int8_t v = -1;
    if (rep < n_replicas) {
        v = in[(size_t)rep * n + (uint32_t)perm[row]];
        if (v != 1 && v != -1) { atomicOr(bad_flag, 1); v = -1; }
    }
    state[(size_t)tile * tile_stride + (size_t)row * kTile + rr] = (uint8_t)v;
}

// internal -> caller layout; replica_sel >= 0 exports that single replica to out[n].
__global__ void k_export(const uint8_t* state, int8_t* out, const int32_t* perm, uint32_t n,
                         unsigned long long tile_stride, int32_t n_replicas, int32_t replica_sel) {
    if (replica_sel >= 0) {
        const unsigned long long row = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
        if (row >= n) return;
        const uint32_t tile = (uint32_t)replica_sel / kTile, rr = (uint32_t)replica_sel % kTile;
        out[(uint32_t)perm[row]] = (int8_t)state[(size_t)tile * tile_stride + row * kTile + rr];
        return;
    }
    const uint32_t tile = blockIdx.y;
    const unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (unsigned long long)n * kTile) return;
    const uint32_t row = (uint32_t)(t >> 5), rr = (uint32_t)(t & 31);
    const int rep = (int)(tile * kTile + rr);
    if (rep < n_replicas)
        out[(size_t)rep * n + (uint32_t)perm[row]] = (int8_t)state[(size_t)tile * tile_stride + (size_t)row * kTile + rr];
}

// Algorithm 1's flip step ("randomly choose and flip N spin glasses"): after a
// sweep of pure local minimisation exactly N DISTINCT spins of every replica are flipped.  The N-subset is drawn by
// Floyd's algorithm: for j = n-N .. n-1: x = floor(u (j+1) / 2^32) with u = philox(seed; ctr = (j - (n-N), T,
// r>>2, FLIPN))[r&3]; x is taken unless it was taken before, then j is.  One warp per replica: the draws are
// sequential by definition, the membership scan over the spins chosen so far is spread over the lanes.
constexpr int kMaxExactN = 4096;
__global__ void __launch_bounds__(32) k_flip_exact(uint8_t* state, const int32_t* inv, uint32_t n, uint32_t N, uint32_t T,
                                                    uint32_t rep0, unsigned long long tile_stride, const PhiloxKeys keys) {
    __shared__ uint32_t chosen[kMaxExactN];
    const uint32_t r = blockIdx.x, rep = rep0 + r, lane = threadIdx.x;
    if (N > n) N = n;
    for (uint32_t k = 0; k < N; ++k) {
        const uint32_t j = n - N + k;
        const uint4 v = philox4x32_10(k, T, rep >> 2, kDomainFlipN, keys);
        const uint32_t u = (rep & 3u) == 0 ? v.x : (rep & 3u) == 1 ? v.y : (rep & 3u) == 2 ? v.z : v.w;
        uint32_t x = (uint32_t)(((unsigned long long)u * (unsigned long long)(j + 1u)) >> 32);
        bool taken = false;
        for (uint32_t c = lane; c < k; c += 32) taken = taken || chosen[c] == x;
        if (__any_sync(0xffffffffu, taken)) x = j;
        __syncwarp();
        if (lane == 0) chosen[k] = x;
        __syncwarp();
    }
    uint8_t* base = state + (size_t)(r / kTile) * tile_stride + (r % kTile);
    for (uint32_t c = lane; c < N; c += 32) {
        uint8_t* q = base + (size_t)(uint32_t)inv[chosen[c]] * kTile;
        *q = (uint8_t)(*q ^ 0xfeu);   // +1 <-> -1; distinct spins, so no two lanes touch the same byte
    }
}

// energy_out / cut_out from an evaluation accumulator (accum = sum_i s_i h_i = 2 E).
__global__ void k_finish_energy(const long long* accum, long long W, int32_t n_replicas, long long* energy_out,
                                long long* cut_out) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_replicas) return;
    const long long E = accum[r] / 2;
    if (energy_out) energy_out[r] = E;
    if (cut_out) cut_out[r] = (W - E) / 2;
}

}  // namespace ising
