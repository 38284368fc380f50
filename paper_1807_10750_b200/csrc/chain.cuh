// Shared-memory chain engine: colour-class Gauss-Seidel levels executed by ONE CTA per group of four replicas, with a
// __syncthreads between colour classes instead of a grid / cluster barrier.
//
// Replicas never interact ("a number of GPU simulations"), so a CTA that owns ALL rows of a
// set of colour classes for four replicas (one 32-bit word of spin bytes per row) needs no other CTA to walk through
// these classes in order.  Two uses:
//   FULL  (k_anneal_small): the whole graph is the chain.  val[row] = the four spin bytes, cells hold every edge; all
//         sweeps x colour classes of an ising_anneal call run without any global synchronisation and, when the packed
//         graph fits shared memory ("resident"), without global traffic inside a sweep except trace / best capture.
//         This is the small-graph regime of the paper's own benchmarks (800 .. 20 000 vertices, Table III).
//   DELTA (tail of k_anneal_gs): the chain rows are the last colour classes of a big graph (few rows, hub-like, a
//         dependent level per class).  Their local fields are first computed by the whole grid from the values all
//         spins hold BEFORE the chain ("bulk" pseudo-phase, h0); the chain then only adds, per row, the corrections
//         w * (new - old) of its LOWER-coloured chain neighbours, which it keeps in shared memory: val[row] = new - old
//         per replica byte (0 / +2 / -2), written when the row is updated and read only by later levels.
// Layout: a chain row's cells hold 4 edges each: four 16-bit LOCAL neighbour ids (uint2) + four int8 weights (one
// word), padded with weight 0.  Rows are cut into CHUNKS (row ranges, 8-row aligned, first cell 4-aligned) that fit
// one shared-memory buffer; a chunk is fetched with 16-byte cp.async by all threads and holds, block after block:
// 16-bit cell pointers relative to the chunk, [DELTA: h0 (int4 per row) and the rows' current spin words], neighbour
// ids, weights.  SEGMENTS = runs of rows of one level inside one chunk; L lanes share a row (its cells strided over
// the lanes, fields summed by a butterfly).  The flip decisions (state-independent) are drawn ahead of the levels, one
// Philox call per row and thread, into a byte per row of shared memory.
#pragma once
#include "common.cuh"
#include "primitives.cuh"

namespace ising {

constexpr int kChainGroups = 8;                 // chain CTAs per replica tile: four replicas (one spin word) each
constexpr uint32_t kChainMaxLocal = 65535;      // local row ids are 16 bit
constexpr int kChainMaxChunks = 96;
constexpr int kChainMaxSegs = 192;
constexpr int kSmallThreadsMax = 512;           // (measured on configs 1-3: 512 threads are as fast as or faster than 1024)

struct ChainSeg {
    uint32_t r0, r1;   // local rows [r0, r1) of one level, inside one chunk
    uint32_t info;     // bits 0-7: log2(lanes per row); bit 8: the level ends with this segment (CTA barrier follows);
                       // bit 9: more rows than the planned CTA has lane groups (a thread walks several rows)
    uint32_t pad;
};
struct ChainChunk {
    uint32_t r0, r1;   // local rows [r0, r1); r0 is a multiple of 8
    uint32_t c0, c1;   // cells [c0, c1); both multiples of 4
    uint32_t ptr_at;   // first entry of this chunk in rel16 (multiple of 8): r1 - r0 + 1 pointers relative to c0
    uint32_t seg0, seg1;
    uint32_t pad;
};

struct ChainView {
    const ChainChunk* chunks;
    const ChainSeg* segs;
    const uint16_t* rel16;
    const uint32_t* orig;    // [n_t_pad] caller id of local row r (Philox counter word 0)
    const uint2* cidx;       // [cells] four 16-bit local neighbour ids
    const uint32_t* cw;      // [cells] four int8 weights
    int* h0;                 // DELTA: [tiles][8][n_t_pad][4] local fields from the pre-chain values (zero between sweeps)
    uint32_t* old;           // DELTA: [tiles][8][n_t_pad] compact copy of the chain rows' spin words
    uint32_t n_chunks, n_segs;
    uint32_t n_t, n_t_pad;   // chain rows, padded to a multiple of 8
    uint32_t row_lo;         // internal row of local row 0
    uint32_t resident;       // FULL: one chunk that stays in shared memory for the whole call
    uint32_t buf_bytes;      // capacity of one chunk buffer
    uint32_t threads;        // CTA size the segments' lanes-per-row were planned for
    uint32_t narrow;         // a sweep's energy increments of all chain rows fit int32
    uint32_t premul;         // the cells hold byte offsets into val[] (n_t_pad <= 16384), else local ids
};

struct ChunkLayout { uint32_t ptr, h0, old, idx, w, bytes; };
__host__ __device__ inline uint32_t chain_align16(uint32_t x) { return (x + 15u) & ~15u; }
__host__ __device__ inline ChunkLayout chunk_layout(uint32_t R, uint32_t Nc, bool delta) {
    ChunkLayout l;
    uint32_t at = 0;
    l.ptr = at;  at += chain_align16(2u * (R + 1u));
    l.h0 = at;   if (delta) at += 16u * R;
    l.old = at;  if (delta) at += chain_align16(4u * R);
    l.idx = at;  at += 8u * Nc;
    l.w = at;    at += 4u * Nc;
    l.bytes = at;
    return l;
}

__device__ __forceinline__ uint2 lds64(uint32_t smem_addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(smem_addr));
    return v;
}
__device__ __forceinline__ uint32_t lds16(uint32_t smem_addr) {
    uint32_t v;
    asm volatile("{ .reg .u16 t; ld.shared.u16 t, [%1]; cvt.u32.u16 %0, t; }" : "=r"(v) : "r"(smem_addr));
    return v;
}

// All threads of the CTA: request chunk `ck` into the buffer at shared address `buf` (one commit group).
template <bool DELTA>
__device__ __forceinline__ void chain_issue_chunk(const ChainView& v, const ChainChunk& ck, uint32_t buf, uint32_t slot,
                                                  uint32_t tid, uint32_t nthr) {
    const uint32_t R = ck.r1 - ck.r0, Nc = ck.c1 - ck.c0;
    const ChunkLayout l = chunk_layout(R, Nc, DELTA);
    const size_t srow = (size_t)slot * v.n_t_pad + ck.r0;
    for (uint32_t off = tid << 4; off < l.bytes; off += nthr << 4) {
        const char* src;
        if (off >= l.w) src = reinterpret_cast<const char*>(v.cw + ck.c0) + (off - l.w);
        else if (off >= l.idx) src = reinterpret_cast<const char*>(v.cidx + ck.c0) + (off - l.idx);
        else if (DELTA && off >= l.old) src = reinterpret_cast<const char*>(v.old + srow) + (off - l.old);
        else if (DELTA && off >= l.h0) src = reinterpret_cast<const char*>(v.h0 + srow * 4) + (off - l.h0);
        else src = reinterpret_cast<const char*>(v.rel16 + ck.ptr_at) + off;
        cp_async16(buf + off, src);
    }
    cp_async_commit();
}

struct ChainRt {             // per sweep
    uint32_t thr, T;
    uint32_t rl0;            // global id of replica 0 of this CTA's word
    int32_t tie_rule;
};

// Flip bits (Alg. 2, reading Q11) of the four replicas rl0 .. rl0+3 of spin `orig` in sweep T.
__device__ __forceinline__ uint32_t chain_flip4(uint32_t orig, const ChainRt& rt, const PhiloxKeys& keys) {
    const uint32_t cw = rt.rl0 >> 2, sh = rt.rl0 & 3u;
    uint32_t m = lt4(philox4x32_10(orig, rt.T, cw, kDomainFlip, keys), rt.thr);
    if (sh) m = ((m | (lt4(philox4x32_10(orig, rt.T, cw + 1u, kDomainFlip, keys), rt.thr) << 4)) >> sh) & 15u;
    return m;
}

// Flip nibbles of local rows [r0, r1) into flip[] (one byte per row), one row per thread.
__device__ __forceinline__ void chain_draw_flips(const ChainView& v, uint32_t flip, uint32_t r0, uint32_t r1,
                                                 const ChainRt& rt, const PhiloxKeys& keys, uint32_t tid, uint32_t nthr) {
    if (rt.thr == 0u) return;
    for (uint32_t r = r0 + tid; r < r1; r += 4u * nthr) {   // four rows at a time: the loads and the Philox chains interleave
        uint32_t o[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) o[j] = r + j * nthr < r1 ? __ldg(v.orig + r + j * nthr) : 0u;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (r + j * nthr < r1) {
                const uint32_t f = chain_flip4(o[j], rt, keys);
                asm volatile("st.shared.u8 [%0], %1;" ::"r"(flip + r + j * nthr), "r"(f) : "memory");
            }
        }
    }
}
__device__ __forceinline__ uint32_t lds8(uint32_t smem_addr) {
    uint32_t v;
    asm volatile("{ .reg .u16 t; ld.shared.u8 t, [%1]; cvt.u32.u16 %0, t; }" : "=r"(v) : "r"(smem_addr));
    return v;
}

// DELTA-only global targets of a chain CTA (its word of every chain row).
struct ChainGlobal {
    uint8_t* state;      // &state[tile][row_lo][4 g]   (row stride kTile)
    uint8_t* best;       // same position in the captured best state
    uint32_t* old;       // compact copy [n_t_pad] of this CTA
    uint32_t cap4;       // capture mask of this CTA's four replicas (improved in the previous sweep)
};
__device__ __forceinline__ uint32_t mapa_u32(uint32_t smem_addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_u32(uint32_t cluster_addr, uint32_t v) {
    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(cluster_addr), "r"(v) : "memory");
}
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// mbarrier hand-off between the two CTAs of a cluster (k_anneal_small, flip producer / level consumer)
__device__ __forceinline__ void mbar_init_cta(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_bar) {   // release at cluster scope
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
// (no data is published: the arriving CTA only says that its loads of a buffer have returned, which the CTA barrier before
// the call has already made certain; a release here would cost a device-wide fence on the critical path)
__device__ __forceinline__ void mbar_arrive_remote_relaxed(uint32_t cluster_bar) {
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {   // acquire at cluster scope
    asm volatile(
        "{\n\t.reg .pred p;\n"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t"
        "@!p bra WAIT_%=;\n\t}"
        ::"r"(bar), "r"(parity) : "memory");
}

// One segment: every row takes its energy-minimising value (L47-49, Q1/Q3), the scheduled flip (L177), and its
// energy increment dE = (a - s) h is added to dE[] (a7; exact because a colour class is an independent set).
// PREMUL: the cells hold BYTE offsets into val[] (local id x 4: chains of at most 16 384 rows), not local ids.
// N32: the energy increments of a thread's rows are added up in 32 bits inside the segment (the chain is `narrow`: all
// its sums fit) and widened once at the end: one IMAD per value (segments of several rows per thread).
template <bool DELTA, bool PREMUL, bool N32 = false>
__device__ __forceinline__ void chain_segment(const ChainSeg sg, const ChainChunk& ck, uint32_t buf, uint32_t val,
                                              uint32_t flip, const ChainRt& rt, const PhiloxKeys& keys, long long (&dE)[4],
                                              const ChainGlobal& cg, uint32_t tid, uint32_t nthr) {
    const uint32_t logL = sg.info & 0xffu, L = 1u << logL, q = tid & (L - 1u);
    const uint32_t rpi = nthr >> logL;
    const ChunkLayout l = chunk_layout(ck.r1 - ck.r0, ck.c1 - ck.c0, DELTA);
    const uint32_t s_lo = sg.r0, s_hi = sg.r1;
    const uint32_t fmask = rt.thr != 0u ? 15u : 0u;
    int e0s = 0, e1s = 0, e2s = 0, e3s = 0;
    uint32_t r = s_lo + (tid >> logL);
    for (uint32_t rw = s_lo + ((tid & ~31u) >> logL); rw < s_hi; rw += rpi, r += rpi) {   // warp-uniform trip count
        // every lane runs the whole update on a valid row (no divergence); the first lane of a live row stores it
        const bool storer = r < s_hi && q == 0u;
        const uint32_t rowc = min(r, s_hi - 1u), lr = rowc - ck.r0;
        const uint32_t p0 = lds16(buf + l.ptr + 2u * lr), p1 = lds16(buf + l.ptr + 2u * lr + 2u);
        const uint32_t f4 = lds8(flip + rowc) & fmask;
        uint32_t oldw;
        int h0 = 0, h1 = 0, h2 = 0, h3 = 0;
        if (DELTA) {
            oldw = lds32(buf + l.old + 4u * lr);
            if (q == 0u) {
                const uint4 hh = lds128(buf + l.h0 + 16u * lr);
                h0 = (int)hh.x; h1 = (int)hh.y; h2 = (int)hh.z; h3 = (int)hh.w;
            }
        } else {
            oldw = lds32(val + 4u * rowc);
        }
        for (uint32_t k = p0 + q; k < p1; k += L) {
            const uint2 ix = lds64(buf + l.idx + 8u * k);
            const uint32_t w = lds32(buf + l.w + 4u * k);
            uint32_t e0, e1, e2, e3;
            if (PREMUL) {
                e0 = lds32(val + (ix.x & 0xffffu)); e1 = lds32(val + (ix.x >> 16));
                e2 = lds32(val + (ix.y & 0xffffu)); e3 = lds32(val + (ix.y >> 16));
            } else {
                e0 = lds32(val + 4u * (ix.x & 0xffffu)); e1 = lds32(val + 4u * (ix.x >> 16));
                e2 = lds32(val + 4u * (ix.y & 0xffffu)); e3 = lds32(val + 4u * (ix.y >> 16));
            }
            uint32_t t0, t1, t2, t3;
            transpose4x4(e0, e1, e2, e3, t0, t1, t2, t3);
            h0 = __dp4a((int)t0, (int)w, h0);
            h1 = __dp4a((int)t1, (int)w, h1);
            h2 = __dp4a((int)t2, (int)w, h2);
            h3 = __dp4a((int)t3, (int)w, h3);
        }
        // (a REDUX per group member mask was measured 3x slower than the butterfly: the groups of a warp are serialised)
        // exactly log2(L) butterfly levels, entered by one jump (the order of the levels does not matter for a sum)
#define ISING_BFLY(o) h0 += __shfl_xor_sync(0xffffffffu, h0, o); h1 += __shfl_xor_sync(0xffffffffu, h1, o); \
                      h2 += __shfl_xor_sync(0xffffffffu, h2, o); h3 += __shfl_xor_sync(0xffffffffu, h3, o);
        if (L > 1u) switch (logL) {
            case 5: ISING_BFLY(16)   // fall through
            case 4: ISING_BFLY(8)    // fall through
            case 3: ISING_BFLY(4)    // fall through
            case 2: ISING_BFLY(2)    // fall through
            case 1: ISING_BFLY(1)    // fall through
            default: break;
        }
#undef ISING_BFLY
        uint32_t a = ~sign_bytes(h0, h1, h2, h3) | 0x01010101u;   // +1 where h < 0, else -1
        if (rt.tie_rule == 1) {                                   // KEEP: h == 0 leaves the spin
            const uint32_t z = (h0 == 0 ? 0xffu : 0u) | (h1 == 0 ? 0xff00u : 0u) | (h2 == 0 ? 0xff0000u : 0u) |
                               (h3 == 0 ? 0xff000000u : 0u);
            a = (a & ~z) | (oldw & z);
        }
        a ^= ((f4 * 0x00204081u) & 0x01010101u) * 0xfeu;
        const uint32_t d2 = storer ? (a << 1) & (a ^ oldw) : 0u;  // a - s per byte: 0, +2, -2
        if (N32) {
            e0s += sbyte(d2, 0) * h0; e1s += sbyte(d2, 1) * h1; e2s += sbyte(d2, 2) * h2; e3s += sbyte(d2, 3) * h3;
        } else {
            asm("mad.wide.s32 %0, %1, %2, %0;" : "+l"(dE[0]) : "r"(sbyte(d2, 0)), "r"(h0));
            asm("mad.wide.s32 %0, %1, %2, %0;" : "+l"(dE[1]) : "r"(sbyte(d2, 1)), "r"(h1));
            asm("mad.wide.s32 %0, %1, %2, %0;" : "+l"(dE[2]) : "r"(sbyte(d2, 2)), "r"(h2));
            asm("mad.wide.s32 %0, %1, %2, %0;" : "+l"(dE[3]) : "r"(sbyte(d2, 3)), "r"(h3));
        }
        if (storer) {
            if (DELTA) {
                sts32(val + 4u * rowc, d2);
                const size_t at = (size_t)rowc * kTile;
                if (d2 != 0u) {
                    *reinterpret_cast<uint32_t*>(cg.state + at) = a;
                    cg.old[rowc] = a;
                }
                if (cg.cap4 != 0u) {   // fused best-state capture: the value the row held after the previous sweep
                    uint32_t* bp = reinterpret_cast<uint32_t*>(cg.best + at);
                    if (cg.cap4 == 15u) {
                        *bp = oldw;
                    } else {
                        const uint32_t km = nibble_to_bytemask(cg.cap4);
                        *bp = (oldw & km) | (__ldcg(bp) & ~km);
                    }
                }
            } else {
                sts32(val + 4u * rowc, a);
            }
        }
    }
    if (N32) { dE[0] += e0s; dE[1] += e1s; dE[2] += e2s; dE[3] += e3s; }
}

// chain_segment<false, PREMUL, true> for segments in which a thread walks SEVERAL rows (throughput-bound levels: config
// 3's checkerboard classes, the big classes of config 2): two rows per trip.  The rows of a level are independent, so
// the two dependent chains (cell pointers -> neighbour offsets -> spin words -> dp4a -> butterfly -> update) interleave.
// A row that has run out of cells rides along on cell 0 of the chunk with weight 0.
template <bool PREMUL>
__device__ __forceinline__ void chain_segment_rows2(const ChainSeg sg, const ChainChunk& ck, uint32_t buf, uint32_t val,
                                                    uint32_t flip, const ChainRt& rt, long long (&dE)[4], uint32_t tid,
                                                    uint32_t nthr) {
    const uint32_t logL = sg.info & 0xffu, L = 1u << logL, q = tid & (L - 1u);
    const uint32_t rpi = nthr >> logL;
    const ChunkLayout l = chunk_layout(ck.r1 - ck.r0, ck.c1 - ck.c0, false);
    const uint32_t s_lo = sg.r0, s_hi = sg.r1;
    const uint32_t fmask = rt.thr != 0u ? 15u : 0u;
    int es0 = 0, es1 = 0, es2 = 0, es3 = 0;
    uint32_t r = s_lo + (tid >> logL);
    for (uint32_t rw = s_lo + ((tid & ~31u) >> logL); rw < s_hi; rw += 2u * rpi, r += 2u * rpi) {   // warp-uniform trip count
        const uint32_t rB = r + rpi;
        const bool stA = r < s_hi && q == 0u, stB = rB < s_hi && q == 0u;
        const uint32_t rowA = min(r, s_hi - 1u), rowB = min(rB, s_hi - 1u);
        const uint32_t lrA = rowA - ck.r0, lrB = rowB - ck.r0;
        const uint32_t p0A = lds16(buf + l.ptr + 2u * lrA), p1A = lds16(buf + l.ptr + 2u * lrA + 2u);
        const uint32_t p0B = lds16(buf + l.ptr + 2u * lrB), p1B = lds16(buf + l.ptr + 2u * lrB + 2u);
        const uint32_t fA = lds8(flip + rowA) & fmask, fB = lds8(flip + rowB) & fmask;
        const uint32_t oldA = lds32(val + 4u * rowA), oldB = lds32(val + 4u * rowB);
        int a0 = 0, a1 = 0, a2 = 0, a3 = 0, b0 = 0, b1 = 0, b2 = 0, b3 = 0;
        uint32_t kA = p0A + q, kB = p0B + q;
        while (kA < p1A || kB < p1B) {
            const bool ha = kA < p1A, hb = kB < p1B;
            const uint32_t ka = ha ? kA : 0u, kb = hb ? kB : 0u;
            const uint2 ix = lds64(buf + l.idx + 8u * ka), jx = lds64(buf + l.idx + 8u * kb);
            uint32_t wa = lds32(buf + l.w + 4u * ka), wb = lds32(buf + l.w + 4u * kb);
            wa = ha ? wa : 0u;
            wb = hb ? wb : 0u;
            uint32_t e0, e1, e2, e3, f0, f1, f2, f3;
            if (PREMUL) {
                e0 = lds32(val + (ix.x & 0xffffu)); e1 = lds32(val + (ix.x >> 16));
                e2 = lds32(val + (ix.y & 0xffffu)); e3 = lds32(val + (ix.y >> 16));
                f0 = lds32(val + (jx.x & 0xffffu)); f1 = lds32(val + (jx.x >> 16));
                f2 = lds32(val + (jx.y & 0xffffu)); f3 = lds32(val + (jx.y >> 16));
            } else {
                e0 = lds32(val + 4u * (ix.x & 0xffffu)); e1 = lds32(val + 4u * (ix.x >> 16));
                e2 = lds32(val + 4u * (ix.y & 0xffffu)); e3 = lds32(val + 4u * (ix.y >> 16));
                f0 = lds32(val + 4u * (jx.x & 0xffffu)); f1 = lds32(val + 4u * (jx.x >> 16));
                f2 = lds32(val + 4u * (jx.y & 0xffffu)); f3 = lds32(val + 4u * (jx.y >> 16));
            }
            uint32_t t0, t1, t2, t3, u0, u1, u2, u3;
            transpose4x4(e0, e1, e2, e3, t0, t1, t2, t3);
            transpose4x4(f0, f1, f2, f3, u0, u1, u2, u3);
            a0 = __dp4a((int)t0, (int)wa, a0); a1 = __dp4a((int)t1, (int)wa, a1);
            a2 = __dp4a((int)t2, (int)wa, a2); a3 = __dp4a((int)t3, (int)wa, a3);
            b0 = __dp4a((int)u0, (int)wb, b0); b1 = __dp4a((int)u1, (int)wb, b1);
            b2 = __dp4a((int)u2, (int)wb, b2); b3 = __dp4a((int)u3, (int)wb, b3);
            kA += L;
            kB += L;
        }
#define ISING_BFLY2(o) a0 += __shfl_xor_sync(0xffffffffu, a0, o); a1 += __shfl_xor_sync(0xffffffffu, a1, o); \
                       a2 += __shfl_xor_sync(0xffffffffu, a2, o); a3 += __shfl_xor_sync(0xffffffffu, a3, o); \
                       b0 += __shfl_xor_sync(0xffffffffu, b0, o); b1 += __shfl_xor_sync(0xffffffffu, b1, o); \
                       b2 += __shfl_xor_sync(0xffffffffu, b2, o); b3 += __shfl_xor_sync(0xffffffffu, b3, o);
        if (L > 1u) switch (logL) {
            case 5: ISING_BFLY2(16)   // fall through
            case 4: ISING_BFLY2(8)    // fall through
            case 3: ISING_BFLY2(4)    // fall through
            case 2: ISING_BFLY2(2)    // fall through
            case 1: ISING_BFLY2(1)    // fall through
            default: break;
        }
#undef ISING_BFLY2
        uint32_t xa = ~sign_bytes(a0, a1, a2, a3) | 0x01010101u;   // +1 where h < 0, else -1
        uint32_t xb = ~sign_bytes(b0, b1, b2, b3) | 0x01010101u;
        if (rt.tie_rule == 1) {                                    // KEEP: h == 0 leaves the spin
            const uint32_t za = (a0 == 0 ? 0xffu : 0u) | (a1 == 0 ? 0xff00u : 0u) | (a2 == 0 ? 0xff0000u : 0u) |
                                (a3 == 0 ? 0xff000000u : 0u);
            const uint32_t zb = (b0 == 0 ? 0xffu : 0u) | (b1 == 0 ? 0xff00u : 0u) | (b2 == 0 ? 0xff0000u : 0u) |
                                (b3 == 0 ? 0xff000000u : 0u);
            xa = (xa & ~za) | (oldA & za);
            xb = (xb & ~zb) | (oldB & zb);
        }
        xa ^= ((fA * 0x00204081u) & 0x01010101u) * 0xfeu;
        xb ^= ((fB * 0x00204081u) & 0x01010101u) * 0xfeu;
        const uint32_t dA = stA ? (xa << 1) & (xa ^ oldA) : 0u, dB = stB ? (xb << 1) & (xb ^ oldB) : 0u;
        es0 += sbyte(dA, 0) * a0 + sbyte(dB, 0) * b0;
        es1 += sbyte(dA, 1) * a1 + sbyte(dB, 1) * b1;
        es2 += sbyte(dA, 2) * a2 + sbyte(dB, 2) * b2;
        es3 += sbyte(dA, 3) * a3 + sbyte(dB, 3) * b3;
        if (stA) sts32(val + 4u * rowA, xa);
        if (stB) sts32(val + 4u * rowB, xb);
    }
    dE[0] += es0; dE[1] += es1; dE[2] += es2; dE[3] += es3;
}

// One pass over all chain levels (one sweep of the chain rows), chunks streamed through two buffers.
// s_chunks / s_segs: the tables in shared memory.  DELTA: h0 of a chunk is cleared once it has landed.
template <bool DELTA, bool PREMUL>
__device__ __forceinline__ void chain_pass_streamed(const ChainView& v, const ChainChunk* s_chunks, const ChainSeg* s_segs,
                                                    uint32_t val, uint32_t flip, uint32_t buf0, uint32_t slot, const ChainRt& rt,
                                                    const PhiloxKeys& keys, long long (&dE)[4], const ChainGlobal& cg,
                                                    uint32_t tid, uint32_t nthr, bool first_issued,
                                                    unsigned long long* dbg = nullptr, uint32_t dbg_stride = 0) {
    const uint32_t bb = v.buf_bytes;
    uint32_t dj = 0;
    auto stamp = [&]() {   // diagnostics: slots 2..7 of consecutive rows of the phase-timing buffer
        if (dbg) { dbg[(size_t)(dj / 6u) * dbg_stride + 2u + dj % 6u] = (unsigned long long)clock64(); ++dj; }
    };
    stamp();
    if (!first_issued) chain_issue_chunk<DELTA>(v, s_chunks[0], buf0, slot, tid, nthr);
    chain_draw_flips(v, flip, s_chunks[0].r0, s_chunks[0].r1, rt, keys, tid, nthr);
    for (uint32_t k = 0; k < v.n_chunks; ++k) {
        const ChainChunk ck = s_chunks[k];
        const uint32_t buf = buf0 + (k & 1u) * bb;
        if (k + 1u < v.n_chunks) {   // next chunk: request it, draw its rows' flips while it is on its way
            chain_issue_chunk<DELTA>(v, s_chunks[k + 1u], buf0 + ((k + 1u) & 1u) * bb, slot, tid, nthr);
            chain_draw_flips(v, flip, s_chunks[k + 1u].r0, s_chunks[k + 1u].r1, rt, keys, tid, nthr);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
        stamp();
        if (DELTA) {
            int4* hz = reinterpret_cast<int4*>(v.h0) + (size_t)slot * v.n_t_pad + ck.r0;
            for (uint32_t i = tid; i < ck.r1 - ck.r0; i += nthr) __stcg(hz + i, make_int4(0, 0, 0, 0));
        }
        bool synced = false;
        for (uint32_t s = ck.seg0; s < ck.seg1; ++s) {
            const ChainSeg sg = s_segs[s];
            chain_segment<DELTA, PREMUL>(sg, ck, buf, val, flip, rt, keys, dE, cg, tid, nthr);
            synced = (sg.info & 0x100u) != 0u;
            if (synced) __syncthreads();
            stamp();
        }
        if (!synced) __syncthreads();   // the buffer is free for the chunk after next
    }
}

// Warp sums of the threads' dE[] into s_wdE[warp][4] (plain stores; the caller adds the warps' slots up after a CTA
// barrier).  narrow: every partial sum of a sweep fits int32 (chain rows x 2 max_i sum_j |w_ij| < 2^31, checked at load):
// one REDUX per value instead of a 64-bit butterfly.
__device__ __forceinline__ void chain_reduce_dE(long long (&dE)[4], long long (*s_wdE)[4], uint32_t tid, bool narrow) {
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        long long x = dE[b];
        if (narrow) {
            x = (long long)__reduce_add_sync(0xffffffffu, (int)x);
        } else {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        }
        if ((tid & 31u) == 0u) s_wdE[tid >> 5][b] = x;
        dE[b] = 0;
    }
}
__device__ __forceinline__ long long chain_sum_dE(const long long (*s_wdE)[4], uint32_t b, uint32_t n_warps) {
    long long x = 0;
    for (uint32_t w = 0; w < n_warps; ++w) x += s_wdE[w][b];
    return x;
}

// ---------------------------------------------------------------------------------------------
// k_anneal_small: a whole ising_anneal call (Gauss-Seidel, int8 weights) for a graph whose chain fits one CTA.
// Grid = tiles x 8 CTAs, one per word of four replicas; CTAs never synchronise with one another.
// ---------------------------------------------------------------------------------------------
struct SmallParams {
    ChainView v;
    uint8_t* state;                 // [tiles][n][32], standard layout: read at start, written at the end
    uint8_t* best;                  // captured best state, standard layout (written at the end)
    uint32_t* best_compact;         // scratch [tiles * 8][bc_stride]: this CTA's words of its best state
    uint32_t bc_stride;
    unsigned long long tile_stride;
    uint32_t n_replicas, rep0;
    int32_t tie_rule;
    uint32_t n_sweeps, sweep_offset;
    const uint32_t* thr;            // DEVICE [n_sweeps]
    long long W;
    const long long* E0;            // [tiles * 32]
    long long* trace;               // [n_sweeps][trace_stride] or nullptr
    unsigned long long trace_stride;
    long long* E_out;
    long long* best_out;
    int32_t* best_sweep_out;
    int32_t resume;
    uint32_t csplit;                // CTAs per word (cluster size): 1, or 2 = levels + flip producer (resident chain only)
    unsigned long long* timing;     // diagnostics (resident chain only): SM-clock stamps of CTA 0 in sweep timing_sweep: sweep start,
                                    // flips drawn, after every segment, dE reduced, cut / best done, capture done; or nullptr
    uint32_t timing_sweep;
    PhiloxKeys keys;
};

// csplit == 2 (resident chain, enough SMs): every word runs on a CLUSTER of two CTAs.  CTA 0 walks the levels; CTA 1 only
// draws the flip decisions -- they do not depend on the spins -- one sweep ahead, straight into CTA 0's shared memory
// (two flip buffers, st.shared::cluster), and hands each buffer over through an mbarrier in CTA 0 (remote arrive, release /
// acquire at cluster scope); CTA 0 gives a buffer back through an mbarrier in CTA 1 once its sweep is done.  The Philox
// work (about half the instructions of a sweep of a low-degree graph) leaves the SM that runs the dependent levels.
template <bool TIMING, bool PREMUL>
__global__ void __launch_bounds__(kSmallThreadsMax, 1) k_anneal_small(const SmallParams p) {
    extern __shared__ __align__(128) uint8_t chain_smem[];
    __shared__ ChainChunk s_chunks[kChainMaxChunks];
    __shared__ ChainSeg s_segs[kChainMaxSegs];
    __shared__ long long s_wdE[kSmallThreadsMax / 32][4];
    __shared__ long long s_E[4], s_bc[4];
    __shared__ int s_bs[4];
    __shared__ uint32_t s_imp;
    __shared__ int s_w32[kSmallThreadsMax / 32][4];   // (narrow sums: the warps' parts, added up by warp 0)
    __shared__ __align__(8) unsigned long long s_full[2], s_empty[2];   // flip buffer b: filled (in CTA 0) / free again (in CTA 1)
    const uint32_t tid = threadIdx.x, nthr = blockDim.x;
    const uint32_t csplit = p.csplit, crank = blockIdx.x % csplit, slot = blockIdx.x / csplit;   // slot = word index
    const uint32_t tile = slot / kChainGroups, g = slot % kChainGroups;
    const uint32_t r_first = tile * kTile + 4u * g;      // first replica of this CTA within the call
    if (r_first >= p.n_replicas) return;                 // no live replica in this word (both CTAs of a cluster leave)
    const ChainView& v = p.v;
    const uint32_t n = v.n_t;
    uint32_t val;   // (opaque to the compiler: it would otherwise re-derive the shared window address wherever it is used)
    asm volatile("{ .reg .u64 t; cvta.to.shared.u64 t, %1; cvt.u32.u64 %0, t; }" : "=r"(val) : "l"(chain_smem));
    const uint32_t flip_bytes = chain_align16(v.n_t_pad);
    const uint32_t flip0 = val + chain_align16(4u * v.n_t_pad);
    const uint32_t buf0 = flip0 + 2u * flip_bytes;
    const uint32_t full0 = (uint32_t)__cvta_generic_to_shared(&s_full[0]), empty0 = (uint32_t)__cvta_generic_to_shared(&s_empty[0]);
    ChainRt rt;
    rt.rl0 = p.rep0 + r_first;
    rt.tie_rule = p.tie_rule;
    if (csplit > 1u) {
        if (tid == 0) {
            mbar_init_cta(full0, nthr); mbar_init_cta(full0 + 8u, nthr);
            mbar_init_cta(empty0, 1u);  mbar_init_cta(empty0 + 8u, 1u);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        cluster_barrier();
        if (crank == 1u) {   // ---- the flip producer
            const uint32_t full_r = mapa_u32(full0, 0u), flip_r = mapa_u32(flip0, 0u);
            uint32_t k = 0;   // sweeps with flips so far (both CTAs count alike)
            for (uint32_t t = 0; t < p.n_sweeps; ++t) {
                rt.thr = __ldg(p.thr + t);
                rt.T = p.sweep_offset + t;
                if (rt.thr == 0u) continue;
                const uint32_t b = k & 1u;
                if (k >= 2u) mbar_wait_cluster(empty0 + 8u * b, ((k >> 1) - 1u) & 1u);   // CTA 0 is done with sweep k - 2
                for (uint32_t r4 = 4u * tid; r4 < n; r4 += 4u * nthr) {   // four rows per thread: one 32-bit store
                    const uint4 o = __ldg(reinterpret_cast<const uint4*>(v.orig + r4));
                    const uint32_t f = chain_flip4(o.x, rt, p.keys) | (chain_flip4(o.y, rt, p.keys) << 8) |
                                       (chain_flip4(o.z, rt, p.keys) << 16) | (chain_flip4(o.w, rt, p.keys) << 24);
                    st_cluster_u32(flip_r + b * flip_bytes + r4, f);
                }
                mbar_arrive_remote(full_r + 8u * b);
                ++k;
            }
            cluster_barrier();   // (CTA 0 may arrive on this CTA's barriers until it is through)
            return;
        }
    }
    const uint32_t empty_r = csplit > 1u ? mapa_u32(empty0, 1u) : 0u;
    uint32_t kf = 0;   // sweeps with flips so far
    uint8_t* const gstate = p.state + (size_t)tile * p.tile_stride + 4u * g;
    uint8_t* const gbest = p.best + (size_t)tile * p.tile_stride + 4u * g;
    uint32_t* const bcomp = p.best_compact + (size_t)slot * p.bc_stride;

    for (uint32_t i = tid; i < v.n_chunks * (uint32_t)(sizeof(ChainChunk) / 4); i += nthr)
        reinterpret_cast<uint32_t*>(s_chunks)[i] = __ldg(reinterpret_cast<const uint32_t*>(v.chunks) + i);
    for (uint32_t i = tid; i < v.n_segs * (uint32_t)(sizeof(ChainSeg) / 4); i += nthr)
        reinterpret_cast<uint32_t*>(s_segs)[i] = __ldg(reinterpret_cast<const uint32_t*>(v.segs) + i);
    for (uint32_t r = tid; r < n; r += nthr) {
        sts32(val + 4u * r, __ldcg(reinterpret_cast<const uint32_t*>(gstate + (size_t)r * kTile)));
        if (p.resume) bcomp[r] = __ldcg(reinterpret_cast<const uint32_t*>(gbest + (size_t)r * kTile));
    }
    if (tid < 4u) {
        s_E[tid] = p.E0[r_first + tid];
        s_bc[tid] = p.resume ? p.best_out[r_first + tid] : (long long)0x8000000000000000ull;
        s_bs[tid] = p.resume ? p.best_sweep_out[r_first + tid] : 0;
    }
    __syncthreads();
    if (v.resident) {
        chain_issue_chunk<false>(v, s_chunks[0], buf0, slot, tid, nthr);
        cp_async_wait<0>();
        __syncthreads();
    }
    ChainGlobal cg{};
    long long dE[4] = {0, 0, 0, 0};
    const uint32_t n_segs = v.n_segs;
    const uint32_t n32_bit = (v.narrow != 0u && nthr == v.threads) ? 0x200u : 0u;   // (bit 9 of a segment was planned for v.threads)
    for (uint32_t t = 0; t < p.n_sweeps; ++t) {
        rt.thr = __ldg(p.thr + t);
        rt.T = p.sweep_offset + t;
        unsigned long long* ts = (TIMING && p.timing && t == p.timing_sweep && blockIdx.x == 0 && tid == 0) ? p.timing : nullptr;
        if (TIMING && ts) *ts++ = (unsigned long long)clock64();
        if (v.resident) {
            const uint32_t fb = kf & 1u, flip = flip0 + fb * flip_bytes;
            if (csplit == 1u) {
                chain_draw_flips(v, flip, 0u, n, rt, p.keys, tid, nthr);
                __syncthreads();
            } else if (rt.thr != 0u) {
                mbar_wait_cluster(full0 + 8u * fb, (kf >> 1) & 1u);   // the producer has filled this sweep's buffer
            }
            if (TIMING && ts) *ts++ = (unsigned long long)clock64();
            const ChainChunk ck = s_chunks[0];
            for (uint32_t s = 0; s < n_segs; ++s) {
                const ChainSeg sg = s_segs[s];
                if (sg.info & n32_bit)   // several rows per thread and all sums fit 32 bits
                    chain_segment_rows2<PREMUL>(sg, ck, buf0, val, flip, rt, dE, tid, nthr);
                else
                    chain_segment<false, PREMUL, false>(sg, ck, buf0, val, flip, rt, p.keys, dE, cg, tid, nthr);
                if (sg.info & 0x100u) __syncthreads();
                if (TIMING && ts) *ts++ = (unsigned long long)clock64();
            }
            if (rt.thr != 0u) {   // (every thread is past the last level: the flip buffer goes back to the producer)
                if (csplit > 1u && tid == nthr - 32u) mbar_arrive_remote_relaxed(empty_r + 8u * fb);
                ++kf;
            }
        } else {
            chain_pass_streamed<false, PREMUL>(v, s_chunks, s_segs, val, flip0, buf0, slot, rt, p.keys, dE, cg, tid, nthr, false);
        }
        if (v.narrow != 0u) {
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const int x = __reduce_add_sync(0xffffffffu, (int)dE[b]);
                if ((tid & 31u) == 0u) s_w32[tid >> 5][b] = x;
                dE[b] = 0;
            }
        } else {
            chain_reduce_dE(dE, s_wdE, tid, false);
        }
        __syncthreads();
        if (TIMING && ts) *ts++ = (unsigned long long)clock64();
        long long dsum = 0;
        if (v.narrow != 0u) {
            if (tid < 32u) {
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const int y = __reduce_add_sync(0xffffffffu, tid < (nthr >> 5) ? s_w32[tid][b] : 0);
                    if (tid == (uint32_t)b) dsum = (long long)y;
                }
            }
        } else if (tid < 4u) {
            dsum = chain_sum_dE(s_wdE, tid, nthr >> 5);
        }
        if (tid < 4u) {   // a7: E, cut = (W - E)/2 (eq. 4), best tracking (strictly greater: the earliest sweep wins)
            const long long E = s_E[tid] + dsum;
            const long long cut = (p.W - E) / 2;
            const bool live = r_first + tid < p.n_replicas;
            const bool improved = live && cut > s_bc[tid];
            s_E[tid] = E;
            if (improved) { s_bc[tid] = cut; s_bs[tid] = (int)rt.T; }
            if (live && p.trace) p.trace[(size_t)t * p.trace_stride + r_first + tid] = cut;
            const uint32_t m = __ballot_sync(0xfu, improved);
            if (tid == 0) s_imp = m;
        }
        __syncthreads();
        if (TIMING && ts) *ts++ = (unsigned long long)clock64();
        const uint32_t imp = s_imp;
        if (imp != 0u) {   // capture the improved replicas' bytes of every row
            const uint32_t km = nibble_to_bytemask(imp);
            for (uint32_t r = tid; r < n; r += nthr) {
                const uint32_t s = lds32(val + 4u * r);
                bcomp[r] = imp == 15u ? s : ((s & km) | (bcomp[r] & ~km));
            }
            __syncthreads();   // the next sweep rewrites val
        }
        if (TIMING && ts) *ts++ = (unsigned long long)clock64();
    }
    // final state and best state back to the standard layout
    for (uint32_t r = tid; r < n; r += nthr) {
        *reinterpret_cast<uint32_t*>(gstate + (size_t)r * kTile) = lds32(val + 4u * r);
        *reinterpret_cast<uint32_t*>(gbest + (size_t)r * kTile) = bcomp[r];
    }
    if (tid < 4u) {
        p.E_out[r_first + tid] = s_E[tid];
        p.best_out[r_first + tid] = s_bc[tid];
        p.best_sweep_out[r_first + tid] = s_bs[tid];
    }
    if (csplit > 1u) cluster_barrier();   // no CTA leaves while its peer may still touch its shared memory
}

// ---------------------------------------------------------------------------------------------
// Chain builder (a1): one warp per chain row scans the row of the caller's CSR and keeps the qualifying neighbours
// (FULL: all; DELTA: chain rows of a lower colour).  Pass 1 counts cells, pass 2 (after the host has cut the rows into
// chunks and fixed the cell pointers) fills them.
// ---------------------------------------------------------------------------------------------
template <bool FILL>
__global__ void k_chain_build(uint32_t n_t, uint32_t row_lo, int delta, const int32_t* perm, const int32_t* inv,
                              const long long* row_ptr, const int32_t* col, const void* w, int wtype,
                              const int32_t* colour, const uint32_t* cptr, uint32_t* counts, uint16_t* idx16,
                              int8_t* w8, uint32_t* orig_out, uint32_t id_shift) {
    const uint32_t r = (uint32_t)(((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    const uint32_t lane = threadIdx.x & 31u;
    if (r >= n_t) return;
    const int32_t orig = perm[row_lo + r];
    const long long b = row_ptr[orig], e = row_ptr[orig + 1];
    const int32_t c_own = delta ? colour[orig] : 0;
    const unsigned long long base_at = FILL ? 4ull * cptr[r] : 0ull;
    uint32_t cnt = 0;
    for (long long at0 = b; at0 < e; at0 += 32) {
        const long long i = at0 + lane;
        bool ok = false;
        uint32_t u = 0;
        int wv = 0;
        if (i < e) {
            const int32_t j = col[i];
            u = (uint32_t)inv[j];
            ok = !delta || (u >= row_lo && colour[j] < c_own);
            wv = wtype == 1 ? (int)reinterpret_cast<const int8_t*>(w)[i] : (int)reinterpret_cast<const int32_t*>(w)[i];
        }
        const uint32_t m = __ballot_sync(0xffffffffu, ok);
        if (FILL && ok) {
            const unsigned long long at = base_at + cnt + __popc(m & ((1u << lane) - 1u));
            idx16[at] = (uint16_t)((u - row_lo) << id_shift);   // (id_shift 2: byte offset into val[])
            w8[at] = (int8_t)wv;
        }
        cnt += __popc(m);
    }
    if (!FILL) {
        if (lane == 0) counts[r] = (cnt + 3u) / 4u;
    } else {
        const unsigned long long end_at = 4ull * cptr[r + 1];   // padding (and the alignment gap before the next chunk)
        for (unsigned long long at = base_at + cnt + lane; at < end_at; at += 32) {
            idx16[at] = (uint16_t)(r << id_shift);
            w8[at] = 0;
        }
        if (lane == 0) orig_out[r] = (uint32_t)orig;
    }
}

}  // namespace ising
