// Sparse annealing sweep and its bookkeeping kernels.
//
// One warp owns one slice (common.cuh): lane = 2*sub_row + half, every lane keeps the
// int32 local fields h_i = sum_j w_ij s_j (eq. (2)) of 16 replicas.  Four
// neighbour sectors are gathered per step (16-byte loads), byte-transposed with PRMT so
// that one dp4a multiplies the four edge weights into one replica's field.  Rows split
// over several sub-rows are finished by a warp-level segmented (butterfly) reduction.
// The epilogue takes the energy-minimising value (L47-49 with the sign reading Q1:
// s_i <- +1 if h_i < 0 else -1), applies the scheduled flip of Algorithm 2 (L177) with the
// stateless Philox word, writes the spin sector and accumulates the energy bookkeeping
// (a7): Gauss-Seidel  dE_i = (a_i - s_i) h_i  (exact because a colour class is an
// independent set), Jacobi / evaluation  s_i h_i  (sum_i s_i h_i = 2 E).
#pragma once
#include "common.cuh"

namespace ising {

// 4x4 byte transpose: in e[j] = bytes (replica 0..3) of edge j; out t[b] = bytes (edge 0..3)
// of replica b.
__device__ __forceinline__ void transpose4x4(uint32_t e0, uint32_t e1, uint32_t e2, uint32_t e3,
                                             uint32_t& t0, uint32_t& t1, uint32_t& t2, uint32_t& t3) {
    const uint32_t x0 = __byte_perm(e0, e1, 0x5140);
    const uint32_t x1 = __byte_perm(e2, e3, 0x5140);
    const uint32_t x2 = __byte_perm(e0, e1, 0x7362);
    const uint32_t x3 = __byte_perm(e2, e3, 0x7362);
    t0 = __byte_perm(x0, x1, 0x5410);
    t1 = __byte_perm(x0, x1, 0x7632);
    t2 = __byte_perm(x2, x3, 0x5410);
    t3 = __byte_perm(x2, x3, 0x7632);
}

__device__ __forceinline__ void field_word(int (&h)[16], int k, uint32_t e0, uint32_t e1, uint32_t e2,
                                           uint32_t e3, uint32_t w) {
    uint32_t t0, t1, t2, t3;
    transpose4x4(e0, e1, e2, e3, t0, t1, t2, t3);
    h[4 * k + 0] = __dp4a((int)t0, (int)w, h[4 * k + 0]);
    h[4 * k + 1] = __dp4a((int)t1, (int)w, h[4 * k + 1]);
    h[4 * k + 2] = __dp4a((int)t2, (int)w, h[4 * k + 2]);
    h[4 * k + 3] = __dp4a((int)t3, (int)w, h[4 * k + 3]);
}

__device__ __forceinline__ int sbyte(uint32_t word, int b) { return (int)(int8_t)(word >> (8 * b)); }

__device__ __forceinline__ void field_word_wide(int (&h)[16], int k, uint32_t e, int w) {
#pragma unroll
    for (int b = 0; b < 4; ++b) h[4 * k + b] += sbyte(e, b) * w;
}

__device__ __forceinline__ uint32_t pick8(const uint4& u, const uint4& v, int idx) {
    uint32_t r = u.x;
    r = idx == 1 ? u.y : r;
    r = idx == 2 ? u.z : r;
    r = idx == 3 ? u.w : r;
    r = idx == 4 ? v.x : r;
    r = idx == 5 ? v.y : r;
    r = idx == 6 ? v.z : r;
    r = idx == 7 ? v.w : r;
    return r;
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

// KIND: kKindGS (in place, one colour class), kKindJacobi (src -> dst), kKindEval (no write).
// WIDE: int32 weights (w4w) and int64 bookkeeping; otherwise int8 weights, dp4a, int32 bookkeeping
// flushed every p.flush_rows rows.
template <int KIND, bool WIDE>
__global__ void __launch_bounds__(kSweepThreads) k_sweep(const SweepParams p) {
    using AccT = typename std::conditional<WIDE, long long, int>::type;
    __shared__ long long s_acc[kTile];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sr = lane >> 1, half = lane & 1;
    const uint32_t tile = blockIdx.y;
    if (threadIdx.x < kTile) s_acc[threadIdx.x] = 0;
    __syncthreads();

    const uint8_t* src = p.src + (size_t)tile * p.tile_stride + half * 16;
    uint8_t* dst = p.dst + (size_t)tile * p.tile_stride + half * 16;
    const uint32_t rep_lane0 = p.rep0 + tile * kTile + half * 16;   // global id of this lane's replica 0

    AccT acc[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) acc[k] = 0;
    uint32_t rows_acc = 0;

    for (uint32_t s = p.slice_begin + blockIdx.x * kWarpsPerCta + warp; s < p.slice_end;
         s += gridDim.x * kWarpsPerCta) {
        const SliceDesc d = p.slices[s];
        int h[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) h[k] = 0;

        if (d.G > 0) {
            const int4* cp = p.col4 + d.off + sr;
            if (!WIDE) {
                const uint32_t* wp = p.w4 + d.off + sr;
                int4 c = ld_stream(cp);
                uint32_t w = ld_stream(wp);
                for (uint32_t g = 0; g < d.G; ++g) {
                    const uint4 e0 = ld_spin(src + (size_t)(uint32_t)c.x * kTile);
                    const uint4 e1 = ld_spin(src + (size_t)(uint32_t)c.y * kTile);
                    const uint4 e2 = ld_spin(src + (size_t)(uint32_t)c.z * kTile);
                    const uint4 e3 = ld_spin(src + (size_t)(uint32_t)c.w * kTile);
                    const uint32_t wc = w;
                    if (g + 1 < d.G) {   // prefetch the next group's indices while the gathers fly
                        c = ld_stream(cp + (size_t)(g + 1) * kSubRows);
                        w = ld_stream(wp + (size_t)(g + 1) * kSubRows);
                    }
                    field_word(h, 0, e0.x, e1.x, e2.x, e3.x, wc);
                    field_word(h, 1, e0.y, e1.y, e2.y, e3.y, wc);
                    field_word(h, 2, e0.z, e1.z, e2.z, e3.z, wc);
                    field_word(h, 3, e0.w, e1.w, e2.w, e3.w, wc);
                }
            } else {
                const int4* wp = p.w4w + d.off + sr;
                for (uint32_t g = 0; g < d.G; ++g) {
                    const int4 c = ld_stream(cp + (size_t)g * kSubRows);
                    const int4 w = ld_stream(wp + (size_t)g * kSubRows);
                    const uint4 e0 = ld_spin(src + (size_t)(uint32_t)c.x * kTile);
                    const uint4 e1 = ld_spin(src + (size_t)(uint32_t)c.y * kTile);
                    const uint4 e2 = ld_spin(src + (size_t)(uint32_t)c.z * kTile);
                    const uint4 e3 = ld_spin(src + (size_t)(uint32_t)c.w * kTile);
                    field_word_wide(h, 0, e0.x, w.x); field_word_wide(h, 1, e0.y, w.x);
                    field_word_wide(h, 2, e0.z, w.x); field_word_wide(h, 3, e0.w, w.x);
                    field_word_wide(h, 0, e1.x, w.y); field_word_wide(h, 1, e1.y, w.y);
                    field_word_wide(h, 2, e1.z, w.y); field_word_wide(h, 3, e1.w, w.y);
                    field_word_wide(h, 0, e2.x, w.z); field_word_wide(h, 1, e2.y, w.z);
                    field_word_wide(h, 2, e2.z, w.z); field_word_wide(h, 3, e2.w, w.z);
                    field_word_wide(h, 0, e3.x, w.w); field_word_wide(h, 1, e3.y, w.w);
                    field_word_wide(h, 2, e3.z, w.w); field_word_wide(h, 3, e3.w, w.w);
                }
            }
        }

        // warp-level segmented reduction over the sub-rows of one row
        const int log_spr = (int)(d.meta & 0xffu);
        const int nrows = (int)(d.meta >> 8);
        for (int lvl = 0; lvl < log_spr; ++lvl) {
#pragma unroll
            for (int k = 0; k < 16; ++k) h[k] += __shfl_xor_sync(0xffffffffu, h[k], 2 << lvl);
        }
        const int rloc = sr >> log_spr;
        const bool owner = ((sr & ((1 << log_spr) - 1)) == 0) && rloc < nrows;
        if (owner) {
            const uint32_t row = d.row0 + (uint32_t)rloc;
            const uint4 so4 = ld_spin(src + (size_t)row * kTile);
            const uint32_t so[4] = {so4.x, so4.y, so4.z, so4.w};
            if (KIND == kKindEval) {
#pragma unroll
                for (int k = 0; k < 4; ++k)
#pragma unroll
                    for (int b = 0; b < 4; ++b) acc[4 * k + b] += (AccT)sbyte(so[k], b) * (AccT)h[4 * k + b];
            } else {
                const uint32_t orig = (uint32_t)p.perm[row];
                const int mis = (int)(rep_lane0 & 3u);
                uint32_t nv[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    uint4 u = make_uint4(0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu), u2 = u;
                    if (p.thr != 0) {
                        const uint32_t cw = (rep_lane0 + 4 * k) >> 2;
                        u = philox4x32_10(orig, p.T, cw, kDomainFlip, p.keys);
                        if (mis) u2 = philox4x32_10(orig, p.T, cw + 1, kDomainFlip, p.keys);
                    }
                    const uint32_t ur[4] = {u.x, u.y, u.z, u.w};
                    uint32_t word = 0;
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        const int hv = h[4 * k + b];
                        const int sold = sbyte(so[k], b);
                        int a = hv < 0 ? 1 : -1;
                        if (p.tie_rule == 1 && hv == 0) a = sold;
                        const uint32_t rnd = mis ? pick8(u, u2, mis + b) : ur[b];
                        if (rnd < p.thr) a = -a;
                        if (KIND == kKindGS) {
                            if (a != sold) acc[4 * k + b] += (AccT)(2 * a) * (AccT)hv;
                        } else {
                            acc[4 * k + b] += (AccT)sold * (AccT)hv;
                        }
                        word |= ((uint32_t)a & 0xffu) << (8 * b);
                    }
                    nv[k] = word;
                }
                *reinterpret_cast<uint4*>(dst + (size_t)row * kTile) = make_uint4(nv[0], nv[1], nv[2], nv[3]);
            }
        }
        if (!WIDE) {
            if (++rows_acc >= p.flush_rows) {   // warp-uniform
                flush_acc(acc, s_acc, lane);
                rows_acc = 0;
            }
        }
    }
    flush_acc(acc, s_acc, lane);
    __syncthreads();
    if (threadIdx.x < kTile) {
        const long long v = s_acc[threadIdx.x];
        if (v != 0)
            atomicAdd(reinterpret_cast<unsigned long long*>(p.accum + (size_t)tile * kTile + threadIdx.x),
                      (unsigned long long)v);
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

__device__ __forceinline__ uint32_t nibble_to_bytemask(uint32_t nib) {
    // bit b of nib -> byte b = 0xff
    uint32_t m = (nib & 1u) | ((nib & 2u) << 7) | ((nib & 4u) << 14) | ((nib & 8u) << 21);
    return m * 0xffu;
}

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
