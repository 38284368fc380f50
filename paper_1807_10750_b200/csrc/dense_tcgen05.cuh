// Dense local-field engine for fully connected instances.
//
// For K_n the local fields of all replicas are one int8 contraction H = J . S (eq. (2), for
// every spin and replica at once; general connectivity L57, Fig. 2 L61): J [n][n] symmetric int8 with zero
// diagonal, S [n][R] spins.  It runs on the 5th-generation tensor cores: tcgen05.mma.kind::i8 issued by
// one thread, both operands K-major in shared memory (A = J rows, B = S^T rows, i.e. the state is kept
// replica-major [R][n] so that K = the neighbour index is contiguous), fed by TMA
// (cp.async.bulk.tensor, 128-byte swizzle) through an mbarrier ring, int32 accumulators in TMEM.
// The epilogue reads the accumulators with tcgen05.ld (one thread = one spin i, 16 replicas at a time)
// and fuses a4-a7 (16 epilogue warps: 4 lane quarters x 4 groups of 64 replicas): energy-minimising value, Philox flip, int8 store of the next state (synchronous
// Jacobi: into the other buffer) and sum_i s_i h_i = 2 E(s) per replica.
//
// One launch = one Jacobi sweep (every sweep needs the complete previous state); one CTA = one
// 128 (spins) x 256 (replicas) output tile, K = n in blocks of 128.
#pragma once
#include <cuda.h>

#include "../../include/ising.h"
#include "common.cuh"
#include "sparse_sweep.cuh"

namespace ising {

constexpr bool kDenseEnabled = true;
constexpr int kDM = 128;        // spins per tile (UMMA M)
constexpr int kDN = 256;        // replicas per tile (UMMA N)
constexpr int kDK = 128;        // K bytes per pipeline stage (one 128-byte swizzle row)
constexpr int kDStages = 4;
constexpr int kDEpiWarps = 16;   // 4 TMEM lane quarters x 4 column groups of 64 replicas
constexpr int kDThreads = 64 + 32 * kDEpiWarps;   // warp 0 TMA, warp 1 MMA, warps 2.. epilogue
constexpr uint32_t kDStageBytesA = kDM * kDK, kDStageBytesB = kDN * kDK;
constexpr uint32_t kDSmemBytes = kDStages * (kDStageBytesA + kDStageBytesB) + 1024 /*align*/ + 256 /*barriers*/;

struct DenseSweepParams {
    const int8_t* src;     // [R_pad][n_pad] state read (also the TMA source of operand B)
    int8_t* dst;           // [R_pad][n_pad] next state (update) -- unused for evaluation
    long long* accum;      // [R_pad] += sum_i s_i h_i
    int* error_flag;       // set when a pipeline wait times out
    uint32_t n, n_pad;
    uint32_t thr, T, rep0;
    int32_t tie_rule;
    int32_t update;        // 1: Jacobi sweep, 0: evaluation only
    PhiloxKeys keys;
};

// ---- PTX wrappers ---------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Bounded wait: a broken pipeline must not hang the GPU.
__device__ __forceinline__ bool mbar_wait(uint64_t* bar, uint32_t parity, int* error_flag) {
    const uint32_t addr = smem_u32(bar);
    for (uint32_t spin = 0; spin < (1u << 24); ++spin) {
        uint32_t done;
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(addr), "r"(parity) : "memory");
        if (done) return true;
    }
    atomicExch(error_flag, 1);
    return false;
}
__device__ __forceinline__ void tma_load_2d(const CUtensorMap* map, uint64_t* bar, void* dst, int x, int y) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
}
// K-major operand tile written by TMA with the 128-byte swizzle: rows of 128 bytes, 8-row atoms of
// 1024 bytes stacked contiguously (stride byte offset 1024); descriptor version 1 (sm_100).
__device__ __forceinline__ uint64_t umma_desc_k128(uint32_t smem_addr) {
    return (uint64_t)((smem_addr & 0x3ffffu) >> 4) | ((uint64_t)(1024u >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// kind::i8 instruction descriptor: D = S32, A = B = signed int8, both K-major, M x N.
__host__ __device__ constexpr uint32_t umma_idesc_i8(int m, int n) {
    return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(m >> 4) << 24);
}

// ---------------------------------------------------------------------------------------------
// k_dense_sweep: one Jacobi sweep (or one evaluation pass) of a K_n instance.
// grid = (n_pad / 128, R_pad / 256); CTA (bx, by) owns spins [128 bx, +128) x replicas [256 by, +256).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kDThreads, 1)
k_dense_sweep(const __grid_constant__ CUtensorMap tm_j, const __grid_constant__ CUtensorMap tm_s,
              const DenseSweepParams p) {
    extern __shared__ uint8_t dsm_raw[];
    uint8_t* dsm = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(dsm_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t* sm_a = dsm;                                         // [stages][128 x 128 B]
    uint8_t* sm_b = dsm + kDStages * kDStageBytesA;              // [stages][256 x 128 B]
    uint64_t* bars = reinterpret_cast<uint64_t*>(dsm + kDStages * (kDStageBytesA + kDStageBytesB));
    uint64_t* full = bars;                    // [stages] TMA -> MMA
    uint64_t* empty = bars + kDStages;        // [stages] MMA -> TMA
    uint64_t* acc_full = bars + 2 * kDStages; // MMA -> epilogue
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * kDStages + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t m0 = blockIdx.x * kDM, n0 = blockIdx.y * kDN;
    const uint32_t num_kb = p.n_pad / kDK;

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < kDStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        mbar_init(acc_full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {   // TMEM: 256 columns of int32 accumulators; this warp also frees them
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(kDN));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        if (lane == 0) {   // ---- TMA producer
            for (uint32_t kb = 0; kb < num_kb; ++kb) {
                const uint32_t s = kb % kDStages, ph = (kb / kDStages) & 1u;
                if (!mbar_wait(&empty[s], ph ^ 1u, p.error_flag)) break;
                mbar_expect_tx(&full[s], kDStageBytesA + kDStageBytesB);
                tma_load_2d(&tm_j, &full[s], sm_a + s * kDStageBytesA, (int)(kb * kDK), (int)m0);
                tma_load_2d(&tm_s, &full[s], sm_b + s * kDStageBytesB, (int)(kb * kDK), (int)n0);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {   // ---- MMA issuer
            constexpr uint32_t idesc = umma_idesc_i8(kDM, kDN);
            bool ok = true;
            for (uint32_t kb = 0; kb < num_kb && ok; ++kb) {
                const uint32_t s = kb % kDStages, ph = (kb / kDStages) & 1u;
                ok = mbar_wait(&full[s], ph, p.error_flag);
                if (!ok) break;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint64_t da = umma_desc_k128(smem_u32(sm_a + s * kDStageBytesA));
                const uint64_t db = umma_desc_k128(smem_u32(sm_b + s * kDStageBytesB));
#pragma unroll
                for (uint32_t k = 0; k < kDK / 32; ++k)   // K = 32 int8 per instruction: +32 B = +2 in the address field
                    umma_i8(tmem_base, da + 2 * k, db + 2 * k, idesc, (kb | k) != 0u ? 1u : 0u);
                umma_commit(&empty[s]);   // frees the stage when these MMAs have read it
            }
            umma_commit(acc_full);        // accumulators complete (arrives even after a time-out)
        }
    } else {
        // ---- epilogue: a warp may only read the TMEM lane quarter q = warp id & 3, i.e. spins m0 + 32 q + lane;
        // the four warps that share a quarter split the 256 replicas of the tile
        const uint32_t q = (uint32_t)warp & 3u;
        const uint32_t row = m0 + q * 32u + (uint32_t)lane;   // caller's vertex id (dense layout keeps caller order)
        const bool live = row < p.n;
        const bool ok = mbar_wait(acc_full, 0u, p.error_flag);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (ok) {
            long long colsum = 0;   // this lane's column (c & 31 == lane) of the current block of 32 replicas
            const uint32_t cg = ((uint32_t)warp - 2u) >> 2;                      // column group of this warp
            constexpr uint32_t kColsPerWarp = (uint32_t)kDN / (kDEpiWarps / 4);  // 64
#pragma unroll 1
            for (uint32_t c0 = cg * kColsPerWarp; c0 < (cg + 1u) * kColsPerWarp; c0 += 16) {
                uint32_t hreg[16];
                tmem_ld16(tmem_base + ((q * 32u) << 16) + c0, hreg);
                int sold[16];
#pragma unroll
                for (int j = 0; j < 16; ++j)
                    sold[j] = (int)p.src[(size_t)(n0 + c0 + j) * p.n_pad + row];   // 32 lanes = 32 consecutive bytes
                const uint32_t rep = p.rep0 + n0 + c0;
                uint32_t flip16 = 0;
                if (p.update) flip16 = finish_flip_mask(flip_mask_part(row, p.T, rep, p.thr, 0u, 1u, p.keys), rep);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const int hv = (int)hreg[j];
                    const int so = sold[j];
                    if (p.update) {
                        int a = hv < 0 ? 1 : -1;                    // a4 (L47-49, Q1/Q3)
                        if (p.tie_rule == 1 && hv == 0) a = so;
                        if ((flip16 >> j) & 1u) a = -a;             // a5 (Alg. 2)
                        if (!live) a = 0;
                        p.dst[(size_t)(n0 + c0 + j) * p.n_pad + row] = (int8_t)a;   // a6: the other buffer
                    }
                    const int part = __reduce_add_sync(0xffffffffu, so * hv);       // a7: sum over 32 spins
                    if (lane == (int)((c0 + j) & 31u)) colsum += part;
                }
                if (c0 & 16u) {   // block of 32 replicas finished
                    if (colsum != 0)
                        atomicAdd(reinterpret_cast<unsigned long long*>(p.accum + n0 + (c0 & ~31u) + lane),
                                  (unsigned long long)colsum);
                    colsum = 0;
                }
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 2) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kDN));
    }
}

// ---------------------------------------------------------------------------------------------
// k_dense_anneal: ALL Jacobi sweeps of one ising_anneal call in one cooperative launch (a8 + a9).
// The product is taken TRANSPOSED: D[replica][spin] = sum_k S[replica][k] J[spin][k] (J is symmetric), i.e. operand A =
// 128 rows of the replica-major state, operand B = 256 rows of J, so that a TMEM lane -- one epilogue thread -- is a
// REPLICA and the accumulator columns are spins.  Then sum_i s_i h_i is a per-thread sum (no warp reductions), the
// thread's new spins are 16 consecutive bytes of its replica's row (one 16-byte store per tcgen05.ld), and its old
// spins are 64 bits in two registers.  (With spins on the lanes the epilogue needed a ballot and a REDUX per replica
// column and took 25 k cycles per sweep against 19 k for the MMAs.)
// grid = (R_pad / 128, n_pad / 256) <= number of SMs.  Per pass t:
//   warp 0 TMA, warp 1 MMA issue as in k_dense_sweep; meanwhile the 16 epilogue warps draw the pass's Philox flips
//   (one call per spin and four replicas, shared by the four lanes of a replica group through shuffles); epilogue:
//   S^(t+1) into the other buffer, sum_i s_i h_i = 2 E(S^t) to a rotating global slot; grid barrier; then every CTA
//   derives, for its 128 replicas, E / cut / best of the candidate S^t (trace row and slot reset by the CTAs of spin
//   block 0) and copies its 256 spins of the improved replicas from S^t into the best state.  The last pass only evaluates.
// ---------------------------------------------------------------------------------------------
struct DenseAnnealParams {
    int8_t* S[2];                   // [R_pad][n_pad] state buffers (S[cur] holds the initial state)
    int8_t* best;                   // [R_pad][n_pad]
    long long* accum;               // [3][R_pad], zero at launch
    long long* E_out;               // [R_pad]
    long long* bestcut;             // [R_pad]
    int32_t* best_sweep;            // [R_pad]
    long long* trace;               // row of this launch's pass 1 candidate (row -1 = pass 0's, if it is a candidate), or nullptr
    unsigned long long trace_stride;
    const uint32_t* thr;            // DEVICE [n_sweeps]
    unsigned int* barrier;          // zero at launch
    int* error_flag;
    uint32_t n, n_pad, r_pad, n_replicas, rep0;
    uint32_t n_sweeps;              // update passes of this launch
    uint32_t sweep_offset;          // absolute index of this launch's first sweep
    int32_t tie_rule;
    int32_t cur;
    int32_t final_eval;             // 1: one more pass that only evaluates the final state
    int32_t first_is_candidate;     // 1: the state this launch starts from is the candidate of the sweep before (chunked call)
    int32_t have_best;              // 1: bestcut / best_sweep hold the bests of earlier chunks
    long long W;
    unsigned long long* timing;     // diagnostics: SM-clock stamps of CTA 0 in pass timing_pass (8 words), or nullptr
    uint32_t timing_pass;
    PhiloxKeys keys;
};

constexpr int kDAM = 128;   // replicas per tile (UMMA M)
constexpr int kDAN = 256;   // spins per tile (UMMA N)

__global__ void __launch_bounds__(kDThreads, 1)
k_dense_anneal(const __grid_constant__ CUtensorMap tm_j, const __grid_constant__ CUtensorMap tm_s0,
               const __grid_constant__ CUtensorMap tm_s1, const DenseAnnealParams p) {
    extern __shared__ uint8_t dsm_raw[];
    uint8_t* dsm = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(dsm_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t* sm_a = dsm;                                         // [stages][128 replicas x 128 B]
    uint8_t* sm_b = dsm + kDStages * kDStageBytesA;              // [stages][256 spins x 128 B]
    uint64_t* bars = reinterpret_cast<uint64_t*>(dsm + kDStages * (kDStageBytesA + kDStageBytesB));
    uint64_t* full = bars;
    uint64_t* empty = bars + kDStages;
    uint64_t* acc_full = bars + 2 * kDStages;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * kDStages + 1);
    __shared__ int s_col[kDAM];                // sum_i s_i h_i over this CTA's 256 spins, per replica
    __shared__ long long s_best[kDAM];
    __shared__ int s_bs[kDAM];
    __shared__ uint8_t s_hb[kDAM];             // a best state exists
    __shared__ uint32_t s_imp[kDAM / 32];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t r0 = blockIdx.x * kDAM, i0 = blockIdx.y * kDAN;   // first replica / first spin of the tile
    const uint32_t num_kb = p.n_pad / kDK;
    const uint32_t n_cta = gridDim.x * gridDim.y;
    const uint32_t n_pass = p.n_sweeps + (p.final_eval ? 1u : 0u);

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < kDStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        mbar_init(acc_full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(kDAN));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    for (uint32_t c = threadIdx.x; c < (uint32_t)kDAM; c += blockDim.x) {
        s_col[c] = 0;
        s_best[c] = p.have_best ? p.bestcut[r0 + c] : 0;
        s_bs[c] = p.have_best ? p.best_sweep[r0 + c] : 0;
        s_hb[c] = p.have_best ? 1 : 0;
    }
    // epilogue thread = replica r0 + 32 q + lane, spins i0 + 64 cg .. + 63: its old spins as 64 bits (bit k = spin 64 cg + k is +1)
    const uint32_t q = (uint32_t)warp & 3u, cg = warp >= 2 ? ((uint32_t)warp - 2u) >> 2 : 0u;
    const uint32_t rloc = q * 32u + (uint32_t)lane;
    const size_t my_row = (size_t)(r0 + rloc) * p.n_pad + i0 + cg * 64u;
    uint32_t old_lo = 0, old_hi = 0;
    if (warp >= 2) {
        const uint4* src = reinterpret_cast<const uint4*>(p.S[p.cur] + my_row);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint4 v = src[k];
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
            uint32_t bits = 0;
#pragma unroll
            for (int b = 0; b < 16; ++b) bits |= (((w[b >> 2] >> (8 * (b & 3))) & 0xffu) == 1u ? 1u : 0u) << b;
            if (k < 2) old_lo |= bits << (16 * k); else old_hi |= bits << (16 * (k - 2));
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot;
    unsigned int epoch = 0;
    bool ok = true;

    for (uint32_t t = 0; t < n_pass; ++t) {
        const int cur = (p.cur + (int)t) & 1;
        const bool update = t < p.n_sweeps;
        const uint32_t kb0 = t * num_kb;
        unsigned long long* ts = (p.timing && t == p.timing_pass && blockIdx.x == 0 && blockIdx.y == 0) ? p.timing : nullptr;
        if (ts && threadIdx.x == 0) ts[0] = (unsigned long long)clock64();
        if (warp == 0) {
            if (lane == 0) {   // ---- TMA producer: A = this tile's 128 replica rows of S^t, B = its 256 rows of J
                asm volatile("fence.proxy.async;" ::: "memory");   // S^t was written by generic-proxy stores of other CTAs
                const CUtensorMap* tms = cur ? &tm_s1 : &tm_s0;
                for (uint32_t kb = 0; kb < num_kb && ok; ++kb) {
                    const uint32_t kk = kb0 + kb, s = kk % kDStages, ph = (kk / kDStages) & 1u;
                    ok = mbar_wait(&empty[s], ph ^ 1u, p.error_flag);
                    if (!ok) break;
                    mbar_expect_tx(&full[s], kDStageBytesA + kDStageBytesB);
                    tma_load_2d(tms, &full[s], sm_a + s * kDStageBytesA, (int)(kb * kDK), (int)r0);
                    tma_load_2d(&tm_j, &full[s], sm_b + s * kDStageBytesB, (int)(kb * kDK), (int)i0);
                }
                if (ts) ts[1] = (unsigned long long)clock64();
            }
        } else if (warp == 1) {
            if (lane == 0) {   // ---- MMA issuer
                constexpr uint32_t idesc = umma_idesc_i8(kDAM, kDAN);
                for (uint32_t kb = 0; kb < num_kb && ok; ++kb) {
                    const uint32_t kk = kb0 + kb, s = kk % kDStages, ph = (kk / kDStages) & 1u;
                    ok = mbar_wait(&full[s], ph, p.error_flag);
                    if (!ok) break;
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint64_t da = umma_desc_k128(smem_u32(sm_a + s * kDStageBytesA));
                    const uint64_t db = umma_desc_k128(smem_u32(sm_b + s * kDStageBytesB));
#pragma unroll
                    for (uint32_t k = 0; k < kDK / 32; ++k)
                        umma_i8(tmem_base, da + 2 * k, db + 2 * k, idesc, (kb | k) != 0u ? 1u : 0u);
                    umma_commit(&empty[s]);
                }
                umma_commit(acc_full);
                if (ts) ts[2] = (unsigned long long)clock64();
            }
        } else {
            // ---- flips of this pass, drawn while the MMAs run: bit k of f = flip spin i0 + 64 cg + k of this replica
            const uint32_t rep = p.rep0 + r0 + rloc;
            const bool rlive = r0 + rloc < p.n_replicas;
            uint32_t f_lo = 0, f_hi = 0;
            const uint32_t thr = update ? __ldg(p.thr + t) : 0u, T = p.sweep_offset + t;
            if (update && thr != 0u) {
                const uint32_t ibase = i0 + cg * 64u;
                if ((p.rep0 & 3u) == 0u) {
                    // the four lanes of a replica group share the calls: lane x draws the spins 4 m + x and keeps, per
                    // spin, the nibble of the four replicas' decisions; then every lane collects its own bit of every nibble
                    const uint32_t x = (uint32_t)lane & 3u;
                    uint32_t n_lo = 0, n_hi = 0;   // nibble m = decisions of spin 4 m + x for replicas 4 g .. 4 g + 3
#pragma unroll 4
                    for (uint32_t m = 0; m < 16u; ++m) {
                        const uint32_t nib = lt4(philox4x32_10(ibase + 4u * m + x, T, rep >> 2, kDomainFlip, p.keys), thr);
                        if (m < 8u) n_lo |= nib << (4u * m); else n_hi |= nib << (4u * (m - 8u));
                    }
#pragma unroll
                    for (uint32_t y = 0; y < 4u; ++y) {   // from lane y of the group: spins 4 m + y, my bit x of every nibble
                        const int srcl = (lane & ~3) | (int)y;
                        const uint32_t a_lo = (__shfl_sync(0xffffffffu, n_lo, srcl) >> x) & 0x11111111u;
                        const uint32_t a_hi = (__shfl_sync(0xffffffffu, n_hi, srcl) >> x) & 0x11111111u;
                        f_lo |= a_lo << y;   // nibble m, bit y  <->  spin 4 m + y  (m < 8)
                        f_hi |= a_hi << y;
                    }
                } else {   // first replica not a multiple of four: every lane draws its own words
                    for (uint32_t k = 0; k < 64u; ++k) {
                        const uint4 u = philox4x32_10(ibase + k, T, rep >> 2, kDomainFlip, p.keys);
                        const uint32_t w = (rep & 3u) == 0u ? u.x : (rep & 3u) == 1u ? u.y : (rep & 3u) == 2u ? u.z : u.w;
                        if (w < thr) { if (k < 32u) f_lo |= 1u << k; else f_hi |= 1u << (k - 32u); }
                    }
                }
            }
            // ---- epilogue
            const bool accok = mbar_wait(acc_full, t & 1u, p.error_flag);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            if (ts && threadIdx.x == 64) ts[3] = (unsigned long long)clock64();
            if (accok) {
                int esum = 0;
                uint32_t hbuf[2][16];
                tmem_ld16(tmem_base + ((q * 32u) << 16) + cg * 64u, hbuf[0]);
#pragma unroll
                for (uint32_t ch = 0; ch < 4; ++ch) {
                    const uint32_t c0 = cg * 64u + 16u * ch;
                    uint32_t (&hreg)[16] = hbuf[ch & 1u];
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    if (ch < 3u) tmem_ld16(tmem_base + ((q * 32u) << 16) + c0 + 16u, hbuf[(ch + 1u) & 1u]);   // next chunk under way
                    const uint32_t old16 = ((ch < 2 ? old_lo : old_hi) >> (16u * (ch & 1u))) & 0xffffu;
                    const uint32_t flip16 = ((ch < 2 ? f_lo : f_hi) >> (16u * (ch & 1u))) & 0xffffu;
                    uint32_t new16 = 0;
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const int hv = (int)hreg[j];
                        const bool opos = (old16 >> j) & 1u;
                        esum += opos ? hv : -hv;                                 // a7: s_i h_i (padding spins: h = 0)
                        bool apos = hv < 0;                                      // a4 (L47-49, Q1/Q3): +1 iff h < 0
                        if (p.tie_rule == 1 && hv == 0) apos = opos;             // KEEP
                        if ((flip16 >> j) & 1u) apos = !apos;                    // a5 (Alg. 2)
                        new16 |= (apos ? 1u : 0u) << j;
                    }
                    if (update) {
                        if (ch < 2) old_lo = (old_lo & ~(0xffffu << (16u * ch))) | (new16 << (16u * ch));
                        else old_hi = (old_hi & ~(0xffffu << (16u * (ch - 2u)))) | (new16 << (16u * (ch - 2u)));
                        // a6: 16 spins of the next state as bytes (+1 = 0x01, -1 = 0xff; padding spins and replicas stay 0)
                        const uint32_t ifirst = i0 + c0;
                        const uint32_t livem = !rlive || ifirst >= p.n ? 0u : (p.n - ifirst >= 16u ? 0xffffu : (1u << (p.n - ifirst)) - 1u);
                        uint32_t out[4];
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const uint32_t m = nibble_to_bytemask((new16 >> (4 * k)) & 15u);
                            out[k] = (0xffffffffu ^ (m & 0xfefefefeu)) & nibble_to_bytemask((livem >> (4 * k)) & 15u);
                        }
                        *reinterpret_cast<uint4*>(p.S[cur ^ 1] + my_row + 16u * ch) = make_uint4(out[0], out[1], out[2], out[3]);
                    }
                }
                if (rlive && esum != 0) atomicAdd(&s_col[rloc], esum);
                asm volatile("fence.proxy.async;" ::: "memory");   // the next pass reads these bytes through TMA
            }
            if (ts && threadIdx.x == 64) ts[4] = (unsigned long long)clock64();
            asm volatile("bar.sync 1, %0;" ::"n"(32 * kDEpiWarps) : "memory");   // the epilogue warps: s_col complete
            {
                const uint32_t c = threadIdx.x - 64u;
                if (c < (uint32_t)kDAM) {
                    const int v = s_col[c];
                    if (v != 0) atomicAdd(reinterpret_cast<unsigned long long*>(p.accum + (size_t)(t % 3u) * p.r_pad + r0 + c),
                                          (unsigned long long)(long long)v);
                    s_col[c] = 0;
                }
            }
        }
        // ---- grid barrier: S^(t+1) and the energy slot are complete everywhere
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (ts && threadIdx.x == 0) ts[5] = (unsigned long long)clock64();
        epoch += n_cta;
        if (threadIdx.x == 0 && n_cta > 1u) {
            asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(p.barrier) : "memory");
            unsigned int v;
            for (uint32_t spin = 0; spin < (1u << 26); ++spin) {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p.barrier) : "memory");
                if ((int)(v - epoch) >= 0) break;
                __nanosleep(40);
            }
        }
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (ts && threadIdx.x == 0) ts[6] = (unsigned long long)clock64();

        // ---- a7: candidate S^t (pass 0: only in a continued chunk): E, cut = (W - E)/2 (eq. 4), best tracking
        const bool candidate = t > 0u || p.first_is_candidate != 0;
        if (threadIdx.x < (uint32_t)kDAM) {
            const uint32_t c = threadIdx.x;
            const long long a = __ldcg(p.accum + (size_t)(t % 3u) * p.r_pad + r0 + c);
            const long long E = a / 2, cut = (p.W - E) / 2;
            const bool liver = r0 + c < p.n_replicas;
            const bool improved = candidate && liver && (!s_hb[c] || cut > s_best[c]);
            if (improved) { s_best[c] = cut; s_bs[c] = (int)(p.sweep_offset + t) - 1; s_hb[c] = 1; }
            const uint32_t m = __ballot_sync(0xffffffffu, improved);
            if (lane == 0) s_imp[c >> 5] = m;
            if (blockIdx.y == 0) {
                p.accum[(size_t)((t + 2u) % 3u) * p.r_pad + r0 + c] = 0;
                p.E_out[r0 + c] = E;
                if (candidate && liver && p.trace) p.trace[((long long)t - 1) * (long long)p.trace_stride + (long long)(r0 + c)] = cut;
            }
        }
        __syncthreads();
        {   // best-state capture: this CTA's 256 spins of every improved replica, from S^t
            const int8_t* src = p.S[cur];
            for (uint32_t i = threadIdx.x; i < (uint32_t)kDAM * 16u; i += blockDim.x) {
                const uint32_t c = i >> 4, k = i & 15u;
                if ((s_imp[c >> 5] >> (c & 31u)) & 1u) {
                    const size_t at = (size_t)(r0 + c) * p.n_pad + i0 + 16u * k;
                    *reinterpret_cast<uint4*>(p.best + at) = __ldcg(reinterpret_cast<const uint4*>(src + at));
                }
            }
        }
        __syncthreads();
        if (ts && threadIdx.x == 0) ts[7] = (unsigned long long)clock64();
    }
    if (blockIdx.y == 0 && threadIdx.x < (uint32_t)kDAM) {
        p.bestcut[r0 + threadIdx.x] = s_best[threadIdx.x];
        p.best_sweep[r0 + threadIdx.x] = s_bs[threadIdx.x];
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 2) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kDAN));
    }
}

// ---------------------------------------------------------------------------------------------
// Small kernels of the dense engine
// ---------------------------------------------------------------------------------------------
// J[i][j] = w_ij from the caller's CSR (one warp per row); J is zero elsewhere (diagonal, padding).
__global__ void k_dense_build_j(int8_t* J, uint32_t n, uint32_t n_pad, const long long* row_ptr, const int32_t* col,
                                const void* w, int wtype) {
    const long long gw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (gw >= n) return;
    for (long long e = row_ptr[gw] + lane; e < row_ptr[gw + 1]; e += 32) {
        const int v = wtype == 1 ? (int)reinterpret_cast<const int8_t*>(w)[e] : reinterpret_cast<const int32_t*>(w)[e];
        J[(size_t)gw * n_pad + (uint32_t)col[e]] = (int8_t)v;
    }
}

// sparse interleaved layout (state[tile][row][32], internal rows) -> dense replica-major [R_pad][n_pad]
__global__ void k_dense_import(int8_t* S, const uint8_t* sparse, const int32_t* perm, uint32_t n, uint32_t n_pad,
                               unsigned long long tile_stride, int32_t n_replicas) {
    const unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;   // (row, rr)
    const uint32_t tile = blockIdx.y;
    if (t >= (unsigned long long)n * kTile) return;
    const uint32_t row = (uint32_t)(t >> 5), rr = (uint32_t)(t & 31);
    const int rep = (int)(tile * kTile + rr);
    if (rep < n_replicas)
        S[(size_t)rep * n_pad + (uint32_t)perm[row]] = (int8_t)sparse[(size_t)tile * tile_stride + (size_t)row * kTile + rr];
}

// dense [R_pad][n_pad] -> caller layout [R][n] (replica_sel >= 0: that one replica to out[n])
__global__ void k_dense_export(const int8_t* S, int8_t* out, uint32_t n, uint32_t n_pad, int32_t n_replicas,
                               int32_t replica_sel) {
    const unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (replica_sel >= 0) {
        if (t < n) out[t] = S[(size_t)replica_sel * n_pad + t];
        return;
    }
    if (t >= (unsigned long long)n * (unsigned long long)n_replicas) return;
    const uint32_t rep = (uint32_t)(t / n), i = (uint32_t)(t % n);
    out[t] = S[(size_t)rep * n_pad + i];
}

// Per replica (one block each): E = accum / 2, cut = (W - E)/2 (eq. 4), trace, best capture of the
// candidate state (a7).  record_only: initial state, no candidate.
__global__ void __launch_bounds__(256) k_dense_sweep_end(const int8_t* S, int8_t* best, long long* accum, long long* E_out,
                                                         long long* bestcut, int32_t* best_sweep, long long* trace_row,
                                                         uint32_t n_pad, long long W, int32_t record_only, int32_t first,
                                                         int32_t T) {
    const uint32_t r = blockIdx.x;
    const long long E = accum[r] / 2;
    const long long cut = (W - E) / 2;
    const bool improved = !record_only && (first || cut > bestcut[r]);
    __syncthreads();   // everyone has read accum / bestcut before thread 0 rewrites them
    if (threadIdx.x == 0) {
        accum[r] = 0;
        E_out[r] = E;
        if (!record_only && trace_row) trace_row[r] = cut;
        if (improved) { bestcut[r] = cut; best_sweep[r] = T; }
    }
    if (!improved) return;
    const uint4* src = reinterpret_cast<const uint4*>(S + (size_t)r * n_pad);
    uint4* dst = reinterpret_cast<uint4*>(best + (size_t)r * n_pad);
    for (uint32_t k = threadIdx.x; k < n_pad / 16; k += blockDim.x) dst[k] = src[k];
}

// ---------------------------------------------------------------------------------------------
// Host side of the engine
// ---------------------------------------------------------------------------------------------
struct DenseEngine {
    uint32_t n = 0, n_pad = 0, r_pad = 0;
    int8_t* J = nullptr;
    int8_t* S[2] = {nullptr, nullptr};
    int8_t* best = nullptr;
    long long* accum = nullptr;
    long long* E = nullptr;
    long long* bestcut = nullptr;
    int32_t* best_sweep = nullptr;
    int* error_flag = nullptr;
    unsigned int* barrier = nullptr;
    int cur = 0;
    CUtensorMap tm_j{}, tm_s[2]{};
    // persistent kernel (k_dense_anneal): cooperative launch of one CTA per tile of the transposed product
    bool persistent = false;
    CUtensorMap tm_sa[2]{}, tm_jb{};    // S as operand A (box of 128 replica rows), J as operand B (box of 256 rows)
    int sm_count = 0;
};

struct DenseAnnealArgs {
    int32_t tie_rule, n_replicas, first_replica;
    PhiloxKeys keys;
    const uint32_t* thresholds;
    int32_t n_sweeps, sweep_offset;
    int64_t* cut_trace;
    long long W;
    bool import_from_sparse;
    const uint8_t* sparse_state;
    const int32_t* perm;
    int8_t* io_stage;
    uint32_t* thr_dev;        // device staging of the thresholds (thr_cap entries), filled by the caller per chunk
    const uint32_t* thr_host;
    uint32_t thr_cap;
    unsigned long long* timing;   // diagnostics (include/ising_debug.h)
    uint32_t timing_pass;
};

inline uint32_t dense_round_up(uint32_t x, uint32_t m) { return (x + m - 1) / m * m; }

inline size_t dense_workspace_bytes(int64_t n, int64_t max_replicas) {
    const size_t n_pad = dense_round_up((uint32_t)n, kDAN), r_pad = dense_round_up((uint32_t)max_replicas, kDN);
    return n_pad * n_pad + 3 * r_pad * n_pad + r_pad * (8 * 5 + 4) + 4096 + 10 * 1024;
}

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 2-D uint8 tensor [rows][cols] (cols contiguous), box = box_rows x 128 bytes, 128-byte swizzle.
inline bool dense_make_map(CUtensorMap* map, void* base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    static PFN_encodeTiled fn = nullptr;
    if (!fn) {
        void* sym = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &q) != cudaSuccess || !sym) {
            (void)cudaGetLastError();
            return false;
        }
        fn = (PFN_encodeTiled)sym;
    }
    const cuuint64_t dims[2] = {cols, rows};
    const cuuint64_t strides[1] = {cols};
    const cuuint32_t box[2] = {(cuuint32_t)kDK, box_rows};
    const cuuint32_t estr[2] = {1, 1};
    return fn(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) ==
           CUDA_SUCCESS;
}

inline DenseEngine* dense_create(int32_t n, int32_t max_replicas, void* mem, size_t bytes, const long long* row_ptr,
                                 const int32_t* col, const void* w, int wtype, cudaStream_t st) {
    DenseEngine* d = new (std::nothrow) DenseEngine();
    if (!d) return nullptr;
    d->n = (uint32_t)n;
    d->n_pad = dense_round_up((uint32_t)n, kDAN);   // 256: a whole number of spin tiles of either kernel
    d->r_pad = dense_round_up((uint32_t)max_replicas, kDN);
    uint8_t* base = (uint8_t*)mem;
    size_t off = 0;
    auto take = [&](size_t b) { void* p = base + off; off = (off + b + 1023) / 1024 * 1024; return p; };
    const size_t sb = (size_t)d->r_pad * d->n_pad;
    d->J = (int8_t*)take((size_t)d->n_pad * d->n_pad);
    d->S[0] = (int8_t*)take(sb);
    d->S[1] = (int8_t*)take(sb);
    d->best = (int8_t*)take(sb);
    d->accum = (long long*)take(3 * 8 * (size_t)d->r_pad);
    d->E = (long long*)take(8 * (size_t)d->r_pad);
    d->bestcut = (long long*)take(8 * (size_t)d->r_pad);
    d->best_sweep = (int32_t*)take(4 * (size_t)d->r_pad);
    d->error_flag = (int*)take(256);
    d->barrier = (unsigned int*)take(256);
    bool ok = off <= bytes;
    ok = ok && cudaMemsetAsync(d->J, 0, (size_t)d->n_pad * d->n_pad, st) == cudaSuccess;
    ok = ok && cudaMemsetAsync(d->S[0], 0, 3 * sb, st) == cudaSuccess;   // S[0], S[1], best are adjacent
    ok = ok && cudaMemsetAsync(d->error_flag, 0, 256, st) == cudaSuccess;
    if (ok) {
        k_dense_build_j<<<(unsigned)(((long long)n * 32 + 255) / 256), 256, 0, st>>>(d->J, d->n, d->n_pad, row_ptr, col, w, wtype);
        ok = dense_make_map(&d->tm_j, d->J, d->n_pad, d->n_pad, kDM) &&
             dense_make_map(&d->tm_s[0], d->S[0], d->r_pad, d->n_pad, kDN) &&
             dense_make_map(&d->tm_s[1], d->S[1], d->r_pad, d->n_pad, kDN);
        ok = ok && cudaFuncSetAttribute(k_dense_sweep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kDSmemBytes) == cudaSuccess;
        ok = ok && cudaFuncSetAttribute(k_dense_anneal, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kDSmemBytes) == cudaSuccess;
    }
    if (ok) {
        int dev = 0, coop = 0;
        ok = cudaGetDevice(&dev) == cudaSuccess &&
             cudaDeviceGetAttribute(&d->sm_count, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
             cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) == cudaSuccess;
        d->persistent = ok && coop != 0;
        // transposed product: A = 128 replica rows of S, B = 256 rows of J
        ok = ok && dense_make_map(&d->tm_sa[0], d->S[0], d->r_pad, d->n_pad, kDAM) &&
             dense_make_map(&d->tm_sa[1], d->S[1], d->r_pad, d->n_pad, kDAM) &&
             dense_make_map(&d->tm_jb, d->J, d->n_pad, d->n_pad, kDAN);
    }
    if (!ok) { (void)cudaGetLastError(); delete d; return nullptr; }
    return d;
}

inline void dense_destroy(DenseEngine* d) { delete d; }

// The persistent path: one cooperative launch per chunk of <= thr_cap sweeps.  Asynchronous: a pipeline time-out raises
// error_flag, which the next synchronising call (dense_best_arrays) reports.
inline ising_status dense_anneal_persistent(DenseEngine* d, const DenseAnnealArgs& a, const dim3 grid, cudaStream_t st,
                                            int64_t* launches) {
    const uint32_t R = (uint32_t)a.n_replicas;
    for (int32_t s0 = 0; s0 < a.n_sweeps; s0 += (int32_t)a.thr_cap) {
        const int32_t ns = std::min<int32_t>((int32_t)a.thr_cap, a.n_sweeps - s0);
        if (cudaMemcpyAsync(a.thr_dev, a.thr_host + s0, 4 * (size_t)ns, cudaMemcpyHostToDevice, st) != cudaSuccess ||
            cudaMemsetAsync(d->accum, 0, 3 * 8 * (size_t)d->r_pad, st) != cudaSuccess ||
            cudaMemsetAsync(d->barrier, 0, 256, st) != cudaSuccess)
            return ISING_ERR_CUDA;
        DenseAnnealParams p{};
        p.S[0] = d->S[0]; p.S[1] = d->S[1]; p.best = d->best; p.accum = d->accum; p.E_out = d->E; p.bestcut = d->bestcut;
        p.best_sweep = d->best_sweep;
        p.trace = a.cut_trace ? (long long*)a.cut_trace + (size_t)s0 * R : nullptr;
        p.trace_stride = R;
        p.thr = a.thr_dev; p.barrier = d->barrier; p.error_flag = d->error_flag;
        p.n = d->n; p.n_pad = d->n_pad; p.r_pad = d->r_pad; p.n_replicas = R; p.rep0 = (uint32_t)a.first_replica;
        p.n_sweeps = (uint32_t)ns; p.sweep_offset = (uint32_t)(a.sweep_offset + s0); p.tie_rule = a.tie_rule; p.cur = d->cur;
        p.final_eval = s0 + ns == a.n_sweeps ? 1 : 0;
        p.first_is_candidate = s0 > 0 ? 1 : 0;
        p.have_best = s0 > 0 ? 1 : 0;
        p.W = a.W; p.keys = a.keys;
        p.timing = s0 == 0 ? a.timing : nullptr; p.timing_pass = a.timing_pass;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = grid;
        cfg.blockDim = dim3(kDThreads);
        cfg.dynamicSmemBytes = kDSmemBytes;
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeCooperative;
        at[0].val.cooperative = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        if (cudaLaunchKernelEx(&cfg, k_dense_anneal, d->tm_jb, d->tm_sa[0], d->tm_sa[1], p) != cudaSuccess) {
            (void)cudaGetLastError();
            return ISING_ERR_CUDA;
        }
        ++*launches;
        d->cur = (d->cur + ns) & 1;
    }
    return ISING_OK;
}

inline ising_status dense_anneal(DenseEngine* d, const DenseAnnealArgs& a, cudaStream_t st, int64_t* launches) {
    const uint32_t R = (uint32_t)a.n_replicas;
    const dim3 grid(d->n_pad / kDM, dense_round_up(R, kDN) / kDN);
    const dim3 pgrid(dense_round_up(R, kDAM) / kDAM, d->n_pad / kDAN);   // tiles of the transposed product
    if (d->persistent && a.n_sweeps > 0 && pgrid.x * pgrid.y <= (unsigned)d->sm_count) {
        if (a.import_from_sparse) {
            d->cur = 0;
            const size_t sb = (size_t)d->r_pad * d->n_pad;
            if (cudaMemsetAsync(d->S[0], 0, 2 * sb, st) != cudaSuccess) return ISING_ERR_CUDA;
            const int tiles = (a.n_replicas + kTile - 1) / kTile;
            k_dense_import<<<dim3((unsigned)(((unsigned long long)d->n * kTile + 255) / 256), tiles), 256, 0, st>>>(
                d->S[0], a.sparse_state, a.perm, d->n, d->n_pad, (unsigned long long)d->n * kTile, a.n_replicas);
            ++*launches;
        }
        return dense_anneal_persistent(d, a, pgrid, st, launches);
    }
    if (a.import_from_sparse) {
        d->cur = 0;
        const size_t sb = (size_t)d->r_pad * d->n_pad;
        if (cudaMemsetAsync(d->S[0], 0, 2 * sb, st) != cudaSuccess) return ISING_ERR_CUDA;
        const int tiles = (a.n_replicas + kTile - 1) / kTile;
        k_dense_import<<<dim3((unsigned)(((unsigned long long)d->n * kTile + 255) / 256), tiles), 256, 0, st>>>(
            d->S[0], a.sparse_state, a.perm, d->n, d->n_pad, (unsigned long long)d->n * kTile, a.n_replicas);
        ++*launches;
    }
    if (cudaMemsetAsync(d->accum, 0, 8 * (size_t)d->r_pad, st) != cudaSuccess) return ISING_ERR_CUDA;
    // pass t reads s^t and yields 2 E(s^t) as a by-product; pass n_sweeps is evaluation only
    for (int32_t t = 0; t <= a.n_sweeps; ++t) {
        DenseSweepParams p{};
        p.src = d->S[d->cur]; p.dst = d->S[d->cur ^ 1]; p.accum = d->accum; p.error_flag = d->error_flag;
        p.n = d->n; p.n_pad = d->n_pad; p.rep0 = (uint32_t)a.first_replica; p.tie_rule = a.tie_rule; p.keys = a.keys;
        p.update = t < a.n_sweeps ? 1 : 0;
        if (p.update) { p.thr = a.thresholds[t]; p.T = (uint32_t)(a.sweep_offset + t); }
        k_dense_sweep<<<grid, kDThreads, kDSmemBytes, st>>>(d->tm_j, d->tm_s[d->cur], p);
        k_dense_sweep_end<<<R, 256, 0, st>>>(d->S[d->cur], d->best, d->accum, d->E, d->bestcut, d->best_sweep,
                                            (t > 0 && a.cut_trace) ? (long long*)a.cut_trace + (size_t)(t - 1) * R : nullptr,
                                            d->n_pad, a.W, t == 0 ? 1 : 0, t == 1 ? 1 : 0, a.sweep_offset + t - 1);
        *launches += 2;
        if (p.update) d->cur ^= 1;
    }
    int err = 0;
    if (cudaMemcpyAsync(&err, d->error_flag, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess)
        return ISING_ERR_CUDA;
    return err ? ISING_ERR_CUDA : ISING_OK;
}

// caller layout [n_replicas][n] of the current (or best) state
inline ising_status dense_export_state(DenseEngine* d, int8_t* out, int32_t n_replicas, bool best, cudaStream_t st) {
    const unsigned long long total = (unsigned long long)d->n * (unsigned long long)n_replicas;
    k_dense_export<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(best ? d->best : d->S[d->cur], out, d->n, d->n_pad,
                                                                    n_replicas, -1);
    return cudaGetLastError() == cudaSuccess ? ISING_OK : ISING_ERR_CUDA;
}
inline ising_status dense_export_one(DenseEngine* d, int8_t* out, int32_t replica, bool best, cudaStream_t st) {
    k_dense_export<<<(unsigned)((d->n + 255) / 256), 256, 0, st>>>(best ? d->best : d->S[d->cur], out, d->n, d->n_pad, 1,
                                                                   replica);
    return cudaGetLastError() == cudaSuccess ? ISING_OK : ISING_ERR_CUDA;
}
inline ising_status dense_best_arrays(DenseEngine* d, long long* bc, int32_t* bs, int32_t R, cudaStream_t st) {
    int err = 0;
    if (cudaMemcpyAsync(bc, d->bestcut, 8 * (size_t)R, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemcpyAsync(bs, d->best_sweep, 4 * (size_t)R, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemcpyAsync(&err, d->error_flag, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return ISING_ERR_CUDA;
    return err ? ISING_ERR_CUDA : ISING_OK;   // (a pipeline time-out of the asynchronous anneal surfaces here)
}

}  // namespace ising
