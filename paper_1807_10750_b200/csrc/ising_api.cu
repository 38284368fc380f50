// C-ABI entry points of the B200 Ising annealer (include/ising.h).
//
// Host side: argument validation, workspace carving, the O(n) slice planning of the
// device layout, and the per-sweep launch sequence.  Every step of the hot path
// (field, argmin, flip, write-back, cut reduction, best capture) runs in the kernels of
// sparse_sweep.cuh / dense_tcgen05.cuh; there is no CPU fallback.
#include <cuda_runtime.h>

#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdint>
#include <cstring>
#include <new>
#include <type_traits>
#include <vector>

#include "../../include/ising.h"
#include "../../include/ising_debug.h"
#include "builder.cuh"
#include "common.cuh"
#include "dense_tcgen05.cuh"
#include "noalloc.cuh"
#include "probe.cuh"
#include "sparse_sweep.cuh"

using namespace ising;

#define CK(call)                                  \
    do {                                          \
        cudaError_t e_ = (call);                  \
        if (e_ != cudaSuccess) {                  \
            (void)cudaGetLastError();             \
            return ISING_ERR_CUDA;                \
        }                                         \
    } while (0)

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct Bump {
    uint8_t* base;
    size_t cap, used;
    bool overflow;
    void* take(size_t bytes) {
        const size_t at = align_up(used);
        if (at + bytes > cap) { overflow = true; used = at + bytes; return nullptr; }
        used = at + bytes;
        return base + at;
    }
};

bool is_device_ptr(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

inline int spr_log2_for_degree(int64_t deg, int sub_row_edges) {
    int l = 0;
    while (l < 4 && ((deg + (1ll << l) - 1) >> l) > sub_row_edges) ++l;
    return l;
}

constexpr int kClusterCtas = 8;       // portable cluster size; 8 x 16 warps per replica tile
constexpr uint32_t kThrCap = 1u << 16;   // thresholds per persistent launch (longer schedules are chunked)

// Upper bounds used by ising_workspace_bytes (any degree distribution).
inline uint64_t bound_slices(int64_t n, int64_t nnz, int64_t C) {
    // full slices of rows with <= 8 edges, full row-split slices (> 64 edges each), one ragged
    // slice per (colour, SPR)
    return (uint64_t)n / 16 + (uint64_t)nnz / 64 + 5 * (uint64_t)(C + 1) + 8;
}
inline uint64_t bound_hubs(int64_t n, int64_t nnz) { return std::min<uint64_t>((uint64_t)n, (uint64_t)nnz / 129 + 1); }   // hub rows have > 128 edges
inline uint64_t bound_cells(int64_t n, int64_t nnz, int64_t C) {
    // two head cells per sub-row of every slice; tail cells only for rows of 129..256 edges (each
    // holds >= 1 edge of a sub-row that is more than half full); hubs: nnz_h/4 + 256 cells of rounding each, at least two groups
    return kHeadGroups * kSubRows * bound_slices(n, nnz, C) + (uint64_t)nnz / 2 +
           (uint64_t)nnz / 4 + 64;
}
constexpr uint64_t kMaxCtas = 1024;

struct SmallArrays {
    long long* accum[2];
    long long* E[2];
    long long* bestcut[2];
    long long* accum_eval;
    long long* out_tmp;    // 2 * max_replicas
    long long* accum3;     // 3 * kMaxPersistReplicas (persistent kernel)
    int32_t* best_sweep;
    uint32_t* thr;         // kThrCap
    unsigned int* barrier;
    int* flag;
};

size_t chain_ws_bound(int64_t n, int64_t nnz, int64_t tiles);

size_t workspace_need(int64_t n, int64_t nnz, int wtype, int64_t max_replicas, int64_t C, bool wide,
                      uint64_t n_slices, uint64_t n_hubs, uint64_t cells, bool with_raw, bool dense) {
    const uint64_t tiles = (uint64_t)(max_replicas + kTile - 1) / kTile;
    const uint64_t phases = (uint64_t)std::max<int64_t>(1, C) + 1;   // (+ 1: the overlap split of class 0)
    size_t s = 0;
    auto add = [&](size_t b) { s = align_up(s) + b; };
    add(sizeof(BuildReport));
    if (with_raw) {
        add(8 * (size_t)(n + 1));
        add(4 * (size_t)nnz);
        add((size_t)wtype * (size_t)nnz);
        add(4 * (size_t)n);
    }
    add(4 * (size_t)n);                       // perm
    add(4 * (size_t)n);                       // inv
    add(4 * (size_t)n);                       // relabelling: second id buffer
    add(4 * 256 * (size_t)((n + kRadixChunk - 1) / kRadixChunk));   // digit histograms
    add(sizeof(RelabelRuns));
    add(12 * (size_t)n);                      // runs of equal (colour, degree)
    add(4 * (size_t)n);                       // colours after the overlap split of class 0
    add(sizeof(SliceDesc) * (size_t)(n_slices + 1));
    add(4 * 16 * (size_t)(n_slices + 1));     // sorig
    add(8 * (size_t)(n_slices + 1));          // slice_aux
    add(8 * kTile * (size_t)tiles * (size_t)(n_hubs + 1));   // hub_acc
    add(4 * (size_t)tiles * (size_t)(n_hubs + 1));           // hub_cnt
    add(sizeof(PhaseRange) * (size_t)(phases * kMaxCtas));
    add(16 * (size_t)(cells + 1));            // col4
    add(4 * (size_t)(cells + 1));             // w4
    if (wide) add(16 * (size_t)(cells + 1));  // w4w
    for (int k = 0; k < 3; ++k) add((size_t)tiles * (size_t)n * kTile);   // state x2, best
    add((size_t)max_replicas * (size_t)n);    // io staging
    for (int k = 0; k < 7; ++k) add(8 * (size_t)tiles * kTile);
    add(16 * (size_t)tiles * kTile);          // out_tmp
    add(8 * 3 * (size_t)kMaxPersistReplicas); // accum3
    add(4 * (size_t)tiles * kTile);           // best_sweep
    add(4 * (size_t)kThrCap);                 // thr
    add(256);                                 // barrier
    add(4 * (size_t)(phases + 1));            // phase_slices
    add(256);                                 // flag
    if (dense) add(dense_workspace_bytes(n, max_replicas));
    add(4 * (size_t)(phases + 2));            // vphase_slices
    if (C > 0) add(chain_ws_bound(n, nnz, (int64_t)tiles));
    return align_up(s) + kAlign;
}

}  // namespace

struct ising_problem {
    int32_t n = 0;
    int64_t nnz = 0;
    int32_t n_colours = 0;
    int32_t max_replicas = 0;
    int32_t tiles_max = 0;
    int64_t W = 0;
    int64_t absw_max = 0;
    bool wide = false;
    // device (inside the caller's workspace)
    int32_t* perm = nullptr;
    int32_t* inv = nullptr;
    SliceDesc* slices = nullptr;
    uint32_t* sorig = nullptr;
    uint32_t* slice_aux = nullptr;       // [n_slices][2] (hub id, part index) of hub-part slices
    bool overlap0 = false;               // chain overlap: virtual phase 0 (the rows of colour class 0 without a chain neighbour) runs
    uint32_t ov_rows = 0;                // for sweep t + 1 beside the chain of sweep t; these are the internal rows [0, ov_rows)
    int cluster_ctas = 0;                // small graph: the persistent kernel runs as one cluster of this many CTAs per replica tile (0: grid)
    unsigned long long* hub_acc = nullptr;   // [n_hubs][tiles_max][32] partial local fields of hub rows
    unsigned int* hub_cnt = nullptr;     // [n_hubs][tiles_max] parts arrived (monotone)
    PhaseRange* ranges = nullptr;
    uint32_t* phase_slices = nullptr;
    int4* col4 = nullptr;
    uint32_t* w4 = nullptr;
    int4* w4w = nullptr;
    uint8_t* state[2] = {nullptr, nullptr};
    uint8_t* best = nullptr;
    int8_t* io_stage = nullptr;
    SmallArrays sm{};
    DenseEngine* dense = nullptr;
    // host bookkeeping
    uint32_t n_slices = 0, n_hubs = 0, n_phases = 1, n_cta = 1;
    uint64_t cells = 0;
    size_t ws_used = 0;
    int cur = 0;
    int parity = 0;
    bool have_state = false;
    bool have_best = false;
    bool state_in_dense = false;         // current / best state live in the dense engine's layout
    int32_t last_R = 0;
    int64_t launches = 0;
    int sm_count = 148;
    bool cooperative = false;
    uint32_t flush_rows = 1;
    unsigned long long* timing = nullptr;   // diagnostics buffer of the next Gauss-Seidel anneal
    // chain engine (chain.cuh): either the whole graph (k_anneal_small) or the tail classes of the persistent kernel
    ChainView chain{};
    bool chain_small = false;
    bool chain_delta = false;
    uint32_t small_threads = 0;
    size_t small_dyn = 0;
    uint32_t small_csplit = 1;              // CTAs per word of four replicas (cluster size) of k_anneal_small
    uint32_t* vphase_slices = nullptr;      // [n_vphases + 1] slice ranges of the persistent kernel's virtual phases
    std::vector<uint32_t> thr_host;         // the call's thresholds (pageable copy: the caller's array is free on return)
    uint32_t n_vphases = 0;
    uint32_t timing_sweep = 0;
};

namespace {

GraphView graph_view(const ising_problem* p) {
    GraphView g{};
    g.col4 = p->col4; g.w4 = p->w4; g.w4w = p->w4w; g.slices = p->slices; g.sorig = p->sorig;
    g.hub_acc = p->hub_acc; g.hub_cnt = p->hub_cnt; g.tiles_max = (uint32_t)p->tiles_max;
    g.ranges = p->ranges; g.phase_slices = p->phase_slices; g.n_cta = p->n_cta; g.n_phases = p->n_phases;
    return g;
}

template <int KIND>
void launch_sweep_kind(ising_problem* p, const SweepParams& sp, cudaStream_t st) {
    if (p->wide) k_sweep<KIND, true><<<p->n_cta, kSweepThreads, 0, st>>>(sp);
    else k_sweep<KIND, false><<<p->n_cta, kSweepThreads, 0, st>>>(sp);
}

// One pass over colour phases [sp.phase_begin, sp.phase_end) for `tiles` replica tiles, in batches of
// kMaxPersistReplicas replicas (the kernels keep per-replica bookkeeping in shared memory).
void launch_sweep(ising_problem* p, int kind, SweepParams sp, int tiles, cudaStream_t st) {
    constexpr int kBatchTiles = kMaxPersistReplicas / kTile;
    for (int t0 = 0; t0 < tiles; t0 += kBatchTiles) {
        SweepParams q = sp;
        q.tiles = (uint32_t)std::min(kBatchTiles, tiles - t0);
        q.src = sp.src + (size_t)t0 * sp.tile_stride;
        q.dst = sp.dst + (size_t)t0 * sp.tile_stride;
        q.accum = sp.accum + (size_t)t0 * kTile;
        q.rep0 = sp.rep0 + (uint32_t)t0 * kTile;
        if (kind == kKindGS) launch_sweep_kind<kKindGS>(p, q, st);
        else if (kind == kKindJacobi) launch_sweep_kind<kKindJacobi>(p, q, st);
        else launch_sweep_kind<kKindEval>(p, q, st);
        p->launches++;
    }
}

SweepParams base_params(const ising_problem* p) {
    SweepParams sp{};
    sp.g = graph_view(p);
    sp.tile_stride = (unsigned long long)p->n * kTile;
    sp.phase_begin = 0;
    sp.phase_end = p->n_phases;
    sp.flush_rows = p->flush_rows;
    return sp;
}

void launch_sweep_end(ising_problem* p, const uint8_t* src, int energy_mode, int first, int32_t T,
                      long long* trace_row, int n_replicas, int tiles, cudaStream_t st) {
    SweepEndParams ep{};
    const int par = p->parity;
    ep.src = src;
    ep.best = p->best;
    ep.accum_in = p->sm.accum[par];
    ep.accum_zero = p->sm.accum[par ^ 1];
    ep.E_in = p->sm.E[par];
    ep.E_out = p->sm.E[par ^ 1];
    ep.best_in = p->sm.bestcut[par];
    ep.best_out = p->sm.bestcut[par ^ 1];
    ep.best_sweep = p->sm.best_sweep;
    ep.trace_row = trace_row;
    ep.tile_stride = (unsigned long long)p->n * kTile;
    ep.units = (unsigned long long)p->n * 2;
    ep.W = p->W;
    ep.n_replicas = n_replicas;
    ep.energy_mode = energy_mode;
    ep.first = first;
    ep.T = T;
    long long bx = (long long)((ep.units + 255) / 256);
    long long cap = ((long long)p->sm_count * 8 + tiles - 1) / tiles;
    if (bx > cap) bx = cap;
    if (bx < 1) bx = 1;
    if (energy_mode == 2) bx = 1;
    k_sweep_end<<<dim3((unsigned)bx, (unsigned)tiles, 1), 256, 0, st>>>(ep);
    p->launches++;
    p->parity ^= 1;
}


// ---- chain engine, host side (chain.cuh) --------------------------------------------------------------
constexpr uint32_t kTailRowsMax = 12288;        // most chain rows the persistent kernel's tail can hold (val <= 48 KB of the 144 KB)
constexpr uint32_t kTailRowsDefault = 1600;     // chain rows of the tail: the chain walks ~150 warp instructions per row and word on ONE
                                                // SM per four replicas, so it pays only for the classes that are pure latency on the grid
                                                // (config 5, us per sweep: 700 rows 199.4, 1600 195.9, 2500 200.4, 4000 206.5, 12288 245.6)
constexpr uint32_t kChainLevelThreads = 384;      // lanes per row: a level keeps about this many threads busy (the row
                                                   // update runs on one lane of L: more lanes, more warps issuing it)
constexpr uint64_t kSmallStreamBytesMax = 1ull << 20;   // a streamed small graph may re-read at most this per sweep and CTA

// Tuning knobs read from the environment exist only in builds with -DISING_TUNING_ENV (never in the shipped library).
inline int64_t tail_rows_limit() {
#ifdef ISING_TUNING_ENV
    if (const char* e = getenv("ISING_TAIL_ROWS")) return std::min<int64_t>(atoll(e), (int64_t)kTailRowsMax);
#endif
    return (int64_t)kTailRowsDefault;
}
inline uint32_t level_threads() {
#ifdef ISING_TUNING_ENV
    if (const char* e = getenv("ISING_LEVEL_THREADS")) return (uint32_t)atoi(e);
#endif
    return kChainLevelThreads;
}
inline uint32_t small_threads_override(uint32_t t) {
#ifdef ISING_TUNING_ENV
    if (const char* e = getenv("ISING_SMALL_THREADS")) return (uint32_t)atoi(e);
#endif
    return t;
}
inline const void* small_kernel(bool timing, bool premul) {
    if (timing) return premul ? (const void*)k_anneal_small<true, true> : (const void*)k_anneal_small<true, false>;
    return premul ? (const void*)k_anneal_small<false, true> : (const void*)k_anneal_small<false, false>;
}
inline uint32_t align4u(uint32_t x) { return (x + 3u) & ~3u; }
inline uint32_t pow2_floor(uint32_t x) { uint32_t r = 1; while (2u * r <= x) r *= 2u; return r; }
inline uint32_t pow2_ceil(uint32_t x) { uint32_t r = 1; while (r < x) r *= 2u; return r; }

struct ChainPlan {
    bool ok = false;
    std::vector<ChainChunk> chunks;
    std::vector<ChainSeg> segs;
    std::vector<uint32_t> cptr;      // [n_t + 1] first cell of every row (a chunk starts at a multiple of 4)
    std::vector<uint16_t> rel16;
    uint32_t cells = 0;
    uint32_t max_chunk_bytes = 0;
    uint64_t total_bytes = 0;
};

// counts[r] = cells of local row r; lvl = ascending local row boundaries of the levels (front 0, back n_t).
ChainPlan plan_chain(const std::vector<uint32_t>& counts, const std::vector<uint32_t>& lvl, uint32_t buf_bytes, bool delta,
                     uint32_t threads) {
    ChainPlan pl;
    const uint32_t n_t = (uint32_t)counts.size();
    pl.cptr.assign((size_t)n_t + 1, 0u);
    uint32_t r0 = 0, cell = 0;
    while (r0 < n_t) {
        ChainChunk ck{};
        ck.r0 = r0;
        ck.c0 = cell;
        uint32_t r1 = r0, nc = 0;
        while (r1 < n_t) {
            const uint32_t step_end = std::min(n_t, r1 + 8u);
            uint32_t add = 0;
            for (uint32_t r = r1; r < step_end; ++r) add += counts[r];
            const uint32_t nc2 = align4u(nc + add);
            if (nc2 > 65532u || chunk_layout(step_end - r0, nc2, delta).bytes > buf_bytes) break;
            r1 = step_end;
            nc += add;
        }
        if (r1 == r0) return pl;   // eight rows do not fit one buffer
        uint32_t at = cell;
        for (uint32_t r = r0; r < r1; ++r) { pl.cptr[r] = at; at += counts[r]; }
        cell += align4u(nc);
        ck.r1 = r1;
        ck.c1 = cell;
        const uint32_t bytes = chunk_layout(r1 - r0, ck.c1 - ck.c0, delta).bytes;
        pl.max_chunk_bytes = std::max(pl.max_chunk_bytes, bytes);
        pl.total_bytes += bytes;
        pl.chunks.push_back(ck);
        r0 = r1;
    }
    pl.cptr[n_t] = cell;
    pl.cells = cell;
    if (pl.chunks.size() > (size_t)kChainMaxChunks) return pl;
    for (ChainChunk& ck : pl.chunks) {
        ck.ptr_at = (uint32_t)pl.rel16.size();
        for (uint32_t r = ck.r0; r < ck.r1; ++r) pl.rel16.push_back((uint16_t)(pl.cptr[r] - ck.c0));
        pl.rel16.push_back((uint16_t)(ck.c1 - ck.c0));
        while (pl.rel16.size() % 8u) pl.rel16.push_back(0);
        ck.seg0 = (uint32_t)pl.segs.size();
        for (size_t j = 0; j + 1 < lvl.size(); ++j) {
            const uint32_t a = lvl[j], b = lvl[j + 1];
            if (b <= a) continue;
            const uint32_t s0 = std::max(a, ck.r0), s1 = std::min(b, ck.r1);
            if (s0 >= s1) continue;
            const uint32_t cells_seg = (s1 == ck.r1 ? ck.c1 : pl.cptr[s1]) - pl.cptr[s0];
            const uint32_t avg = (cells_seg + (s1 - s0) - 1u) / (s1 - s0);
            uint32_t L = std::min<uint32_t>(32u, pow2_ceil(std::max(1u, avg)));
            L = std::min(L, pow2_floor(std::max(1u, std::min(threads, level_threads()) / (b - a))));
            uint32_t logL = 0;
            while ((1u << logL) < L) ++logL;
            ChainSeg sg{};
            sg.r0 = s0; sg.r1 = s1;
            sg.info = logL | (b <= ck.r1 ? 0x100u : 0u) | ((s1 - s0) > (threads >> logL) ? 0x200u : 0u);
            pl.segs.push_back(sg);
        }
        ck.seg1 = (uint32_t)pl.segs.size();
    }
    while (pl.rel16.size() % 8u) pl.rel16.push_back(0);
    if (pl.segs.size() > (size_t)kChainMaxSegs) return pl;
    pl.ok = true;
    return pl;
}

// Upper bound of what the chain arrays take in the workspace (either use).
size_t chain_ws_bound(int64_t n, int64_t nnz, int64_t tiles) {
    const uint64_t nt = (uint64_t)std::min<int64_t>(n, (int64_t)kChainMaxLocal);
    const uint64_t cells = (uint64_t)nnz / 4 + nt + 4ull * kChainMaxChunks + 8;
    const uint64_t tl = (uint64_t)std::min<int64_t>(tiles, kMaxPersistReplicas / kTile);
    size_t b = 0;
    auto add = [&](size_t x) { b = align_up(b) + x; };
    add(4 * (nt + 2));                                   // counts / cell pointers
    add(2 * (nt + 1 + 8ull * (kChainMaxChunks + 1)));    // rel16
    add(4 * (nt + 16));                                  // orig
    add(8 * cells);
    add(4 * cells);
    add(sizeof(ChainChunk) * kChainMaxChunks);
    add(sizeof(ChainSeg) * kChainMaxSegs);
    add(tl * kChainGroups * ((uint64_t)kTailRowsMax + 8) * 16);   // h0
    add(tl * kChainGroups * ((uint64_t)kTailRowsMax + 8) * 4);    // old
    return align_up(b) + kAlign;
}

ising_status check_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return ISING_ERR_UNSUPPORTED_DEVICE; }
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return ISING_ERR_UNSUPPORTED_DEVICE;
    }
    return major == 10 ? ISING_OK : ISING_ERR_UNSUPPORTED_DEVICE;
}

}  // namespace

extern "C" {

const char* ising_status_string(ising_status s) {
    switch (s) {
        case ISING_OK: return "ok";
        case ISING_ERR_NULL_ARG: return "null argument";
        case ISING_ERR_BAD_SHAPE: return "bad shape / out-of-range index / bad enum";
        case ISING_ERR_UNSORTED_OR_DUP: return "row columns not strictly ascending";
        case ISING_ERR_SELF_LOOP: return "self loop";
        case ISING_ERR_ASYMMETRIC: return "graph or weights not symmetric";
        case ISING_ERR_BAD_COLOURING: return "colouring out of range or not proper";
        case ISING_ERR_FIELD_OVERFLOW: return "max_i sum_j |w_ij| >= 2^31";
        case ISING_ERR_TOO_MANY_REPLICAS: return "too many replicas";
        case ISING_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
        case ISING_ERR_NO_COLOURING_FOR_GS: return "Gauss-Seidel mode needs a colouring";
        case ISING_ERR_UNSUPPORTED_DEVICE: return "no sm_100 (B200) device";
        case ISING_ERR_CUDA: return "CUDA error";
        case ISING_ERR_BAD_SPINS: return "spin value is neither +1 nor -1";
        case ISING_ERR_NO_STATE: return "no state yet";
        default: return "unknown status";
    }
}

ising_status ising_workspace_bytes(int32_t n, int64_t nnz, int32_t wtype, int32_t max_replicas,
                                   int32_t n_colours, size_t* bytes_out) {
    if (!bytes_out) return ISING_ERR_NULL_ARG;
    if (n <= 0 || nnz < 0 || n_colours < 0 || (wtype != ISING_W_INT8 && wtype != ISING_W_INT32))
        return ISING_ERR_BAD_SHAPE;
    if (max_replicas < 1 || max_replicas > 65536) return ISING_ERR_TOO_MANY_REPLICAS;
    const bool dense = kDenseEnabled && nnz == (int64_t)n * (n - 1) && n >= 2;
    *bytes_out = workspace_need(n, nnz, wtype, max_replicas, n_colours, wtype == ISING_W_INT32,
                                bound_slices(n, nnz, n_colours + 1), bound_hubs(n, nnz), bound_cells(n, nnz, n_colours + 1), true,
                                dense);
    return ISING_OK;
}

}  // extern "C"

namespace {
ising_status load_csr_impl(int32_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx,
                           const void* weights, int32_t wtype, const int32_t* colour, int32_t n_colours,
                           int32_t max_replicas, void* workspace, size_t workspace_bytes, int32_t flags,
                           void* stream, ising_problem** out) {
    if (!out || !row_ptr || !workspace || (nnz > 0 && (!col_idx || !weights))) return ISING_ERR_NULL_ARG;
    if (n <= 0 || nnz < 0 || n_colours < 0 || (wtype != ISING_W_INT8 && wtype != ISING_W_INT32))
        return ISING_ERR_BAD_SHAPE;
    if ((colour == nullptr) != (n_colours == 0)) return ISING_ERR_BAD_COLOURING;
    if (max_replicas < 1 || max_replicas > 65536) return ISING_ERR_TOO_MANY_REPLICAS;
    if (ising_status s = check_device()) return s;
    if ((reinterpret_cast<uintptr_t>(workspace) & (kAlign - 1)) != 0 || !is_device_ptr(workspace))
        return ISING_ERR_BAD_SHAPE;   // not 256-byte aligned device memory
    cudaStream_t st = (cudaStream_t)stream;
#ifdef ISING_TUNING_ENV
    const bool lt_on = getenv("ISING_LOAD_TIMING") != nullptr;
    auto lt_t0 = std::chrono::steady_clock::now();
    auto LT = [&](const char* what) {
        if (!lt_on) return;
        if (getenv("ISING_LOAD_TIMING_SYNC")) cudaStreamSynchronize(st);
        auto t = std::chrono::steady_clock::now();
        fprintf(stderr, "  [load] %-28s %8.3f ms\n", what, std::chrono::duration<double, std::milli>(t - lt_t0).count());
        lt_t0 = t;
    };
#else
    auto LT = [](const char*) {};
#endif

    Bump ws{(uint8_t*)workspace, workspace_bytes, 0, false};
    BuildReport* d_rep = (BuildReport*)ws.take(sizeof(BuildReport));
    if (ws.overflow) return ISING_ERR_WORKSPACE_TOO_SMALL;

    // ---- bring the raw CSR to the device (staged in the workspace when it is host memory): row_ptr and colour first,
    // the relabelling needs nothing else
    const bool rp_dev = is_device_ptr(row_ptr), ci_dev = nnz == 0 || is_device_ptr(col_idx);
    const bool w_dev = nnz == 0 || is_device_ptr(weights), co_dev = colour && is_device_ptr(colour);
    const long long* d_row_ptr = (const long long*)row_ptr;
    const int32_t* d_col = col_idx;
    const void* d_w = weights;
    const int32_t* d_colour = colour;
    if (!rp_dev) {
        void* b = ws.take(8 * (size_t)(n + 1));
        if (!b) return ISING_ERR_WORKSPACE_TOO_SMALL;
        CK(cudaMemcpyAsync(b, row_ptr, 8 * (size_t)(n + 1), cudaMemcpyHostToDevice, st));
        d_row_ptr = (const long long*)b;
    }
    if (colour && !co_dev) {
        void* b = ws.take(4 * (size_t)n);
        if (!b) return ISING_ERR_WORKSPACE_TOO_SMALL;
        CK(cudaMemcpyAsync(b, colour, 4 * (size_t)n, cudaMemcpyHostToDevice, st));
        d_colour = (const int32_t*)b;
    }
    CK(cudaMemsetAsync(d_rep, 0, sizeof(BuildReport), st));
    k_check_rowptr<<<(unsigned)((n + 1 + 255) / 256), 256, 0, st>>>(d_row_ptr, n, nnz, d_rep);

    // ---- relabelling on the device (builder.cuh), on a stream of its own: it overlaps the copies of col_idx / weights
    int32_t C = n_colours > 0 ? n_colours : 1;   // (+ 1 after the overlap split of class 0, below)
    struct Side {   // the side stream and its fork event
        cudaStream_t s = nullptr;
        cudaEvent_t e = nullptr;
        ~Side() { if (s) (void)cudaStreamSynchronize(s); if (e) cudaEventDestroy(e); if (s) cudaStreamDestroy(s); }   // (its work reads the workspace)
    } side;
    CK(cudaStreamCreateWithFlags(&side.s, cudaStreamNonBlocking));
    CK(cudaEventCreateWithFlags(&side.e, cudaEventDisableTiming));
    CK(cudaEventRecord(side.e, st));
    CK(cudaStreamWaitEvent(side.s, side.e, 0));
    auto bits_of = [](uint64_t x) { uint32_t b = 0; while (x) { ++b; x >>= 1; } return b; };
    RelabelKey rk{};
    rk.row_ptr = d_row_ptr; rk.colour = d_colour; rk.n = n; rk.n_colours = C;
    rk.dbits = std::max(1u, bits_of((uint64_t)(n - 1)));
    const uint32_t key_bits = rk.dbits + bits_of((uint64_t)(C - 1));
    const uint32_t passes = std::max(1u, (key_bits + 7u) / 8u);
    const uint32_t n_chunks = (uint32_t)(((int64_t)n + kRadixChunk - 1) / kRadixChunk);
    int32_t* d_perm = (int32_t*)ws.take(4 * (size_t)n);
    int32_t* d_inv = (int32_t*)ws.take(4 * (size_t)n);
    uint32_t* d_ids = (uint32_t*)ws.take(4 * (size_t)n);
    uint32_t* d_hist = (uint32_t*)ws.take(4 * 256 * (size_t)n_chunks);
    RelabelRuns* d_runs = (RelabelRuns*)ws.take(sizeof(RelabelRuns));
    uint32_t* d_run_rows = (uint32_t*)ws.take(12 * (size_t)n);
    if (ws.overflow) return ISING_ERR_WORKSPACE_TOO_SMALL;
    auto enqueue_relabel = [&](const RelabelKey& key, uint32_t n_passes, cudaStream_t s) -> ising_status {
        const unsigned cb = (n_chunks + 3u) / 4u;
        const uint32_t* src = nullptr;
        for (uint32_t ps = 0; ps < n_passes; ++ps) {   // (the last pass lands in d_perm)
            uint32_t* dst = ((n_passes - ps) & 1u) ? (uint32_t*)d_perm : d_ids;
            k_radix_hist<<<cb, 128, 0, s>>>(key, src, 8u * ps, n_chunks, d_hist);
            k_radix_scan<<<1, 1024, 0, s>>>(d_hist, 256u * n_chunks);
            k_radix_scatter<<<cb, 128, 0, s>>>(key, src, dst, 8u * ps, n_chunks, d_hist);
            src = dst;
        }
        CK(cudaMemsetAsync(d_runs, 0, sizeof(RelabelRuns), s));
        k_relabel_finish<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(key, (const uint32_t*)d_perm, d_inv, d_runs, d_run_rows,
                                                                    (uint32_t)n);
        return ISING_OK;
    };
    if (ising_status s = enqueue_relabel(rk, passes, side.s)) return s;
    // (meanwhile, on the caller's stream: the edges)
    if (!ci_dev) {
        void* b = ws.take(4 * (size_t)nnz);
        if (!b) return ISING_ERR_WORKSPACE_TOO_SMALL;
        CK(cudaMemcpyAsync(b, col_idx, 4 * (size_t)nnz, cudaMemcpyHostToDevice, st));
        d_col = (const int32_t*)b;
    }
    if (!w_dev) {
        void* b = ws.take((size_t)wtype * (size_t)nnz);
        if (!b) return ISING_ERR_WORKSPACE_TOO_SMALL;
        CK(cudaMemcpyAsync(b, weights, (size_t)wtype * (size_t)nnz, cudaMemcpyHostToDevice, st));
        d_w = b;
    }
    LT("copies + relabel enqueued");
    // the one small read-back of the planning: row_ptr verdict + the runs of equal (colour, degree)
    BuildReport rep{};
    RelabelRuns runs_hdr{};
    const size_t runs_first = std::min<size_t>((size_t)n, 32768);
    std::vector<uint32_t> run_rows(3 * runs_first);
    auto fetch_runs = [&](cudaStream_t s) -> ising_status {
        CK(cudaMemcpyAsync(&rep, d_rep, sizeof(rep), cudaMemcpyDeviceToHost, s));
        CK(cudaMemcpyAsync(&runs_hdr, d_runs, sizeof(runs_hdr), cudaMemcpyDeviceToHost, s));
        CK(cudaMemcpyAsync(run_rows.data(), d_run_rows, 12 * runs_first, cudaMemcpyDeviceToHost, s));
        CK(cudaStreamSynchronize(s));
        CK(cudaGetLastError());
        if (runs_hdr.count > runs_first) {
            run_rows.resize(3 * (size_t)runs_hdr.count);
            CK(cudaMemcpy(run_rows.data(), d_run_rows, 12 * (size_t)runs_hdr.count, cudaMemcpyDeviceToHost));
        }
        return ISING_OK;
    };
    if (ising_status s = fetch_runs(side.s)) return s;
    if (rep.err_mask) { (void)cudaStreamSynchronize(st); return ISING_ERR_BAD_SHAPE; }   // (the copies read the caller's arrays)
    LT("relabel done (runs on host)");
    // ---- validate on the device (row_ptr is sound from here on); the report is read before anything is packed.
    // (Launched below, behind the overlap split and its relabelling: the host waits for those, not for the validation.)
    auto enqueue_validate = [&]() {
        const long long warps = n;
        const unsigned blocks = (unsigned)((warps * 32 + 255) / 256);
        k_validate<<<blocks, 256, 0, st>>>(n, d_row_ptr, d_col, d_w, wtype, d_colour, n_colours, d_rep);
    };
    auto read_report = [&]() -> ising_status {
        CK(cudaMemcpyAsync(&rep, d_rep, sizeof(rep), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        CK(cudaGetLastError());
        if (rep.kinds != 0) rep.err_mask |= 1u << ISING_ERR_ASYMMETRIC;   // (k_validate: an entry without a mirror in a longer row)
        for (int code : {ISING_ERR_BAD_SHAPE, ISING_ERR_UNSORTED_OR_DUP, ISING_ERR_SELF_LOOP, ISING_ERR_ASYMMETRIC,
                         ISING_ERR_BAD_COLOURING, ISING_ERR_FIELD_OVERFLOW})
            if (rep.err_mask & (1u << code)) return code;
        return ISING_OK;
    };

    // ---- O(slices) planning on the host, from the runs: internal rows [run_start[q], run_start[q + 1]) have degree
    // run_deg[q]; a run never crosses a colour boundary
    size_t n_runs = 0;
    std::vector<int64_t> run_start, run_deg;
    std::vector<int64_t> cstart;                         // internal rows of colour c: [cstart[c], cstart[c+1])
    auto sort_runs = [&]() {
        n_runs = runs_hdr.count;
        run_start.assign(n_runs + 1, 0);
        run_deg.assign(n_runs + 1, 0);
        cstart.assign((size_t)C + 1, 0);
        std::vector<uint64_t> order(n_runs);             // (first row << 32 | run index), sorted by first row
        for (size_t q = 0; q < n_runs; ++q) order[q] = ((uint64_t)run_rows[3 * q] << 32) | q;
        std::sort(order.begin(), order.end());
        for (size_t q = 0; q < n_runs; ++q) {
            const size_t r = (size_t)(order[q] & 0xffffffffu);
            const int64_t k0 = run_rows[3 * r], k1 = q + 1 < n_runs ? (int64_t)(order[q + 1] >> 32) : (int64_t)n;
            const uint32_t c = std::min<uint32_t>(run_rows[3 * r + 1], (uint32_t)C - 1u);
            run_start[q] = k0;
            run_deg[q] = run_rows[3 * r + 2];
            cstart[(size_t)c + 1] += k1 - k0;
        }
        run_start[n_runs] = n;
        for (size_t k = 1; k < cstart.size(); ++k) cstart[k] += cstart[k - 1];
    };
    sort_runs();
    LT("runs sorted");
    // Tail chain (chain.cuh, DELTA): the last colour classes of a big graph hold few, hub-like rows and cost a grid
    // barrier plus a dependent unit each (config 5: 14 of 22 phases, 8 % of the edges, 29 % of the sweep).  If the
    // classes c_tail .. C-1 hold at most kTailRows rows in all, the persistent kernel computes their fields in ONE
    // bulk pseudo-phase and walks the classes inside one CTA per four replicas.  Graphs small enough for
    // k_anneal_small are wholly a chain and need no tail.
    auto tail_start = [&]() {
        int32_t ct = C;
        if (colour && C >= 3 && !(flags & ISING_LOAD_NO_TAIL_CHAIN)) {
            const int64_t tail_rows = tail_rows_limit();
            int32_t c = C;
            while (c > 1 && (int64_t)n - cstart[(size_t)c - 1] <= tail_rows) --c;
            if (C - c >= 2) ct = c;
        }
        return ct;
    };
    int32_t c_tail = tail_start();
    // Chain overlap: while the chain (8 CTAs per tile) finishes sweep t, the other CTAs already update, for sweep
    // t + 1, the rows of colour class 0 that have no neighbour among the chain's rows (builder.cuh k_split_class0: they
    // become a colour class of their own in front of the rest of class 0; same Gauss-Seidel result).  Needs the edges on
    // the device, so the relabelling is repeated on the caller's stream behind the copies.
    bool split0 = false;
    if (c_tail < C && (int64_t)n > (int64_t)kChainMaxLocal && !(flags & ISING_LOAD_NO_OVERLAP)) {
        int32_t* d_colour2 = (int32_t*)ws.take(4 * (size_t)n);
        if (ws.overflow) { (void)cudaStreamSynchronize(st); return ISING_ERR_WORKSPACE_TOO_SMALL; }
        k_split_class0<<<(unsigned)(((long long)n * 32 + 255) / 256), 256, 0, st>>>(n, d_row_ptr, d_col, d_colour, C, c_tail, d_colour2);
        C += 1;
        RelabelKey rk2 = rk;
        rk2.colour = d_colour2; rk2.n_colours = C;
        const uint32_t passes2 = std::max(1u, (rk.dbits + bits_of((uint64_t)(C - 1)) + 7u) / 8u);
        if (ising_status s = enqueue_relabel(rk2, passes2, st)) { (void)cudaStreamSynchronize(st); return s; }
        if (ising_status s = fetch_runs(st)) { (void)cudaStreamSynchronize(st); return s; }
        sort_runs();
        c_tail = tail_start();
        split0 = true;
        LT("overlap split + second relabel");
    }
    enqueue_validate();
    // ---- work units: hubs (rows above kHubDegree, one CTA each) and slices (one warp each)
    int sm_count = 148, coop = 0;
    {
        int dev = 0;
        CK(cudaGetDevice(&dev));
        CK(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));
        CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    }
    std::vector<SliceDesc> slices;
    std::vector<uint32_t> slice_aux;                            // per slice: (hub id, part index) of hub-part slices
    slices.reserve((size_t)n / 3 + 1024);
    slice_aux.reserve(2 * ((size_t)n / 3 + 1024));
    std::vector<uint32_t> slice_begin((size_t)C + 1, 0);
    uint64_t tail_cells = 0;
    uint32_t n_hub_rows = 0;
    bool too_many_parts = false;
    // Edges per sub-row before a row is split over more sub-rows: 16 keeps the instruction count per edge low
    // (throughput-bound colour phases); 8 keeps every row inside the prefetched head cells, i.e. one gather round
    // trip per phase (latency-bound phases: fewer units than HALF the warps on the GPU; measured on config 5 in ms
    // per 500 sweeps: threshold 2x the warps 112.9, 1x 110.8, 1/2 109.6, 1/3 109.6, 1/4 109.9).  Chosen per colour phase.
    // A row of more than 16 sub-rows x sub_row_edges edges (a hub) is cut into P balanced PARTS of <= 128 edges, one slice each,
    // whose partial fields meet in hub_acc (integer atomics); the part that arrives last finishes the row.
    const uint64_t tiles_all = (uint64_t)((max_replicas + kTile - 1) / kTile);
    auto emit_colour = [&](int32_t c, int32_t k, int sub_row_edges) {   // rows k.. of colour c -> slices; returns the next row
        const int64_t part_cells_max = (int64_t)kSubRows * (sub_row_edges / 4);
        const int32_t k_end = (int32_t)cstart[(size_t)c + 1];
        size_t ri = (size_t)(std::upper_bound(run_start.begin(), run_start.end(), (int64_t)k) - run_start.begin()) - 1;   // run of row k
        int64_t same_l_end = k;   // rows [k, same_l_end) share this row's sub-row split
        while (k < k_end) {
            while (run_start[ri + 1] <= k) ++ri;
            const int64_t deg = run_deg[ri];
            const int64_t groups = (deg + 3) / 4;
            if (groups > part_cells_max) {
                // parts of at most 128 edges in every phase: a part lives in the prefetched head cells alone (measured
                // on config 5: 256-edge parts in the 16-edge phases 109.6 ms, 128-edge parts 108.9 ms; cutting the rows
                // of 129-256 edges into two parts as well: 113.4 ms)
                const int64_t part_size = kSubRows * kHeadGroups;
                const int64_t P = (groups + part_size - 1) / part_size;
                const int64_t cpp = (groups + P - 1) / P;
                if (P > 0x7fff) too_many_parts = true;   // packed arrival count / biased sum of part_finish
                for (int64_t q = 0; q < P; ++q) {
                    SliceDesc d;
                    d.off = 0;
                    d.row0 = (uint32_t)k;
                    d.G = (uint32_t)((cpp + kSubRows - 1) / kSubRows);
                    d.meta = 4u | (1u << 8) | ((uint32_t)P << 16);
                    slices.push_back(d);
                    slice_aux.push_back(n_hub_rows);
                    slice_aux.push_back((uint32_t)q);
                }
                ++n_hub_rows;
                ++k;
                continue;
            }
            const int l = spr_log2_for_degree(deg, sub_row_edges);
            const int rps = kSubRows >> l;
            if (same_l_end <= k) {   // (degrees descend inside a colour: the rows of one split are a stretch of runs)
                size_t rj = ri + 1;
                while (run_start[rj] < k_end && spr_log2_for_degree(run_deg[rj], sub_row_edges) == l) ++rj;
                same_l_end = std::min<int64_t>(run_start[rj], k_end);
            }
            const int nr = (int)std::min<int64_t>(rps, same_l_end - k);
            const int64_t G = std::max<int64_t>(1, (groups + (1ll << l) - 1) >> l);
            SliceDesc d;
            d.off = 0;
            d.row0 = (uint32_t)k;
            d.G = (uint32_t)G;
            d.meta = (uint32_t)l | ((uint32_t)nr << 8);
            slices.push_back(d);
            slice_aux.push_back(0u);
            slice_aux.push_back(0u);
            k += nr;
        }
        return k;
    };
    {
        int32_t k = 0;
        for (int32_t c = 0; c < C; ++c) {
            slice_begin[c] = (uint32_t)slices.size();
            const size_t mark = slices.size();
            const uint32_t hub_mark = n_hub_rows;
            const int32_t k_end = emit_colour(c, k, kSubRowEdges);
            uint64_t sub8_units = (uint64_t)sm_count * kWarpsPerCta / 2;   // latency-bound phase: less than half a round of the grid's warps
#ifdef ISING_TUNING_ENV
            if (const char* e = getenv("ISING_SUB8_UNITS")) sub8_units = (uint64_t)atoll(e);
#endif
            if (c < c_tail &&   // (the tail classes are throughput work of the bulk pseudo-phase)
                (uint64_t)(slices.size() - mark) * tiles_all < sub8_units) {
                slices.resize(mark);
                slice_aux.resize(2 * mark);
                n_hub_rows = hub_mark;
                emit_colour(c, k, kHeadGroups * 4);
            }
            k = k_end;
        }
        slice_begin[C] = (uint32_t)slices.size();
        for (const SliceDesc& d : slices) tail_cells += (uint64_t)(d.G > (uint32_t)kHeadGroups ? d.G - kHeadGroups : 0u) * kSubRows;
    }
    LT("slices");
    if (too_many_parts) { (void)cudaStreamSynchronize(st); return ISING_ERR_BAD_SHAPE; }   // the copies read the caller's arrays
    const uint64_t head_cells = (uint64_t)slices.size() * kSubRows * kHeadGroups;
    const uint64_t cells = head_cells + tail_cells;
    if (cells > 0xffffffffull) { (void)cudaStreamSynchronize(st); return ISING_ERR_BAD_SHAPE; }
    {
        uint64_t at = head_cells;
        for (SliceDesc& d : slices) {
            d.off = (uint32_t)at;
            at += (uint64_t)(d.G > (uint32_t)kHeadGroups ? d.G - kHeadGroups : 0u) * kSubRows;
        }
    }

    // ---- static split of every colour phase over the CTAs of the grid (launch-per-phase kernels; the persistent
    // kernel deals the units out itself).  Cost unit: executed warp instructions (ncu source counters,
    // profiles/): a slice costs ~430 + 70 per group + 45 per butterfly level + 120 per dependent tail group.
    auto slice_cost = [](const SliceDesc& d) {
        const double G = (double)d.G, l = (double)(d.meta & 0xffu);
        return 430.0 + 70.0 * G + 45.0 * l + 120.0 * std::max(0.0, G - (double)kHeadGroups);
    };
    // Grid size: small graphs are latency-bound (one dependent gather chain per phase), so every (slice, tile)
    // unit of the largest phase gets its own CTA, up to one CTA per SM (measured on configs 1-3: spreading the
    // units beats the cheaper barrier of a smaller grid).
    uint32_t n_cta = 1;
    {
        const uint64_t tiles_max = (uint64_t)(max_replicas + kTile - 1) / kTile;
        uint64_t units = 1;
        for (int32_t c = 0; c < C; ++c)
            units = std::max<uint64_t>(units, (uint64_t)(slice_begin[c + 1] - slice_begin[c]) * tiles_max);
        n_cta = (uint32_t)std::min<uint64_t>(units, (uint64_t)std::min<int>(sm_count, (int)kMaxCtas));
    }
    uint32_t max_phase_slices = 0;
    for (int32_t c = 0; c < C; ++c) max_phase_slices = std::max(max_phase_slices, slice_begin[c + 1] - slice_begin[c]);
    std::vector<PhaseRange> ranges((size_t)C * n_cta);
    for (int32_t c = 0; c < C; ++c) {
        double total = 0;
        for (uint32_t q = slice_begin[c]; q < slice_begin[c + 1]; ++q) total += slice_cost(slices[q]);
        uint32_t pos = slice_begin[c];
        const uint32_t end = slice_begin[c + 1];
        double remaining = total;
        for (uint32_t b = 0; b < n_cta; ++b) {
            PhaseRange& r = ranges[(size_t)c * n_cta + b];
            const double target = remaining / (double)(n_cta - b);
            double mine = 0;
            r.s0 = pos;
            if (b + 1 == n_cta) {
                while (pos < end) mine += slice_cost(slices[pos++]);
            } else {
                while (pos < end) {
                    const double cs = slice_cost(slices[pos]);
                    if (mine + 0.5 * cs > target) break;
                    mine += cs;
                    ++pos;
                }
            }
            r.s1 = pos;
            remaining -= mine;
        }
    }

    LT("ranges");
    if (ising_status s = read_report()) return s;
    LT("wait for validation report");
    const bool wide = rep.max_abs_w > 127 || (uint64_t)rep.absw_max * 2ull >= (1ull << 31);
    const bool complete = n >= 2 && nnz == (int64_t)n * (n - 1);
    const bool want_dense = kDenseEnabled && complete && !(flags & ISING_LOAD_NO_DENSE) && rep.max_abs_w <= 127;

    ising_problem* p = new (std::nothrow) ising_problem();
    if (!p) return ISING_ERR_CUDA;
    p->n = n; p->nnz = nnz; p->n_colours = n_colours; p->max_replicas = max_replicas;
    p->tiles_max = (max_replicas + kTile - 1) / kTile;
    p->W = rep.w_sum / 2; p->absw_max = rep.absw_max; p->wide = wide;
    p->n_slices = (uint32_t)slices.size(); p->n_hubs = n_hub_rows; p->cells = cells;
    // latency-bound graphs whose biggest phase fits two rounds of one cluster's warps: cluster barrier instead of grid barrier
    p->cluster_ctas = (max_phase_slices <= 2u * kClusterCtas * kWarpsPerCta && !(flags & ISING_LOAD_NO_CLUSTER)) ? kClusterCtas : 0;   // (16-CTA clusters measured
    // slower on config 3: 108 vs 73 ms, the eight clusters do not all fit at once)
    p->n_phases = (uint32_t)C; p->n_cta = n_cta; p->sm_count = sm_count; p->cooperative = coop != 0;
    p->flush_rows = wide ? 0x7fffffffu
                         : (uint32_t)std::max<int64_t>(1, ((1ll << 31) - 1) / std::max<int64_t>(1, 2 * rep.absw_max));

    const size_t tiles = (size_t)p->tiles_max;
    p->perm = d_perm;
    p->inv = d_inv;
    p->slices = (SliceDesc*)ws.take(sizeof(SliceDesc) * (slices.size() + 1));
    p->sorig = (uint32_t*)ws.take(4 * kSubRows * (slices.size() + 1));
    p->slice_aux = (uint32_t*)ws.take(8 * (slices.size() + 1));
    p->hub_acc = (unsigned long long*)ws.take(8 * kTile * tiles * ((size_t)n_hub_rows + 1));
    p->hub_cnt = (unsigned int*)ws.take(4 * tiles * ((size_t)n_hub_rows + 1));
    p->ranges = (PhaseRange*)ws.take(sizeof(PhaseRange) * ranges.size());
    p->col4 = (int4*)ws.take(16 * ((size_t)cells + 1));
    p->w4 = (uint32_t*)ws.take(4 * ((size_t)cells + 1));
    if (wide) p->w4w = (int4*)ws.take(16 * ((size_t)cells + 1));
    p->state[0] = (uint8_t*)ws.take(tiles * (size_t)n * kTile);
    p->state[1] = (uint8_t*)ws.take(tiles * (size_t)n * kTile);
    p->best = (uint8_t*)ws.take(tiles * (size_t)n * kTile);
    p->io_stage = (int8_t*)ws.take((size_t)max_replicas * (size_t)n);
    for (int k = 0; k < 2; ++k) {
        p->sm.accum[k] = (long long*)ws.take(8 * tiles * kTile);
        p->sm.E[k] = (long long*)ws.take(8 * tiles * kTile);
        p->sm.bestcut[k] = (long long*)ws.take(8 * tiles * kTile);
    }
    p->sm.accum_eval = (long long*)ws.take(8 * tiles * kTile);
    p->sm.out_tmp = (long long*)ws.take(16 * tiles * kTile);
    p->sm.accum3 = (long long*)ws.take(8 * 3 * (size_t)kMaxPersistReplicas);
    p->sm.best_sweep = (int32_t*)ws.take(4 * tiles * kTile);
    p->sm.thr = (uint32_t*)ws.take(4 * (size_t)kThrCap);
    p->sm.barrier = (unsigned int*)ws.take(256);
    p->phase_slices = (uint32_t*)ws.take(4 * ((size_t)C + 1));
    p->sm.flag = (int*)ws.take(256);
    void* dense_mem = nullptr;
    size_t dense_bytes = 0;
    if (want_dense) {
        dense_bytes = dense_workspace_bytes(n, max_replicas);
        dense_mem = ws.take(dense_bytes);
    }
    if (ws.overflow) { delete p; return ISING_ERR_WORKSPACE_TOO_SMALL; }
    p->ws_used = ws.used;

    auto fail = [&](ising_status s) { delete p; return s; };
#define CKP(call) do { if ((call) != cudaSuccess) { (void)cudaGetLastError(); return fail(ISING_ERR_CUDA); } } while (0)
    CKP(cudaMemcpyAsync(p->ranges, ranges.data(), sizeof(PhaseRange) * ranges.size(), cudaMemcpyHostToDevice, st));
    CKP(cudaMemcpyAsync(p->phase_slices, slice_begin.data(), 4 * ((size_t)C + 1), cudaMemcpyHostToDevice, st));
    if (!slices.empty()) {
        CKP(cudaMemcpyAsync(p->slices, slices.data(), sizeof(SliceDesc) * slices.size(), cudaMemcpyHostToDevice, st));
        CKP(cudaMemcpyAsync(p->slice_aux, slice_aux.data(), 4 * slice_aux.size(), cudaMemcpyHostToDevice, st));
        const unsigned blocks = (unsigned)(((long long)slices.size() * 32 + 255) / 256);
        k_pack<<<blocks, 256, 0, st>>>(p->slices, p->slice_aux, (uint32_t)slices.size(), p->perm, p->inv, d_row_ptr,
                                       d_col, d_w, wtype, p->col4, p->w4, p->w4w, p->sorig);
    }
    CKP(cudaMemsetAsync(p->hub_acc, 0, 8 * kTile * tiles * ((size_t)n_hub_rows + 1), st));
    CKP(cudaMemsetAsync(p->hub_cnt, 0, 4 * tiles * ((size_t)n_hub_rows + 1), st));
    if (want_dense) {
        p->dense = dense_create(n, max_replicas, dense_mem, dense_bytes, d_row_ptr, d_col, d_w, wtype, st);
        if (!p->dense) return fail(ISING_ERR_CUDA);
    }

    LT("uploads + pack enqueued");
    // ---- chain engine (chain.cuh): the whole graph (k_anneal_small) or the tail classes of the persistent kernel
    p->vphase_slices = (uint32_t*)ws.take(4 * ((size_t)C + 2));
    if (ws.overflow) return fail(ISING_ERR_WORKSPACE_TOO_SMALL);
    const bool persistent_ok = colour && !wide && coop != 0;
    const bool try_small = colour && !wide && (int64_t)n <= (int64_t)kChainMaxLocal && !(flags & ISING_LOAD_NO_SMALL);
    const bool try_tail = persistent_ok && c_tail < C && p->cluster_ctas == 0 &&
                          n_cta >= (uint32_t)kChainGroups * (uint32_t)std::min<int>(p->tiles_max, kMaxPersistReplicas / kTile);
    for (int pass = 0; pass < 2; ++pass) {   // the whole graph as a chain if it fits one CTA, else the tail classes
        const bool delta = pass == 1;
        if (delta ? (p->chain_small || !try_tail) : !try_small) continue;
        const uint32_t row_lo = delta ? (uint32_t)cstart[(size_t)c_tail] : 0u;
        const uint32_t n_t = (uint32_t)n - row_lo, n_t_pad = (n_t + 7u) & ~7u;
        std::vector<uint32_t> lvl;
        for (int32_t c = delta ? c_tail : 0; c <= C; ++c) lvl.push_back((uint32_t)cstart[(size_t)c] - row_lo);
        uint32_t* d_cnt = (uint32_t*)ws.take(4 * ((size_t)n_t + 2));
        if (ws.overflow) return fail(ISING_ERR_WORKSPACE_TOO_SMALL);
        const unsigned cb = (unsigned)(((unsigned long long)n_t * 32 + 255) / 256);
        k_chain_build<false><<<cb, 256, 0, st>>>(n_t, row_lo, delta ? 1 : 0, p->perm, p->inv, d_row_ptr, d_col, d_w, wtype,
                                                 d_colour, nullptr, d_cnt, nullptr, nullptr, nullptr, 0u);
        std::vector<uint32_t> counts(n_t);
        CKP(cudaMemcpyAsync(counts.data(), d_cnt, 4 * (size_t)n_t, cudaMemcpyDeviceToHost, st));
        CKP(cudaStreamSynchronize(st));
        int smem_optin = 0;
        {
            int dev = 0;
            CKP(cudaGetDevice(&dev));
            CKP(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        }
        const bool premul = n_t_pad <= 16384u;   // 16-bit cells can hold id x 4 (the tail chain always: kTailRowsMax)
        ChainPlan pl;
        bool resident = false;
        uint32_t threads = kSweepThreads, buf_bytes = 0;
        // val[] + flip[] (k_anneal_small: two flip buffers)
        const uint32_t val_bytes = chain_align16(4u * n_t_pad) + chain_align16(n_t_pad) * (delta ? 1u : 2u);
        if (delta) {
            buf_bytes = val_bytes < kChainSmemBytes ? ((kChainSmemBytes - val_bytes) / 2u) & ~15u : 0u;
            if (buf_bytes >= 4096u) pl = plan_chain(counts, lvl, buf_bytes, true, threads);
        } else {
            // CTA size: enough threads to give every row of the widest level min(32, its cells) lanes
            uint64_t want = 128;
            for (size_t j = 0; j + 1 < lvl.size(); ++j) {
                const uint32_t rows = lvl[j + 1] - lvl[j];
                if (!rows) continue;
                uint64_t cells = 0;
                for (uint32_t r = lvl[j]; r < lvl[j + 1]; ++r) cells += counts[r];
                const uint32_t avg = (uint32_t)((cells + rows - 1) / rows);
                want = std::max<uint64_t>(want, (uint64_t)rows * std::min<uint32_t>(4u, pow2_ceil(std::max(1u, avg))));
            }
            threads = (uint32_t)std::min<uint64_t>((uint64_t)kSmallThreadsMax, pow2_ceil((uint32_t)std::min<uint64_t>(want, 4096)));
            threads = small_threads_override(std::max(threads, 256u));
            cudaFuncAttributes fa{};
            CKP(cudaFuncGetAttributes(&fa, k_anneal_small<true, false>));
            const int64_t cap = (int64_t)smem_optin - (int64_t)fa.sharedSizeBytes - (int64_t)val_bytes - 256;
            if (cap >= 8192) {
                pl = plan_chain(counts, lvl, (uint32_t)cap & ~15u, false, threads);
                resident = pl.ok && pl.chunks.size() == 1;
                buf_bytes = resident ? (pl.max_chunk_bytes + 15u) & ~15u : 0u;
                if (!resident) {
                    buf_bytes = ((uint32_t)(cap / 2)) & ~15u;
                    pl = plan_chain(counts, lvl, buf_bytes, false, threads);
                    if (pl.ok && pl.total_bytes > kSmallStreamBytesMax) pl.ok = false;
                    if (pl.ok) buf_bytes = (pl.max_chunk_bytes + 15u) & ~15u;
                }
            }
        }
        if (pl.ok) {
            uint32_t* d_cptr = d_cnt;   // (same buffer: n_t + 1 entries)
            uint16_t* d_rel = (uint16_t*)ws.take(2 * (pl.rel16.size() + 8));
            uint32_t* d_orig = (uint32_t*)ws.take(4 * ((size_t)n_t_pad + 16));
            uint2* d_cidx = (uint2*)ws.take(8 * ((size_t)pl.cells + 4));
            uint32_t* d_cw = (uint32_t*)ws.take(4 * ((size_t)pl.cells + 4));
            ChainChunk* d_chunks = (ChainChunk*)ws.take(sizeof(ChainChunk) * pl.chunks.size());
            ChainSeg* d_segs = (ChainSeg*)ws.take(sizeof(ChainSeg) * pl.segs.size());
            int* d_h0 = nullptr;
            uint32_t* d_old = nullptr;
            const size_t tl = (size_t)std::min<int>(p->tiles_max, kMaxPersistReplicas / kTile);
            if (delta) {
                d_h0 = (int*)ws.take(tl * kChainGroups * (size_t)n_t_pad * 16);
                d_old = (uint32_t*)ws.take(tl * kChainGroups * (size_t)n_t_pad * 4);
            }
            if (ws.overflow) return fail(ISING_ERR_WORKSPACE_TOO_SMALL);
            CKP(cudaMemcpyAsync(d_cptr, pl.cptr.data(), 4 * pl.cptr.size(), cudaMemcpyHostToDevice, st));
            CKP(cudaMemcpyAsync(d_rel, pl.rel16.data(), 2 * pl.rel16.size(), cudaMemcpyHostToDevice, st));
            CKP(cudaMemcpyAsync(d_chunks, pl.chunks.data(), sizeof(ChainChunk) * pl.chunks.size(), cudaMemcpyHostToDevice, st));
            CKP(cudaMemcpyAsync(d_segs, pl.segs.data(), sizeof(ChainSeg) * pl.segs.size(), cudaMemcpyHostToDevice, st));
            CKP(cudaMemsetAsync(d_orig, 0, 4 * ((size_t)n_t_pad + 16), st));
            if (delta) CKP(cudaMemsetAsync(d_h0, 0, tl * kChainGroups * (size_t)n_t_pad * 16, st));
            k_chain_build<true><<<cb, 256, 0, st>>>(n_t, row_lo, delta ? 1 : 0, p->perm, p->inv, d_row_ptr, d_col, d_w, wtype,
                                                    d_colour, d_cptr, nullptr, reinterpret_cast<uint16_t*>(d_cidx),
                                                    reinterpret_cast<int8_t*>(d_cw), d_orig, premul ? 2u : 0u);
            ChainView& v = p->chain;
            v.chunks = d_chunks; v.segs = d_segs; v.rel16 = d_rel; v.orig = d_orig; v.cidx = d_cidx; v.cw = d_cw;
            v.h0 = d_h0; v.old = d_old;
            v.n_chunks = (uint32_t)pl.chunks.size(); v.n_segs = (uint32_t)pl.segs.size();
            v.n_t = n_t; v.n_t_pad = n_t_pad; v.row_lo = row_lo; v.resident = resident ? 1u : 0u;
            v.buf_bytes = buf_bytes; v.threads = threads; v.premul = premul ? 1u : 0u;
            v.narrow = (uint64_t)n_t * 2ull * (uint64_t)rep.absw_max < (1ull << 31) ? 1u : 0u;
            if (delta) {
                p->chain_delta = true;
                p->overlap0 = split0;
                p->ov_rows = split0 ? (uint32_t)cstart[1] : 0u;
            } else {
                p->chain_small = true;
                p->small_threads = threads;
                p->small_dyn = (size_t)val_bytes + (size_t)buf_bytes * (resident ? 1u : 2u);
                // a resident chain may run on clusters of two CTAs per word (levels + flip producer) when an anneal call
                // leaves enough SMs free: decided per call
                p->small_csplit = (resident && !(flags & ISING_LOAD_NO_CLUSTER)) ? 2u : 1u;
            }
            CKP(cudaStreamSynchronize(st));   // the plan's host vectors die here
        }
    }
    LT("chain plan + build");
    {
        // virtual phases of the persistent kernel: the colour phases, or (tail chain) the phases before the tail plus
        // ONE bulk pseudo-phase holding every slice of the tail classes
        std::vector<uint32_t> vps;
        const int32_t c_cut = p->chain_delta ? c_tail : C;
        for (int32_t c = 0; c <= c_cut; ++c) vps.push_back(slice_begin[(size_t)c]);
        if (p->chain_delta) vps.push_back(slice_begin[(size_t)C]);
        p->n_vphases = (uint32_t)vps.size() - 1u;
        CKP(cudaMemcpyAsync(p->vphase_slices, vps.data(), 4 * vps.size(), cudaMemcpyHostToDevice, st));
        CKP(cudaStreamSynchronize(st));
    }
    p->ws_used = ws.used;
    CKP(cudaFuncSetAttribute(k_anneal_gs<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kAnnealDynSmem));
    CKP(cudaFuncSetAttribute(k_anneal_gs<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kAnnealDynSmem));
    CKP(cudaFuncSetAttribute(k_anneal_gs<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kAnnealDynSmem));
    CKP(cudaStreamSynchronize(st));   // the host vectors die at return
    CKP(cudaGetLastError());
    LT("final sync");
#undef CKP
    *out = p;
    return ISING_OK;
}

}  // namespace

extern "C" {

ising_status ising_load_csr(int32_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx,
                            const void* weights, int32_t wtype, const int32_t* colour, int32_t n_colours,
                            int32_t max_replicas, void* workspace, size_t workspace_bytes, int32_t flags,
                            void* stream, ising_problem** out) {
    ising_status s;
    try {
        s = load_csr_impl(n, nnz, row_ptr, col_idx, weights, wtype, colour, n_colours, max_replicas, workspace,
                          workspace_bytes, flags, stream, out);
    } catch (...) {   // std::bad_alloc of the host-side planning: no exception crosses the C ABI
        s = ISING_ERR_CUDA;
    }
    // on error, copies enqueued from the caller's (possibly pinned) arrays have finished before the call returns:
    // the inputs may be freed on return either way
    if (s != ISING_OK) { (void)cudaStreamSynchronize((cudaStream_t)stream); (void)cudaGetLastError(); }
    return s;
}

ising_status ising_anneal(ising_problem* p, int32_t mode, int32_t tie_rule, int32_t n_replicas,
                          int32_t first_replica, uint64_t seed, const uint32_t* thresholds, int32_t n_sweeps,
                          int32_t sweep_offset, int32_t init_mode, const int8_t* init_spins, int64_t* cut_trace,
                          void* stream) {
    if (!p) return ISING_ERR_NULL_ARG;
    if (mode < 0 || mode > 3 || tie_rule < 0 || tie_rule > 1 || init_mode < 0 || init_mode > 2 || n_sweeps < 0 ||
        sweep_offset < 0 || first_replica < 0)
        return ISING_ERR_BAD_SHAPE;
    if (n_replicas < 1 || n_replicas > p->max_replicas) return ISING_ERR_TOO_MANY_REPLICAS;
    if (n_sweeps > 0 && !thresholds) return ISING_ERR_NULL_ARG;
    if (init_mode == ISING_INIT_GIVEN && !init_spins) return ISING_ERR_NULL_ARG;
    if ((mode == ISING_MODE_GS || mode == ISING_MODE_EXACT_N) && p->n_colours == 0) return ISING_ERR_NO_COLOURING_FOR_GS;
    if (mode == ISING_MODE_EXACT_N)
        for (int32_t t = 0; t < n_sweeps; ++t)
            if (thresholds[t] > (uint32_t)kMaxExactN) return ISING_ERR_BAD_SHAPE;
    if (init_mode == ISING_INIT_CONTINUE && (!p->have_state || p->last_R != n_replicas)) return ISING_ERR_NO_STATE;
    if (cut_trace && !is_device_ptr(cut_trace)) return ISING_ERR_BAD_SHAPE;
    cudaStream_t st = (cudaStream_t)stream;
    const int tiles = (n_replicas + kTile - 1) / kTile;
    const uint32_t n = (uint32_t)p->n;
    const unsigned long long tile_stride = (unsigned long long)n * kTile;
    const PhiloxKeys keys = philox_make_keys(seed);
    const bool use_dense = p->dense && mode == ISING_MODE_JACOBI;

    // ---- a2: initial state (into the sparse layout; the dense engine imports from it)
    if (p->state_in_dense && !(use_dense && init_mode == ISING_INIT_CONTINUE)) {
        // the state of the previous call lives in the dense layout: bring it back first
        if (init_mode == ISING_INIT_CONTINUE) {
            if (ising_status s = dense_export_state(p->dense, p->io_stage, n_replicas, /*best=*/false, st)) return s;
            CK(cudaMemsetAsync(p->sm.flag, 0, sizeof(int), st));
            k_import<<<dim3((unsigned)(((unsigned long long)n * kTile + 255) / 256), tiles), 256, 0, st>>>(
                p->state[p->cur], p->io_stage, p->perm, n, tile_stride, n_replicas, p->sm.flag);
            p->launches++;
        }
        p->state_in_dense = false;
    }
    if (init_mode == ISING_INIT_PHILOX) {
        p->cur = 0;
        k_init_philox<<<dim3((unsigned)((2ull * n + 255) / 256), tiles), 256, 0, st>>>(p->state[0], p->perm, n,
                                                                                     tile_stride, (uint32_t)first_replica, keys);
        p->launches++;
    } else if (init_mode == ISING_INIT_GIVEN) {
        const int8_t* d_in = init_spins;
        if (!is_device_ptr(init_spins)) {
            CK(cudaMemcpyAsync(p->io_stage, init_spins, (size_t)n_replicas * n, cudaMemcpyHostToDevice, st));
            d_in = p->io_stage;
        }
        p->cur = 0;
        CK(cudaMemsetAsync(p->sm.flag, 0, sizeof(int), st));
        k_import<<<dim3((unsigned)(((unsigned long long)n * kTile + 255) / 256), tiles), 256, 0, st>>>(
            p->state[0], d_in, p->perm, n, tile_stride, n_replicas, p->sm.flag);
        p->launches++;
        int bad = 0;
        CK(cudaMemcpyAsync(&bad, p->sm.flag, sizeof(int), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        if (bad) { p->have_state = false; return ISING_ERR_BAD_SPINS; }
    }
    p->have_state = true;
    p->last_R = n_replicas;
    p->have_best = false;
    if (n_sweeps == 0) { CK(cudaGetLastError()); return ISING_OK; }

    try {
        p->thr_host.assign(thresholds, thresholds + n_sweeps);
    } catch (...) {
        return ISING_ERR_CUDA;
    }
    const size_t small_bytes = 8 * (size_t)tiles * kTile;
    CK(cudaMemsetAsync(p->sm.accum[0], 0, small_bytes, st));
    CK(cudaMemsetAsync(p->sm.accum[1], 0, small_bytes, st));
    CK(cudaMemsetAsync(p->sm.bestcut[0], 0, small_bytes, st));
    CK(cudaMemsetAsync(p->sm.bestcut[1], 0, small_bytes, st));
    p->parity = 0;

    if (use_dense) {
        DenseAnnealArgs a{};
        a.tie_rule = tie_rule; a.n_replicas = n_replicas; a.first_replica = first_replica; a.keys = keys;
        a.thresholds = p->thr_host.data(); a.n_sweeps = n_sweeps; a.sweep_offset = sweep_offset; a.cut_trace = cut_trace;
        a.W = p->W;
        a.import_from_sparse = !(p->state_in_dense && init_mode == ISING_INIT_CONTINUE);
        a.sparse_state = p->state[p->cur]; a.perm = p->perm; a.io_stage = p->io_stage;
        a.thr_dev = p->sm.thr; a.thr_host = p->thr_host.data(); a.thr_cap = kThrCap;
        a.timing = p->timing; a.timing_pass = p->timing_sweep;
        ising_status s = dense_anneal(p->dense, a, st, &p->launches);
        if (s) return s;
        p->state_in_dense = true;
        p->have_best = true;
        CK(cudaGetLastError());
        return ISING_OK;
    }

    SweepParams sp = base_params(p);
    sp.rep0 = (uint32_t)first_replica;
    sp.tie_rule = tie_rule;
    sp.keys = keys;

    if (mode == ISING_MODE_GS && p->chain_small) {
        // small graph (chain.cuh, FULL): initial energy from the definition, then ONE launch of independent CTAs (one per
        // word of four replicas) per chunk of <= kThrCap sweeps; no grid-wide synchronisation at all
        CK(cudaMemsetAsync(p->sm.accum_eval, 0, small_bytes, st));
        SweepParams ev = sp;
        ev.src = p->state[p->cur]; ev.dst = p->state[p->cur]; ev.accum = p->sm.accum_eval;
        launch_sweep(p, kKindEval, ev, tiles, st);
        k_finish_energy<<<(unsigned)((tiles * kTile + 255) / 256), 256, 0, st>>>(p->sm.accum_eval, p->W, tiles * kTile,
                                                                              p->sm.E[0], nullptr);
        p->launches++;
        int dev_sms = 0;
        {
            int dev = 0;
            CK(cudaGetDevice(&dev));
            CK(cudaDeviceGetAttribute(&dev_sms, cudaDevAttrMultiProcessorCount, dev));
        }
        const uint32_t csplit = (p->small_csplit > 1u && 2 * (int64_t)tiles * kChainGroups <= (int64_t)dev_sms) ? 2u : 1u;
        const void* small_fn = small_kernel(p->timing != nullptr, p->chain.premul != 0u);
        CK(cudaFuncSetAttribute(small_fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->small_dyn));
        for (int32_t s0 = 0; s0 < n_sweeps; s0 += (int32_t)kThrCap) {
            const int32_t ns = std::min<int32_t>((int32_t)kThrCap, n_sweeps - s0);
            CK(cudaMemcpyAsync(p->sm.thr, p->thr_host.data() + s0, 4 * (size_t)ns, cudaMemcpyHostToDevice, st));
            SmallParams a{};
            a.v = p->chain;
            a.state = p->state[p->cur];
            a.best = p->best;
            a.best_compact = reinterpret_cast<uint32_t*>(p->state[p->cur ^ 1]);
            a.bc_stride = n;
            a.tile_stride = tile_stride;
            a.n_replicas = (uint32_t)n_replicas;
            a.rep0 = (uint32_t)first_replica;
            a.tie_rule = tie_rule;
            a.n_sweeps = (uint32_t)ns;
            a.sweep_offset = (uint32_t)(sweep_offset + s0);
            a.thr = p->sm.thr;
            a.W = p->W;
            a.E0 = p->sm.E[0];
            a.trace = cut_trace ? (long long*)cut_trace + (size_t)s0 * n_replicas : nullptr;
            a.trace_stride = (unsigned long long)n_replicas;
            a.E_out = p->sm.E[0];
            a.best_out = p->sm.bestcut[0];
            a.best_sweep_out = p->sm.best_sweep;
            a.resume = s0 > 0 ? 1 : 0;
            a.timing = s0 == 0 ? p->timing : nullptr;
            a.timing_sweep = p->timing_sweep;
            a.keys = keys;
            a.csplit = csplit;
            {
                cudaLaunchConfig_t cfg{};
                cfg.gridDim = dim3((unsigned)(tiles * kChainGroups) * csplit);
                cfg.blockDim = dim3(p->small_threads);
                cfg.dynamicSmemBytes = p->small_dyn;
                cfg.stream = st;
                cudaLaunchAttribute at[1];
                at[0].id = cudaLaunchAttributeClusterDimension;
                at[0].val.clusterDim.x = csplit; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
                cfg.attrs = at;
                cfg.numAttrs = csplit > 1u ? 1 : 0;
                void* args[1] = {&a};
                CK(cudaLaunchKernelExC(&cfg, small_fn, args));
            }
            p->launches++;
        }
        p->parity = 0;
    } else if (mode == ISING_MODE_GS && !p->wide && p->cooperative) {
        // the hot path: initial energy from the definition (evaluation pass), then ONE persistent
        // cooperative launch per batch of <= kMaxPersistReplicas (512) replicas and chunk of <= kThrCap sweeps
        CK(cudaMemsetAsync(p->sm.accum_eval, 0, small_bytes, st));
        SweepParams ev = sp;
        ev.src = p->state[p->cur]; ev.dst = p->state[p->cur]; ev.accum = p->sm.accum_eval;
        launch_sweep(p, kKindEval, ev, tiles, st);
        k_finish_energy<<<(unsigned)((tiles * kTile + 255) / 256), 256, 0, st>>>(p->sm.accum_eval, p->W, tiles * kTile,
                                                                              p->sm.E[0], nullptr);
        p->launches++;
        constexpr int kBatchTiles = kMaxPersistReplicas / kTile;
        for (int t0 = 0; t0 < tiles; t0 += kBatchTiles) {
            const int bt = std::min(kBatchTiles, tiles - t0);
            for (int32_t s0 = 0; s0 < n_sweeps; s0 += (int32_t)kThrCap) {
                const int32_t ns = std::min<int32_t>((int32_t)kThrCap, n_sweeps - s0);
                CK(cudaMemcpyAsync(p->sm.thr, p->thr_host.data() + s0, 4 * (size_t)ns, cudaMemcpyHostToDevice, st));
                CK(cudaMemsetAsync(p->sm.accum3, 0, 8 * 3 * (size_t)kMaxPersistReplicas, st));
                CK(cudaMemsetAsync(p->sm.barrier, 0, 256, st));
                AnnealParams a{};
                a.g = graph_view(p);
                a.state = p->state[p->cur] + (size_t)t0 * tile_stride;
                a.best = p->best + (size_t)t0 * tile_stride;
                a.tile_stride = tile_stride;
                a.n = n;
                a.tiles = (uint32_t)bt;
                a.n_replicas = (uint32_t)std::min(bt * kTile, n_replicas - t0 * kTile);
                a.rep0 = (uint32_t)first_replica + (uint32_t)t0 * kTile;
                a.tie_rule = tie_rule;
                a.flush_rows = p->flush_rows;
                a.n_sweeps = (uint32_t)ns;
                a.sweep_offset = (uint32_t)(sweep_offset + s0);
                a.thr = p->sm.thr;
                a.W = p->W;
                a.E0 = p->sm.E[0] + (size_t)t0 * kTile;
                a.accum = p->sm.accum3;
                a.trace = cut_trace ? (long long*)cut_trace + (size_t)s0 * n_replicas + (size_t)t0 * kTile : nullptr;
                a.trace_stride = (unsigned long long)n_replicas;
                a.E_out = p->sm.E[0] + (size_t)t0 * kTile;
                a.best_out = p->sm.bestcut[0] + (size_t)t0 * kTile;
                a.best_sweep_out = p->sm.best_sweep + (size_t)t0 * kTile;
                a.barrier = p->sm.barrier;
                a.vphase_slices = p->vphase_slices;
                a.n_vphases = p->n_vphases;
                a.chain_on = p->chain_delta ? 1u : 0u;
                a.chain = p->chain;
                const bool overlap = p->overlap0 && 2 * kChainGroups * bt <= (int)p->n_cta;   // (the phase runs on the CTAs that are not chain CTAs)
                a.ov_rows = p->ov_rows;
                a.alt = p->state[p->cur ^ 1] + (size_t)t0 * tile_stride;
                a.resume = s0 > 0 ? 1 : 0;
                a.timing = (t0 == 0 && s0 == 0) ? p->timing : nullptr;
                a.timing_sweep = p->timing_sweep;
                a.keys = keys;
                bool cluster = p->cluster_ctas > 0 && !p->timing;   // (the phase-timing diagnostics belong to the grid kernel)
                if (cluster) {
                    // small graph: one cluster of kClusterCtas CTAs per replica tile, hardware cluster barrier
                    cudaLaunchConfig_t cfg{};
                    cfg.gridDim = dim3((unsigned)(bt * p->cluster_ctas));
                    cfg.blockDim = dim3(kSweepThreads);
                    cfg.dynamicSmemBytes = kAnnealDynSmem;
                    cfg.stream = st;
                    cudaLaunchAttribute at[1];
                    at[0].id = cudaLaunchAttributeClusterDimension;
                    at[0].val.clusterDim.x = (unsigned)p->cluster_ctas; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
                    cfg.attrs = at;
                    cfg.numAttrs = 1;
                    CK(cudaLaunchKernelEx(&cfg, k_anneal_gs<true, false>, a));
                } else {
                    void* args[] = {&a};
                    CK(cudaLaunchCooperativeKernel(overlap ? (const void*)k_anneal_gs<false, true> : (const void*)k_anneal_gs<false, false>,
                                                   dim3(p->n_cta), dim3(kSweepThreads), args, kAnnealDynSmem, st));
                }
                p->launches++;
            }
        }
        p->parity = 0;
    } else if (mode == ISING_MODE_GS) {
        // wide (int32) weights: one launch per colour phase; incremental dE per phase
        SweepParams ev = sp;
        ev.src = p->state[p->cur]; ev.dst = p->state[p->cur]; ev.accum = p->sm.accum[p->parity];
        launch_sweep(p, kKindEval, ev, tiles, st);
        launch_sweep_end(p, p->state[p->cur], 2, 0, 0, nullptr, n_replicas, tiles, st);
        for (int32_t t = 0; t < n_sweeps; ++t) {
            SweepParams q = sp;
            q.src = p->state[p->cur]; q.dst = p->state[p->cur];
            q.accum = p->sm.accum[p->parity];
            q.thr = thresholds[t]; q.T = (uint32_t)(sweep_offset + t);
            for (int32_t c = 0; c < (int32_t)p->n_phases; ++c) {
                q.phase_begin = (uint32_t)c; q.phase_end = (uint32_t)c + 1;
                launch_sweep(p, kKindGS, q, tiles, st);
            }
            launch_sweep_end(p, p->state[p->cur], 0, t == 0, sweep_offset + t,
                             cut_trace ? (long long*)cut_trace + (size_t)t * n_replicas : nullptr, n_replicas, tiles, st);
        }
    } else if (mode == ISING_MODE_JACOBI) {
        // pass t reads s^t and yields 2E(s^t) as a by-product; pass n_sweeps is evaluation only
        for (int32_t t = 0; t <= n_sweeps; ++t) {
            SweepParams q = sp;
            q.src = p->state[p->cur]; q.dst = p->state[p->cur ^ 1];
            q.accum = p->sm.accum[p->parity];
            if (t < n_sweeps) {
                q.thr = thresholds[t]; q.T = (uint32_t)(sweep_offset + t);
                launch_sweep(p, kKindJacobi, q, tiles, st);
            } else {
                launch_sweep(p, kKindEval, q, tiles, st);
            }
            if (t == 0) launch_sweep_end(p, p->state[p->cur], 2, 0, 0, nullptr, n_replicas, tiles, st);
            else launch_sweep_end(p, p->state[p->cur], 1, t == 1, sweep_offset + t - 1,
                                  cut_trace ? (long long*)cut_trace + (size_t)(t - 1) * n_replicas : nullptr,
                                  n_replicas, tiles, st);
            if (t < n_sweeps) p->cur ^= 1;
        }
    } else if (mode == ISING_MODE_EXACT_N) {
        // Algorithm 1 (L77-99): a sweep of pure local minimisation (one launch per colour phase, no flips), then
        // exactly N_t distinct spins per replica are flipped, then an evaluation pass for the cut
        for (int32_t t = 0; t < n_sweeps; ++t) {
            SweepParams q = sp;
            q.src = p->state[p->cur]; q.dst = p->state[p->cur];
            q.accum = p->sm.accum_eval;   // increments of the minimisation sweep: not used, the cut is evaluated below
            q.thr = 0u; q.T = (uint32_t)(sweep_offset + t);
            for (int32_t c = 0; c < (int32_t)p->n_phases; ++c) {
                q.phase_begin = (uint32_t)c; q.phase_end = (uint32_t)c + 1;
                launch_sweep(p, kKindGS, q, tiles, st);
            }
            if (thresholds[t] > 0u) {
                k_flip_exact<<<(unsigned)n_replicas, 32, 0, st>>>(p->state[p->cur], p->inv, n, thresholds[t], q.T,
                                                                 (uint32_t)first_replica, tile_stride, keys);
                p->launches++;
            }
            SweepParams ev = sp;
            ev.src = p->state[p->cur]; ev.dst = p->state[p->cur]; ev.accum = p->sm.accum[p->parity];
            launch_sweep(p, kKindEval, ev, tiles, st);
            launch_sweep_end(p, p->state[p->cur], 1, t == 0, sweep_offset + t,
                             cut_trace ? (long long*)cut_trace + (size_t)t * n_replicas : nullptr, n_replicas, tiles, st);
        }
    } else {
        // paper-like racy in-place update of all spins (L158), then an evaluation pass for the cut
        for (int32_t t = 0; t < n_sweeps; ++t) {
            SweepParams q = sp;
            q.src = p->state[p->cur]; q.dst = p->state[p->cur];
            q.accum = p->sm.accum_eval;   // meaningless under races; discarded
            q.thr = thresholds[t]; q.T = (uint32_t)(sweep_offset + t);
            launch_sweep(p, kKindGS, q, tiles, st);
            SweepParams ev = sp;
            ev.src = p->state[p->cur]; ev.dst = p->state[p->cur]; ev.accum = p->sm.accum[p->parity];
            launch_sweep(p, kKindEval, ev, tiles, st);
            launch_sweep_end(p, p->state[p->cur], 1, t == 0, sweep_offset + t,
                             cut_trace ? (long long*)cut_trace + (size_t)t * n_replicas : nullptr, n_replicas, tiles, st);
        }
    }
    p->have_best = true;
    CK(cudaGetLastError());
    return ISING_OK;
}

ising_status ising_energy_cut(ising_problem* p, const int8_t* spins, int32_t n_replicas, int64_t* energy_out,
                              int64_t* cut_out, void* stream) {
    if (!p) return ISING_ERR_NULL_ARG;
    if (n_replicas < 1 || n_replicas > p->max_replicas) return ISING_ERR_TOO_MANY_REPLICAS;
    if (!spins && (!p->have_state || n_replicas != p->last_R)) return ISING_ERR_NO_STATE;
    cudaStream_t st = (cudaStream_t)stream;
    const int tiles = (n_replicas + kTile - 1) / kTile;
    const uint32_t n = (uint32_t)p->n;
    const unsigned long long tile_stride = (unsigned long long)n * kTile;
    const uint8_t* eval_state = nullptr;
    uint8_t* scratch = p->state[p->cur ^ 1];
    if (spins || p->state_in_dense) {
        const int8_t* d_in = spins;
        if (!spins) {
            if (ising_status s = dense_export_state(p->dense, p->io_stage, n_replicas, false, st)) return s;
            d_in = p->io_stage;
        } else if (!is_device_ptr(spins)) {
            CK(cudaMemcpyAsync(p->io_stage, spins, (size_t)n_replicas * n, cudaMemcpyHostToDevice, st));
            d_in = p->io_stage;
        }
        CK(cudaMemsetAsync(p->sm.flag, 0, sizeof(int), st));
        k_import<<<dim3((unsigned)(((unsigned long long)n * kTile + 255) / 256), tiles), 256, 0, st>>>(
            scratch, d_in, p->perm, n, tile_stride, n_replicas, p->sm.flag);
        p->launches++;
        int bad = 0;
        CK(cudaMemcpyAsync(&bad, p->sm.flag, sizeof(int), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        if (bad) return ISING_ERR_BAD_SPINS;
        eval_state = scratch;
    } else {
        eval_state = p->state[p->cur];
    }
    CK(cudaMemsetAsync(p->sm.accum_eval, 0, 8 * (size_t)tiles * kTile, st));
    SweepParams ev = base_params(p);
    ev.src = eval_state; ev.dst = const_cast<uint8_t*>(eval_state); ev.accum = p->sm.accum_eval;
    launch_sweep(p, kKindEval, ev, tiles, st);
    const bool e_host = energy_out && !is_device_ptr(energy_out);
    const bool c_host = cut_out && !is_device_ptr(cut_out);
    long long* d_e = energy_out ? (e_host ? p->sm.out_tmp : (long long*)energy_out) : nullptr;
    long long* d_c = cut_out ? (c_host ? p->sm.out_tmp + (size_t)tiles * kTile : (long long*)cut_out) : nullptr;
    k_finish_energy<<<(unsigned)((n_replicas + 255) / 256), 256, 0, st>>>(p->sm.accum_eval, p->W, n_replicas, d_e, d_c);
    p->launches++;
    if (e_host) CK(cudaMemcpyAsync(energy_out, d_e, 8 * (size_t)n_replicas, cudaMemcpyDeviceToHost, st));
    if (c_host) CK(cudaMemcpyAsync(cut_out, d_c, 8 * (size_t)n_replicas, cudaMemcpyDeviceToHost, st));
    if (e_host || c_host) CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    return ISING_OK;
}

ising_status ising_best_state(ising_problem* p, int32_t replica, int8_t* spins_out, int64_t* cut_out,
                              int32_t* sweep_out, int32_t* replica_out, void* stream) {
    if (!p) return ISING_ERR_NULL_ARG;
    if (!p->have_best) return ISING_ERR_NO_STATE;
    if (replica < -1 || replica >= p->last_R) return ISING_ERR_BAD_SHAPE;
    cudaStream_t st = (cudaStream_t)stream;
    const int R = p->last_R;
    std::vector<long long> bc;
    std::vector<int32_t> bs;
    try {
        bc.resize((size_t)R);
        bs.resize((size_t)R);
    } catch (...) {
        return ISING_ERR_CUDA;
    }
    if (p->state_in_dense) {
        if (ising_status s = dense_best_arrays(p->dense, bc.data(), bs.data(), R, st)) return s;
    } else {
        CK(cudaMemcpyAsync(bc.data(), p->sm.bestcut[p->parity], 8 * (size_t)R, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(bs.data(), p->sm.best_sweep, 4 * (size_t)R, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    int sel = replica;
    if (sel < 0) {
        sel = 0;
        for (int r = 1; r < R; ++r)
            if (bc[r] > bc[sel]) sel = r;
    }
    if (spins_out) {
        const bool host_out = !is_device_ptr(spins_out);
        int8_t* d_out = host_out ? p->io_stage : spins_out;
        if (p->state_in_dense) {
            if (ising_status s = dense_export_one(p->dense, d_out, sel, /*best=*/true, st)) return s;
        } else {
            k_export<<<(unsigned)((p->n + 255) / 256), 256, 0, st>>>(p->best, d_out, p->perm, (uint32_t)p->n,
                                                                    (unsigned long long)p->n * kTile, R, sel);
        }
        p->launches++;
        if (host_out) CK(cudaMemcpyAsync(spins_out, d_out, (size_t)p->n, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    if (cut_out) *cut_out = bc[sel];
    if (sweep_out) *sweep_out = bs[sel];
    if (replica_out) *replica_out = sel;
    CK(cudaGetLastError());
    return ISING_OK;
}

ising_status ising_current_state(ising_problem* p, int8_t* spins_out, int32_t n_replicas, void* stream) {
    if (!p || !spins_out) return ISING_ERR_NULL_ARG;
    if (!p->have_state || n_replicas != p->last_R) return ISING_ERR_NO_STATE;
    cudaStream_t st = (cudaStream_t)stream;
    const bool host_out = !is_device_ptr(spins_out);
    int8_t* d_out = host_out ? p->io_stage : spins_out;
    const int tiles = (n_replicas + kTile - 1) / kTile;
    if (p->state_in_dense) {
        if (ising_status s = dense_export_state(p->dense, d_out, n_replicas, false, st)) return s;
    } else {
        k_export<<<dim3((unsigned)(((unsigned long long)p->n * kTile + 255) / 256), tiles), 256, 0, st>>>(
            p->state[p->cur], d_out, p->perm, (uint32_t)p->n, (unsigned long long)p->n * kTile, n_replicas, -1);
    }
    p->launches++;
    if (host_out) {
        CK(cudaMemcpyAsync(spins_out, d_out, (size_t)n_replicas * p->n, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    CK(cudaGetLastError());
    return ISING_OK;
}

ising_status ising_problem_info(const ising_problem* p, int32_t what, int64_t* value_out) {
    if (!p || !value_out) return ISING_ERR_NULL_ARG;
    switch (what) {
        case 0: *value_out = p->n; break;
        case 1: *value_out = p->nnz; break;
        case 2: *value_out = p->n_colours; break;
        case 3: *value_out = p->max_replicas; break;
        case 4: *value_out = p->W; break;
        case 5: *value_out = p->dense ? 1 : 0; break;
        case 6: *value_out = p->launches; break;
        case 7: *value_out = p->absw_max; break;
        case 8: *value_out = (int64_t)p->ws_used; break;
        case 9: *value_out = p->n_slices; break;
        case 10: *value_out = (int64_t)p->cells * 4; break;
        case 11: *value_out = p->n_hubs; break;
        case 12: *value_out = p->n_cta; break;
        case 13: *value_out = p->chain_small ? 4 : !(p->n_colours > 0 && !p->wide && p->cooperative) ? 0
                                  : p->chain_delta ? 3 : p->cluster_ctas > 0 ? 2 : 1; break;
        case 14: *value_out = (p->chain_small || p->chain_delta) ? p->chain.n_t : 0; break;
        case 15: *value_out = p->n_vphases; break;
        case 16: *value_out = (p->chain_small || p->chain_delta) ? p->chain.n_chunks : 0; break;
        case 17: *value_out = (p->chain_small || p->chain_delta) ? p->chain.resident : 0; break;
        case 18: *value_out = p->chain_small ? p->small_csplit : 0; break;
        case 19: *value_out = p->overlap0 ? (int64_t)p->ov_rows : 0; break;
        default: return ISING_ERR_BAD_SHAPE;
    }
    return ISING_OK;
}

ising_status ising_debug_phase_timing(ising_problem* p, uint64_t* stamps, int32_t sweep) {
    if (!p) return ISING_ERR_NULL_ARG;
    if (sweep < 0 || (stamps && !is_device_ptr(stamps))) return ISING_ERR_BAD_SHAPE;
    p->timing = (unsigned long long*)stamps;
    p->timing_sweep = (uint32_t)sweep;
    return ISING_OK;
}

ising_status ising_debug_probe_l2(void* scratch, size_t bytes, double* gather_gbs, double* gather16_gbs, double* stream_gbs,
                                  void* stream) {
    if (!scratch || !gather_gbs || !gather16_gbs || !stream_gbs) return ISING_ERR_NULL_ARG;
    if (bytes < (1u << 20) || !is_device_ptr(scratch)) return ISING_ERR_BAD_SHAPE;
    if (ising_status s = check_device()) return s;
    cudaStream_t st = (cudaStream_t)stream;
    size_t use = 1u << 20;
    while (use * 2 <= bytes && use < ((size_t)1 << 31)) use *= 2;
    int sm = 148;
    {
        int dev = 0;
        CK(cudaGetDevice(&dev));
        CK(cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev));
    }
    uint32_t* sink = reinterpret_cast<uint32_t*>(scratch);   // (never written: the kernels' results cannot match the magic value)
    const uint32_t sectors_mask = (uint32_t)(use / 32) - 1u, per_pair = 2048, blocks = (unsigned)sm * 4, passes = 16;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    float ms_g = 0, ms_s = 0, ms_g4 = 0;
    for (int rep = 0; rep < 3; ++rep) {   // the last of three runs counts (the first brings the buffer into L2)
        CK(cudaEventRecord(e0, st));
        k_probe_gather<<<blocks, 512, 0, st>>>((const uint4*)scratch, sectors_mask, per_pair, sink);
        CK(cudaEventRecord(e1, st));
        CK(cudaEventSynchronize(e1));
        CK(cudaEventElapsedTime(&ms_g, e0, e1));
        float ms_4 = 0;
        CK(cudaEventRecord(e0, st));
        k_probe_gather4<<<blocks, 512, 0, st>>>((const uint32_t*)scratch, sectors_mask, per_pair, sink);
        CK(cudaEventRecord(e1, st));
        CK(cudaEventSynchronize(e1));
        CK(cudaEventElapsedTime(&ms_4, e0, e1));
        ms_g4 = ms_4;
        CK(cudaEventRecord(e0, st));
        k_probe_stream<<<blocks, 512, 0, st>>>((const uint4*)scratch, (uint32_t)(use / 16), passes, sink);
        CK(cudaEventRecord(e1, st));
        CK(cudaEventSynchronize(e1));
        CK(cudaEventElapsedTime(&ms_s, e0, e1));
    }
    CK(cudaEventDestroy(e0));
    CK(cudaEventDestroy(e1));
    CK(cudaGetLastError());
    *gather16_gbs = (double)blocks * 256.0 * per_pair * 32.0 / (ms_g * 1e-3) / 1e9;   // 16-byte lanes: 256 pairs per CTA
    const double g4 = (double)blocks * 64.0 * per_pair * 32.0 / (ms_g4 * 1e-3) / 1e9;      // 4-byte lanes: 64 groups per CTA
    *gather_gbs = std::max(*gather16_gbs, g4);
    *stream_gbs = (double)use * passes / (ms_s * 1e-3) / 1e9;
    return ISING_OK;
}

// include/ising_noalloc.h: no handle, no workspace, no allocation; scratch = g_noalloc_scratch (noalloc.cuh, this
// translation unit), its device address taken with cudaGetSymbolAddress once per device.
ising_status ising_energy_cut_noalloc(int32_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx,
                                      const void* weights, int32_t wtype, const int8_t* spins, int32_t n_replicas,
                                      int64_t* energy_out, int64_t* cut_out, void* stream) {
    if (!row_ptr || !spins || (nnz > 0 && (!col_idx || !weights))) return ISING_ERR_NULL_ARG;
    if (n <= 0 || nnz < 0 || (wtype != ISING_W_INT8 && wtype != ISING_W_INT32)) return ISING_ERR_BAD_SHAPE;
    if (n_replicas < 1 || n_replicas > kNoAllocMaxReplicas) return ISING_ERR_TOO_MANY_REPLICAS;   // the scratch holds no more
    if (ising_status s = check_device()) return s;
    long long* scratch = noalloc_scratch_ptr();
    if (!scratch) return ISING_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)stream;
    k_noalloc_clear<<<(unsigned)((n_replicas + 255) / 256), 256, 0, st>>>(scratch, n_replicas);
    const unsigned row_blocks = (unsigned)std::min<long long>(((long long)n + 7) / 8, 2048);
    k_noalloc_accumulate<<<dim3(row_blocks, (unsigned)n_replicas), 256, 0, st>>>(
        n, reinterpret_cast<const long long*>(row_ptr), col_idx, weights, wtype, spins, scratch);
    k_noalloc_finish<<<(unsigned)((n_replicas + 255) / 256), 256, 0, st>>>(
        scratch, n_replicas, reinterpret_cast<long long*>(energy_out), reinterpret_cast<long long*>(cut_out));
    CK(cudaGetLastError());
    return ISING_OK;
}

ising_status ising_free(ising_problem* p) {
    if (p) {
        if (p->dense) dense_destroy(p->dense);
        delete p;
    }
    return ISING_OK;
}

}  // extern "C"
