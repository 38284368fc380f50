// Device CSR builder: validation of the caller's graph and packing into
// the sliced, relabelled, replica-tile-friendly layout of common.cuh.  The paper leaves the
// storage of its "generally connected" model unstated (Fig. 2 L61) and only
// says the graph is copied to the device once (L138); everything here is this library's.
#pragma once
#include "common.cuh"

namespace ising {

struct BuildReport {
    unsigned int err_mask;     // bit k set = ISING_ERR_k seen
    int max_abs_w;             // max |w|
    long long w_sum;           // sum over directed entries (= 2 W)
    long long absw_max;        // max_i sum_j |w_ij|
    long long kinds;           // entries towards a shorter row minus entries towards a longer row (0 in a symmetric graph)
};

__device__ __forceinline__ long long load_w(const void* w, int wtype, long long e) {
    return wtype == 1 ? (long long)reinterpret_cast<const int8_t*>(w)[e]
                      : (long long)reinterpret_cast<const int32_t*>(w)[e];
}

// row_ptr[0] == 0, row_ptr[n] == nnz, monotone non-decreasing
__global__ void k_check_rowptr(const long long* row_ptr, int32_t n, long long nnz, BuildReport* rep) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    bool bad = false;
    const long long v = row_ptr[i];
    if (i == 0 && v != 0) bad = true;
    if (i == n && v != nnz) bad = true;
    if (v < 0 || v > nnz) bad = true;
    if (i < n && row_ptr[i + 1] < v) bad = true;
    if (bad) atomicOr(&rep->err_mask, 1u << 2);
}

// ---------------------------------------------------------------------------------------------
// Relabelling on the device: internal row order = colour ascending, then degree descending, then caller id ascending
// (the order the slices are cut from).  A stable LSD radix sort of the caller ids on the key
//     colour << dbits | (2^dbits - 1 - degree),        dbits = bits of n - 1 (>= any degree),
// eight bits a pass; the key is recomputed from row_ptr / colour in every pass (three gathers per row: nothing next to
// the edge traffic of the load), so only the ids move.  Garbage row_ptr / colour values are clamped: the sort never
// leaves its arrays, and the validation report rejects the graph afterwards.
// ---------------------------------------------------------------------------------------------
constexpr int kRadixChunk = 2048;   // rows per warp and pass

struct RelabelKey {
    const long long* row_ptr;
    const int32_t* colour;   // or nullptr
    int32_t n, n_colours;
    uint32_t dbits;
    __device__ __forceinline__ uint32_t degree(uint32_t v) const {
        const long long d = row_ptr[v + 1] - row_ptr[v];
        const long long cap = (1ll << dbits) - 1;
        return (uint32_t)(d < 0 ? 0 : (d > cap ? cap : d));
    }
    __device__ __forceinline__ uint32_t colour_of(uint32_t v) const {
        if (!colour) return 0u;
        const int32_t c = colour[v];
        return (uint32_t)(c < 0 ? 0 : (c >= n_colours ? n_colours - 1 : c));
    }
    __device__ __forceinline__ unsigned long long key(uint32_t v) const {
        return ((unsigned long long)colour_of(v) << dbits) | (unsigned long long)(((1u << dbits) - 1u) - degree(v));
    }
};

// ids == nullptr: the identity (first pass)
__global__ void k_radix_hist(RelabelKey rk, const uint32_t* ids, uint32_t shift, uint32_t n_chunks, uint32_t* hist) {
    __shared__ uint32_t s_cnt[4][256];
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    const uint32_t chunk = blockIdx.x * 4u + warp;
    for (uint32_t d = lane; d < 256u; d += 32u) s_cnt[warp][d] = 0u;
    __syncwarp();
    if (chunk < n_chunks) {
        const uint32_t lo = chunk * (uint32_t)kRadixChunk, hi = min((uint32_t)rk.n, lo + (uint32_t)kRadixChunk);
        for (uint32_t k = lo + lane; k < hi; k += 32u) {
            const uint32_t v = ids ? ids[k] : k;
            atomicAdd(&s_cnt[warp][(uint32_t)(rk.key(v) >> shift) & 255u], 1u);
        }
        __syncwarp();
        for (uint32_t d = lane; d < 256u; d += 32u) hist[(size_t)d * n_chunks + chunk] = s_cnt[warp][d];
    }
}
// exclusive scan of hist[256 * n_chunks] in place (digit-major), one CTA
__global__ void k_radix_scan(uint32_t* hist, uint32_t total) {
    __shared__ uint32_t s_part[1024];
    const uint32_t t = threadIdx.x, per = (total + 1023u) / 1024u;
    const uint32_t lo = min(total, t * per), hi = min(total, lo + per);
    uint32_t sum = 0;
    for (uint32_t k = lo; k < hi; ++k) sum += hist[k];
    s_part[t] = sum;
    __syncthreads();
    for (uint32_t o = 1; o < 1024u; o <<= 1) {
        const uint32_t x = t >= o ? s_part[t - o] : 0u;
        __syncthreads();
        s_part[t] += x;
        __syncthreads();
    }
    uint32_t run = s_part[t] - sum;
    for (uint32_t k = lo; k < hi; ++k) {
        const uint32_t c = hist[k];
        hist[k] = run;
        run += c;
    }
}
// stable scatter: a warp walks its chunk in order, 32 rows a step; rows of one digit keep their order (match_any)
__global__ void k_radix_scatter(RelabelKey rk, const uint32_t* ids, uint32_t* out, uint32_t shift, uint32_t n_chunks,
                                const uint32_t* offs) {
    __shared__ uint32_t s_off[4][256];
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    const uint32_t chunk = blockIdx.x * 4u + warp;
    if (chunk >= n_chunks) return;
    for (uint32_t d = lane; d < 256u; d += 32u) s_off[warp][d] = offs[(size_t)d * n_chunks + chunk];
    __syncwarp();
    const uint32_t lo = chunk * (uint32_t)kRadixChunk, hi = min((uint32_t)rk.n, lo + (uint32_t)kRadixChunk);
    for (uint32_t k0 = lo; k0 < hi; k0 += 32u) {
        const uint32_t k = k0 + lane;
        const bool act = k < hi;
        const uint32_t v = act ? (ids ? ids[k] : k) : 0u;
        const uint32_t d = act ? (uint32_t)(rk.key(v) >> shift) & 255u : 256u + lane;   // (idle lanes: a group of their own)
        const uint32_t m = __match_any_sync(0xffffffffu, d);
        const uint32_t rank = __popc(m & ((1u << lane) - 1u));
        if (act) out[s_off[warp][d] + rank] = v;
        __syncwarp();
        if (act && rank == 0u) s_off[warp][d] += __popc(m);
        __syncwarp();
    }
}
// perm -> inv, and the runs of equal (colour, degree) along the internal order: (first row, colour, degree), unordered
struct RelabelRuns {
    unsigned int count;
    unsigned int pad;
};
__global__ void k_relabel_finish(RelabelKey rk, const uint32_t* perm, int32_t* inv, RelabelRuns* runs, uint32_t* run_rows,
                                 uint32_t cap) {
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= (uint32_t)rk.n) return;
    const uint32_t v = perm[k];
    inv[v] = (int32_t)k;
    const unsigned long long key = rk.key(v);
    if (k == 0u || rk.key(perm[k - 1u]) != key) {
        const uint32_t at = atomicAdd(&runs->count, 1u);
        if (at < cap) {
            run_rows[3u * at] = k;
            run_rows[3u * at + 1u] = (uint32_t)(key >> rk.dbits);
            run_rows[3u * at + 2u] = ((1u << rk.dbits) - 1u) - (uint32_t)(key & ((1ull << rk.dbits) - 1ull));
        }
    }
}

// Overlap split (ising_api.cu, "chain overlap"): colour class 0 is cut into the rows WITHOUT a neighbour among the tail
// chain's classes (colour >= c_tail; new colour 0) and the rest (new colour 1); every other class moves up by one.  Both
// halves of class 0 are independent sets, so this is a valid colouring with the same Gauss-Seidel result (the order
// inside a class is irrelevant), and the first half can be updated for sweep t + 1 while the chain still finishes
// sweep t: none of its rows reads or is read by a chain row.  One warp per row; only class-0 rows look at their edges.
__global__ void k_split_class0(int32_t n, const long long* row_ptr, const int32_t* col, const int32_t* colour,
                               int32_t n_colours, int32_t c_tail, int32_t* colour2) {
    const long long gw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (gw >= n) return;
    const int32_t i = (int32_t)gw;
    const int32_t c = colour[i];
    if (c != 0) {
        if (lane == 0) colour2[i] = (c < 0 ? 0 : (c >= n_colours ? n_colours - 1 : c)) + 1;   // (garbage is rejected by k_validate)
        return;
    }
    bool adj = false;
    long long b = row_ptr[i], e = row_ptr[i + 1];
    if (b < 0 || e < b) { b = 0; e = 0; }
    for (long long k = b + lane; k < e && !adj; k += 32) {
        const int32_t j = col[k];
        if (j >= 0 && j < n) adj = colour[j] >= c_tail;
    }
    adj = __any_sync(0xffffffffu, adj);
    if (lane == 0) colour2[i] = adj ? 1 : 0;
}

// One warp per row: column range / order / self loops, symmetry, colouring, sum_j |w_ij|.
// Symmetry: entry (i, j) is looked up in row j (binary search) only when row j is not longer than row i; the entries
// whose row j is longer are counted instead.  Every looked-up entry of the first kind (deg j < deg i) names a distinct
// entry of the second kind as its mirror, so "all look-ups succeed and both kinds are equally many" means that every
// entry has its mirror with the same weight -- and the searches run in the SHORT rows (a power-law graph's edges
// mostly lead to hubs, whose rows cost 14-17 dependent probes each).
__global__ void k_validate(int32_t n, const long long* row_ptr, const int32_t* col, const void* w, int wtype,
                           const int32_t* colour, int32_t n_colours, BuildReport* rep) {
    __shared__ unsigned int s_err;
    __shared__ int s_maxabs;
    __shared__ long long s_absw, s_wsum, s_kinds;
    if (threadIdx.x == 0) { s_err = 0u; s_maxabs = 0; s_absw = 0; s_wsum = 0; s_kinds = 0; }
    __syncthreads();
    const long long gw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    unsigned int err = 0;
    long long absw = 0, wsum = 0, kinds = 0;   // kinds: entries towards a shorter row minus entries towards a longer one
    int maxabs = 0;
    if (gw < n) {
        const int32_t i = (int32_t)gw;
        const long long b = row_ptr[i], e = row_ptr[i + 1];
        int ci = 0;
        if (colour) {
            ci = colour[i];
            if (ci < 0 || ci >= n_colours) err |= 1u << 6;
        }
        for (long long idx = b + lane; idx < e; idx += 32) {
            const int32_t j = col[idx];
            if (j < 0 || j >= n) { err |= 1u << 2; continue; }
            if (j == i) err |= 1u << 4;
            if (idx > b && col[idx - 1] >= j) err |= 1u << 3;
            const long long wv = load_w(w, wtype, idx);
            long long lo = row_ptr[j];
            const long long end_j = row_ptr[j + 1];
            if (end_j - lo > e - b) {
                --kinds;
            } else {
                if (end_j - lo < e - b) ++kinds;
                long long hi = end_j;   // find i in row j
                while (lo < hi) {
                    const long long mid = (lo + hi) >> 1;
                    if (col[mid] < i) lo = mid + 1; else hi = mid;
                }
                if (lo >= end_j || col[lo] != i || load_w(w, wtype, lo) != wv) err |= 1u << 5;
            }
            if (colour && colour[j] == ci) err |= 1u << 6;
            const long long aw = wv < 0 ? -wv : wv;
            absw += aw;
            wsum += wv;
            if (aw > maxabs) maxabs = (int)(aw > 0x7fffffffll ? 0x7fffffffll : aw);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        absw += __shfl_xor_sync(0xffffffffu, absw, o);
        wsum += __shfl_xor_sync(0xffffffffu, wsum, o);
        kinds += __shfl_xor_sync(0xffffffffu, kinds, o);
        maxabs = max(maxabs, __shfl_xor_sync(0xffffffffu, maxabs, o));
        err |= __shfl_xor_sync(0xffffffffu, err, o);
    }
    if (lane == 0) {   // the rows of a block meet in shared memory: one set of global atomics per block
        if (absw >= (1ll << 31)) err |= 1u << 7;
        if (err) atomicOr(&s_err, err);
        atomicMax(&s_absw, absw);
        atomicMax(&s_maxabs, maxabs);
        if (wsum != 0) atomicAdd(reinterpret_cast<unsigned long long*>(&s_wsum), (unsigned long long)wsum);
        if (kinds != 0) atomicAdd(reinterpret_cast<unsigned long long*>(&s_kinds), (unsigned long long)kinds);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_err) atomicOr(&rep->err_mask, s_err);
        atomicMax(&rep->absw_max, s_absw);
        atomicMax(&rep->max_abs_w, s_maxabs);
        if (s_wsum != 0) atomicAdd(reinterpret_cast<unsigned long long*>(&rep->w_sum), (unsigned long long)s_wsum);
        if (s_kinds != 0) atomicAdd(reinterpret_cast<unsigned long long*>(&rep->kinds), (unsigned long long)s_kinds);
    }
}

// One warp per slice: fill the cells of the slice (head cells for groups 0 and 1, tail cells for
// the rest) and the per-sub-row caller ids (hub parts: caller id, hub id, part index).  Cell (g, sr) holds group q = g * SPR + part of row
// row0 + (sr >> log_spr), part = sr & (SPR - 1); edges 4q .. 4q+3.
__device__ __forceinline__ void store_cell(int4* col4, uint32_t* w4, int4* w4w, size_t at, const int (&cc)[4],
                                           const int (&ww)[4]) {
    col4[at] = make_int4(cc[0], cc[1], cc[2], cc[3]);
    if (w4w) w4w[at] = make_int4(ww[0], ww[1], ww[2], ww[3]);
    else w4[at] = ((uint32_t)ww[0] & 0xffu) | (((uint32_t)ww[1] & 0xffu) << 8) |
                  (((uint32_t)ww[2] & 0xffu) << 16) | (((uint32_t)ww[3] & 0xffu) << 24);
}

__device__ __forceinline__ void fetch_group(const int32_t* inv, const int32_t* col, const void* w, int wtype,
                                            long long b, long long deg, long long q, int pad, int (&cc)[4],
                                            int (&ww)[4]) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const long long e = 4 * q + j;
        cc[j] = pad;
        ww[j] = 0;
        if (e < deg) {
            cc[j] = inv[col[b + e]];
            ww[j] = (int)load_w(w, wtype, b + e);
        }
    }
}

__global__ void k_pack(const SliceDesc* slices, const uint32_t* slice_aux, uint32_t n_slices, const int32_t* perm,
                       const int32_t* inv, const long long* row_ptr, const int32_t* col, const void* w, int wtype,
                       int4* col4, uint32_t* w4, int4* w4w, uint32_t* sorig) {
    const long long gw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (gw >= n_slices) return;
    const SliceDesc d = slices[gw];
    const int log_spr = (int)(d.meta & 0xffu), nrows = (int)((d.meta >> 8) & 0xffu);
    const uint32_t parts = d.meta >> 16;
    const uint32_t spr = 1u << log_spr;
    if (parts != 0u) {
        // part `part` of a hub row: cells [part * cpp, min((part + 1) * cpp, groups)) of the row, cell l of the
        // part at (g, sr) = (l / 16, l % 16)
        const uint32_t hub = slice_aux[2 * gw], part = slice_aux[2 * gw + 1];
        const int32_t orig = perm[d.row0];
        const long long b = row_ptr[orig], deg = row_ptr[orig + 1] - b;
        const long long groups = (deg + 3) / 4, cpp = (groups + parts - 1) / parts;
        const long long first = (long long)part * cpp;
        const long long mine = groups - first < cpp ? groups - first : cpp;   // may be <= 0 for a trailing part
        if (lane < kSubRows)
            sorig[(size_t)gw * kSubRows + lane] = lane == 0 ? (uint32_t)orig : lane == 1 ? hub : lane == 2 ? part : 0xffffffffu;
        const uint32_t Gs = d.G > (uint32_t)kHeadGroups ? d.G : (uint32_t)kHeadGroups;
        for (uint32_t cell = lane; cell < Gs * kSubRows; cell += 32) {
            const uint32_t g = cell / kSubRows, sr = cell % kSubRows;
            int cc[4] = {(int)d.row0, (int)d.row0, (int)d.row0, (int)d.row0};
            int ww[4] = {0, 0, 0, 0};
            if ((long long)cell < mine) fetch_group(inv, col, w, wtype, b, deg, first + cell, (int)d.row0, cc, ww);
            const size_t at = g < kHeadGroups ? ((size_t)gw * kHeadGroups + g) * kSubRows + sr
                                              : (size_t)d.off + (size_t)(g - kHeadGroups) * kSubRows + sr;
            store_cell(col4, w4, w4w, at, cc, ww);
        }
        return;
    }
    if (lane < kSubRows) {
        const uint32_t rloc = (uint32_t)lane >> log_spr;
        sorig[(size_t)gw * kSubRows + lane] = (int)rloc < nrows ? (uint32_t)perm[d.row0 + rloc] : 0xffffffffu;
    }
    const unsigned long long cells = (unsigned long long)d.G * kSubRows;
    for (unsigned long long cell = lane; cell < cells; cell += 32) {
        const uint32_t g = (uint32_t)(cell / kSubRows), sr = (uint32_t)(cell % kSubRows);
        const uint32_t rloc = sr >> log_spr, part = sr & (spr - 1);
        const int pad = (int)((int)rloc < nrows ? d.row0 + rloc : d.row0);
        int cc[4] = {pad, pad, pad, pad};
        int ww[4] = {0, 0, 0, 0};
        if ((int)rloc < nrows) {
            const int32_t orig = perm[d.row0 + rloc];
            const long long b = row_ptr[orig], deg = row_ptr[orig + 1] - b;
            fetch_group(inv, col, w, wtype, b, deg, (long long)g * spr + part, pad, cc, ww);
        }
        const size_t at = g < kHeadGroups ? ((size_t)gw * kHeadGroups + g) * kSubRows + sr
                                          : (size_t)d.off + (size_t)(g - kHeadGroups) * kSubRows + sr;
        store_cell(col4, w4, w4w, at, cc, ww);
    }
    if (d.G < kHeadGroups && lane < kSubRows) {   // unused head cells: all padding
        const uint32_t rloc = (uint32_t)lane >> log_spr;
        const int pad = (int)((int)rloc < nrows ? d.row0 + rloc : d.row0);
        const int cc[4] = {pad, pad, pad, pad};
        const int ww[4] = {0, 0, 0, 0};
        for (uint32_t g = d.G; g < kHeadGroups; ++g)
            store_cell(col4, w4, w4w, ((size_t)gw * kHeadGroups + g) * kSubRows + lane, cc, ww);
    }
}

}  // namespace ising
