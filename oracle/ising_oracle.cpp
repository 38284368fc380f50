// ===========================================================================
// CPU ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct implementation of the annealing sweep of
// arXiv 1807.10750 ("GPU Ising Computing for Combinatorial Optimization
// Problems in VLSI Physical Design"), written from PAPER.md and the readings in
// SURVEY.md 8(c) / DESIGN.md.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may call it.  It shares NO
// code with the CUDA path (own Philox, own CSR walk, energy always from the
// definition, never the delta-E shortcut) and never imports it.
//
// What it follows, in the paper's order and notation:
//   * Algorithm 2: while F_p > 0: for all sigma_i:
//       sigma_i <- argmin H(sigma_i); flip sigma_i with probability F_p; reduce F_p.
//     Read as exactly M = len(thr) sweeps (Q7), F_p supplied per sweep as a uint32
//     threshold (Q6), flip applied immediately after the spin's own update (Q5).
//   * Algorithm 1 (L77-99) gives the sequential sweep used as the update ORDER:
//     vertices in (colour, id) order ("gs"), or all from the sweep-start state
//     ("jacobi") (Q8).
//   * eq. (2) (L45-49) local update: sigma_i from the sign of S; with the max-cut
//     mapping of eq. (4)/(5) (L119-128) read as minimising
//     E(s) = +sum_{i<j} w_ij s_i s_j (Q1), so h_i = sum_j w_ij s_j and the
//     energy-minimising value is a_i = +1 if h_i < 0 else -1; tie h_i = 0 -> -1
//     (MINUS, the literal "otherwise" branch of L49) or unchanged (KEEP) (Q3).
//   * eq. (4) (L119): cut = 1/2 sum_{i<j} w_ij (1 - x_i x_j) = (W - E)/2.
//   * RNG (Q11): Philox4x32-10, key = 64-bit seed, counter =
//     (spin id, absolute sweep, replica>>2, domain), word = replica & 3;
//     flip iff word < thr[t] (unsigned, strict).  DOMAIN_FLIP = 0, DOMAIN_INIT = 1.
//   * Algorithm 1's own flip step (L92), mode 2: after a sweep of pure minimisation flip
//     exactly N = thr[t] distinct spins (Floyd's subset sampling on Philox words, DOMAIN_FLIPN = 2).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors,
// brute force over all 2^n cuts (n <= 20), cut identity vs an independent
// "edges whose endpoints differ" count, zero-temperature monotonicity and 1-flip
// local optimum, torus and K_n closed forms, flip-rate statistics, order
// invariance inside a colour class, batch/sweep split invariance.
// The trajectory itself (which spins at which sweep) is "parity unpinned" by the
// paper (it prints no trace; its runs are racy, L247): the oracle DEFINES it.
//
// Build: g++ -O2 -std=c++17 -shared -fPIC -pthread -o liboracle.so ising_oracle.cpp
// ===========================================================================
#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <thread>
#include <vector>

namespace {

constexpr uint32_t DOMAIN_FLIP = 0;
constexpr uint32_t DOMAIN_INIT = 1;
constexpr uint32_t DOMAIN_FLIPN = 2;   // Algorithm 1's exact-N flip step: counter word 0 = draw index

// Philox4x32-10 (Salmon et al., "Parallel random numbers: as easy as 1, 2, 3").
// One round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0));
// key bumped by the Weyl constants between rounds.
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

uint32_t philox_word(uint64_t seed, uint32_t spin, uint32_t sweep, uint32_t replica, uint32_t domain) {
    uint32_t ctr[4] = {spin, sweep, replica >> 2, domain};
    uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
    uint32_t out[4];
    philox4x32_10(ctr, key, out);
    return out[replica & 3];
}

struct Graph {
    int32_t n;
    const int64_t* row_ptr;
    const int32_t* col;
    const int8_t* w8;    // exactly one of w8 / w32 is non-null
    const int32_t* w32;
    int64_t weight(int64_t e) const { return w8 ? (int64_t)w8[e] : (int64_t)w32[e]; }
};

// E(s) = sum_{i<j} w_ij s_i s_j  (eq. (3)/(5) with J = -w, Q1; each pair once, Q9)
int64_t energy(const Graph& g, const int8_t* s) {
    int64_t E = 0;
    for (int32_t i = 0; i < g.n; ++i)
        for (int64_t e = g.row_ptr[i]; e < g.row_ptr[i + 1]; ++e)
            if (g.col[e] > i) E += g.weight(e) * (int64_t)s[i] * (int64_t)s[g.col[e]];
    return E;
}

// W = sum_{i<j} w_ij
int64_t total_weight(const Graph& g) {
    int64_t W = 0;
    for (int32_t i = 0; i < g.n; ++i)
        for (int64_t e = g.row_ptr[i]; e < g.row_ptr[i + 1]; ++e)
            if (g.col[e] > i) W += g.weight(e);
    return W;
}

// h_i = sum_j w_ij s_j  (eq. (2), S = -h_i under Q1)
int64_t local_field(const Graph& g, const int8_t* s, int32_t i) {
    int64_t h = 0;
    for (int64_t e = g.row_ptr[i]; e < g.row_ptr[i + 1]; ++e) h += g.weight(e) * (int64_t)s[g.col[e]];
    return h;
}

struct AnnealArgs {
    Graph g;
    const int32_t* order;     // [n] visiting order for GS (vertices sorted by (colour, id)); unused in Jacobi
    int32_t mode;             // 0 GS (Algorithm 2), 1 Jacobi (Algorithm 2), 2 GS + exact-N flips (Algorithm 1)
    int32_t tie_rule;         // 0 MINUS, 1 KEEP
    int32_t n_replicas;
    int32_t first_replica;
    uint64_t seed;
    const uint32_t* thr;      // [n_sweeps]
    int32_t n_sweeps;
    int32_t sweep_offset;
    const int8_t* init_spins; // [R][n] or null -> Philox INIT
    int8_t* final_spins;      // [R][n] or null
    int64_t* trace;           // [n_sweeps][R] or null
    int64_t* best_cut;        // [R] or null
    int32_t* best_sweep;      // [R] or null
    int8_t* best_spins;       // [R][n] or null
    int64_t W;
};

int8_t update_value(int64_t h, int8_t old, int32_t tie_rule) {
    if (h < 0) return +1;
    if (h > 0) return -1;
    return tie_rule == 1 ? old : (int8_t)-1;
}

void anneal_replica(const AnnealArgs& a, int32_t r) {
    const Graph& g = a.g;
    const int32_t n = g.n;
    const uint32_t rep = (uint32_t)(a.first_replica + r);
    std::vector<int8_t> s(n), nxt(a.mode == 1 ? n : 0), best(n);
    for (int32_t i = 0; i < n; ++i) {
        if (a.init_spins) s[i] = a.init_spins[(size_t)r * n + i];
        else s[i] = (philox_word(a.seed, (uint32_t)i, 0u, rep, DOMAIN_INIT) & 1u) ? +1 : -1;
    }
    bool have_best = false;
    int64_t bc = 0;
    int32_t bs = -1;
    for (int32_t t = 0; t < a.n_sweeps; ++t) {
        const uint32_t T = (uint32_t)(a.sweep_offset + t);
        const uint32_t thr = a.thr[t];
        if (a.mode == 2) {
            // Algorithm 1 (L77-99): a sweep of pure local minimisation in the sequential order, then "randomly
            // choose and flip N spin glasses" (L92): N = thr[t] DISTINCT spins (clamped to n), drawn as a uniform
            // N-subset by Floyd's algorithm: for j = n-N .. n-1: x = uniform integer in [0, j]; take x unless it
            // was taken already, then take j.  The integer comes from one Philox word u (counter =
            // (draw index, sweep, replica>>2, DOMAIN_FLIPN), word replica&3) as floor(u (j+1) / 2^32).
            for (int32_t k = 0; k < n; ++k) {
                const int32_t i = a.order[k];
                s[i] = update_value(local_field(g, s.data(), i), s[i], a.tie_rule);
            }
            const int64_t N = std::min<int64_t>((int64_t)thr, (int64_t)n);
            std::vector<int32_t> chosen;
            for (int64_t j = (int64_t)n - N; j < (int64_t)n; ++j) {
                const uint32_t u = philox_word(a.seed, (uint32_t)(j - ((int64_t)n - N)), T, rep, DOMAIN_FLIPN);
                int32_t x = (int32_t)(((uint64_t)u * (uint64_t)(j + 1)) >> 32);
                bool taken = false;
                for (int32_t c : chosen) taken = taken || c == x;
                if (taken) x = (int32_t)j;
                chosen.push_back(x);
            }
            for (int32_t c : chosen) s[c] = (int8_t)-s[c];
        } else if (a.mode == 0) {
            for (int32_t k = 0; k < n; ++k) {
                const int32_t i = a.order[k];
                int8_t v = update_value(local_field(g, s.data(), i), s[i], a.tie_rule);
                if (philox_word(a.seed, (uint32_t)i, T, rep, DOMAIN_FLIP) < thr) v = (int8_t)-v;
                s[i] = v;   // in place: later vertices see it
            }
        } else {
            for (int32_t i = 0; i < n; ++i) {
                int8_t v = update_value(local_field(g, s.data(), i), s[i], a.tie_rule);
                if (philox_word(a.seed, (uint32_t)i, T, rep, DOMAIN_FLIP) < thr) v = (int8_t)-v;
                nxt[i] = v;
            }
            s.swap(nxt);
        }
        const int64_t E = energy(g, s.data());            // from scratch every sweep
        const int64_t cut = (a.W - E) / 2;                 // W - E is always even
        if (a.trace) a.trace[(size_t)t * a.n_replicas + r] = cut;
        if (!have_best || cut > bc) {                       // strict: earliest sweep wins
            have_best = true; bc = cut; bs = (int32_t)T; best = s;
        }
    }
    if (a.final_spins) std::memcpy(a.final_spins + (size_t)r * n, s.data(), n);
    if (a.best_cut) a.best_cut[r] = have_best ? bc : 0;
    if (a.best_sweep) a.best_sweep[r] = bs;
    if (a.best_spins && have_best) std::memcpy(a.best_spins + (size_t)r * n, best.data(), n);
}

}  // namespace

extern "C" {

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
    philox4x32_10(ctr, key, out);
}

// Energy E = sum_{i<j} w s_i s_j and cut = (W - E)/2 of given states [R][n].
int32_t oracle_energy_cut(int32_t n, const int64_t* row_ptr, const int32_t* col, const void* w, int32_t wtype,
                          const int8_t* spins, int32_t n_replicas, int64_t* energy_out, int64_t* cut_out) {
    Graph g{n, row_ptr, col, wtype == 1 ? (const int8_t*)w : nullptr, wtype == 4 ? (const int32_t*)w : nullptr};
    if (!g.w8 && !g.w32) return 1;
    const int64_t W = total_weight(g);
    for (int32_t r = 0; r < n_replicas; ++r) {
        const int64_t E = energy(g, spins + (size_t)r * n);
        if (energy_out) energy_out[r] = E;
        if (cut_out) cut_out[r] = (W - E) / 2;
    }
    return 0;
}

// Local fields h_i of one state (for the local-optimum pin).
int32_t oracle_local_fields(int32_t n, const int64_t* row_ptr, const int32_t* col, const void* w, int32_t wtype,
                            const int8_t* spins, int64_t* h_out) {
    Graph g{n, row_ptr, col, wtype == 1 ? (const int8_t*)w : nullptr, wtype == 4 ? (const int32_t*)w : nullptr};
    if (!g.w8 && !g.w32) return 1;
    for (int32_t i = 0; i < n; ++i) h_out[i] = local_field(g, spins, i);
    return 0;
}

// The annealer.  n_threads > 1 only spreads independent replicas over host threads
// (timing convenience; every replica is still computed by the single-threaded code above).
int32_t oracle_anneal(int32_t n, const int64_t* row_ptr, const int32_t* col, const void* w, int32_t wtype,
                      const int32_t* order, int32_t mode, int32_t tie_rule,
                      int32_t n_replicas, int32_t first_replica, uint64_t seed,
                      const uint32_t* thr, int32_t n_sweeps, int32_t sweep_offset,
                      const int8_t* init_spins, int8_t* final_spins, int64_t* trace,
                      int64_t* best_cut, int32_t* best_sweep, int8_t* best_spins, int32_t n_threads) {
    AnnealArgs a;
    a.g = Graph{n, row_ptr, col, wtype == 1 ? (const int8_t*)w : nullptr, wtype == 4 ? (const int32_t*)w : nullptr};
    if (!a.g.w8 && !a.g.w32) return 1;
    if ((mode == 0 || mode == 2) && !order) return 2;
    a.order = order; a.mode = mode; a.tie_rule = tie_rule;
    a.n_replicas = n_replicas; a.first_replica = first_replica; a.seed = seed;
    a.thr = thr; a.n_sweeps = n_sweeps; a.sweep_offset = sweep_offset;
    a.init_spins = init_spins; a.final_spins = final_spins; a.trace = trace;
    a.best_cut = best_cut; a.best_sweep = best_sweep; a.best_spins = best_spins;
    a.W = total_weight(a.g);
    if (n_threads <= 1) {
        for (int32_t r = 0; r < n_replicas; ++r) anneal_replica(a, r);
    } else {
        std::vector<std::thread> pool;
        for (int32_t th = 0; th < n_threads; ++th)
            pool.emplace_back([&a, th, n_threads, n_replicas]() {
                for (int32_t r = th; r < n_replicas; r += n_threads) anneal_replica(a, r);
            });
        for (auto& t : pool) t.join();
    }
    return 0;
}

// Brute force over all 2^n states (n <= 24): plain enumeration, the cut of every state from the
// definition (energy() above); the first state reaching the maximum is returned.
int32_t oracle_bruteforce_maxcut(int32_t n, const int64_t* row_ptr, const int32_t* col, const void* w,
                                 int32_t wtype, int64_t* max_cut_out, int8_t* argmax_spins_out) {
    if (n > 24 || n < 1) return 1;
    Graph g{n, row_ptr, col, wtype == 1 ? (const int8_t*)w : nullptr, wtype == 4 ? (const int32_t*)w : nullptr};
    if (!g.w8 && !g.w32) return 1;
    const int64_t W = total_weight(g);
    std::vector<int8_t> s(n);
    int64_t best = INT64_MIN;
    for (uint32_t code = 0; code < (1u << n); ++code) {
        for (int32_t i = 0; i < n; ++i) s[i] = ((code >> i) & 1u) ? +1 : -1;
        const int64_t cut = (W - energy(g, s.data())) / 2;
        if (cut > best) {
            best = cut;
            if (argmax_spins_out) std::memcpy(argmax_spins_out, s.data(), n);
        }
    }
    *max_cut_out = best;
    return 0;
}

}  // extern "C"
