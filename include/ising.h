/*
 * ising.h -- C ABI of the B200-native Ising max-cut annealer.
 *
 * The operation is the annealing sweep of arXiv 1807.10750 ("GPU Ising Computing for
 * Combinatorial Optimization Problems in VLSI Physical Design"); citations are
 * PAPER.md line numbers plus section / equation / algorithm:
 *
 *   problem    weighted graph G=(V,E), integer w_ij in; x_i in {+1,-1} and the cut
 *              value  cut = 1/2 sum_{i<j} w_ij (1 - x_i x_j)  out      (L117-122, eq. 4)
 *   mapping    sigma_i = x_i, couplings from w_ij, no external field   (L124-128, eq. 5);
 *              the quantity minimised is E(s) = +sum_{i<j} w_ij s_i s_j, so that
 *              cut = (W - E)/2 with W = sum_{i<j} w_ij  (reading Q1)
 *   update     h_i = sum_j w_ij s_j ; s_i <- +1 if h_i < 0 else -1     (L43-49, eq. 2)
 *   annealing  Algorithm 2 (L164-184): for every sweep, every spin takes its
 *              energy-minimising value and is then flipped with probability F_p;
 *              F_p is lowered after every sweep.  Here F_p is a caller-supplied
 *              uint32 threshold per sweep and the flip test is
 *              Philox4x32-10(key=seed; ctr=(spin id, absolute sweep, replica>>2, 0))[replica&3] < thr.
 *   order      the paper leaves the order inside a sweep to thread scheduling
 *              (L158); this library offers deterministic orders only:
 *              colour-class Gauss-Seidel (sequential in (colour, id) order) and
 *              synchronous Jacobi (every spin from the sweep-start state).
 *
 * All arithmetic is integer; results are bit-exact and independent of launch geometry.
 *
 * Conventions
 *   - Pointers marked "host|device" may be either; the library inspects them with
 *     cudaPointerGetAttributes.  "device" pointers must be device memory of the
 *     current device.  "host" pointers are plain host memory.
 *   - Caller-facing spin arrays are replica-major [n_replicas][n] int8, values +1 / -1,
 *     indexed by the CALLER's vertex ids.  The replica-interleaved layout is internal.
 *   - The library allocates no device memory: everything lives in the workspace the
 *     caller passes to ising_load_csr (e.g. a torch uint8 tensor), borrowed until
 *     ising_free.  Inputs of ising_load_csr are copied and may be freed on return.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *     ising_load_csr is synchronous (it validates on the device and reads back the
 *     verdict).  ising_anneal / ising_energy_cut enqueue work on `stream` and return;
 *     outputs in DEVICE memory are ready when the stream has drained.  Outputs in HOST
 *     memory are written before the call returns (the call synchronises the stream).
 *   - Every function returns an ising_status; 0 is success.  On error no output is
 *     written.  No exceptions, no abort().  A device fault surfaces as ISING_ERR_CUDA
 *     on the call that observes it.
 *   - A handle is not thread-safe; distinct handles are independent.
 *   - There is no CPU fallback: on a machine without an sm_100 device every compute
 *     entry point returns ISING_ERR_UNSUPPORTED_DEVICE.
 */
#ifndef ISING_B200_H
#define ISING_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ising_problem ising_problem; /* opaque */
typedef int32_t ising_status;

enum {
    ISING_OK = 0,
    ISING_ERR_NULL_ARG = 1,
    ISING_ERR_BAD_SHAPE = 2,          /* n<=0, nnz<0, row_ptr not monotone / wrong ends, col out of range, bad enum,
                                         workspace not 256-byte aligned device memory */
    ISING_ERR_UNSORTED_OR_DUP = 3,    /* a row's columns are not strictly ascending */
    ISING_ERR_SELF_LOOP = 4,
    ISING_ERR_ASYMMETRIC = 5,         /* (i,j) present without (j,i), or w(i,j) != w(j,i) */
    ISING_ERR_BAD_COLOURING = 6,      /* colour out of [0,n_colours) or two neighbours share a colour */
    ISING_ERR_FIELD_OVERFLOW = 7,     /* max_i sum_j |w_ij| >= 2^31 */
    ISING_ERR_TOO_MANY_REPLICAS = 8,
    ISING_ERR_WORKSPACE_TOO_SMALL = 9,
    ISING_ERR_NO_COLOURING_FOR_GS = 10,
    ISING_ERR_UNSUPPORTED_DEVICE = 11,
    ISING_ERR_CUDA = 12,
    ISING_ERR_BAD_SPINS = 13,         /* a caller-supplied spin is neither +1 nor -1 */
    ISING_ERR_NO_STATE = 14           /* continue / current-state request before any state exists */
};

/* update order (Q8) */
enum { ISING_MODE_GS = 0, ISING_MODE_JACOBI = 1, ISING_MODE_RACY = 2, ISING_MODE_EXACT_N = 3 };
/* tie rule when h_i == 0 (L49: "If S=0, it can take any value"; Q3) */
enum { ISING_TIE_MINUS = 0, ISING_TIE_KEEP = 1 };
/* initial state (L82 / L169 "initialize all sigma_i"; Q4) */
enum { ISING_INIT_PHILOX = 0, ISING_INIT_GIVEN = 1, ISING_INIT_CONTINUE = 2 };
/* weight element type of the CSR passed to ising_load_csr */
enum { ISING_W_INT8 = 1, ISING_W_INT32 = 4 };
/* load flags */
enum {
    ISING_LOAD_DEFAULT = 0,
    ISING_LOAD_NO_DENSE = 1,      /* never build the dense tcgen05 engine, even for a complete graph */
    /* Gauss-Seidel engine selection (results never depend on it; the default picks the fastest that applies):       */
    ISING_LOAD_NO_SMALL = 2,      /* do not run a small graph wholly inside one CTA per four replicas (shared memory)   */
    ISING_LOAD_NO_CLUSTER = 4,    /* no thread-block clusters: neither one per replica tile, nor pairs of CTAs sharing   */
                                  /* the rows of a small graph in the shared-memory engine                               */
    ISING_LOAD_NO_TAIL_CHAIN = 8, /* big graph: every colour class is a grid-wide phase (no shared-memory tail chain)    */
    ISING_LOAD_NO_OVERLAP = 16    /* tail chain: do not update the chain-free rows of colour class 0 for sweep t + 1 while */
                                  /* the chain finishes sweep t (the chain runs alone, as in the build before)            */
};

/*
 * Upper bound of the device workspace ising_load_csr needs for a graph with these
 * dimensions (any degree distribution), in bytes.  n_colours = 0 for a Jacobi-only
 * problem.  Host-only computation; works without a GPU.
 */
ising_status ising_workspace_bytes(int32_t n, int64_t nnz, int32_t wtype, int32_t max_replicas,
                                   int32_t n_colours, size_t* bytes_out);

/*
 * Ingest a symmetric integer-weighted graph in CSR form and build the device layout
 * ("connections ... able to connect to any other spin",
 * L138 host->device offload model).
 *
 *   n, nnz       vertices, directed entries (= 2 * #edges)
 *   row_ptr      int64 [n+1], host|device; row_ptr[0] = 0, row_ptr[n] = nnz
 *   col_idx      int32 [nnz], host|device; each row strictly ascending, no self loops
 *   weights      int8 [nnz] (wtype = ISING_W_INT8) or int32 [nnz] (ISING_W_INT32), host|device;
 *                w(i,j) == w(j,i); zero weights are allowed
 *   colour       int32 [n] proper colouring with values in [0, n_colours), host|device;
 *                NULL (and n_colours = 0) -> the problem supports Jacobi / racy modes only
 *   max_replicas largest n_replicas any later call will pass (1 .. 65536)
 *   workspace    DEVICE memory, 256-byte aligned (else ISING_ERR_BAD_SHAPE), workspace_bytes long (else
 *                ISING_ERR_WORKSPACE_TOO_SMALL), borrowed until ising_free
 *   flags        ISING_LOAD_*
 *   out          receives the handle (host object; free with ising_free)
 *
 * A complete graph (nnz == n(n-1)) with int8-range weights additionally gets the dense
 * engine (J as an int8 matrix, local fields J.S on tcgen05 tensor cores), used by
 * ISING_MODE_JACOBI.  Limits: a row may hold at most 32767 x 128 edges (ISING_ERR_BAD_SHAPE beyond).
 * Synchronous.  Errors: every ISING_ERR_* above.
 */
ising_status ising_load_csr(int32_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx,
                            const void* weights, int32_t wtype, const int32_t* colour,
                            int32_t n_colours, int32_t max_replicas, void* workspace,
                            size_t workspace_bytes, int32_t flags, void* stream, ising_problem** out);

/*
 * Run n_sweeps annealing sweeps on n_replicas independent replicas (Algorithm 2,
 * PAPER.md L164-184; replicas = the "number of GPU simulations" of L239 run side by side).
 *
 *   mode           ISING_MODE_GS (needs a colouring), ISING_MODE_JACOBI, ISING_MODE_RACY
 *                  (paper-like unordered in-place update, L158; not deterministic), or
 *                  ISING_MODE_EXACT_N (Algorithm 1, L77-99; needs a colouring): every sweep is pure local
 *                  minimisation in colour-class order, then exactly N = thresholds[t] (<= 4096, clamped
 *                  to n) DISTINCT spins per replica are flipped, drawn as a uniform N-subset by Floyd's
 *                  algorithm on Philox words (counter = (draw index, sweep, replica>>2, 2))
 *   tie_rule       ISING_TIE_*
 *   n_replicas     1 .. max_replicas; replica r of this call has global id first_replica + r,
 *                  which is what enters the Philox counter
 *   seed           Philox key
 *   thresholds     uint32 [n_sweeps], HOST; flip iff philox_word < thresholds[t] (ISING_MODE_EXACT_N: the
 *                  number of spins to flip after sweep t)
 *   sweep_offset   absolute index of this call's first sweep (enters the Philox counter)
 *   init_mode      ISING_INIT_PHILOX: s_i = (philox(ctr=(i,0,r>>2,1))[r&3] & 1) ? +1 : -1
 *                  ISING_INIT_GIVEN: copy init_spins; ISING_INIT_CONTINUE: keep the handle's state
 *   init_spins     int8 [n_replicas][n], host|device, or NULL unless ISING_INIT_GIVEN
 *   cut_trace      int64 [n_sweeps][n_replicas], DEVICE, or NULL: cut after every sweep
 *
 * After every sweep the cut of every replica is evaluated (eq. 4) and the best state seen
 * in THIS call is captured (strictly greater cut wins, so the earliest sweep wins ties).
 * Asynchronous on `stream` (except ISING_INIT_GIVEN, which reads back a validity flag of the given spins).
 * `thresholds` is copied before the call returns.  n_sweeps == 0 only (re)initialises the state.
 */
ising_status ising_anneal(ising_problem* p, int32_t mode, int32_t tie_rule, int32_t n_replicas,
                          int32_t first_replica, uint64_t seed, const uint32_t* thresholds,
                          int32_t n_sweeps, int32_t sweep_offset, int32_t init_mode,
                          const int8_t* init_spins, int64_t* cut_trace, void* stream);

/*
 * Energy E = sum_{i<j} w_ij s_i s_j (eq. 3/5 under reading Q1) and cut = (W - E)/2 (eq. 4)
 * of given states, from the definition (a full edge reduction, not the incremental value
 * the annealer tracks).
 *
 *   spins        int8 [n_replicas][n], host|device, or NULL = the handle's current state
 *   energy_out   int64 [n_replicas], host|device, or NULL
 *   cut_out      int64 [n_replicas], host|device, or NULL
 */
ising_status ising_energy_cut(ising_problem* p, const int8_t* spins, int32_t n_replicas,
                              int64_t* energy_out, int64_t* cut_out, void* stream);

/*
 * Best state captured by the last ising_anneal call.
 *
 *   replica      0 .. n_replicas-1 of that call, or -1 = the replica with the largest best
 *                cut (lowest replica index wins ties)
 *   spins_out    int8 [n], host|device, or NULL
 *   cut_out      int64, HOST, or NULL
 *   sweep_out    int32, HOST, or NULL: absolute sweep after which the state was seen
 *   replica_out  int32, HOST, or NULL: the replica chosen
 * Synchronises `stream`.
 */
ising_status ising_best_state(ising_problem* p, int32_t replica, int8_t* spins_out, int64_t* cut_out,
                              int32_t* sweep_out, int32_t* replica_out, void* stream);

/*
 * Current (final) state of the last ising_anneal call.
 *   spins_out    int8 [n_replicas][n], host|device
 * Synchronises `stream` when spins_out is host memory.
 */
ising_status ising_current_state(ising_problem* p, int8_t* spins_out, int32_t n_replicas, void* stream);

/*
 * Properties of a loaded problem (host-side bookkeeping, no device work).
 *   what: 0 n, 1 nnz, 2 n_colours, 3 max_replicas, 4 W = sum_{i<j} w_ij, 5 dense engine built (0/1),
 *         6 kernels launched by this handle so far, 7 max_i sum_j |w_ij|, 8 workspace bytes in use,
 *         9 slices of the sparse layout, 10 padded edge slots of the sparse layout, 11 hub rows,
 *         12 CTAs of the persistent grid, 13 Gauss-Seidel engine (0 launch per phase, 1 persistent grid, 2 persistent
 *         clusters, 3 persistent grid + shared-memory tail chain, 4 shared-memory chain for the whole graph),
 *         14 rows of the shared-memory chain, 15 virtual phases of the persistent kernel,
 *         16 chunks of the chain, 17 1 if the chain is resident in shared memory,
 *         18 CTAs per word of four replicas of the small-graph engine (cluster size),
 *         19 rows of colour class 0 updated beside the tail chain (chain overlap; 0 = off)
 */
ising_status ising_problem_info(const ising_problem* p, int32_t what, int64_t* value_out);

/* Release the handle (the workspace returns to the caller).  NULL is allowed. */
ising_status ising_free(ising_problem* p);

/* Static, never-NULL description of a status code. */
const char* ising_status_string(ising_status s);

#ifdef __cplusplus
}
#endif
#endif /* ISING_B200_H */
