/*
 * ising_noalloc.h -- an entry point of the B200-native Ising annealer that allocates NOTHING.
 *
 * Why: some callers cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it) and have no workspace to hand to ising_load_csr.  ising_energy_cut_noalloc evaluates
 *     E = sum_{i<j} w_ij s_i s_j   (eq. (3)/(5), L53/L124, sign reading Q1 of DESIGN.md)
 *     cut = (W - E) / 2,  W = sum_{i<j} w_ij   (eq. (4))
 * of given spin states straight from the caller's CSR, without a handle and without a workspace: its scratch (one
 * int64 accumulator per replica + W) is a file-scope `static __device__ __align__(256)` array inside the library.
 *
 * Limits and rules:
 *   - n_replicas <= ISING_NOALLOC_MAX_REPLICAS (1024); more is rejected with ISING_ERR_TOO_MANY_REPLICAS and nothing is
 *     launched.  n and nnz are not limited by the scratch (it does not grow with the graph).
 *   - The scratch costs ISING_NOALLOC_SCRATCH_BYTES (8448 bytes) of device memory on every GPU that loads the library,
 *     until the process exits.
 *   - The call never calls cudaMalloc / cudaFree / any allocating routine, never synchronises, and enqueues three
 *     kernels on `stream` (clear, accumulate, finish).  The scratch is cleared by the call itself: nothing depends on
 *     what an earlier call left there.
 *   - ALL calls on one GPU share the scratch: two calls that overlap on the GPU (different streams, or graphs
 *     replayed concurrently) RACE and give wrong results.  Calls on one stream are ordered and safe.
 *   - Every pointer is DEVICE memory.  The graph is not validated (use ising_load_csr for that): it must be the
 *     symmetric CSR of ising.h (both directions stored, no self loops), spins must be +1 / -1.
 *   - Results are exact integers, identical to ising_energy_cut on the same graph and spins.
 */
#ifndef ISING_B200_NOALLOC_H
#define ISING_B200_NOALLOC_H

#include "ising.h"

#ifdef __cplusplus
extern "C" {
#endif

enum {
    ISING_NOALLOC_MAX_REPLICAS = 1024,
    ISING_NOALLOC_SCRATCH_BYTES = 8 * (1024 + 32)   /* accumulators + the W slot, padded to 256 bytes */
};

/*
 *   n, nnz       vertices, directed entries (both directions of every edge are stored)
 *   row_ptr      int64 [n + 1], DEVICE
 *   col_idx      int32 [nnz], DEVICE
 *   weights      int8 or int32 [nnz] (wtype = ISING_W_INT8 / ISING_W_INT32), DEVICE
 *   spins        int8 [n_replicas][n], +1 / -1, DEVICE
 *   energy_out   int64 [n_replicas], DEVICE, or NULL
 *   cut_out      int64 [n_replicas], DEVICE, or NULL
 * Asynchronous on `stream`.  Errors: NULL_ARG, BAD_SHAPE (n <= 0, nnz < 0, bad wtype), TOO_MANY_REPLICAS
 * (n_replicas < 1 or > ISING_NOALLOC_MAX_REPLICAS), UNSUPPORTED_DEVICE, CUDA.
 */
ising_status ising_energy_cut_noalloc(int32_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx,
                                      const void* weights, int32_t wtype, const int8_t* spins, int32_t n_replicas,
                                      int64_t* energy_out, int64_t* cut_out, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* ISING_B200_NOALLOC_H */
