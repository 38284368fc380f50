// Dense local-field engine for fully connected instances -- interface.
// (placeholder until the tcgen05 kernel lands: kDenseEnabled = false keeps K_n on the sparse path)
#pragma once
#include "common.cuh"
#include "../../include/ising.h"

namespace ising {

constexpr bool kDenseEnabled = false;

struct DenseEngine;

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
};

inline size_t dense_workspace_bytes(int64_t, int64_t) { return 0; }
inline DenseEngine* dense_create(int32_t, int32_t, void*, size_t, const long long*, const int32_t*, const void*, int,
                                 cudaStream_t) { return nullptr; }
inline void dense_destroy(DenseEngine*) {}
inline ising_status dense_anneal(DenseEngine*, const DenseAnnealArgs&, cudaStream_t, int64_t*) { return ISING_ERR_CUDA; }
inline ising_status dense_export_state(DenseEngine*, int8_t*, int32_t, bool, cudaStream_t) { return ISING_ERR_CUDA; }
inline ising_status dense_export_one(DenseEngine*, int8_t*, int32_t, bool, cudaStream_t) { return ISING_ERR_CUDA; }
inline ising_status dense_best_arrays(DenseEngine*, long long*, int32_t*, int32_t, cudaStream_t) { return ISING_ERR_CUDA; }

}  // namespace ising
