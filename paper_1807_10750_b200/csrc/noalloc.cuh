// ising_energy_cut_noalloc (include/ising_noalloc.h): energy / cut of given states straight from the caller's CSR,
// for callers that may not allocate.  No handle, no workspace: the only scratch is the file-scope device array below
// (8448 bytes on every GPU that loads the library, until exit).  Shares no state with the rest of the library.
//
// E = sum_{i<j} w_ij s_i s_j (eq. (3)/(5), reading Q1) = 1/2 sum_i s_i h_i with h_i = sum_j w_ij s_j (eq. (2),
// L45); cut = (W - E)/2 (eq. (4)), W = 1/2 sum over the stored (directed) entries.
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>

#include "../../include/ising_noalloc.h"

namespace ising {

constexpr int kNoAllocMaxReplicas = ISING_NOALLOC_MAX_REPLICAS;
constexpr int kNoAllocSlots = kNoAllocMaxReplicas + 32;   // [0, R): sum_i s_i h_i per replica; slot kNoAllocMaxReplicas: sum of the stored weights
static_assert(sizeof(long long) * kNoAllocSlots == ISING_NOALLOC_SCRATCH_BYTES, "header and scratch size disagree");

// The scratch.  In HOST code this name is only a stand-in for the symbol, not a device address: the host side takes
// the address once per device with cudaGetSymbolAddress (noalloc_scratch_ptr below) and passes it to the kernels.
static __device__ __align__(256) long long g_noalloc_scratch[kNoAllocSlots];

// Every call starts from zero: nothing depends on what the previous call left in the scratch.
__global__ void k_noalloc_clear(long long* scratch, int n_replicas) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_replicas) scratch[i] = 0;
    if (i == 0) scratch[kNoAllocMaxReplicas] = 0;
}

// grid = (row blocks, replicas); one warp per row at a time, lanes over the row's entries.
__global__ void __launch_bounds__(256) k_noalloc_accumulate(int32_t n, const long long* row_ptr, const int32_t* col,
                                                            const void* w, int wtype, const int8_t* spins,
                                                            long long* scratch) {
    __shared__ long long s_part[8], s_wpart[8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int r = blockIdx.y;
    const int8_t* s = spins + (size_t)r * (size_t)n;
    long long acc = 0, wsum = 0;
    for (long long i = (long long)blockIdx.x * 8 + warp; i < n; i += (long long)gridDim.x * 8) {
        const long long b = row_ptr[i], e = row_ptr[i + 1];
        long long h = 0;
        for (long long k = b + lane; k < e; k += 32) {
            const long long wv = wtype == 1 ? (long long)reinterpret_cast<const int8_t*>(w)[k]
                                            : (long long)reinterpret_cast<const int32_t*>(w)[k];
            h += wv * (long long)s[col[k]];
            wsum += wv;
        }
        acc += (long long)s[i] * h;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        acc += __shfl_xor_sync(0xffffffffu, acc, o);
        wsum += __shfl_xor_sync(0xffffffffu, wsum, o);
    }
    if (lane == 0) { s_part[warp] = acc; s_wpart[warp] = wsum; }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long a = 0, ws = 0;
        for (int k = 0; k < 8; ++k) { a += s_part[k]; ws += s_wpart[k]; }
        if (a != 0) atomicAdd(reinterpret_cast<unsigned long long*>(scratch + r), (unsigned long long)a);
        if (r == 0 && ws != 0)
            atomicAdd(reinterpret_cast<unsigned long long*>(scratch + kNoAllocMaxReplicas), (unsigned long long)ws);
    }
}

__global__ void k_noalloc_finish(const long long* scratch, int n_replicas, long long* energy_out, long long* cut_out) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_replicas) return;
    const long long E = scratch[r] / 2;                       // sum_i s_i h_i counts every edge twice
    const long long W = scratch[kNoAllocMaxReplicas] / 2;     // so does the sum over the stored entries
    if (energy_out) energy_out[r] = E;
    if (cut_out) cut_out[r] = (W - E) / 2;
}

// Device address of the scratch on the CURRENT device, taken once per device (cudaGetSymbolAddress allocates
// nothing: the array is part of the loaded module).  nullptr on failure.
inline long long* noalloc_scratch_ptr() {
    constexpr int kMaxDevices = 64;
    static std::atomic<long long*> cache[kMaxDevices];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
    if (dev >= 0 && dev < kMaxDevices) {
        if (long long* p = cache[dev].load(std::memory_order_acquire)) return p;
    }
    long long* ptr = nullptr;
    if (cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_noalloc_scratch) != cudaSuccess || !ptr) {
        (void)cudaGetLastError();
        return nullptr;
    }
    if (dev >= 0 && dev < kMaxDevices) cache[dev].store(ptr, std::memory_order_release);
    return ptr;
}

}  // namespace ising
