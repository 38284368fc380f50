// Bandwidth probes behind include/ising_debug.h (measurement only, never on the product path): what the L2 of this
// GPU sustains for the two access patterns of the sparse sweep -- random 32-byte sector gathers from a state-sized
// array (the 512 MB of neighbour gathers per sweep of config 5 are L2 hits) and a streaming read of an
// L2-resident buffer.  bench.py reports them as roofline.l2_* beside the HBM figure of MEASURED_PEAKS.json.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace ising {

// Every lane pair reads `per_pair` random 32-byte sectors (two 16-byte L2 loads, like the sweep's gathers), eight in
// flight per lane; indices from a counter hash (no index traffic).
__global__ void __launch_bounds__(512) k_probe_gather(const uint4* buf, uint32_t sectors_mask, uint32_t per_pair, uint32_t* sink) {
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, pair = tid >> 1, half = tid & 1u;
    uint32_t acc = 0;
    for (uint32_t k = 0; k < per_pair; k += 8) {
        uint4 v[8];
#pragma unroll
        for (uint32_t j = 0; j < 8; ++j) {
            uint32_t x = (pair * 0x9E3779B9u) ^ ((k + j) * 0x85EBCA6Bu);
            x ^= x >> 15; x *= 0x2C1B3C6Du; x ^= x >> 12; x *= 0x297A2D39u; x ^= x >> 15;
            v[j] = __ldcg(buf + (size_t)(x & sectors_mask) * 2u + half);
        }
#pragma unroll
        for (uint32_t j = 0; j < 8; ++j) acc += v[j].x ^ v[j].w;
    }
    if (acc == 0x12345678u) *sink = acc;
}

// The same sectors with 4-byte loads: eight consecutive lanes read the eight words of one sector (four sectors per
// warp instruction instead of sixteen).
__global__ void __launch_bounds__(512) k_probe_gather4(const uint32_t* buf, uint32_t sectors_mask, uint32_t per_group, uint32_t* sink) {
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, grp = tid >> 3, word = tid & 7u;
    uint32_t acc = 0;
    for (uint32_t k = 0; k < per_group; k += 8) {
        uint32_t v[8];
#pragma unroll
        for (uint32_t j = 0; j < 8; ++j) {
            uint32_t x = (grp * 0x9E3779B9u) ^ ((k + j) * 0x85EBCA6Bu);
            x ^= x >> 15; x *= 0x2C1B3C6Du; x ^= x >> 12; x *= 0x297A2D39u; x ^= x >> 15;
            v[j] = __ldcg(buf + (size_t)(x & sectors_mask) * 8u + word);
        }
#pragma unroll
        for (uint32_t j = 0; j < 8; ++j) acc += v[j];
    }
    if (acc == 0x12345678u) *sink = acc;
}

// Every thread streams 16-byte words of the (L2-resident) buffer, grid-strided, `passes` times.
__global__ void __launch_bounds__(512) k_probe_stream(const uint4* buf, uint32_t n16, uint32_t passes, uint32_t* sink) {
    uint32_t acc = 0;
    for (uint32_t p = 0; p < passes; ++p)
        for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += gridDim.x * blockDim.x) {
            const uint4 v = __ldcg(buf + i);
            acc += v.x ^ v.w;
        }
    if (acc == 0x12345678u) *sink = acc;
}

}  // namespace ising
