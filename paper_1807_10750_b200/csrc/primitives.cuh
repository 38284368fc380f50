// Small device primitives shared by the sweep kernels (sparse_sweep.cuh) and the shared-memory chain engine
// (chain.cuh): byte transposes feeding dp4a, sign / mask helpers, cp.async and shared-memory accessors.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

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

__device__ __forceinline__ uint32_t nibble_to_bytemask(uint32_t nib) {
    // bit b of nib -> byte b = 0xff (the four copies of nib at shifts 0, 7, 14, 21 do not overlap)
    return ((nib * 0x00204081u) & 0x01010101u) * 0xffu;
}

__device__ __forceinline__ uint32_t lt4(const uint4& u, uint32_t thr) {
    return (u.x < thr ? 1u : 0u) | (u.y < thr ? 2u : 0u) | (u.z < thr ? 4u : 0u) | (u.w < thr ? 8u : 0u);
}

__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
    uint32_t r;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(sel));
    return r;
}
// byte b of the result = 0xff if v_b < 0 else 0x00 (PRMT sign replication of the top bytes)
__device__ __forceinline__ uint32_t sign_bytes(int v0, int v1, int v2, int v3) {
    const uint32_t t0 = prmt((uint32_t)v0, (uint32_t)v1, 0xfbfbu);
    const uint32_t t1 = prmt((uint32_t)v2, (uint32_t)v3, 0xfbfbu);
    return prmt(t0, t1, 0x5410u);
}

__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void* gptr) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
// 16 bytes if `real`, else no global access at all: the slot is zero-filled (cp.async with src-size 0)
__device__ __forceinline__ void cp_async16_if(uint32_t smem_addr, const void* gptr, bool real) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_addr), "l"(gptr), "r"(real ? 16 : 0) : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void* gptr) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(gptr));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ uint4 lds128(uint32_t smem_addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(smem_addr));
    return v;
}

__device__ __forceinline__ void cp_async4(uint32_t smem_addr, const void* gptr) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ uint32_t lds32(uint32_t smem_addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(smem_addr));
    return v;
}
__device__ __forceinline__ void sts32(uint32_t smem_addr, uint32_t v) {
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(smem_addr), "r"(v) : "memory");
}

}  // namespace ising
