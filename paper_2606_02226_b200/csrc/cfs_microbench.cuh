// cfs_microbench.cuh -- roofline denominators measured in the same run (BASELINE north_star:
// "the slower of FP32/INT issue at peak ... and the L2-atomic rate measured by a microbenchmark
// in the same run").  Each kernel does `ops` operations per thread; the caller times the stream.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cfs {

// cheap counter hash -> uniformly random bin (2 IMAD + 2 shift/xor per op, far below the
// cost of the memory operation it addresses)
__device__ __forceinline__ uint32_t mb_hash(uint32_t x)
{
    x *= 0x9E3779B1u;
    x ^= x >> 15;
    x *= 0x85EBCA77u;
    x ^= x >> 13;
    return x;
}

__device__ __forceinline__ uint32_t mb_bin(uint32_t h, uint32_t n_bins)
{
    return __umulhi(h, n_bins);   // uniform on [0, n_bins)
}

template <int KIND>
__global__ void mb_mem_kernel(void *buf, uint32_t n_bins, uint64_t ops)
{
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t ctr = tid * 0x632BE5ABu + 1u;
    unsigned long long sink = 0;
    for (uint64_t i = 0; i < ops; ++i) {
        ctr += 0x9E3779B9u;
        const uint32_t b = mb_bin(mb_hash(ctr), n_bins);
        if (KIND == 0) {
            asm volatile("red.global.add.u32 [%0], %1;" :: "l"(reinterpret_cast<uint32_t *>(buf) + b), "r"(1u) : "memory");
        } else if (KIND == 1) {
            asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};"
                         :: "l"(reinterpret_cast<float *>(buf) + 4 * (size_t)b), "f"(1.0f), "f"(2.0f), "f"(3.0f), "f"(1.0f) : "memory");
        } else if (KIND == 2) {
            // keys decrease with i so that most atomics really write (worst case for the depth path)
            const unsigned long long key = ((unsigned long long)(0x7F000000u - (uint32_t)i) << 32) | tid;
            atomicMin(reinterpret_cast<unsigned long long *>(buf) + b, key);
        } else if (KIND == 3) {
            sink += __ldcg(reinterpret_cast<const unsigned long long *>(buf) + b);
        }
    }
    if (KIND == 3 && sink == 0x1234567ull) reinterpret_cast<unsigned long long *>(buf)[0] = sink;
}

__global__ void mb_atoms_kernel(void *buf, uint32_t n_bins, uint64_t ops)
{
    extern __shared__ uint32_t sh[];
    for (uint32_t i = threadIdx.x; i < n_bins; i += blockDim.x) sh[i] = 0;
    __syncthreads();
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t ctr = tid * 0x632BE5ABu + 1u;
    for (uint64_t i = 0; i < ops; ++i) {
        ctr += 0x9E3779B9u;
        atomicAdd(&sh[mb_bin(mb_hash(ctr), n_bins)], 1u);
    }
    __syncthreads();
    if (threadIdx.x == 0 && sh[0] == 0xFFFFFFFFu) reinterpret_cast<uint32_t *>(buf)[0] = 1;
}

// ALU kinds: 8 independent dependent-chains per thread, 8 ops per loop trip per chain
template <int KIND>
__global__ void mb_alu_kernel(void *buf, uint64_t ops)
{
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
    float f[8];
    uint32_t u[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { f[j] = 1.0f + 1e-3f * (float)(tid + j); u[j] = tid * 8u + j + 1u; }
    const float a = 0.999f, b = 1e-4f;
    const uint64_t trips = ops / 64;
    for (uint64_t i = 0; i < trips; ++i) {
#pragma unroll
        for (int rep = 0; rep < 8; ++rep) {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                if (KIND == 5) f[j] = __fmaf_rn(f[j], a, b);
                else if (KIND == 6) { const uint64_t p = (uint64_t)u[j] * 0xD2511F53u; u[j] = (uint32_t)(p >> 32) ^ (uint32_t)p; }
                else if (KIND == 7) u[j] = (u[j] ^ u[(j + 1) & 7]) ^ (uint32_t)i;
                else if (KIND == 8) f[j] = __sinf(f[j]);
            }
        }
    }
    float fs = 0.f; uint32_t us = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { fs += f[j]; us ^= u[j]; }
    if (fs == 123.456f || us == 0x12345u) reinterpret_cast<uint32_t *>(buf)[0] = us + (uint32_t)fs;
}

__global__ void mb_stream_kernel(void *buf, uint64_t n_vec)
{
    const uint4 *v = reinterpret_cast<const uint4 *>(buf);
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint32_t acc = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += stride) {
        const uint4 q = __ldcs(v + i);
        acc ^= q.x ^ q.y ^ q.z ^ q.w;
    }
    if (acc == 0x9876543u) reinterpret_cast<uint32_t *>(buf)[0] = acc;
}

}  // namespace cfs
