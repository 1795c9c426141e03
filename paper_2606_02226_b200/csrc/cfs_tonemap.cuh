// cfs_tonemap.cuh -- log-density tone map (DESIGN R10).  HBM-bound: reads the
// image twice (max pass + map pass; the second read hits L2 for images below 126 MB) and writes
// W*H*4 bytes.  Not in the paper; fractal-flame convention.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cfs {

constexpr int kToneThreads = 256;

// count of pixel i as float: HIST value or RGBA alpha
template <int MODE>
__device__ __forceinline__ float tone_count(const void *img, size_t i)
{
    if (MODE == 0) return (float)__ldg(reinterpret_cast<const uint32_t *>(img) + i);
    return __ldg(reinterpret_cast<const float *>(img) + 4 * i + 3);
}

// pass 1: n_max.  Non-negative floats order like their bit patterns -> one atomicMax(u32) per CTA.
template <int MODE>
__global__ void __launch_bounds__(kToneThreads) tone_max_kernel(const void *img, size_t n, uint32_t *scratch)
{
    float m = 0.0f;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    if (MODE == 0) {
        // 128-bit loads over the u32 histogram
        const uint4 *v = reinterpret_cast<const uint4 *>(img);
        const size_t n4 = n / 4;
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
            const uint4 q = __ldg(v + i);
            m = fmaxf(m, (float)max(max(q.x, q.y), max(q.z, q.w)));
        }
        for (size_t i = n4 * 4 + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
            m = fmaxf(m, tone_count<0>(img, i));
    } else {
        const float4 *v = reinterpret_cast<const float4 *>(img);
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
            m = fmaxf(m, __ldg(v + i).w);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xFFFFFFFFu, m, o));
    __shared__ float sm[kToneThreads / 32];
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < kToneThreads / 32; ++i) m = fmaxf(m, sm[i]);
        if (m > 0.0f) atomicMax(scratch, __float_as_uint(m));
    }
}

__device__ __forceinline__ uint32_t tone_byte(float v)
{
    v = fminf(fmaxf(v, 0.0f), 1.0f);   // NaN -> 0 (fmaxf returns the non-NaN operand)
    return (uint32_t)__float2int_rd(__fmaf_rn(255.0f, v, 0.5f));
}

// pass 2: one pixel per thread.
template <int MODE>
__global__ void __launch_bounds__(kToneThreads)
tone_map_kernel(const void *img, size_t n, const uint32_t *scratch, float inv_gamma, float colour_scale,
                uint32_t *out)
{
    const float nmax = __uint_as_float(__ldg(scratch));
    const float inv_lmax = 1.0f / log1pf(nmax);
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        if (MODE == 0) {
            const float c = tone_count<0>(img, i);
            uint32_t o = 0;
            if (c > 0.0f) {
                const float L = log1pf(c) * inv_lmax;
                const uint32_t g = tone_byte(powf(L, inv_gamma));
                o = g | (g << 8) | (g << 16) | (tone_byte(L) << 24);
            }
            out[i] = o;
        } else {
            const float4 a = __ldg(reinterpret_cast<const float4 *>(img) + i);
            uint32_t o = 0;
            if (a.w > 0.0f) {
                const float L = log1pf(a.w) * inv_lmax;
                const float sc = colour_scale * powf(L, inv_gamma) / a.w;
                o = tone_byte(a.x * sc) | (tone_byte(a.y * sc) << 8) | (tone_byte(a.z * sc) << 16) |
                    (tone_byte(L) << 24);
            }
            out[i] = o;
        }
    }
}

// DEPTH: resolve = colour word, empty -> 0
__global__ void __launch_bounds__(kToneThreads)
tone_depth_kernel(const unsigned long long *buf, size_t n, uint32_t *out)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const unsigned long long v = __ldg(buf + i);
        out[i] = (v == 0xFFFFFFFFFFFFFFFFull) ? 0u : (uint32_t)v;
    }
}

}  // namespace cfs
