// cfs_hiz.cuh -- Hi-Z map of the depth splat stage (sm_100a).
//
// The 3-D depth path (BASELINE configs[4]: "nearest-point depth test via 64-bit packed
// (float depth | rgba8) atomicMin") pays one random 32-byte L2 sector per splat for its pre-test
// load, and an SM can issue about one such request per clock: measured, that request rate -- not
// the atomics, of which a solid needs few -- bounds the direct variant.  Almost all of those loads
// only confirm that the splat is occluded.  A coarse, conservative copy of the depth image that
// fits shared memory answers the same question on the SM:
//
//   hz[block] = max over the pixels of a 2^shift x 2^shift block of (depth bits >> 16),
//
// built by hiz_build_kernel from a snapshot of the image after a first small slice of the points.
// The image only ever decreases (atomicMin), so the snapshot bound stays an upper bound for the
// rest of the render and `(bits(d) >> 16) > hz[block]` proves `key > image[pixel]`: skipping that
// splat cannot change the result.  Depths are positive floats, so their bit patterns order like
// the values; an empty pixel (all ones) gives 0xFFFF, which culls nothing.
#pragma once
#ifndef __CUDACC_RTC__
#include <cuda_runtime.h>
#include <stdint.h>
#endif

#include "cfs_params.h"

namespace cfs {

// one CTA of (2^shift)^2 threads per Hi-Z block (shift <= 5), one pixel per thread
__global__ void hiz_build_kernel(const unsigned long long *__restrict__ image, int W, int H, uint32_t shift,
                                 uint32_t nbx, uint16_t *__restrict__ hz)
{
    const uint32_t bx = blockIdx.x % nbx, by = blockIdx.x / nbx;
    const uint32_t side = 1u << shift;
    const uint32_t tx = threadIdx.x & (side - 1u), ty = threadIdx.x >> shift;
    const uint32_t px = (bx << shift) + tx, py = (by << shift) + ty;
    uint32_t v = 0u;
    if (px < (uint32_t)W && py < (uint32_t)H)
        v = (uint32_t)(__ldcg(image + (size_t)py * (size_t)W + px) >> 48);     // depth bits >> 16
    v = __reduce_max_sync(0xFFFFFFFFu, v);
    __shared__ uint32_t s_max[32];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31u) >> 5;
    if (lane == 0) s_max[warp] = v;
    __syncthreads();
    if (warp == 0) {
        uint32_t m = (lane < nwarps) ? s_max[lane] : 0u;
        m = __reduce_max_sync(0xFFFFFFFFu, m);
        if (lane == 0) hz[blockIdx.x] = (uint16_t)m;
    }
}

}  // namespace cfs
