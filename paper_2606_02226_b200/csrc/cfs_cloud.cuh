// cfs_cloud.cuh -- the stored-cloud generator (BASELINE configs[3]) as a streaming kernel (sm_100a).
//
// A stored cloud is one 16-byte record per point, read once (row 1 of SURVEY 8(a)), so the record stream is the only
// HBM traffic of the render and the kernel must keep enough bytes in flight to cover HBM latency: Little's law
// at 6.5 TB/s x ~1 us is ~6.5 MB, i.e. ~44 KB per SM.  A thread that loads its own record and then works on it
// holds 16 bytes in flight, and the r01j capture showed exactly that: 28 % issue-active, 47 long-scoreboard
// stall cycles per issue.  Here the stream is moved by the copy engine of each SM instead:
//
//   one elected thread per CTA issues cp.async.bulk (1-D TMA: global -> shared, completion counted in bytes on
//   an mbarrier, L2 evict-first hint so the stream does not push the image out of L2) for chunks of
//   kCloudChunk records into a ring of kCloudStages shared-memory stages; all threads wait on the stage's
//   mbarrier, take their records with conflict-free LDS.128, run chain -> bounds -> pixel -> reduction on
//   kCloudChunk / kCloudThreads independent records each, and a CTA barrier hands the stage back for the
//   refill.  Two CTAs per SM, so one CTA's barrier is hidden behind the other's arithmetic; with 3 stages of 32 KB
//   that is 128 KB in flight per SM.
//
// What the stream cannot hide is the splat itself: one L2 reduction per record, and the L2 executes ~190 G of
// them per second -- 2^24 records need >= 87 us there against 41 us for the 268 MB of records at the measured
// HBM rate (DESIGN "rooflines").
#pragma once
#include "cfs_render.cuh"

namespace cfs {

// launch shape: measured flat on configs[3] (151.6 - 160.8 us over 128..1024 threads x 8..1 CTAs per SM, chunks of
// 512..4096 records, 2..6 stages): the render is bound by the L2 slices, not by the shape of the stream
constexpr int kCloudThreads = 512;
constexpr int kCloudCtasPerSm = 2;
constexpr uint32_t kCloudChunk = 2048;      // records per stage (32 KB)
constexpr int kCloudStages = 3;
constexpr uint32_t kCloudSmemBytes = (uint32_t)kCloudStages * kCloudChunk * 16u;

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}"
        :: "r"(bar), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared::cta of this CTA, bytes a multiple of 16, completion on `bar`
__device__ __forceinline__ void bulk_load(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar, uint64_t policy)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy) : "memory");
}

// SPLAT: SPLAT_HIST_DIRECT, SPLAT_RGBA or SPLAT_DEPTH (the direct sinks; the other variants of a cloud render run
// on render_kernel<GEN = 1>)
template <int DIM, int SPLAT, uint32_t SIG, int TRIG, int OPT>
__global__ void __launch_bounds__(kCloudThreads, kCloudCtasPerSm)
cloud_kernel(const __grid_constant__ RenderParams prm)
{
    extern __shared__ __align__(128) uint32_t s_dyn[];        // the ring: kCloudStages x kCloudChunk records
    __shared__ __align__(8) unsigned long long s_bar[kCloudStages];
    const uint32_t ring = (uint32_t)__cvta_generic_to_shared(s_dyn);
    const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(s_bar);
    // a cloud render has no generator tables: the reference only keeps the signature of the shared splat code
    // (the direct sinks of a GEN = 1 render never touch it)
    const SharedTables &s = *reinterpret_cast<const SharedTables *>(s_dyn);

    const uint64_t n_chunks = (prm.n_points + kCloudChunk - 1) / kCloudChunk;
    const float4 *cloud = reinterpret_cast<const float4 *>(prm.cloud) + (prm.point_offset - prm.cloud_base);
    uint64_t policy = 0;
    auto chunk_bytes = [&](uint64_t c) -> uint32_t {
        const uint64_t left = prm.n_points - c * kCloudChunk;
        return (uint32_t)(left < kCloudChunk ? left : kCloudChunk) * 16u;
    };
    if (threadIdx.x == 0) {
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
#pragma unroll
        for (int st = 0; st < kCloudStages; ++st) mbar_init(bar0 + 8u * st, 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
        for (int st = 0; st < kCloudStages; ++st) {            // prologue: fill the ring
            const uint64_t c = (uint64_t)blockIdx.x + (uint64_t)st * gridDim.x;
            if (c < n_chunks) {
                mbar_expect_tx(bar0 + 8u * st, chunk_bytes(c));
                bulk_load(ring + (uint32_t)st * kCloudChunk * 16u, cloud + c * kCloudChunk, chunk_bytes(c), bar0 + 8u * st, policy);
            }
        }
    }
    __syncthreads();
    const Sm sm = {0u, ring, 0u};
    const BinRegs br = {};

    uint32_t n_in = 0, n_drop = 0;
    uint32_t stage = 0, parity = 0;
    for (uint64_t c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        mbar_wait(bar0 + 8u * stage, parity);
        const uint32_t n_rec = chunk_bytes(c) >> 4;
        CFS_CHECK(stage < (uint32_t)kCloudStages && n_rec >= 1u && n_rec <= kCloudChunk);
        const uint32_t base = ring + stage * kCloudChunk * 16u;
        const uint64_t p0 = prm.point_offset + c * kCloudChunk;
        constexpr int kPer = kCloudChunk / kCloudThreads;      // independent records per thread: the ILP of the chain
        float4 rec[kPer];
#pragma unroll
        for (int j = 0; j < kPer; ++j) rec[j] = lds_v4(base + 16u * (threadIdx.x + (uint32_t)j * kCloudThreads));
#pragma unroll
        for (int j = 0; j < kPer; ++j) {
            const uint32_t r = threadIdx.x + (uint32_t)j * kCloudThreads;
            const bool have = r < n_rec;
            const uint64_t p = p0 + r;
            float gx = rec[j].x, gy = rec[j].y, gz = (DIM == 3) ? rec[j].z : 0.0f;
            const uint32_t dropped = chain_and_splat<DIM, 1, SPLAT, SIG, TRIG, OPT>(prm, s, sm, s_dyn, gx, gy, gz, 0, __float_as_uint(rec[j].w), have, true, br,
                                                                                StepCtx{(uint32_t)p, (uint32_t)(p >> 32), 0});
            if (have) { n_drop += dropped; n_in += (uint32_t)prm.n_branches - dropped; }
        }
        __syncthreads();                                        // every thread has its records of this stage in registers
        if (threadIdx.x == 0) {
            const uint64_t cn = c + (uint64_t)kCloudStages * gridDim.x;
            if (cn < n_chunks) {
                mbar_expect_tx(bar0 + 8u * stage, chunk_bytes(cn));
                bulk_load(base, cloud + cn * kCloudChunk, chunk_bytes(cn), bar0 + 8u * stage, policy);
            }
        }
        if (++stage == kCloudStages) { stage = 0; parity ^= 1u; }
    }

    if (prm.counters) {
        __shared__ unsigned long long s_cnt[2][32];
        unsigned long long a = n_in, b = n_drop;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_xor_sync(0xFFFFFFFFu, a, o);
            b += __shfl_xor_sync(0xFFFFFFFFu, b, o);
        }
        if ((threadIdx.x & 31) == 0) { s_cnt[0][threadIdx.x >> 5] = a; s_cnt[1][threadIdx.x >> 5] = b; }
        __syncthreads();
        if (threadIdx.x < 2) {
            unsigned long long v = 0;
            for (int i = 0; i < (int)(blockDim.x >> 5); ++i) v += s_cnt[threadIdx.x][i];
            if (v) atomicAdd(prm.counters + threadIdx.x, v);
        }
    }
}

}  // namespace cfs
