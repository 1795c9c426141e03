// cfs_select.cuh -- run-time -> compile-time selection helpers shared by the kernel translation units
#pragma once
#include "cfs_registry.h"
#include "cfs_cloud.cuh"
#include "cfs_render.cuh"

namespace cfs {

// SPLATS: bit mask of SplatKind values to instantiate for this (DIM, GEN, AFF, SIG, TRIG)
template <int DIM, int GEN, int AFF, uint32_t SIG, int TRIG, unsigned SPLATS>
render_fn select_splat(int splat)
{
    // a stored cloud with a direct sink streams through cloud_kernel (bulk-async record ring); the host
    // launches it with its own shape (cfs_api.cu is_cloud_stream)
#define CFS_CASE(K)                                                                   \
    if constexpr ((SPLATS >> K) & 1u) {                                               \
        if constexpr (GEN == 1 && (K == SPLAT_HIST_DIRECT || K == SPLAT_RGBA || K == SPLAT_DEPTH)) { \
            if (splat == K) return cloud_kernel<DIM, K, SIG, TRIG, 0>;                   \
        } else {                                                                      \
            if (splat == K) return render_kernel<DIM, GEN, AFF, K, SIG, TRIG, 0>;        \
        }                                                                             \
    }
    CFS_CASE(SPLAT_HIST_DIRECT)
    CFS_CASE(SPLAT_HIST_SHARED)
    CFS_CASE(SPLAT_HIST_WARPAGG)
    if constexpr (GEN == 0) { CFS_CASE(SPLAT_HIST_CLUSTER) }
    CFS_CASE(SPLAT_RGBA)
    if constexpr (DIM == 3) { CFS_CASE(SPLAT_DEPTH) }
    if constexpr (DIM == 3 && GEN == 0) { CFS_CASE(SPLAT_DEPTH_HIZ) }
    if constexpr (GEN == 0) { CFS_CASE(SPLAT_BIN) }
#undef CFS_CASE
    return nullptr;
}

// (gen, aff) -> template arguments; the cloud generator has no affine table (AFF_GENERAL slot)
template <int DIM, uint32_t SIG, int TRIG, unsigned SPLATS>
render_fn select_render(int gen, int aff, int splat)
{
    if (gen == 1) return select_splat<DIM, 1, AFF_GENERAL, SIG, TRIG, SPLATS>(splat);
    if (aff == AFF_CIRCLE) {   // PAPER Eq. 1 generator: 2-D, chain interpreter only (no kernel per signature)
        if constexpr (DIM == 2 && SIG == kChainGeneric) return select_splat<2, 0, AFF_CIRCLE, SIG, TRIG, SPLATS>(splat);
        else return nullptr;
    }
    if (aff == AFF_DIAG) return select_splat<DIM, 0, AFF_DIAG, SIG, TRIG, SPLATS>(splat);
    return select_splat<DIM, 0, AFF_GENERAL, SIG, TRIG, SPLATS>(splat);
}

template <int DIM, uint32_t SIG, int TRIG>
render_fn select_trace(int gen, int aff)
{
    if (gen == 1) return trace_kernel<DIM, 1, AFF_GENERAL, SIG, TRIG>;
    if (aff == AFF_CIRCLE) {
        if constexpr (DIM == 2 && SIG == kChainGeneric) return trace_kernel<2, 0, AFF_CIRCLE, SIG, TRIG>;
        else return nullptr;
    }
    if (aff == AFF_DIAG) return trace_kernel<DIM, 0, AFF_DIAG, SIG, TRIG>;
    return trace_kernel<DIM, 0, AFF_GENERAL, SIG, TRIG>;
}

constexpr unsigned kSplatsAll = (1u << SPLAT_HIST_DIRECT) | (1u << SPLAT_HIST_SHARED) | (1u << SPLAT_HIST_WARPAGG) | (1u << SPLAT_HIST_CLUSTER) |
                                (1u << SPLAT_RGBA) | (1u << SPLAT_DEPTH) | (1u << SPLAT_BIN) | (1u << SPLAT_DEPTH_HIZ);
constexpr unsigned kSplatsDirect = (1u << SPLAT_HIST_DIRECT) | (1u << SPLAT_RGBA) | (1u << SPLAT_DEPTH) | (1u << SPLAT_BIN) | (1u << SPLAT_DEPTH_HIZ);

}  // namespace cfs
