// cfs_render.cuh -- the fused sampler + pick + map + chain + colour + splat kernel (sm_100a).
//
// One thread owns one point at a time ("a single point chooses a single function at
// random every step"); the per-thread state is 3 floats of generator state, 3 of the copy and 4
// Philox words ("less than ten floating-point values stored per thread").
// Nothing but the output image is written to global memory.
//
// Template axes: DIM 2|3, GEN 0 = IFS / 1 = stored cloud, AFF table form, SPLAT sink, SIG chain
// signature (kChainGeneric = interpreter, else the chain is compiled in), TRIG sin/cos evaluation.
#pragma once
#include "cfs_bin.cuh"
#include "cfs_device.cuh"

namespace cfs {

// ---------------------------------------------------------------------------------------------
// splat sinks (row 7).  `pix >= 0` is guaranteed by the caller.
__device__ __forceinline__ void red_add_v4_f32(float *addr, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};"
                 :: "l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

__device__ __forceinline__ void red_add_u32(uint32_t *addr, uint32_t v)
{
    asm volatile("red.global.add.u32 [%0], %1;" :: "l"(addr), "r"(v) : "memory");
}

// cluster histogram: bin `pix` lives in the shared memory of CTA rank pix >> slice_shift of this
// cluster; one remote shared-memory reduction through DSMEM, no L2 traffic
__device__ __forceinline__ void splat_hist_cluster(uint32_t s_hist_addr, uint32_t slice_shift, int pix)
{
    const uint32_t rank = (uint32_t)pix >> slice_shift;
    const uint32_t local = s_hist_addr + 4u * ((uint32_t)pix & ((1u << slice_shift) - 1u));
    uint32_t remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local), "r"(rank));
    asm volatile("red.relaxed.cluster.shared::cluster.add.u32 [%0], 1;" :: "r"(remote) : "memory");
}

__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release;\n\tbarrier.cluster.wait.acquire;" ::: "memory");
}

__device__ __forceinline__ void splat_hist_warpagg(uint32_t *hist, int pix, bool valid)
{
    // ballot/match aggregation of same-pixel hits before the atomic (BASELINE north_star).
    const unsigned act = __ballot_sync(0xFFFFFFFFu, valid);
    if (!valid) return;
    const unsigned peers = __match_any_sync(act, pix);
    const int leader = __ffs(peers) - 1;
    if ((int)(threadIdx.x & 31) == leader) red_add_u32(hist + pix, (uint32_t)__popc(peers));
}

__device__ __forceinline__ void splat_depth(unsigned long long *buf, int pix, float depth, uint32_t rgba8)
{
    // key = bits(d) << 32 | rgba8; d > 0 so unsigned order = float order (DESIGN R8).
    const unsigned long long key = ((unsigned long long)__float_as_uint(depth) << 32) | rgba8;
    // The buffer only ever decreases, so a stale read can cause a redundant atomic but never a
    // wrong skip; most splats of a solid are occluded and stop at this load.
    const unsigned long long cur = __ldcg(buf + pix);
    if (key < cur) atomicMin(buf + pix, key);
}

template <int DIM, int GEN, int SPLAT, int OPT>
__device__ __forceinline__ uint32_t splat_q(const RenderParams &prm, const SharedTables &s, const Sm &sm, uint32_t *s_hist,
                                            float qx, float qy, float qz, bool alive, int k, uint32_t point_rgba8,
                                            bool have, const BinRegs &br, bool bin_direct_half);

// one branch of a compiled one-to-many chain, then the branches after it: every branch gets its own
// copy of the generated point and its own splat; the structure is fixed at compile time
template <int DIM, int GEN, int SPLAT, uint32_t SIG, int TRIG, int OPT, int M>
__device__ __forceinline__ uint32_t branches_static(const RenderParams &prm, const SharedTables &s, const Sm &sm, uint32_t *s_hist,
                                                    float gx, float gy, float gz, int k, uint32_t point_rgba8, bool have,
                                                    const BinRegs &br, const StepCtx &ctx, bool bin_direct_half)
{
    float qx = gx, qy = gy, qz = gz;
    const bool alive = chain_static<DIM, SIG, TRIG, M, OPT>(prm, ctx, qx, qy, qz);
    uint32_t dropped = splat_q<DIM, GEN, SPLAT, OPT>(prm, s, sm, s_hist, qx, qy, qz, alive, k, point_rgba8, have, br, bin_direct_half);
    constexpr int next = sig_next_branch(SIG, M);
    if constexpr (next >= 0)
        dropped += branches_static<DIM, GEN, SPLAT, SIG, TRIG, OPT, next>(prm, s, sm, s_hist, gx, gy, gz, k, point_rgba8, have, br, ctx, bin_direct_half);
    return dropped;
}

// rows 5-7 for one generated point: copy -> chain -> pixel -> reduction.  `k` is the map applied
// in this iteration (colour rule MAP_INDEX), `point_rgba8` the record colour (POINT).
// Returns the number of dropped splats (dead or out of bounds).  Fig. 2(C) reuse: a run-time option of the
// interpreter (prm.reuse), a compile-time one (OPT_REUSE) of a kernel compiled for the chain.
template <int DIM, int GEN, int SPLAT, uint32_t SIG, int TRIG, int OPT>
__device__ __forceinline__ uint32_t chain_and_splat(const RenderParams &prm, const SharedTables &s, const Sm &sm, uint32_t *s_hist,
                                                    float &gx, float &gy, float &gz, int k, uint32_t point_rgba8,
                                                    bool have, bool past_burn_in, const BinRegs &br, const StepCtx &ctx,
                                                    bool bin_direct_half = false)
{
    if constexpr (SIG != kChainGeneric && sig_has_branch(SIG)) {
        return branches_static<DIM, GEN, SPLAT, SIG, TRIG, OPT, 0>(prm, s, sm, s_hist, gx, gy, gz, k, point_rgba8, have, br, ctx, bin_direct_half);
    }
    if (SIG == kChainGeneric && prm.n_branches > 1) {
        // one-to-many ("many objects from a single primitive"): every BRANCH of the chain
        // gets its own copy of the generated point and its own splat.  The markers sit in the parameter
        // block, so the loop structure is warp-uniform; only dead lanes skip steps.
        float qx = gx, qy = gy, qz = gz;
        bool alive = true;
        uint32_t dropped = 0u;
        for (int m = 0; m <= prm.n_chain; ++m) {
            if (m == prm.n_chain || prm.chain[m].type == T_BRANCH) {
                dropped += splat_q<DIM, GEN, SPLAT, OPT>(prm, s, sm, s_hist, qx, qy, qz, alive, k, point_rgba8, have, br, bin_direct_half);
                qx = gx; qy = gy; qz = gz; alive = true;
            } else if (alive) {
                alive = chain_step_dyn<DIM, TRIG>(prm, prm.chain[m], ctx, qx, qy, qz);
            }
        }
        return dropped;
    }
    float qx = gx, qy = gy, qz = gz;            // the copy of Fig. 2(B)
    const bool alive = apply_chain<DIM, SIG, TRIG, OPT>(prm, ctx, qx, qy, qz);
    if ((SIG == kChainGeneric) ? (prm.reuse != 0) : ((OPT & OPT_REUSE) != 0)) {    // Fig. 2(C): the same point is reused
        gx = qx; gy = qy; gz = qz;
        if (!past_burn_in) return 0u;
    }
    return splat_q<DIM, GEN, SPLAT, OPT>(prm, s, sm, s_hist, qx, qy, qz, alive, k, point_rgba8, have, br, bin_direct_half);
}

// rows 6-7 for one chain output: bounds -> pixel -> reduction.  Returns 1 when the splat was dropped.
template <int DIM, int GEN, int SPLAT, int OPT>
__device__ __forceinline__ uint32_t splat_q(const RenderParams &prm, const SharedTables &s, const Sm &sm, uint32_t *s_hist,
                                            float qx, float qy, float qz, bool alive, int k, uint32_t point_rgba8,
                                            bool have, const BinRegs &br, bool bin_direct_half)
{
    const bool ok = alive && have && in_bounds<OPT>(prm, qx, qy);
    if (SPLAT == SPLAT_HIST_WARPAGG) {
        splat_hist_warpagg(reinterpret_cast<uint32_t *>(prm.image), ok ? pixel_of(prm, qx, qy) : -1, ok);
        return (have && !ok) ? 1u : 0u;
    }
    if (!ok) return 1u;
    if (SPLAT == SPLAT_DEPTH_HIZ) {
        // Hi-Z pre-test in shared memory: a splat whose depth bits exceed the block's upper bound is
        // certainly occluded (the bound comes from a snapshot of an image that only decreases), so
        // it never leaves the SM.  ~95 % of the splats of a solid stop here (DESIGN "Hi-Z variant").
        uint32_t px, py;
        pixel_xy(prm, qx, qy, px, py);
        CFS_CHECK((py >> prm.hiz.shift) * prm.hiz.nbx + (px >> prm.hiz.shift) < prm.hiz.nbx * prm.hiz.nby);
        const uint32_t bound = lds_u16(sm.dyn + 2u * ((py >> prm.hiz.shift) * prm.hiz.nbx + (px >> prm.hiz.shift)));
        if ((__float_as_uint(qz) >> 16) > bound) return 0u;
        splat_depth(reinterpret_cast<unsigned long long *>(prm.image), (int)(py * (uint32_t)prm.W + px), qz,
                    lds_u32(sm.tab + CFS_SM_OFF(pal8) + 4u * (uint32_t)k));
        return 0u;
    }
    const int pix = (SPLAT == SPLAT_BIN) ? bin_pixel_of(br, qx, qy) : pixel_of<OPT>(prm, qx, qy);
    CFS_CHECK((uint32_t)pix < (uint32_t)prm.W * (uint32_t)prm.H);
    if (SPLAT == SPLAT_HIST_DIRECT) {
        red_add_u32(reinterpret_cast<uint32_t *>(prm.image) + pix, 1u);
    } else if (SPLAT == SPLAT_HIST_SHARED) {
        atomicAdd(&s_hist[pix], 1u);
    } else if (SPLAT == SPLAT_HIST_CLUSTER) {
        splat_hist_cluster((uint32_t)__cvta_generic_to_shared(s_hist), prm.slice_shift, pix);
    } else if (SPLAT == SPLAT_RGBA) {
        float *dst = reinterpret_cast<float *>(prm.image) + 4 * (size_t)pix;
        if (GEN == 1) {   // colour of the point record, integer-valued (DESIGN R9)
            red_add_v4_f32(dst, (float)(point_rgba8 & 0xFFu), (float)((point_rgba8 >> 8) & 0xFFu),
                           (float)((point_rgba8 >> 16) & 0xFFu), 1.0f);
        } else {          // colour of the map applied in this iteration
            const float4 c = lds_v4(sm.tab + CFS_SM_OFF(palette) + 16u * (uint32_t)k);
            red_add_v4_f32(dst, c.x, c.y, c.z, c.w);                    // c.w = 1 (load_tables)
        }
    } else if (SPLAT == SPLAT_DEPTH) {
        splat_depth(reinterpret_cast<unsigned long long *>(prm.image), pix, qz,
                    GEN == 1 ? point_rgba8 : lds_u32(sm.tab + CFS_SM_OFF(pal8) + 4u * (uint32_t)k));
    } else if (SPLAT == SPLAT_BIN) {
        if (bin_direct_half) {      // hybrid stage on the interpreter path: this iteration's splat goes straight to L2 (warp-uniform)
            if (prm.color_rule == 0) {
                red_add_u32(reinterpret_cast<uint32_t *>(prm.image) + pix, 1u);
            } else {
                const float4 c = lds_v4(sm.tab + CFS_SM_OFF(palette) + 16u * (uint32_t)k);
                red_add_v4_f32(reinterpret_cast<float *>(prm.image) + 4 * (size_t)pix, c.x, c.y, c.z, c.w);
            }
        } else {
            bin_append(prm, s, br, pix, k);
        }
    }
    return 0u;
}

// rows 6-7 of the four iterations of one steady-state Philox block, binned.  HYBRID: iterations 0
// and 2 of the block splat straight to L2 (red.global), 1 and 3 go through the tile bins -- pass 1 is
// bound by instruction issue and pass 2 by shared-memory atomics while the L2 reduction units would
// idle, so half of the splats are given to them (a direct splat costs ~5 instructions against ~11
// for record + append, and pass 2 halves).  Any split is a correct result: HIST sums are exact,
// RGBA sums are order-free (DESIGN R8).  Straight-line code: every reduction, atomic and store is predicated.
// Returns the number of dropped splats.
template <int DIRECT_MASK, bool RGBA, bool UNCLAMPED = false, bool ALL_HAVE = false>
__device__ __forceinline__ uint32_t bin_block_splat(const RenderParams &prm, const SharedTables &s, const Sm &sm, const BinRegs &br,
                                                    const float (&X)[4], const float (&Y)[4], const int (&K)[4],
                                                    const bool (&ok)[4])
{
    // In stages, so that the shared-memory atomics of the block are in flight TOGETHER: as one loop (record ->
    // atomic -> store per splat) every store waited for its own atomic in turn, 7 % of the stall samples of pass 1
    // (short scoreboard at the slot compare, profiles/r02 source view).  The asm statements are volatile, so their
    // order here is their order in the kernel: reductions, then the atomics, then the stores.
    // UNCLAMPED = OPT_NO_DROP: `ok` is `have` (nothing to count: the caller counts a thread without a point as
    // nothing); ALL_HAVE: every thread has a point, so `ok` is true and every predicate below folds away.
    int pix[4];
    uint32_t tile[4] = {0u, 0u, 0u, 0u}, rec[4] = {0u, 0u, 0u, 0u}, slot[4] = {0u, 0u, 0u, 0u};
    uint32_t dropped = 0u;
#pragma unroll
    for (int j = 0; j < 4; ++j) {      // out-of-bounds coordinates are clamped by the pixel rule: always a valid tile
        pix[j] = bin_pixel_of<UNCLAMPED>(br, X[j], Y[j]);
        CFS_CHECK((uint32_t)pix[j] < (uint32_t)prm.W * (uint32_t)prm.H);
        CFS_CHECK(!ALL_HAVE || ok[j]);
        if (!UNCLAMPED && !ok[j]) ++dropped;   // counted here, so that no `ok` outlives its splat
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (!((DIRECT_MASK >> j) & 1)) continue;   // straight to L2: one predicated reduction, no branch
        if (RGBA) {
            const float4 c = lds_v4(sm.tab + CFS_SM_OFF(palette) + 16u * (uint32_t)K[j]);     // (r, g, b, 1): load_tables
            float *dst = reinterpret_cast<float *>(prm.image) + 4 * (size_t)(uint32_t)pix[j];
            if (ALL_HAVE)
                asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" :: "l"(dst), "f"(c.x), "f"(c.y), "f"(c.z), "f"(c.w) : "memory");
            else
                asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %5, 0;\n\t"
                             "@p red.global.add.v4.f32 [%0], {%1, %2, %3, %4};\n\t}"
                             :: "l"(dst), "f"(c.x), "f"(c.y), "f"(c.z), "f"(c.w), "r"((uint32_t)ok[j]) : "memory");
        } else {
            uint32_t *dst = reinterpret_cast<uint32_t *>(prm.image) + (uint32_t)pix[j];
            if (ALL_HAVE)
                asm volatile("red.global.add.u32 [%0], 1;" :: "l"(dst) : "memory");
            else
                asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %1, 0;\n\t@p red.global.add.u32 [%0], 1;\n\t}"
                             :: "l"(dst), "r"((uint32_t)ok[j]) : "memory");
        }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {      // a slot in the staging row of the tile (a dropped splat: in the lane's dummy row, "full")
        if ((DIRECT_MASK >> j) & 1) continue;
        bin_record_of(br, pix[j], RGBA ? K[j] : 0, tile[j], rec[j]);
        slot[j] = bin_take_slot(br, ALL_HAVE || ok[j], tile[j], rec[j]);
    }
    bool fine = true;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if ((DIRECT_MASK >> j) & 1) continue;
        fine &= bin_store_record(br, tile[j], rec[j], slot[j]);
    }
    if (!fine) {   // a staging row was full (or a splat was dropped): live records go straight to L2 -- the pixel and the
                   // colour index are still in registers, so an overflow costs one reduction, not a division (rows of hot
                   // tiles may overflow now and then: that is what lets the drain interval be long)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (((DIRECT_MASK >> j) & 1) || slot[j] < br.cap || !ok[j]) continue;
            if (RGBA && br.ktp != 0u) {      // (the run-time test: kernels linked ahead of time run HIST renders through the RGBA body, ktp = 0)
                const float4 c = lds_v4(sm.tab + CFS_SM_OFF(palette) + 16u * (uint32_t)K[j]);
                bin_red_add_v4_f32(reinterpret_cast<float *>(prm.image) + 4 * (size_t)(uint32_t)pix[j], c.x, c.y, c.z, c.w);
            } else {
                bin_red_add_u32(reinterpret_cast<uint32_t *>(prm.image) + (uint32_t)pix[j], 1u);
            }
        }
    }
    return dropped;
}

// four iterations served by one Philox block (DESIGN R1: word it & 3 of block it >> 2).
// CHECKED = false: the caller guarantees burn_in <= it0 and it0 + 4 <= iterations, so the body
// has no per-iteration tests (the steady state of a render); CHECKED = true handles burn-in
// and the ragged last block.
template <int DIM, int GEN, int AFF, int SPLAT, uint32_t SIG, int TRIG, int OPT, bool CHECKED>
__device__ __forceinline__ uint32_t iterate_block(const RenderParams &prm, const SharedTables &s, const Sm &sm, uint32_t *s_hist,
                                                  uint32_t plo, uint32_t phi, int it0, float &gx, float &gy, float &gz,
                                                  bool have, BinLane &bl, const BinRegs &br)
{
    const U4 w = philox4x32_10(plo, phi, (uint32_t)it0 >> 2, DOMAIN_PICK, prm);
    uint32_t dropped = 0;
    constexpr bool kReuse = (SIG != kChainGeneric) && (OPT & OPT_REUSE) != 0;
    if constexpr (!CHECKED && SIG != kChainGeneric && SPLAT == SPLAT_BIN && !sig_has_branch(SIG) && !kReuse) {
        // ALU-bound variant: the generator recurrence is short (LDS + FMAs), the chain and pixel
        // arithmetic of the four iterations are independent of one another once the four generator
        // states exist -- written as straight-line stages so that the four dependent chains
        // (LDS -> FMA -> MUFU -> FMA -> F2I -> ATOMS) can interleave.  (The same staging of the four
        // depth-buffer loads of SPLAT_DEPTH was measured slower, 324 vs 309 ms on configs[4]: that
        // path is bound by the SM-to-L2 request rate, not by load latency.)
        float X[4], Y[4], Z[4];
        int K[4];
        bool ok[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t u = (j == 0) ? w.x : (j == 1) ? w.y : (j == 2) ? w.z : w.w;
            K[j] = pick_index<OPT>(u, sm, prm);
            apply_gen<DIM, AFF>(K[j], sm, prm, gx, gy, gz);
            X[j] = gx; Y[j] = gy; Z[j] = gz;                 // the copies of Fig. 2(B)
        }
        // a thread without a point carries NaN coordinates (render_kernel), which fail every bounds test: no `have` here
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const bool alive = apply_chain<DIM, SIG, TRIG, OPT>(prm, StepCtx{plo, phi, it0 + j}, X[j], Y[j], Z[j]);
            if constexpr ((OPT & OPT_NO_DROP) != 0) {
                // the host has proved every splat alive and in bounds: only a thread without a point (NaN) holds back
                CFS_CHECK(!have || bin_in_bounds<false>(br, X[j], Y[j]));
                CFS_CHECK((OPT & OPT_ALL_HAVE) == 0 || have);
                ok[j] = have;
            } else {
                ok[j] = alive && bin_in_bounds<(OPT & OPT_SYM_BOUNDS) != 0>(br, X[j], Y[j]);
            }
        }
        if constexpr ((OPT & OPT_BIN_FIXED) != 0) {
            // compiled for this render's split and output: one straight-line body
            dropped += bin_block_splat<(OPT >> OPT_BIN_MASK_SHIFT) & 15, (OPT & OPT_BIN_RGBA) != 0, (OPT & OPT_NO_DROP) != 0,
                                       (OPT & OPT_NO_DROP) != 0 && (OPT & OPT_ALL_HAVE) != 0>(prm, s, sm, br, X, Y, K, ok);
        } else {
            // warp-uniform choice of one of three straight-line bodies (hybrid RGBA / hybrid HIST / pure bins); any
            // non-zero mask runs as "every other splat" here -- the exact mask is a compiled-in option
            if (prm.bin.hybrid) {
                if (prm.color_rule != 0) dropped += bin_block_splat<5, true>(prm, s, sm, br, X, Y, K, ok);
                else                     dropped += bin_block_splat<5, false>(prm, s, sm, br, X, Y, K, ok);
            } else {
                dropped += bin_block_splat<0, true>(prm, s, sm, br, X, Y, K, ok);    // br.ktp = 0 for HIST: k is ignored
            }
        }
    } else if constexpr (!CHECKED && SIG != kChainGeneric && SPLAT == SPLAT_DEPTH_HIZ && !sig_has_branch(SIG) && !kReuse) {
        // Hi-Z depth splats of a steady-state block in stages: the four chains, bounds tests and Hi-Z tests first, then the
        // pre-test loads of the survivors back to back, then the compares -- one exposed L2 latency per block instead
        // of four (the render is bound by instruction issue, and the sequential form spent a quarter of its stall
        // samples waiting for each load in turn: profiles/r02c).
        float X[4], Y[4], Z[4];
        int K[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t u = (j == 0) ? w.x : (j == 1) ? w.y : (j == 2) ? w.z : w.w;
            K[j] = pick_index<OPT>(u, sm, prm);
            apply_gen<DIM, AFF>(K[j], sm, prm, gx, gy, gz);
            X[j] = gx; Y[j] = gy; Z[j] = gz;                 // the copies of Fig. 2(B)
        }
        unsigned long long *buf = reinterpret_cast<unsigned long long *>(prm.image);
        uint32_t pix[4];
        bool sv[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const bool alive = apply_chain<DIM, SIG, TRIG, OPT>(prm, StepCtx{plo, phi, it0 + j}, X[j], Y[j], Z[j]);
            const bool ok = alive && in_bounds<OPT>(prm, X[j], Y[j]);
            if (!ok) ++dropped;
            uint32_t px, py;
            pixel_xy<OPT>(prm, X[j], Y[j], px, py);          // clamped (or proved inside): a valid pixel and block even for a dropped splat
            CFS_CHECK((py >> prm.hiz.shift) * prm.hiz.nbx + (px >> prm.hiz.shift) < prm.hiz.nbx * prm.hiz.nby);
            const uint32_t bound = lds_u16(sm.dyn + 2u * ((py >> prm.hiz.shift) * prm.hiz.nbx + (px >> prm.hiz.shift)));
            sv[j] = ok && !((__float_as_uint(Z[j]) >> 16) > bound);
            pix[j] = py * (uint32_t)prm.W + px;
        }
        unsigned long long cur[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {                        // the survivors' pre-test loads, all in flight together
            cur[j] = 0ull;
            if (sv[j]) cur[j] = __ldcg(buf + pix[j]);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            // cur = 0 where no load was issued, and a live splat's depth bits are > 0 (d > near >= 0): under OPT_NO_DROP
            // (every splat proved alive) the depth compare alone tells a candidate, without re-testing `sv`
            CFS_CHECK((OPT & OPT_NO_DROP) == 0 || __float_as_uint(Z[j]) > 0u);
            if (((OPT & OPT_NO_DROP) != 0 || sv[j]) && __float_as_uint(Z[j]) <= (uint32_t)(cur[j] >> 32)) {      // else the key is larger whatever its colour
                const unsigned long long key = ((unsigned long long)__float_as_uint(Z[j]) << 32) | lds_u32(sm.tab + CFS_SM_OFF(pal8) + 4u * (uint32_t)K[j]);
                if (key < cur[j]) atomicMin(buf + pix[j], key);
            }
        }
    } else {
#pragma unroll(CHECKED ? 1 : 4)
        for (int j = 0; j < 4; ++j) {
            const int it = it0 + j;
            if (CHECKED && it >= prm.iterations) break;
            const uint32_t u = (j == 0) ? w.x : (j == 1) ? w.y : (j == 2) ? w.z : w.w;
            const int k = pick_index<OPT>(u, sm, prm);
            apply_gen<DIM, AFF>(k, sm, prm, gx, gy, gz);
            const bool past = !CHECKED || it >= prm.burn_in;
            // hybrid stage (DESIGN "hybrid"): iterations 0 and 2 of a steady-state block splat straight to L2
            const bool direct_half = SPLAT == SPLAT_BIN && !CHECKED && ((prm.bin.hybrid >> j) & 1u) != 0u;
            if (past || (SIG == kChainGeneric && prm.reuse) || kReuse)
                dropped += chain_and_splat<DIM, GEN, SPLAT, SIG, TRIG, OPT>(prm, s, sm, s_hist, gx, gy, gz, k, 0u, have, past, br,
                                                                       StepCtx{plo, phi, it}, direct_half);
        }
    }
    // the staging rows of SPLAT_BIN are drained by the caller, between runs of blocks (render_kernel): a run then is a
    // loop of its own whose invariants -- the Philox round keys above all -- stay in uniform registers
    return dropped;
}

// ---------------------------------------------------------------------------------------------
// the kernel
template <int DIM, int GEN, int AFF, int SPLAT, uint32_t SIG, int TRIG, int OPT>
__global__ void __launch_bounds__(SPLAT == SPLAT_BIN ? kBinThreads : SPLAT == SPLAT_HIST_CLUSTER ? kClusterThreads :
                                  SPLAT == SPLAT_DEPTH_HIZ ? kHizThreads : kRenderThreads,
                                  SPLAT == SPLAT_BIN ? kBinCtasPerSm : SPLAT == SPLAT_DEPTH_HIZ ? kHizCtasPerSm : 0)
render_kernel(const __grid_constant__ RenderParams prm)
{
    __shared__ SharedTables s;
    extern __shared__ __align__(16) uint32_t s_hist[];   // SPLAT_HIST_SHARED: histogram; SPLAT_BIN: staging
    CFS_CHECK_ENTRY();
    if (GEN == 0) load_tables(s, prm);
    if (SPLAT == SPLAT_HIST_SHARED)
        for (uint32_t i = threadIdx.x; i < prm.hist_bins; i += blockDim.x) s_hist[i] = 0u;
    if (SPLAT == SPLAT_HIST_CLUSTER) {   // this CTA's slice; nobody may touch a peer's slice before it is cleared
        for (uint32_t i = threadIdx.x; i < (1u << prm.slice_shift); i += blockDim.x) s_hist[i] = 0u;
        cluster_sync_all();
    }
    if (SPLAT == SPLAT_DEPTH_HIZ) {      // the Hi-Z map of this render phase: 16-byte vectors, L2 -> shared memory
        const uint4 *src = reinterpret_cast<const uint4 *>(prm.hiz.hz);
        uint4 *dst = reinterpret_cast<uint4 *>(s_hist);
        for (uint32_t i = threadIdx.x; i < prm.hiz.n_pad / 8u; i += blockDim.x) dst[i] = __ldcg(src + i);
    }
    __shared__ Sm s_sm;
    sm_publish(&s_sm, s, s_hist);
    BinLane bl = {0u, 0u, 0u};
    BinRegs br = {};
    __shared__ BinRegs s_br;
    if (SPLAT == SPLAT_BIN) {
        // through shared memory on purpose: values read back from memory stay in registers for the
        // whole kernel, whereas values derived from the parameter block are re-derived (constant
        // loads + shifts) at every use, ~10 extra instructions per splat
        if (threadIdx.x == 0) s_br = bin_regs_init(prm, s_hist);   // the staging rows; this lane's tile state
        for (uint32_t i = threadIdx.x; i < prm.bin.n_tiles + kBinDummy; i += blockDim.x)
            s_hist[i] = (i < prm.bin.n_tiles) ? 0u : prm.bin.cap;   // fill counters; the dummy ones read "full"
        bin_lane_init(prm, bl);
    }
    __syncthreads();
    if (SPLAT == SPLAT_BIN) { br = s_br; br.dummy += threadIdx.x & 31u; }
    const Sm sm = sm_read(&s_sm, prm);

    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const int I = prm.iterations, B = prm.burn_in;
    const int it_fast0 = min((B + 3) & ~3, I & ~3), it_fast1 = I & ~3;   // steady-state Philox blocks: [it_fast0, it_fast1)
    uint32_t n_in = 0, n_drop = 0;
    int until = (SPLAT == SPLAT_BIN) ? (int)prm.bin.check_every : 0;

    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; ; i += stride) {
        // SPLAT_HIST_WARPAGG uses full-warp collectives inside: keep whole warps in the loop
        const bool have = i < prm.n_points;
        if (SPLAT == SPLAT_HIST_WARPAGG) { if (!__any_sync(0xFFFFFFFFu, have)) break; }
        else if (SPLAT == SPLAT_BIN) { if (i - threadIdx.x >= prm.n_points) break; }   // whole CTAs: barriers inside
        else if (!have) break;
        const uint64_t p = prm.point_offset + i;
        float gx, gy, gz = 0.0f;
        uint32_t dropped = 0;

        if (GEN == 1) {   // stored cloud: one coalesced 128-bit load per point (row 1), one splat
            float4 rec = make_float4(0.f, 0.f, 0.f, 0.f);
            if (have) rec = __ldcs(reinterpret_cast<const float4 *>(prm.cloud) + (p - prm.cloud_base));
            gx = rec.x; gy = rec.y; gz = (DIM == 3) ? rec.z : 0.0f;
            dropped = chain_and_splat<DIM, GEN, SPLAT, SIG, TRIG, OPT>(prm, s, sm, s_hist, gx, gy, gz, 0,
                                                                  __float_as_uint(rec.w), have, true, br,
                                                                  StepCtx{(uint32_t)p, (uint32_t)(p >> 32), 0});
        } else {
            const uint32_t plo = (uint32_t)p, phi = (uint32_t)(p >> 32);
            {
                const U4 w = philox4x32_10(plo, phi, 0u, DOMAIN_INIT, prm);
                gx = u24_to_pm1(w.x);
                gy = u24_to_pm1(w.y);
                if (DIM == 3) gz = u24_to_pm1(w.z);
                // SPLAT_BIN keeps whole CTAs in the loop (barriers inside): a thread without a point carries NaN, which
                // every map hands on and every bounds test rejects -- no `have` predicate in the steady-state body
                if (SPLAT == SPLAT_BIN && !have) gx = __int_as_float(0x7FC00000);
            }
            // blocks touching burn-in or the ragged end take the checked path, the rest the lean one
            int it0 = 0;
            if (SPLAT == SPLAT_BIN) {
                // every thread of the CTA is at the same it0 (whole CTAs in the loop), so `until` -- Philox blocks left
                // before the staging rows are drained, counted across the points a thread renders -- is CTA-uniform
#pragma unroll 1
                for (; it0 < it_fast0; it0 += 4) {
                    dropped += iterate_block<DIM, GEN, AFF, SPLAT, SIG, TRIG, OPT, true>(prm, s, sm, s_hist, plo, phi, it0, gx, gy, gz, have, bl, br);
                    if (--until == 0) { bin_fence_async(); __syncthreads(); bin_drain(prm, s, br, bl, false); __syncthreads(); until = (int)prm.bin.check_every; }
                }
#pragma unroll 1
                while (it0 < it_fast1) {                   // runs of steady-state blocks up to the next drain
                    const int run = min((it_fast1 - it0) >> 2, until);
                    const int stop = it0 + 4 * run;
#pragma unroll 1
                    for (; it0 < stop; it0 += 4)
                        dropped += iterate_block<DIM, GEN, AFF, SPLAT, SIG, TRIG, OPT, false>(prm, s, sm, s_hist, plo, phi, it0, gx, gy, gz, have, bl, br);
                    until -= run;
                    if (until == 0) { bin_fence_async(); __syncthreads(); bin_drain(prm, s, br, bl, false); __syncthreads(); until = (int)prm.bin.check_every; }
                }
#pragma unroll 1
                for (; it0 < I; it0 += 4) {
                    dropped += iterate_block<DIM, GEN, AFF, SPLAT, SIG, TRIG, OPT, true>(prm, s, sm, s_hist, plo, phi, it0, gx, gy, gz, have, bl, br);
                    if (--until == 0) { bin_fence_async(); __syncthreads(); bin_drain(prm, s, br, bl, false); __syncthreads(); until = (int)prm.bin.check_every; }
                }
            } else {
#pragma unroll 1
                for (; it0 < it_fast0; it0 += 4)
                    dropped += iterate_block<DIM, GEN, AFF, SPLAT, SIG, TRIG, OPT, true>(prm, s, sm, s_hist, plo, phi, it0, gx, gy, gz, have, bl, br);
#pragma unroll 1
                for (; it0 < it_fast1; it0 += 4)
                    dropped += iterate_block<DIM, GEN, AFF, SPLAT, SIG, TRIG, OPT, false>(prm, s, sm, s_hist, plo, phi, it0, gx, gy, gz, have, bl, br);
#pragma unroll 1
                for (; it0 < I; it0 += 4)
                    dropped += iterate_block<DIM, GEN, AFF, SPLAT, SIG, TRIG, OPT, true>(prm, s, sm, s_hist, plo, phi, it0, gx, gy, gz, have, bl, br);
            }
        }
        if (have) { n_drop += dropped; n_in += (uint32_t)(I - B) * (uint32_t)prm.n_branches - dropped; }
    }

    if (SPLAT == SPLAT_BIN) {           // write out what is left in the staging rows
        bin_fence_async();
        __syncthreads();
        bin_drain(prm, s, br, bl, true);
    }
    if (SPLAT == SPLAT_HIST_CLUSTER) {  // all peers done with my slice, then merge it (red.global, non-zero bins)
        cluster_sync_all();
        uint32_t rank;
        asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
        uint32_t *hist = reinterpret_cast<uint32_t *>(prm.image);
        const uint32_t base = rank << prm.slice_shift;
        for (uint32_t i = threadIdx.x; i < (1u << prm.slice_shift) && base + i < prm.hist_bins; i += blockDim.x) {
            const uint32_t v = s_hist[i];
            if (v) red_add_u32(hist + base + i, v);
        }
    }
    if (SPLAT == SPLAT_HIST_SHARED) {   // merge the private histogram (red.global, non-zero bins only)
        __syncthreads();
        uint32_t *hist = reinterpret_cast<uint32_t *>(prm.image);
        for (uint32_t i = threadIdx.x; i < prm.hist_bins; i += blockDim.x) {
            const uint32_t v = s_hist[i];
            if (v) red_add_u32(hist + i, v);
        }
    }
    if (prm.counters) {   // block-level reduction: two atomics per CTA (same-address L2 atomics serialise)
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

// ---------------------------------------------------------------------------------------------
// parity instrument: same device functions, records instead of splatting (SURVEY 8(c) S10 i, ii)
template <int DIM, int GEN, int AFF, uint32_t SIG, int TRIG>
__global__ void __launch_bounds__(kRenderThreads)
trace_kernel(const __grid_constant__ RenderParams prm)
{
    __shared__ SharedTables s;
    if (GEN == 0) load_tables(s, prm);
    __shared__ Sm s_sm;
    sm_publish(&s_sm, s, &s_sm);
    __syncthreads();
    const Sm sm = sm_read(&s_sm, prm);
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < prm.n_points; i += stride) {
        const uint64_t p = prm.point_offset + i;
        float gx, gy, gz = 0.0f;
        if (GEN == 1) {
            const float4 rec = __ldcs(reinterpret_cast<const float4 *>(prm.cloud) + (p - prm.cloud_base));
            gx = rec.x; gy = rec.y; gz = (DIM == 3) ? rec.z : 0.0f;
        } else {
            const U4 w = philox4x32_10((uint32_t)p, (uint32_t)(p >> 32), 0u, DOMAIN_INIT, prm);
            gx = u24_to_pm1(w.x);
            gy = u24_to_pm1(w.y);
            if (DIM == 3) gz = u24_to_pm1(w.z);
        }
        float qx = 0.f, qy = 0.f, qz = 0.f;
        bool alive = false;
        U4 w = {0, 0, 0, 0};
        for (int it = 0; it < prm.iterations; ++it) {
            if (GEN == 0) {
                if ((it & 3) == 0)
                    w = philox4x32_10((uint32_t)p, (uint32_t)(p >> 32), (uint32_t)it >> 2, DOMAIN_PICK, prm);
                const uint32_t u = w.x;
                w.x = w.y; w.y = w.z; w.z = w.w;
                const int k = pick_index(u, sm, prm);
                if (prm.tr_picks) prm.tr_picks[i * (uint64_t)prm.iterations + it] = (uint8_t)k;
                apply_gen<DIM, AFF>(k, sm, prm, gx, gy, gz);
            }
            if (it < prm.burn_in && !prm.reuse) continue;
            qx = gx; qy = gy; qz = gz;
            alive = apply_chain<DIM, SIG, TRIG>(prm, StepCtx{(uint32_t)p, (uint32_t)(p >> 32), it}, qx, qy, qz);
            if (prm.reuse) { gx = qx; gy = qy; gz = qz; }
        }
        if (prm.tr_g) { prm.tr_g[3 * i] = gx; prm.tr_g[3 * i + 1] = gy; prm.tr_g[3 * i + 2] = gz; }
        if (prm.tr_q) { prm.tr_q[3 * i] = qx; prm.tr_q[3 * i + 1] = qy; prm.tr_q[3 * i + 2] = qz; }
        if (prm.tr_alive) prm.tr_alive[i] = alive ? 1 : 0;
    }
}

}  // namespace cfs
