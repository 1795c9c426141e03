// cfs_params.h -- kernel parameter block of the CFS hot path (host fills it, device reads it).
//
// Everything a render needs travels BY VALUE in the launch ("a few bytes for necessary function
// arguments"): no device-side table allocation, launches are asynchronous and
// graph-capturable.  ~5.5 KB, inside the 32 KB parameter space of sm_70+ / CUDA >= 12.1.
#pragma once
#include <stdint.h>

namespace cfs {

constexpr int kMaxFuncs = 64;
constexpr int kMaxChain = 8;

// affine table forms (bit-identical results, DESIGN R4: fma(0,y,b) == b)
enum AffForm : int { AFF_GENERAL = 0, AFF_DIAG = 1 };
// splat variants compiled into the render kernel
enum SplatKind : int {
    SPLAT_HIST_DIRECT = 0,   // red.global.add.u32
    SPLAT_HIST_SHARED = 1,   // atom.shared.add.u32 into a per-CTA histogram, merged by red.global
    SPLAT_HIST_WARPAGG = 2,  // __match_any_sync aggregation, then red.global.add.u32
    SPLAT_RGBA = 3,          // red.global.add.v4.f32
    SPLAT_DEPTH = 4,         // ld.global.cg pre-test + atom.global.min.u64
    SPLAT_NONE = 5           // trace kernel
};

struct ChainStep {
    int32_t type;      // cfs_xform_type after host resolution (ROTATE_Z -> AFFINE)
    float p[12];       // resolved at t.  AFFINE: as cfs_func; PINHOLE: fx fy cam_z near
};

struct RenderParams {
    uint64_t n_points, point_offset;
    uint32_t rk[10][2];          // Philox round keys: key + r*(0x9E3779B9, 0xBB67AE85)
    int32_t iterations, burn_in;
    int32_t W, H;
    float xmin, xmax, ymin, ymax;
    float sx, ox, sy, oy;        // pixel map: px = floor(fma(x, sx, ox))
    void *image;
    const void *cloud;
    unsigned long long *counters;
    // trace outputs (trace kernel only)
    uint8_t *tr_picks;
    float *tr_g, *tr_q;
    uint8_t *tr_alive;

    int32_t dim, n_funcs, n_chain, color_rule, reuse;
    int32_t pick_shift;          // >= 0: k = u >> pick_shift (equal power-of-two thresholds)
    int32_t n_thr;               // thresholds below 2^32 (k = #{j < n_thr : u >= T[j]})
    int32_t pick_steps;          // max thresholds inside one 2^24 bucket of u
    uint32_t points_per_thread;  // shared-hist persistent grid
    uint32_t hist_bins;          // W*H (shared-hist variant)

    ChainStep chain[kMaxChain];
    uint32_t T[kMaxFuncs];       // thresholds (u32), T[j >= n_thr] = 0xFFFFFFFF
    uint8_t lut[256];            // lut[b] = #{j < n_thr : T[j] <= b << 24}
    float coef[kMaxFuncs * 12];  // GENERAL dim2: rows of 8 (a00 a01 b0 0 | a10 a11 b1 0);
                                 // GENERAL dim3: rows of 12 (a00 a01 a02 b0 | ... );
                                 // DIAG dim2: rows of 4 (sx sy bx by); DIAG dim3: rows of 8
                                 // (sx sy sz 0 | bx by bz 0)
    float palette[kMaxFuncs * 4];
    uint32_t pal8[kMaxFuncs];    // palette rounded to rgba8 (DEPTH mode)
};

}  // namespace cfs
