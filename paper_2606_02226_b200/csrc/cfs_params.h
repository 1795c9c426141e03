// cfs_params.h -- kernel parameter block of the CFS hot path (host fills it, device reads it).
//
// Everything a render needs travels BY VALUE in the launch ("a few bytes for necessary function
// arguments"): no device-side table allocation, launches are asynchronous and
// graph-capturable.  ~5.5 KB, inside the 32 KB parameter space of sm_70+ / CUDA >= 12.1.
#pragma once
#ifdef __CUDACC_RTC__
// run-time compilation (cfs_jit.cu): NVRTC has no host headers; the fixed-width types are spelled out
typedef signed char int8_t;
typedef unsigned char uint8_t;
typedef short int16_t;
typedef unsigned short uint16_t;
typedef int int32_t;
typedef unsigned int uint32_t;
typedef long long int64_t;
typedef unsigned long long uint64_t;
#else
#include <stdint.h>
#endif

#ifdef __CUDACC__
#define CFS_HD __host__ __device__
#else
#define CFS_HD
#endif

namespace cfs {

constexpr int kMaxFuncs = 64;
constexpr int kMaxChain = 8;
constexpr int kRenderThreads = 256;   // CTA size of the render / trace kernels
constexpr int kClusterThreads = 512;  // CTA size of the cluster-histogram variant (one CTA per SM, 16 warps)
constexpr int kClusterSize = 8;       // CTAs per cluster (portable maximum)

// affine table forms (bit-identical results, DESIGN R4: fma(0,y,b) == b)
enum AffForm : int { AFF_GENERAL = 0, AFF_DIAG = 1, AFF_CIRCLE = 2 /* PAPER Eq. 1 maps: one row (f_id, r2 flag, -, -) per map */,
                     AFF_USCALE = 3 /* DIAG maps that all share one scale (sx, sy, sz): the table holds the translations only,
                                       one row (bx by bz -) per map, the scale travels as prm.uscale -- half the table reads
                                       of AFF_DIAG, bit-identical results (run-time compiled kernels) */ };
// transcendental evaluation of the non-affine chain steps: libdevice sincosf/sinf/cosf (<= 2 ulp)
// or the MUFU special-function unit (sin.approx/cos.approx, abs. error ~2^-21 on [-pi, pi])
enum TrigKind : int { TRIG_ACCURATE = 0, TRIG_FAST = 1, TRIG_RUNTIME = 2 /* prm.fast_trig decides (interpreter) */ };
// chain signature: 4 bits per step, (type + 1) of step m in bits [4m, 4m+4), 0 terminates.
// A kernel compiled for a signature has the chain unrolled with every parameter a fixed constant
// operand; kChainGeneric selects the interpreter (unrolled to kMaxChain steps, warp-uniform switch).
constexpr uint32_t kChainGeneric = 0xFFFFFFFFu;
CFS_HD constexpr uint32_t chain_sig(int a = -1, int b = -1, int c = -1, int d = -1)
{
    return (uint32_t)(a + 1) | ((uint32_t)(b + 1) << 4) | ((uint32_t)(c + 1) << 8) | ((uint32_t)(d + 1) << 12);
}
// type of step m of a signature, -1 past its end
CFS_HD constexpr int sig_step(uint32_t sig, int m)
{
    return (sig == kChainGeneric || m < 0 || m >= kMaxChain) ? -1 : (int)((sig >> (4 * m)) & 15u) - 1;
}
// kernel options compiled in (template argument OPT of render_kernel / cloud_kernel)
enum KernelOpt : int {
    OPT_REUSE = 1,         // Fig. 2(C): the chain output is fed back into the generator (compiled chains; the interpreter reads prm.reuse)
    OPT_PICK_SHIFT = 2,    // equal power-of-two thresholds: k = u >> prm.pick_shift, nothing else compiled in
    OPT_PICK_LUT1 = 4,     // at most one threshold per 2^24 bucket of u: one table read + one compare, no loop
    OPT_PICK_MULHI = 8,    // equal thresholds T_j = floor((j + 1) 2^32 / n), n not a power of two: k = (u n + n - 1) >> 32 (64-bit product)
    OPT_BIN_RGBA = 16,     // tile bins: records carry the colour index (RGBA + MAP_INDEX); with OPT_BIN_FIXED only
    OPT_BIN_FIXED = 32,    // tile bins: OPT_BIN_RGBA and the direct mask below are the truth (else prm.bin.hybrid / prm.color_rule decide at run time)
    OPT_SYM_BOUNDS = 64,   // xmin == -xmax and ymin == -ymax: the closed-bounds test is |x| <= xmax && |y| <= ymax (two compares)
    OPT_PICK_CMP2 = 128,   // at most two thresholds: k = (u >= T[0]) + (u >= T[1]), two compares against the parameter block, no table read
    OPT_RCP_NORMAL = 4096, // PINHOLE: the host has PROVED 2^-126 <= d < 2^126 for every live splat (bounded attractor, near >= 2^-100), so
                           // 1/d is the four-instruction normal-range sequence of the correctly rounded reciprocal, without its range test
    OPT_NO_DROP = 8192,    // the host has PROVED (same bound, with a margin against rounding) that every splat is alive and inside the image
                           // bounds: no near test, no bounds test, nothing to count as dropped
    OPT_ALL_HAVE = 16384,  // tile bins: every chunk of the render is a whole number of CTAs (n_points a multiple of kBinThreads), so no
                           // thread of pass 1 is ever without a point: no `have` predicate, select or dummy counter in the append
    OPT_BIN_MASK_SHIFT = 8 // bits 8..11, with OPT_BIN_FIXED: iteration j of a steady-state block splats straight to L2 when bit j is set
};
// true when the signature holds a BRANCH separator (type 8): one-to-many splatting
CFS_HD constexpr bool sig_has_branch(uint32_t sig)
{
    if (sig == kChainGeneric) return false;
    for (int m = 0; m < kMaxChain; ++m)
        if (sig_step(sig, m) == 8) return true;
    return false;
}
// true when a step of the signature evaluates sin/cos (types 1 SWIRL, 2 SINUSOIDAL, 4 TWIST_Z,
// 5 BEND, 7 STRETCH_COS); the generic signature may
CFS_HD constexpr bool sig_has_trig(uint32_t sig)
{
    if (sig == kChainGeneric) return true;
    for (int m = 0; m < 8; ++m) {
        const int code = (int)((sig >> (4 * m)) & 15u);
        if (code == 0) break;
        const int t = code - 1;
        if (t == 1 || t == 2 || t == 4 || t == 5 || t == 7) return true;
    }
    return false;
}
// splat variants compiled into the render kernel
enum SplatKind : int {
    SPLAT_HIST_DIRECT = 0,   // red.global.add.u32
    SPLAT_HIST_SHARED = 1,   // atom.shared.add.u32 into a per-CTA histogram, merged by red.global
    SPLAT_HIST_WARPAGG = 2,  // __match_any_sync aggregation, then red.global.add.u32
    SPLAT_RGBA = 3,          // red.global.add.v4.f32
    SPLAT_DEPTH = 4,         // ld.global.cg pre-test + atom.global.min.u64
    SPLAT_NONE = 5,          // trace kernel
    SPLAT_HIST_CLUSTER = 7,  // histogram distributed over the shared memory of a thread-block cluster
                             // (red.shared::cluster.add.u32 through DSMEM), merged by red.global
    SPLAT_DEPTH_HIZ = 8,     // SPLAT_DEPTH behind a coarse conservative depth map (Hi-Z) held in shared memory
    SPLAT_BIN = 6            // tile-binned: records partitioned by image tile into a block pool
                             // (pass 1), accumulated per tile in shared memory (pass 2)
};

// tile-binned splat stage (DESIGN "binned variant").  A record is one uint16:
// (colour index) * (pixels per tile) + (pixel index inside the tile), i.e. directly the index of the
// shared-memory counter pass 2 increments (a tile has at most 3 * 2^14 = 49152 counters).  The pool is a set of fixed-size blocks; a block belongs to
// one (CTA, tile) while it is filled and is listed under its tile when it is allocated.
constexpr uint32_t kBinBlockRecords = 1024;    // records per pool block (2 KiB)
constexpr uint32_t kBinGrain = 8;              // records per 128-bit vector: a drained row is padded to whole vectors with the DUMMY record
constexpr uint32_t kBinDrainMin = 64;          // a row is drained when it holds at least this many records (a 128-byte store or longer)
constexpr uint32_t kBinTailShift = 11;         // tails word: blocks << 11 | records in the last block (<= 1024)
constexpr uint32_t kBinRowPad = 16;            // bytes between two staging rows beyond their records: rows 2 * cap bytes long would all start on bank 0, and
                                               // with interleaved tiles all rows fill in step, so the stores of a warp met on a few banks (4.15 wavefronts
                                               // per STS); 16 bytes of skew per row spread them (rows stay 16-byte aligned for the bulk copy)
constexpr uint32_t kBinDummy = 32;             // dummy fill counters behind cnt[n_tiles], one per lane: pre-set to the row capacity, they take
                                               // the dropped splats -- "row full" for free, so a dropped splat stores nothing and needs no predicate
constexpr uint32_t kBinInvalid = 0xFFFFFFFFu;  // tile has no block (pool or list exhausted): direct splats
constexpr int kBinThreads = 1024;              // CTA size of pass 1 and CTAs per SM.  2 x 512 threads (half-length staging rows, one CTA computing
constexpr int kBinCtasPerSm = 1;               // while the other is at its flush barrier) measured no better: configs[1] 2.97 against 2.95 ms, configs[2]
                                               // 6.74 against 6.12 ms per frame -- the barrier stall of the flush is skew, which the slower warps fill
constexpr int kBinAccThreads = 1024;           // CTA size of pass 2 (one CTA per SM: the tile fills shared memory)

// Hi-Z pre-test of the depth splat (DESIGN "Hi-Z variant").  hz[by * nbx + bx] is an upper bound of
// (depth bits >> 16) over the 2^shift x 2^shift pixel block (bx, by), taken from a snapshot of the
// depth image; the image only decreases, so the bound stays valid for the rest of the render.
constexpr int kHizThreads = 576;               // CTA size of the Hi-Z render kernel, two CTAs per SM: 56 registers per thread, no spills (configs[4], ms: 512x2 132.3, 576x2 129.4, 640x2 130.8, 704x2 136.0, 768x2 135.2 with 40 registers and spills, 512x3 141.7, 1024x1 slower still)
constexpr int kHizCtasPerSm = 2;
constexpr uint32_t kHizMaxBytes = 96 * 1024;   // per CTA, in shared memory
struct HizParams {
    const uint16_t *hz;    // nbx * nby entries (device)
    uint32_t shift, nbx, nby, n_pad;   // n_pad = entries rounded up to a multiple of 8 (copied as 16-byte vectors)
};

struct BinParams {
    uint16_t *pool;        // nb * kBinBlockRecords records
    uint32_t *list;        // [n_tiles][grid][lcap] block ids listed by pass-1 CTA c for a tile
    uint32_t *tails;       // [n_tiles][grid] (blocks listed) << kBinTailShift | records in the last block
    uint32_t *ctrl;        // [0] = blocks handed out, [1] = records splatted directly (statistics)
    uint32_t nb, lcap, n_tiles;
    uint32_t grid;         // CTAs of pass 1
    uint32_t tile_pixels;  // pixels (counters per colour slot) of a tile: ceil(W H / n_tiles)
    uint32_t tshift, tmask; // n_tiles = 2^tshift, tmask = n_tiles - 1: pixel p belongs to tile p & tmask and is its pixel p >> tshift (tiles are INTERLEAVED)
    uint32_t nk;           // colour slots per pixel: 1 = HIST, else the number of functions (<= 16)
    uint32_t cap;          // staging records per tile in shared memory (multiple of 64, >= 320)
    uint32_t drain_min;    // a staging row is drained when it holds at least this many records (multiple of 8)
    uint32_t check_every;  // the staging rows are drained every check_every Philox blocks (4 iterations each) of the CTA
    uint32_t split;        // pass 2: CTAs per tile
    uint32_t hybrid;       // 4-bit mask: iteration j of every steady-state Philox block splats straight to L2 when bit j is set
                           // (0 = pure bins, 5 = every other splat: the hybrid stage)
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
    const void *cloud;           // record p of the whole cloud is cloud[p - cloud_base]
    uint64_t cloud_base;
    unsigned long long *counters;
    // trace outputs (trace kernel only)
    uint8_t *tr_picks;
    float *tr_g, *tr_q;
    uint8_t *tr_alive;

    int32_t dim, n_funcs, n_chain, color_rule, reuse, fast_trig;
    int32_t aff_form;            // AffForm of the coefficient table below
    float uscale[3];             // AFF_USCALE: the scale all maps share
    int32_t n_branches;          // 1 + BRANCH markers in the chain: splats per generated point and iteration
    int32_t pick_shift;          // >= 0: k = u >> pick_shift (equal power-of-two thresholds)
    int32_t n_thr;               // thresholds below 2^32 (k = #{j < n_thr : u >= T[j]})
    int32_t pick_steps;          // max thresholds inside one 2^24 bucket of u
    uint32_t coef_rows;          // 16-byte coefficient rows in use (n_funcs x rows per map)
    uint32_t coef_kstride, coef_rstride; // bytes between the first rows of two maps / between the rows of one map
    uint32_t coef_cshift;        // log2(copies of each coefficient row in shared memory), bank-conflict-free table reads
    uint32_t points_per_thread;  // shared-hist persistent grid
    uint32_t hist_bins;          // W*H (shared-hist and cluster-hist variants)
    uint32_t slice_shift;        // cluster-hist: bins per CTA = 1 << slice_shift, bin b lives in CTA rank b >> slice_shift

    BinParams bin;               // SPLAT_BIN only
    HizParams hiz;               // SPLAT_DEPTH_HIZ only

    ChainStep chain[kMaxChain];
    uint32_t T[kMaxFuncs];       // thresholds (u32), T[j >= n_thr] = 0xFFFFFFFF
    uint32_t lut[256][2];        // bucket b of the top byte of u: { ~m, m = (first threshold inside the bucket) - 1, or 0xFFFFFFFF
                                 // when the bucket holds none;  #{j < n_thr : T[j] <= b << 24} }.  k = lut[b][1] + (u > m),
                                 // and u > m is the carry of u + ~m
                                 // is the pick when no bucket holds two thresholds; further ones are walked in T[]
    float coef[kMaxFuncs * 12];  // GENERAL dim2: rows of 8 (a00 a01 b0 0 | a10 a11 b1 0);
                                 // GENERAL dim3: rows of 12 (a00 a01 a02 b0 | ... );
                                 // DIAG dim2: rows of 4 (sx sy bx by); DIAG dim3: rows of 8
                                 // (sx sy sz 0 | bx by bz 0)
    float palette[kMaxFuncs * 4];
    uint32_t pal8[kMaxFuncs];    // palette rounded to rgba8 (DEPTH mode)
};

}  // namespace cfs
