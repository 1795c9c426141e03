/* cfs.h -- C ABI of the B200-native Composable Function System (CFS) hot path.
 *
 * What it computes (arxiv/paper_2606_02226, "Composable function systems as a general-purpose
 * rendering framework"; citations "PAPER L<n>" are lines of the paper's text, "DESIGN R<n>" are
 * the readings listed in DESIGN.md where the paper is silent):
 *
 *   chaos game: every point picks one function of the generator IFS at
 *   random each step and applies it; a COPY of the point (Fig. 1, L77 Fig. 2(B)) runs
 *   through the ordered chain of later, possibly non-affine, transforms and
 *   is splatted / histogrammed into the output image; colours show the function
 *   that produced the point.  The generator may instead be a stored point cloud
 *   (PAPER L25, L206).
 *
 * All kernels are hand-written CUDA for sm_100a.  There is no CPU fallback: every entry point
 * that does work needs a CUDA device and returns CFS_ERR_CUDA without one.
 *
 * Conventions
 *   - plain C types only; pointers named d_* are DEVICE pointers, h_* are HOST pointers.
 *   - every call returns cfs_status; nothing throws, aborts or prints.  cfs_last_error() gives
 *     a thread-local message for the last non-OK status on the calling thread.
 *   - cfs_create copies everything it is given; the caller keeps ownership of its arrays.
 *   - cfs_render / cfs_tonemap / cfs_trace / cfs_microbench are asynchronous on `cuda_stream`
 *     (a cudaStream_t passed as void*; NULL = the legacy default stream) and never synchronise.
 *     They allocate no device memory (only the output image lives in global
 *     memory); tables travel in the kernel parameter block.
 *   - images are caller-owned and caller-cleared (0 for HIST/RGBA, all-ones bytes for DEPTH);
 *     renders ACCUMULATE, so frames, point sub-ranges and GPUs compose by sum / min.
 */
#ifndef CFS_H
#define CFS_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CFS_MAX_FUNCS 64
#define CFS_MAX_CHAIN 8

typedef struct cfs_system cfs_system; /* opaque, host-side, owned by the library */

typedef enum {
    CFS_OK = 0,
    CFS_ERR_INVALID_ARG = 1,
    CFS_ERR_UNSUPPORTED = 2,
    CFS_ERR_CUDA = 3,
    CFS_ERR_NOMEM = 4
} cfs_status;

/* generator: an IFS solved by the chaos game, or a stored cloud */
typedef enum { CFS_GEN_IFS = 0, CFS_GEN_CLOUD = 1 } cfs_gen_kind;
/* generator function types.  AFFINE params: dim 2: a00 a01 a10 a11 b0 b1;
 * dim 3: a00..a22 row-major, then b0 b1 b2.  x' = fma(a00,x,fma(a01,y,b0)) etc. (DESIGN R4).
 * CIRCLE_HALF (dim 2 only; every function of the generator must then be CIRCLE_HALF) is PAPER Eq. 1
 * (L47-60), the non-affine circle IFS whose two maps send the unit disc to its top / bottom half:
 * params[0] = f_id (0 or 1), params[1] != 0 selects the r^2 reading.  r = sqrt(x^2+y^2), theta = atan2(y,x)
 * wrapped to [0, 2 pi), theta2 = pi (r + f_id) [flag: pi (r^2 + f_id)], r2 = sqrt(theta / 2 pi),
 * (x', y') = (r2 cos theta2, r2 sin theta2) (DESIGN R13; the printed equation is garbled).  f_id is
 * DATA (a table entry), so the two maps share one code path: no divergence from the random choice. */
typedef enum { CFS_F_AFFINE = 0, CFS_F_CIRCLE_HALF = 1 } cfs_func_type;
typedef struct { int32_t type; float prob; float params[12]; } cfs_func;

/* chain transform types (applied to the copy, in order).  Effective parameter i of a step is
 * (float)((double)p0[i] + (double)t*(double)p1[i]), resolved on the host once per render.
 *   AFFINE      params as cfs_func AFFINE
 *   SWIRL       r2 = x^2+y^2; (x,y) rotated by r2                         (BASELINE cfg 1)
 *   SINUSOIDAL  (sin x, sin y), z kept                                    (BASELINE cfg 2)
 *   ROTATE_Z    p[0] = angle; resolved on the host to an AFFINE rotation  (BASELINE cfg 2)
 *   TWIST_Z     (x,y) rotated by p[0]*z                                   (BASELINE cfg 3)
 *   BEND        (x,y) rotated by p[0]*x (input x)                         (DESIGN R6)
 *   PINHOLE     p = (fov_y degrees, cam_z, near): d = z-cam_z; dropped unless d > near;
 *               x' = (fx*x)*(1/d), y' = (fy*y)*(1/d), z' = d; fy = 1/tan(fov/2), fx = fy*H/W
 *   STRETCH_COS x' = 2x, y' = y - cos x                                   (PAPER Eq. 2)
 *   BRANCH      not a transform: ends one branch of the chain and starts the next.  Every branch is applied
 *               to its own copy of the generated point and splatted, so a point drives M splats per iteration
 *               ("many objects from a single primitive"); the image equals the sum (DEPTH: the
 *               min) of the M single-chain renders.  Not with reuse; DEPTH needs every branch to end in PINHOLE.
 *               Runs on the chain interpreter, or compiled in with CFS_FLAG_JIT; cfs_trace does not serve it.
 *   SCATTER     p = (D, rx, ry, rz), D a whole number in [1, 2^20]: PRNG-placed duplicates of an object
 *               (DESIGN R14).  The copy moves onto duplicate d = floor(w D / 2^32), w = word it & 3
 *               of Philox(seed; point lo, point hi, it >> 2, domain 2); its offset is (u(v0) rx, u(v1) ry, u(v2) rz)
 *               with v = Philox(seed; d, 0, 0, domain 3) and u the 24-bit map to [-1, 1) of the point init --
 *               a pure function of (seed, d), nothing is stored.  Exact float32 (one multiply, one add per
 *               coordinate).  Runs on the chain interpreter, or compiled in with CFS_FLAG_JIT. */
typedef enum {
    CFS_T_AFFINE = 0, CFS_T_SWIRL = 1, CFS_T_SINUSOIDAL = 2, CFS_T_ROTATE_Z = 3,
    CFS_T_TWIST_Z = 4, CFS_T_BEND = 5, CFS_T_PINHOLE = 6, CFS_T_STRETCH_COS = 7, CFS_T_BRANCH = 8,
    CFS_T_SCATTER = 9
} cfs_xform_type;
typedef struct { int32_t type; float p0[12]; float p1[12]; } cfs_xform;

/* colour rule and output layer (BASELINE cfg 0-4) */
typedef enum { CFS_COLOR_NONE = 0, CFS_COLOR_MAP_INDEX = 1, CFS_COLOR_POINT = 2 } cfs_color_rule;
typedef enum {
    CFS_OUT_HIST_U32 = 0,        /* uint32[H*W]: hits                                    */
    CFS_OUT_RGBA_F32 = 1,        /* float[H*W*4]: sum of (r,g,b,1), 16-byte aligned      */
    CFS_OUT_DEPTH_RGBA8_U64 = 2  /* uint64[H*W]: min of (bits(depth)<<32 | rgba8)        */
} cfs_out_mode;

/* splat-stage variant (BASELINE north_star: "two variants chosen by image size") */
typedef enum {
    CFS_VARIANT_AUTO = 0,        /* chosen from mode and image bytes                                  */
    CFS_VARIANT_DIRECT = 1,      /* one L2 reduction per splat (red.global / atom.global.min.u64)     */
    CFS_VARIANT_SHARED_HIST = 2, /* HIST only, W*H*4 <= cfs_shared_hist_max_bytes(): per-CTA shared   */
                                 /* histogram, merged with red.global                                 */
    CFS_VARIANT_WARP_AGG = 3,    /* DIRECT + __match_any_sync aggregation of same-pixel hits (HIST)   */
    CFS_VARIANT_CLUSTER_HIST = 5,/* HIST, IFS generator, W*H*4 <= 8 x (shared memory of a CTA): the histogram is   */
                                 /* distributed over the shared memory of 8-CTA thread-block clusters, splats are */
                                 /* red.shared::cluster through DSMEM, slices merged with red.global              */
    CFS_VARIANT_DEPTH_HIZ = 6,   /* DEPTH, IFS generator, needs d_scratch of cfs_hiz_scratch_bytes(): a coarse        */
                                 /* conservative depth map (max of depth bits >> 16 per pixel block), rebuilt from   */
                                 /* the image after the first slices of the points and held in shared memory, lets   */
                                 /* occluded splats stop on the SM instead of paying a random L2 load; same image    */
    CFS_VARIANT_BINNED = 4       /* HIST, or RGBA + MAP_INDEX with <= 16 functions, IFS generator:    */
                                 /* splats are partitioned by image tile through d_scratch (one       */
                                 /* 2-byte record each), then every tile is accumulated in shared     */
                                 /* memory and merged with red.global; no L2 atomic per splat         */
} cfs_variant;

/* render flags.
 *   FAST_TRIG: the non-affine chain steps evaluate sin/cos on the special-function unit (MUFU
 *   sin.approx / cos.approx, absolute error ~2^-21 on [-pi, pi], growing with |argument|) instead
 *   of the <= 2 ulp sincosf.  Within the 1e-4 coordinate tolerance of BASELINE north_star for the
 *   bounded arguments of contractive systems; the default is the accurate evaluation.
 *   INTERPRET_CHAIN: never use a kernel compiled for the chain's signature; run the chain
 *   interpreter (same device functions, same results; for tests and comparisons).
 *   BIN_PASS1_ONLY: measurement instrument of the BINNED variant: run pass 1 (sample + bin) and
 *   skip pass 2, so the two passes can be timed apart with events; the image is NOT updated
 *   (with BIN_HYBRID it receives the direct half only).
 *   BIN_HYBRID: the BINNED variant sends one splat in four (iteration 0 of each Philox block of four) straight
 *   to L2 with red.global and the rest through the tile bins, so that the L2 reduction units, the issue slots of
 *   pass 1 and the shared-memory atomics of pass 2 are all busy.  Same image (HIST sums are exact; RGBA sums are
 *   order-free, DESIGN R8).  CFS_VARIANT_AUTO sets it whenever it chooses the tile bins; CFS_VARIANT_BINNED takes
 *   it from the caller.  (Round 1 sent every other splat; with the leaner pass 2 of round 2 one in four measured
 *   ahead on configs[2] and level on configs[1], DESIGN "hybrid".)
 *   JIT: run-time specialisation (the chain is spliced into one fused kernel at run time; here by
 *   NVRTC).  The render uses a kernel compiled in this process for exactly this system -- dimension, generator
 *   form, splat sink, the chain unrolled with every step's type fixed, BRANCH / SCATTER / reuse / the Eq. 1
 *   generator included -- instead of the ahead-of-time kernels (which exist for the BASELINE chains only) or the
 *   chain interpreter.  The first use of a kernel pays its compilation (cfs_specialize() does it ahead of the
 *   render and reports the time; PAPER L200 quotes 0.745 s against 0.0215 s per frame for the paper's own
 *   system); kernels are cached in the process and, when $CFS_JIT_CACHE names a directory, on disk.  Same
 *   device functions, same results as the other two ways.  UNSUPPORTED when NVRTC cannot be loaded. */
typedef enum { CFS_FLAG_FAST_TRIG = 1, CFS_FLAG_INTERPRET_CHAIN = 2, CFS_FLAG_BIN_PASS1_ONLY = 4, CFS_FLAG_JIT = 8,
               CFS_FLAG_BIN_HYBRID = 0x100 } cfs_render_flags;

/* one 16-byte record of a stored cloud (BASELINE cfg 3); rgba8 = r | g<<8 | b<<16 | a<<24 */
typedef struct { float x, y, z; uint32_t rgba8; } cfs_cloud_rec;

/* cfs_create -- the generator IFS (per-function type id, parameters, selection probabilities),
 * the ordered transform chain and the colouring rule (BASELINE north_star).
 *   dim 2|3.  funcs/n_funcs: 1..CFS_MAX_FUNCS, ignored for CLOUD.  chain/n_chain: 0..CFS_MAX_CHAIN.
 *   palette_rgba: n_funcs*4 floats (integer-valued 0..255 by convention, DESIGN R9), required for
 *   MAP_INDEX, else NULL.  reuse != 0 selects Fig. 2(C) composition (chain output fed back).
 * Errors: INVALID_ARG for bad dims/counts/types, prob < 0 / NaN / sum <= 0, rule mismatch
 * (COLOR_POINT needs CLOUD; MAP_INDEX needs IFS + palette). Host only: no device work. */
cfs_status cfs_create(cfs_system **out, int32_t dim, int32_t gen_kind,
                      const cfs_func *funcs, int32_t n_funcs,
                      const cfs_xform *chain, int32_t n_chain,
                      int32_t color_rule, const float *palette_rgba, int32_t reuse);
void cfs_destroy(cfs_system *sys);

typedef struct {
    uint64_t n_points;      /* 0 is a no-op                                                     */
    uint64_t point_offset;  /* first global point id (sub-range renders, multi-GPU sharding)    */
    uint64_t seed;          /* Philox key                                                       */
    int32_t iterations;     /* >= 1; CLOUD: must be 1                                           */
    int32_t burn_in;        /* 0 <= burn_in < iterations; CLOUD: 0                              */
    int32_t width, height;  /* width*height <= 2^31-1                                           */
    float xmin, xmax, ymin, ymax; /* closed bounds; row 0 is ymin (DESIGN R8)                   */
    float t;                /* frame parameter                                                  */
    int32_t out_mode;       /* cfs_out_mode                                                     */
    int32_t variant;        /* cfs_variant                                                      */
    int32_t flags;          /* OR of cfs_render_flags; 0 = accurate sin/cos, compiled chain     */
    void *d_image;          /* device, caller-owned, caller-cleared, accumulates                */
    const void *d_cloud;    /* device, CLOUD only: record p of the WHOLE cloud is d_cloud[p]    */
    uint64_t *d_counters;   /* optional device u64[2]: += in-bounds splats, += dropped splats   */
    void *d_scratch;        /* optional device scratch of the BINNED variant, caller-owned; its  */
    uint64_t scratch_bytes; /* contents are garbage afterwards.  cfs_binned_scratch_bytes() is    */
                            /* what renders all points in one chunk; less means more chunks       */
} cfs_render_args;

/* cfs_render -- the hot path: sampler + pick + map + chain + colour + splat, one kernel launch
 * (BINNED: a memset and two launches per chunk of points).
 * Errors: INVALID_ARG, UNSUPPORTED (variant impossible for the mode
 * or image), CUDA (launch failure; message holds the CUDA error string). */
cfs_status cfs_render(const cfs_system *sys, const cfs_render_args *args, void *cuda_stream);

/* cfs_specialize -- compile now (NVRTC, sm_100a) and cache every kernel a cfs_render of this system with these
 * arguments and CFS_FLAG_JIT may launch (the direct sink of the output mode, the tile-bin pass 1 where the bins can
 * serve, the Hi-Z kernel for DEPTH), so that no render pays for compilation.  *out_compile_ms (optional) receives
 * the milliseconds this call spent compiling and loading (0 when everything was cached already).  Needs a
 * CUDA device (the module is loaded into its context).  PAPER L37, L182, L200.
 * Errors: INVALID_ARG as cfs_render; UNSUPPORTED when NVRTC cannot be loaded or the compilation fails (message). */
cfs_status cfs_specialize(const cfs_system *sys, const cfs_render_args *args, double *out_compile_ms);
/* cfs_jit_check -- test instrument, no device needed: compile the kernel a CFS_FLAG_JIT render of this system would
 * use for one splat sink (splat_kind < 0: the direct sink of args->out_mode; 6: the tile-bin pass 1; 8: the Hi-Z
 * depth kernel) to sm_100a SASS and drop it.  Outputs (optional): size of the cubin, milliseconds NVRTC took. */
cfs_status cfs_jit_check(const cfs_system *sys, const cfs_render_args *args, int32_t splat_kind,
                         uint64_t *out_cubin_bytes, double *out_ms);
/* kernels compiled at run time by this process so far and the milliseconds that took (either may be NULL) */
void cfs_jit_stats(uint64_t *out_kernels_compiled, double *out_total_ms);

/* bytes of d_scratch with which CFS_VARIANT_BINNED renders args->n_points in ONE chunk (pass 1 +
 * pass 2); 0 when the variant cannot serve this system / output mode / image, or without a device.
 * With scratch memory given, CFS_VARIANT_AUTO takes the binned path in its hybrid form (CFS_FLAG_BIN_HYBRID)
 * for large renders it can serve (at least one 1024-point CTA per SM and 2^27 splats) -- where it was
 * measured faster than the L2 atomic rate allows -- and the direct path otherwise. */
uint64_t cfs_binned_scratch_bytes(const cfs_system *sys, const cfs_render_args *args);

/* bytes of d_scratch CFS_VARIANT_DEPTH_HIZ needs for a width x height depth image (host arithmetic,
 * no device needed); 0 when the image is too large for a shared-memory Hi-Z map (> 96 KiB at
 * 32 x 32-pixel blocks).  CFS_VARIANT_AUTO takes this path for DEPTH renders of an IFS with at least 2^30 splats
 * when d_scratch holds that many bytes: the direct path is bound by the SM-to-L2 request rate, this one by
 * instruction issue -- level as linked ahead of time, ahead when compiled for the system (CFS_FLAG_JIT). */
uint64_t cfs_hiz_scratch_bytes(int32_t width, int32_t height);

/* cfs_render_depth_noalloc -- the Hi-Z depth render (CFS_VARIANT_DEPTH_HIZ) for callers that cannot allocate device
 * memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): its scratch -- the
 * Hi-Z map -- lives in a file-scope `static __device__` array of CFS_NOALLOC_SCRATCH_BYTES inside the library, which
 * every GPU that loads the library holds until the process exits.  The call allocates nothing: no cudaMalloc /
 * cudaFree, no run-time compilation or module load (CFS_FLAG_JIT and $CFS_FORCE_JIT are refused: INVALID_ARG; the
 * kernels are the ones linked ahead of time), only a memset of the map and kernel launches on `cuda_stream`.
 *   args  as for cfs_render: d_image (u64[width*height], cleared to 2^64 - 1 by the caller), d_counters (optional),
 *         n_points, point_offset, ...; out_mode must be CFS_OUT_DEPTH_RGBA8_U64 and the system an IFS (UNSUPPORTED
 *         otherwise); variant, d_scratch and scratch_bytes are IGNORED.
 *   limit cfs_hiz_scratch_bytes(width, height) must be non-zero and <= CFS_NOALLOC_SCRATCH_BYTES -- i.e. at most
 *         49152 blocks of 32 x 32 pixels, e.g. up to 7000 x 7000 -- else INVALID_ARG with both numbers in
 *         cfs_last_error().
 *   result identical, pixel for pixel and in the counters, to cfs_render with CFS_VARIANT_DEPTH_HIZ (and DIRECT).
 * The array is SHARED by every call on a device and keeps the last call's contents; the call clears what it reads
 * (the map is reset to "nothing culled" first), so a stale map cannot leak into a render -- but two calls that
 * overlap on the GPU (different streams, no dependency) RACE on it: serialise them.  The first call on a device
 * resolves the array's device address (cudaGetSymbolAddress) and lets CUDA load the kernels; make it before capture. */
#define CFS_NOALLOC_SCRATCH_BYTES (96 * 1024 + 256)
cfs_status cfs_render_depth_noalloc(const cfs_system *sys, const cfs_render_args *args, void *cuda_stream);

/* the tile plan of the BINNED variant for an image and a device shape, host arithmetic only (no device
 * needed; test instrument): out = { tiles (a power of two), pixels per tile, shift, mask (the tiles are
 * interleaved: pixel p belongs to tile p & mask and is its pixel p >> shift), colour slots per pixel, staging
 * records per tile, drain interval in iterations, pass-2 CTAs per tile }.  UNSUPPORTED when the variant cannot serve the image. */
cfs_status cfs_binned_plan(int32_t width, int32_t height, int32_t out_mode, int32_t n_funcs, int32_t sms,
                           int32_t smem_per_block_optin, uint32_t out[8]);

/* cfs_host_resolve -- test instrument, HOST arithmetic only (no device needed; d_image / d_cloud are ignored):
 * what cfs_render resolves on the host for this system and these arguments before it launches, so that each
 * value can be checked against a hand-worked number (tests/golden/host_resolved.txt).
 *   sx, ox, sy, oy   pixel map px = floor(fma(x, sx, ox)) (DESIGN R8): sx = (float)(W / (xmax - xmin)),
 *                    ox = (float)(-xmin W / (xmax - xmin)), evaluated in double
 *   chain_type/p     the chain at frame parameter t: AFFINE parameters (float)((double)p0 + (double)t (double)p1);
 *                    ROTATE_Z resolved to the AFFINE [c -s; s c] (3-D: about z), c = (float)cos(theta), s likewise;
 *                    PINHOLE as (fx, fy, cam_z, near), fy = (float)(1 / tan(fov/2)), fx = (float)(that H / W);
 *                    TWIST_Z / BEND p[0]; SCATTER (D, rx, ry, rz)
 *   pick_form        how a kernel compiled for this system (CFS_FLAG_JIT) evaluates k = #{j : u >= T_j}: 0 table + walk,
 *                    1 shift (equal power-of-two thresholds), 2 two compares, 3 table + one compare, 4 one multiply,
 *                    k = (u n + n - 1) >> 32, taken only when T_j == floor((j + 1) 2^32 / n) for every j
 *   proved           what the host has PROVED about this render and compiles into a CFS_FLAG_JIT kernel as a dropped test
 *                    (bounded attractor pushed through the chain, DESIGN "proved options"): bit 0 = every PINHOLE
 *                    depth is a normal float (the reciprocal's short sequence is the correctly rounded one), bit 1 =
 *                    every splat is alive and lands strictly inside the image (no bounds test, no drop count, no clamp)
 *   thresholds       T_j of DESIGN R2 (n_thresholds of them lie below 2^32), pal8 the palette packed to rgba8:
 *                    byte = floor(v + 0.5) clamped to [0, 255], NaN -> 0, r | g<<8 | b<<16 | a<<24 (DESIGN R9)
 * Errors: as cfs_render's validation (INVALID_ARG). */
typedef struct {
    float sx, ox, sy, oy;
    int32_t n_chain, n_funcs, n_thresholds, pick_form;
    int32_t chain_type[CFS_MAX_CHAIN];
    float chain_p[CFS_MAX_CHAIN][12];
    uint32_t thresholds[CFS_MAX_FUNCS];
    uint32_t pal8[CFS_MAX_FUNCS];
    int32_t proved, pad_;
} cfs_resolved;
cfs_status cfs_host_resolve(const cfs_system *sys, const cfs_render_args *args, cfs_resolved *out);

/* cfs_render_host -- same path with HOST buffers (end-to-end entry point): copies h_cloud to the
 * device (CLOUD), clears a device image, renders [point_offset, +n_points), copies the image to
 * h_image (layout of out_mode) and the counters to h_counters (u64[2], optional); synchronises
 * the stream before returning.  args->d_image/d_cloud/d_counters are ignored.  Scratch device
 * buffers are cached in the system handle and freed by cfs_destroy. */
cfs_status cfs_render_host(cfs_system *sys, const cfs_render_args *args, void *h_image,
                           const cfs_cloud_rec *h_cloud, uint64_t *h_counters, void *cuda_stream);

/* cfs_render_rgba8_host -- the whole path end to end with HOST buffers, to the paper's output format: as
 * cfs_render_host, then cfs_resolve_rgba8(gamma, colour_scale, n_max) on the device image, and only the width*height
 * RGBA8888 words travel back (h_rgba8), with the counters (optional) and this image's measured n_max (h_n_max,
 * optional, float; untouched for DEPTH).  Synchronises the stream before returning.  Device buffers (image, cloud,
 * scratch of at most 1 GiB, rgba8) are cached in the system handle and freed by cfs_destroy: the one exception to
 * "the library allocates nothing" (DESIGN "what differs"), confined to the two *_host convenience entry points. */
cfs_status cfs_render_rgba8_host(cfs_system *sys, const cfs_render_args *args, float gamma, float colour_scale,
                                 float n_max, uint32_t *h_rgba8, const cfs_cloud_rec *h_cloud,
                                 uint64_t *h_counters, float *h_n_max, void *cuda_stream);

/* cfs_resolve_rgba8 -- the paper's output layer (an RGBA8888 image) from the accumulator in ONE kernel
 * launch: log-density tone map (DESIGN R10; fractal-flame convention): n = count (HIST value /
 * RGBA alpha), n_max = max n; n = 0 -> 0; L = log(1+n)/log(1+n_max);
 * v_c = clamp(colour_scale * acc_c/n * L^(1/gamma), 0, 1) (HIST: v = L^(1/gamma)); alpha = L;
 * byte = floor(255 v + 0.5).  DEPTH: out = low 32 bits, empty -> 0 (gamma, colour_scale, n_max, d_scratch unused).
 *   n_max > 0 : the maximum to map with is GIVEN (an animation passes the previous frame's): a single pass, every
 *               accumulator is read once.  The pass also measures this image's own maximum.
 *   n_max == 0: the maximum is measured first, inside the same (cooperative) launch; the second read of the image
 *               comes from L2.
 *   n_max < 0 : map with the maximum the PREVIOUS call on this d_scratch measured (its word 0; at least 1), with no
 *               host round trip: frame k of an animation is mapped with frame k-1's maximum, in a single pass.
 * d_scratch: >= 16 bytes of device memory, 4-byte aligned; afterwards word 0 holds the bits of this image's n_max as a
 * float (0 for an empty image), words 1-3 are garbage.  d_rgba8_out: width*height uint32.  Asynchronous on the stream.
 * Errors: INVALID_ARG (NULL pointers, sizes, gamma <= 0, non-finite values), CUDA. */
cfs_status cfs_resolve_rgba8(const void *d_image, int32_t out_mode, int32_t width, int32_t height,
                             float gamma, float colour_scale, float n_max, uint32_t *d_rgba8_out, void *d_scratch,
                             void *cuda_stream);

/* cfs_tonemap -- cfs_resolve_rgba8 with the maximum measured inside (n_max = 0): BASELINE north_star "cfs_tonemap
 * does log-density tone mapping".  One memset and one kernel on the stream; d_scratch >= 8 bytes. */
cfs_status cfs_tonemap(const void *d_image, int32_t out_mode, int32_t width, int32_t height,
                       float gamma, float colour_scale, uint32_t *d_rgba8_out, void *d_scratch,
                       void *cuda_stream);

/* cfs_trace -- parity instrument (same device functions as cfs_render, no splat): per point the
 * pick sequence d_picks[n_points*iterations] (u8), the final generator state d_final_g[n*3],
 * the final chain output d_final_q[n*3] and its alive flag d_alive[n] (u8).  Any may be NULL. */
cfs_status cfs_trace(const cfs_system *sys, const cfs_render_args *args, uint8_t *d_picks,
                     float *d_final_g, float *d_final_q, uint8_t *d_alive, void *cuda_stream);

/* cfs_microbench -- roofline denominators measured in the same run (BASELINE north_star).
 * Launches `blocks` x `threads` threads each doing `ops_per_thread` operations of `kind`;
 * the caller times the stream.  Memory kinds address `footprint_bytes` of d_buf uniformly at
 * random (hash of a per-thread counter); ALU kinds ignore d_buf except for one sink store (ops_per_thread is
 * rounded down to a multiple of 256 there). */
typedef enum {
    CFS_MB_RED_ADD_U32 = 0,     /* red.global.add.u32, random 4-byte bins                */
    CFS_MB_RED_ADD_V4F32 = 1,   /* red.global.add.v4.f32, random 16-byte pixels          */
    CFS_MB_ATOM_MIN_U64 = 2,    /* atom.global.min.u64 (result unused), random bins      */
    CFS_MB_LD_U64 = 3,          /* ld.global.cg.u64 at random bins (depth pre-test)      */
    CFS_MB_ATOMS_ADD_U32 = 4,   /* atom.shared.add.u32 over footprint_bytes of shared    */
    CFS_MB_FFMA = 5,            /* FFMA, 8 independent dependent chains, one SASS instruction per op */
    CFS_MB_IMAD_WIDE = 6,       /* IMAD.WIDE.U32 chains (Philox core), one instruction per op        */
    CFS_MB_LOP3 = 7,            /* LOP3.LUT chains, one instruction per op                           */
    CFS_MB_MUFU = 8,            /* MUFU.RSQ chains (special-function unit), one instruction per op   */
    CFS_MB_STREAM_LD128 = 9,    /* coalesced 128-bit loads over footprint_bytes                      */
    CFS_MB_STREAM_RED_V4F32 = 10 /* the stored cloud's shape: per op one streamed 16-byte record (the first
                                    blocks*threads*ops*16 bytes of d_buf) + one red.global.add.v4.f32 at a random
                                    pixel of the footprint_bytes that follow them                                */
} cfs_microbench_kind;
cfs_status cfs_microbench(int32_t kind, void *d_buf, uint64_t footprint_bytes,
                          uint64_t ops_per_thread, int32_t blocks, int32_t threads,
                          void *cuda_stream);

/* largest W*H*4 the SHARED_HIST variant accepts on the current device (0 without a device) */
uint64_t cfs_shared_hist_max_bytes(void);
/* kernels launched by this library on the calling thread since the last reset (bench accounting) */
uint64_t cfs_launch_count(int32_t reset);
const char *cfs_last_error(void);
const char *cfs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CFS_H */
