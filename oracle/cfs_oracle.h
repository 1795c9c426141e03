/* cfs_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU restatement of the hot path of the Composable
 * Function System (CFS) method of arxiv/paper_2606_02226 ("Composable function
 * systems as a general-purpose rendering framework", J. Schloss): chaos-game
 * sampler -> composed transform chain on a copy of the point -> splat.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may use anything in this directory.  It shares no code, header,
 * table or constant generator with the CUDA path under paper_2606_02226_b200/.
 *
 * Citations: "PAPER L<n>" = line n of /root/reference/PAPER.md; "DESIGN R<n>" =
 * reading n in DESIGN.md (where the paper is silent); "BJ" = BASELINE.json.
 *
 * Pins (tests/test_oracle_*.py): Philox known answers, threshold brute force,
 * affine fixed points, the cfg-0 closed form (pixel = word of the last 9 picks),
 * uniform invariant density (chi-square), conservation, removed regions
 * (Sierpinski / carpet / Menger), word enumeration up to length 8, chain
 * invariants, depth buffer vs brute force, tone-map closed forms.
 * Parity unpinned: the AS-PRINTED reading of the paper's Eq. 1 circle map
 * (ORC_F_CIRCLE_HALF with params[1] == 0; DESIGN R13): the equation is garbled in
 * the source, so beyond the invariants of PAPER L60, the polar-swap structure and
 * nine hand-worked values nothing fixes it.  Its r^2 reading (params[1] != 0) is
 * pinned by its closed-form uniform invariant density.  Everything else is pinned.
 */
#ifndef CFS_ORACLE_H
#define CFS_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_GEN_IFS = 0, ORC_GEN_CLOUD = 1 };
enum { ORC_F_AFFINE = 0, ORC_F_CIRCLE_HALF = 1 };
enum {
    ORC_T_AFFINE = 0, ORC_T_SWIRL = 1, ORC_T_SINUSOIDAL = 2, ORC_T_ROTATE_Z = 3,
    ORC_T_TWIST_Z = 4, ORC_T_BEND = 5, ORC_T_PINHOLE = 6, ORC_T_STRETCH_COS = 7,
    ORC_T_BRANCH = 8,  /* not a transform: ends one branch of the chain and starts the next */
    ORC_T_SCATTER = 9  /* PRNG-placed duplicates; p = (D, rx, ry, rz); DESIGN R14 */
};
enum { ORC_COLOR_NONE = 0, ORC_COLOR_MAP_INDEX = 1, ORC_COLOR_POINT = 2 };
enum { ORC_OUT_HIST_U32 = 0, ORC_OUT_RGBA = 1, ORC_OUT_DEPTH_U64 = 2 };
enum { ORC_DOMAIN_PICK = 0, ORC_DOMAIN_INIT = 1, ORC_DOMAIN_AUX = 2, ORC_DOMAIN_PLACE = 3 };

/* generator function: AFFINE params, dim 2: a00 a01 a10 a11 b0 b1;
 * dim 3: a00..a22 row-major then b0 b1 b2.
 * CIRCLE_HALF (PAPER Eq. 1; dim 2 only): params[0] = f_id (0 -> top half, 1 -> bottom half of
 * the unit disc), params[1] != 0 selects the r^2 reading of theta_2 (DESIGN R13).  PARITY UNPINNED
 * beyond the invariants the paper states (L60): Eq. 1 is garbled in the source. */
typedef struct { int32_t type; float prob; float params[12]; } orc_func;
/* chain transform: effective parameter i = (float)((double)p0[i] + (double)t*(double)p1[i]) */
typedef struct { int32_t type; float p0[12]; float p1[12]; } orc_xform;

typedef struct {
    int32_t dim;          /* 2 | 3 */
    int32_t gen_kind;     /* ORC_GEN_* */
    int32_t n_funcs;      /* IFS only */
    int32_t n_chain;
    int32_t color_rule;   /* ORC_COLOR_* */
    int32_t reuse;        /* 0: Fig. 2(B) copy-then-transform; 1: Fig. 2(C) feed chain output back */
    const orc_func *funcs;
    const orc_xform *chain;
    const float *palette; /* n_funcs*4 floats (r,g,b,a), MAP_INDEX only */
} orc_system;

typedef struct { float x, y, z; uint32_t rgba8; } orc_cloud_rec;

typedef struct {
    uint64_t n_points, point_offset, seed;
    int32_t iterations, burn_in;
    int32_t width, height;
    float xmin, xmax, ymin, ymax, t;
    int32_t out_mode;     /* ORC_OUT_* */
    int32_t pad_;
    void *image;          /* HIST: uint32[W*H]; RGBA: double[W*H*4]; DEPTH: uint64[W*H]; accumulates */
    const orc_cloud_rec *cloud; /* CLOUD only: record p of the whole cloud is cloud[p] */
    uint64_t *counters;   /* optional u64[2]: in-bounds splats, dropped; accumulates */
} orc_render_args;

/* S2: Philox4x32-10 */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* S3: thresholds T[0..n-1] (T[n-1] = 2^32) from float probabilities; returns 0 or -1 if invalid */
int orc_thresholds(const float *prob, int n, uint64_t *T);
int orc_pick(uint32_t u, const uint64_t *T, int n);
/* pick of point p at iteration it (keyed word, then orc_pick) */
uint32_t orc_pick_word(uint64_t seed, uint64_t p, uint32_t it);
/* SCATTER step (DESIGN R14): q += the offset of the duplicate drawn for (seed, p, it); prm = (D, rx, ry, rz) */
void orc_scatter(uint64_t seed, uint64_t p, uint32_t it, const float *prm, int dim, float q[3]);
/* S4 */
void orc_init_point(uint64_t seed, uint64_t p, int dim, float g[3]);
/* S5 */
void orc_apply_func(const orc_func *f, int dim, float g[3]);
/* S6: one chain step with parameters already resolved at t; returns alive */
int orc_apply_xform(int type, const float *prm, int dim, float q[3]);
/* resolve the parameters of one chain step at frame parameter t; type_out may differ
 * from x->type (ROTATE_Z resolves to AFFINE). aspect = H/W for PINHOLE. */
void orc_resolve_xform(const orc_xform *x, int dim, float t, int width, int height,
                       int *type_out, float prm_out[12]);
/* S7: pixel index or -1 if out of bounds */
int64_t orc_pixel(float x, float y, float xmin, float xmax, float ymin, float ymax, int W, int H);

/* S1: the whole path. Returns 0, or -1 on invalid arguments. */
int orc_render(const orc_system *sys, const orc_render_args *a);
/* S10(i),(ii): per-point pick sequences [n_points*iterations], final generator
 * state [n_points*3], final chain output [n_points*3] and its alive flag. Any may be NULL. */
int orc_trace(const orc_system *sys, const orc_render_args *a, uint8_t *picks,
              float *final_g, float *final_q, uint8_t *final_alive);
/* S9. image as produced by the GPU path: HIST uint32, RGBA float32[4], DEPTH uint64 */
int orc_tonemap(const void *image, int out_mode, int W, int H, float gamma, float colour_scale,
                uint32_t *rgba8_out);

#ifdef __cplusplus
}
#endif
#endif
