/* cfs_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see cfs_oracle.h).
 *
 * Step-by-step CPU statement of the chaos game with a composed transform chain.
 * The method is a randomised iteration, so the oracle IS the algorithm in the
 * paper's order: choose a function at random, apply it, copy the point, run the
 * copy through the later transforms, splat.
 * Build: gcc -O2 -ffp-contract=off -shared -fPIC cfs_oracle.c -lm
 * (-ffp-contract=off: every fused multiply-add below is an explicit fmaf()).
 */
#include "cfs_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------- S2: Philox4x32-10
 * BJ north_star: "RNG and pick are fixed as Philox4x32 keyed by (seed, point,
 * iteration)".  Round function as published (Salmon et al., SC'11): two 32x32->64
 * products with the constants below, key bumped by the Weyl constants each round. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* DESIGN R1: counter = (p lo, p hi, block, domain), key = (seed lo, seed hi). */
static void keyed_block(uint64_t seed, uint64_t p, uint32_t block, uint32_t domain, uint32_t out[4])
{
    uint32_t ctr[4] = { (uint32_t)(p & 0xFFFFFFFFu), (uint32_t)(p >> 32), block, domain };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    orc_philox4x32_10(ctr, key, out);
}

/* DESIGN R1: PICK domain, one block per 4 iterations, word it&3 -- still a pure
 * function of (seed, point, iteration) as BJ requires. */
uint32_t orc_pick_word(uint64_t seed, uint64_t p, uint32_t it)
{
    uint32_t w[4];
    keyed_block(seed, p, it >> 2, ORC_DOMAIN_PICK, w);
    return w[it & 3];
}

/* "duplication" of an object by an on-the-fly PRNG (the stars of Fig. 4), no per-thread
 * allocation.  The paper gives no rule; DESIGN R14 [PROPOSED]: a SCATTER step with parameters
 * (D, rx, ry, rz) moves the copy onto one of D duplicates of the object,
 *     d      = floor(w * D / 2^32),  w = word it&3 of Philox(seed; p lo, p hi, it>>2, AUX),
 *     offset = (u(v0) rx, u(v1) ry, u(v2) rz),  v = Philox(seed; d, 0, 0, PLACE),  u = the 24-bit map of S4,
 *     q     += offset          (one float multiply and one float add per coordinate; z only in 3-D).
 * The D offsets are a pure function of (seed, d): nothing is stored. */
void orc_scatter(uint64_t seed, uint64_t p, uint32_t it, const float *prm, int dim, float q[3])
{
    uint32_t w[4], v[4];
    keyed_block(seed, p, it >> 2, ORC_DOMAIN_AUX, w);
    const uint32_t D = (uint32_t)prm[0];
    const uint32_t d = (uint32_t)(((uint64_t)w[it & 3] * (uint64_t)D) >> 32);
    keyed_block(seed, (uint64_t)d, 0, ORC_DOMAIN_PLACE, v);
    for (int c = 0; c < (dim == 3 ? 3 : 2); ++c) {
        const float u = (float)(v[c] >> 8) * 0x1p-23f - 1.0f;
        const float o = u * prm[1 + c];
        q[c] = q[c] + o;
    }
}

/* ---------------------------------------------------------------- S3: function pick
 * PAPER L17 "chooses a single function at random"; BJ "selection probabilities".
 * DESIGN R2: cumulative sums in double, T_j = floor(c_j / c_{n-1} * 2^32), T_{n-1} = 2^32,
 * k = #{ j < n-1 : u >= T_j }. */
int orc_thresholds(const float *prob, int n, uint64_t *T)
{
    if (n < 1) return -1;
    double total = 0.0;
    for (int j = 0; j < n; ++j) {
        if (!(prob[j] >= 0.0f) || isinf(prob[j])) return -1;   /* negative or NaN */
        total += (double)prob[j];
    }
    if (!(total > 0.0)) return -1;
    double c = 0.0;
    for (int j = 0; j < n; ++j) {
        c += (double)prob[j];
        T[j] = (uint64_t)floor(c / total * 4294967296.0);
    }
    T[n - 1] = 4294967296ull;
    return 0;
}

int orc_pick(uint32_t u, const uint64_t *T, int n)
{
    int k = 0;
    for (int j = 0; j < n - 1; ++j)
        if ((uint64_t)u >= T[j]) ++k;
    return k;
}

/* ---------------------------------------------------------------- S4: initial point
 * PAPER L41 "a single point randomly chosen in real space"; BJ cfg 0 "uniform in [-1,1]^2".
 * DESIGN R3: 24-bit uniform, every step exact in float32. */
void orc_init_point(uint64_t seed, uint64_t p, int dim, float g[3])
{
    uint32_t w[4];
    keyed_block(seed, p, 0, ORC_DOMAIN_INIT, w);
    g[0] = (float)(w[0] >> 8) * 0x1p-23f - 1.0f;
    g[1] = (float)(w[1] >> 8) * 0x1p-23f - 1.0f;
    g[2] = (dim == 3) ? (float)(w[2] >> 8) * 0x1p-23f - 1.0f : 0.0f;
}

/* ---------------------------------------------------------------- S5: generator map
 * "each function f_n maps some position P_n on to some new position P_{n+1}";
 * BJ cfg 0: f_i(p) = 0.5 p + 0.5 c_i.  Affine maps as nested single-rounding FMAs. */
static void affine_apply(const float *m, int dim, float v[3])
{
    float x = v[0], y = v[1], z = v[2];
    if (dim == 2) {
        v[0] = fmaf(m[0], x, fmaf(m[1], y, m[4]));
        v[1] = fmaf(m[2], x, fmaf(m[3], y, m[5]));
        /* z unchanged (0 for 2-D systems) */
    } else {
        v[0] = fmaf(m[0], x, fmaf(m[1], y, fmaf(m[2], z, m[9])));
        v[1] = fmaf(m[3], x, fmaf(m[4], y, fmaf(m[5], z, m[10])));
        v[2] = fmaf(m[6], x, fmaf(m[7], y, fmaf(m[8], z, m[11])));
    }
}

/* PAPER Eq. 1 (L49-58), the non-affine circle IFS: "functions to map the circle on to either the
 * top or bottom half of itself" (L60).  As printed, with the reading of DESIGN R13:
 *     r = sqrt(x^2 + y^2),  theta = atan(y/x) taken as the full-circle angle in [0, 2 pi),
 *     theta_2 = pi (r + f_id)        [flag: pi (r^2 + f_id)],
 *     r_2 = sqrt(theta / (2 pi)),
 *     x_2 = r_2 cos theta_2,  y_2 = r_2 sin theta_2      (the source prints "r^2": a mangled r_2).
 * Non-affine, hence tolerance-checked: evaluated in double on the float input, each output rounded
 * once (DESIGN R5).  z is left alone. */
static void circle_half_apply(const float *prm, float v[3])
{
    static const double PI = 3.14159265358979323846;
    const double x = (double)v[0], y = (double)v[1];
    const double fid = (double)prm[0];
    const double r = sqrt(x * x + y * y);
    double th = atan2(y, x);
    if (th < 0.0) th += 2.0 * PI;
    const double th2 = PI * ((prm[1] != 0.0f ? r * r : r) + fid);
    const double r2 = sqrt(th / (2.0 * PI));
    v[0] = (float)(r2 * cos(th2));
    v[1] = (float)(r2 * sin(th2));
}

void orc_apply_func(const orc_func *f, int dim, float g[3])
{
    if (f->type == ORC_F_CIRCLE_HALF) circle_half_apply(f->params, g);
    else affine_apply(f->params, dim, g);
}

/* ---------------------------------------------------------------- S6: chain transforms
 * arbitrary (non-affine) spatial transforms applied to a copy of
 * the point before it is written.  DESIGN R5: non-affine steps are evaluated in
 * double from the float inputs and each output coordinate is rounded once to float;
 * AFFINE and PINHOLE are float32 with a fixed association (bit-exact contract). */
static float resolve1(float p0, float p1, float t)
{
    return (float)((double)p0 + (double)t * (double)p1);
}

void orc_resolve_xform(const orc_xform *x, int dim, float t, int width, int height,
                       int *type_out, float prm[12])
{
    memset(prm, 0, 12 * sizeof(float));
    *type_out = x->type;
    switch (x->type) {
    case ORC_T_AFFINE:
        for (int i = 0; i < 12; ++i) prm[i] = resolve1(x->p0[i], x->p1[i], t);
        break;
    case ORC_T_ROTATE_Z: {
        /* angle in double, resolved once per render to an AFFINE [c -s; s c], b = 0 */
        double th = (double)x->p0[0] + (double)t * (double)x->p1[0];
        float c = (float)cos(th), s = (float)sin(th);
        *type_out = ORC_T_AFFINE;
        if (dim == 2) {
            prm[0] = c; prm[1] = -s; prm[2] = s; prm[3] = c; prm[4] = 0.0f; prm[5] = 0.0f;
        } else {
            prm[0] = c; prm[1] = -s; prm[2] = 0.0f;
            prm[3] = s; prm[4] = c;  prm[5] = 0.0f;
            prm[6] = 0.0f; prm[7] = 0.0f; prm[8] = 1.0f;
        }
        break;
    }
    case ORC_T_TWIST_Z:
    case ORC_T_BEND:
        prm[0] = resolve1(x->p0[0], x->p1[0], t);
        break;
    case ORC_T_PINHOLE: {
        /* params: fov_y (degrees), cam_z, near.  f = 1/tan(fov/2), fx = f*H/W */
        double fov = (double)x->p0[0] + (double)t * (double)x->p1[0];
        double f = 1.0 / tan(fov * (3.14159265358979323846 / 180.0) * 0.5);
        prm[0] = (float)(f * (double)height / (double)width);
        prm[1] = (float)f;
        prm[2] = resolve1(x->p0[1], x->p1[1], t);
        prm[3] = resolve1(x->p0[2], x->p1[2], t);
        break;
    }
    default: /* SWIRL, SINUSOIDAL, STRETCH_COS: no parameters */
        break;
    }
}

int orc_apply_xform(int type, const float *prm, int dim, float q[3])
{
    double x = q[0], y = q[1], z = q[2];
    switch (type) {
    case ORC_T_AFFINE:
        affine_apply(prm, dim, q);
        return 1;
    case ORC_T_SWIRL: {             /* BJ cfg 1 */
        double r2 = x * x + y * y, c = cos(r2), s = sin(r2);
        q[0] = (float)(x * c - y * s);
        q[1] = (float)(x * s + y * c);
        return 1;
    }
    case ORC_T_SINUSOIDAL:          /* BJ cfg 2 */
        q[0] = (float)sin(x);
        q[1] = (float)sin(y);
        return 1;
    case ORC_T_TWIST_Z: {           /* BJ cfg 3: rotate (x,y) by p*z */
        double a = (double)prm[0] * z, c = cos(a), s = sin(a);
        q[0] = (float)(x * c - y * s);
        q[1] = (float)(x * s + y * c);
        return 1;
    }
    case ORC_T_BEND: {              /* DESIGN R6: rotate (x,y) by kappa*x (input x) */
        double a = (double)prm[0] * x, c = cos(a), s = sin(a);
        q[0] = (float)(x * c - y * s);
        q[1] = (float)(x * s + y * c);
        return 1;
    }
    case ORC_T_PINHOLE: {           /* DESIGN R7: float32, IEEE division, fixed association */
        float d = q[2] - prm[2];
        if (!(d > prm[3])) return 0;
        float r = 1.0f / d;
        q[0] = (prm[0] * q[0]) * r;
        q[1] = (prm[1] * q[1]) * r;
        q[2] = d;
        return 1;
    }
    case ORC_T_STRETCH_COS:         /* PAPER L62-67, Eq. 2: x2 = 2x, y2 = y - cos(x) */
        q[0] = (float)(2.0 * x);
        q[1] = (float)(y - cos(x));
        return 1;
    default:
        return 0;
    }
}

/* ---------------------------------------------------------------- S7: pixel rule
 * PAPER L43 "the point is then splat or histogrammed on to screen" (no rule given).
 * DESIGN R8: closed bounds, floor of an FMA, clamp to the last pixel, row 0 = ymin. */
typedef struct { float sx, ox, sy, oy; } pixmap;

static pixmap make_pixmap(float xmin, float xmax, float ymin, float ymax, int W, int H)
{
    pixmap m;
    double wx = (double)xmax - (double)xmin, wy = (double)ymax - (double)ymin;
    m.sx = (float)((double)W / wx);
    m.ox = (float)(-(double)xmin * (double)W / wx);
    m.sy = (float)((double)H / wy);
    m.oy = (float)(-(double)ymin * (double)H / wy);
    return m;
}

static int64_t pixel_of(const pixmap *m, float x, float y, float xmin, float xmax,
                        float ymin, float ymax, int W, int H)
{
    if (!(x >= xmin && x <= xmax && y >= ymin && y <= ymax)) return -1;  /* NaN -> out */
    int px = (int)floorf(fmaf(x, m->sx, m->ox));
    int py = (int)floorf(fmaf(y, m->sy, m->oy));
    if (px < 0) px = 0;
    if (px > W - 1) px = W - 1;
    if (py < 0) py = 0;
    if (py > H - 1) py = H - 1;
    return (int64_t)py * W + px;
}

int64_t orc_pixel(float x, float y, float xmin, float xmax, float ymin, float ymax, int W, int H)
{
    pixmap m = make_pixmap(xmin, xmax, ymin, ymax, W, H);
    return pixel_of(&m, x, y, xmin, xmax, ymin, ymax, W, H);
}

/* ---------------------------------------------------------------- S8: colour
 * "the colors indicate the function used on each individual point to land
 * on its final position".  DESIGN R9: colours are integer-valued 0..255 floats. */
static uint32_t pack_rgba8(const float *c)
{
    uint32_t out = 0;
    for (int i = 0; i < 4; ++i) {
        float v = floorf(c[i] + 0.5f);
        if (!(v >= 0.0f)) v = 0.0f;
        if (v > 255.0f) v = 255.0f;
        out |= (uint32_t)v << (8 * i);
    }
    return out;
}

/* ---------------------------------------------------------------- validation */
static int validate(const orc_system *s, const orc_render_args *a)
{
    if (!s || !a) return -1;
    if (s->dim != 2 && s->dim != 3) return -1;
    if (s->n_chain < 0 || s->n_chain > 8) return -1;
    if (s->gen_kind == ORC_GEN_IFS) {
        if (s->n_funcs < 1 || s->n_funcs > 64 || !s->funcs) return -1;
        if (a->iterations < 1 || a->burn_in < 0 || a->burn_in >= a->iterations) return -1;
        if (s->color_rule == ORC_COLOR_POINT) return -1;
        if (s->color_rule == ORC_COLOR_MAP_INDEX && !s->palette) return -1;
    } else if (s->gen_kind == ORC_GEN_CLOUD) {
        if (a->iterations != 1 || a->burn_in != 0) return -1;
        if (a->n_points && !a->cloud) return -1;
        if (s->color_rule == ORC_COLOR_MAP_INDEX) return -1;
    } else return -1;
    if (a->width < 1 || a->height < 1 || (int64_t)a->width * a->height > 2147483647ll) return -1;
    if (!(a->xmax > a->xmin) || !(a->ymax > a->ymin)) return -1;
    if (a->out_mode == ORC_OUT_HIST_U32) { /* colour ignored */ }
    else if (a->out_mode == ORC_OUT_RGBA) { if (s->color_rule == ORC_COLOR_NONE) return -1; }
    else if (a->out_mode == ORC_OUT_DEPTH_U64) {
        if (s->color_rule == ORC_COLOR_NONE || s->dim != 3) return -1;
        if (s->n_chain < 1) return -1;
        for (int m = 0; m <= s->n_chain; ++m)        /* every branch ends in PINHOLE */
            if ((m == s->n_chain || s->chain[m].type == ORC_T_BRANCH) && (m == 0 || s->chain[m - 1].type != ORC_T_PINHOLE)) return -1;
    } else return -1;
    return 0;
}

/* ---------------------------------------------------------------- S7 + S8: one splat */
static void splat_one(const orc_system *s, const orc_render_args *a, const pixmap *pm, const float q[3], int alive,
                      int k, uint32_t point_rgba8, uint64_t *n_in, uint64_t *n_drop)
{
    int64_t pix = alive ? pixel_of(pm, q[0], q[1], a->xmin, a->xmax, a->ymin, a->ymax, a->width, a->height) : -1;
    if (pix < 0) { ++*n_drop; return; }
    ++*n_in;
    if (a->out_mode == ORC_OUT_HIST_U32) {
        ((uint32_t *)a->image)[pix] += 1u;
    } else if (a->out_mode == ORC_OUT_RGBA) {
        double *acc = (double *)a->image + 4 * pix;
        if (s->color_rule == ORC_COLOR_MAP_INDEX) {
            const float *c = s->palette + 4 * k;
            acc[0] += (double)c[0]; acc[1] += (double)c[1]; acc[2] += (double)c[2];
        } else {
            acc[0] += (double)(point_rgba8 & 0xFFu);
            acc[1] += (double)((point_rgba8 >> 8) & 0xFFu);
            acc[2] += (double)((point_rgba8 >> 16) & 0xFFu);
        }
        acc[3] += 1.0;
    } else {
        /* BJ cfg 4: nearest-point depth test via packed (float depth | rgba8) min */
        uint32_t col = (s->color_rule == ORC_COLOR_MAP_INDEX) ? pack_rgba8(s->palette + 4 * k) : point_rgba8;
        uint32_t dbits;
        memcpy(&dbits, &q[2], 4);
        uint64_t key = ((uint64_t)dbits << 32) | col;
        uint64_t *buf = (uint64_t *)a->image + pix;
        if (key < *buf) *buf = key;
    }
}

/* ---------------------------------------------------------------- S1: the loop */
static int run(const orc_system *s, const orc_render_args *a, int do_splat, uint8_t *picks,
               float *final_g, float *final_q, uint8_t *final_alive)
{
    if (validate(s, a)) return -1;
    uint64_t T[64];
    if (s->gen_kind == ORC_GEN_IFS) {
        float prob[64];
        for (int j = 0; j < s->n_funcs; ++j) {
            if (s->funcs[j].type != ORC_F_AFFINE && !(s->funcs[j].type == ORC_F_CIRCLE_HALF && s->dim == 2)) return -1;
            prob[j] = s->funcs[j].prob;
        }
        if (orc_thresholds(prob, s->n_funcs, T)) return -1;
    }
    int ctype[8];
    float cprm[8][12];
    for (int m = 0; m < s->n_chain; ++m) {
        if (s->chain[m].type < 0 || s->chain[m].type > ORC_T_SCATTER) return -1;
        if (s->chain[m].type == ORC_T_SCATTER) {       /* parameters at t like any other step; D in [1, 2^20] */
            for (int i = 0; i < 4; ++i)
                cprm[m][i] = (float)((double)s->chain[m].p0[i] + (double)a->t * (double)s->chain[m].p1[i]);
            if (!(cprm[m][0] >= 1.0f && cprm[m][0] <= 1048576.0f) || cprm[m][0] != (float)(uint32_t)cprm[m][0]) return -1;
            ctype[m] = ORC_T_SCATTER;
            continue;
        }
        if (s->chain[m].type == ORC_T_BRANCH) {
            if (s->reuse) return -1;              /* which branch would be fed back? */
            ctype[m] = ORC_T_BRANCH;
            continue;
        }
        orc_resolve_xform(&s->chain[m], s->dim, a->t, a->width, a->height, &ctype[m], cprm[m]);
    }
    pixmap pm = make_pixmap(a->xmin, a->xmax, a->ymin, a->ymax, a->width, a->height);
    uint64_t n_in = 0, n_drop = 0;

    for (uint64_t i = 0; i < a->n_points; ++i) {
        uint64_t p = a->point_offset + i;
        float g[3], q[3] = { 0.0f, 0.0f, 0.0f };
        int alive = 0;
        uint32_t point_rgba8 = 0;
        if (s->gen_kind == ORC_GEN_CLOUD) {       /* any source of points */
            g[0] = a->cloud[p].x; g[1] = a->cloud[p].y;
            g[2] = (s->dim == 3) ? a->cloud[p].z : 0.0f;
            point_rgba8 = a->cloud[p].rgba8;
        } else {
            orc_init_point(a->seed, p, s->dim, g);
        }
        for (int32_t it = 0; it < a->iterations; ++it) {
            int k = 0;
            if (s->gen_kind == ORC_GEN_IFS) {
                k = orc_pick(orc_pick_word(a->seed, p, (uint32_t)it), T, s->n_funcs);
                if (picks) picks[i * (uint64_t)a->iterations + (uint64_t)it] = (uint8_t)k;
                orc_apply_func(&s->funcs[k], s->dim, g);
            }
            if (it < a->burn_in && !s->reuse) continue;
            /* PAPER L77 / Fig. 2(B): a copy of the point goes through the chain.  PAPER L192-198 ("many
             * objects from a single primitive"): a chain may hold several BRANCHes; each is applied to its
             * own copy of the generated point and splatted, so one point drives M splats per iteration. */
            for (int m0 = 0; m0 <= s->n_chain; ) {
                q[0] = g[0]; q[1] = g[1]; q[2] = g[2];
                alive = 1;
                int m = m0;
                for (; m < s->n_chain && ctype[m] != ORC_T_BRANCH; ++m)
                    if (alive) {
                        if (ctype[m] == ORC_T_SCATTER) orc_scatter(a->seed, p, (uint32_t)it, cprm[m], s->dim, q);
                        else alive = orc_apply_xform(ctype[m], cprm[m], s->dim, q);
                    }
                m0 = m + 1;                       /* past the BRANCH marker (or past the end) */
                if (s->reuse) {                   /* Fig. 2(C): the same point is reused (single branch) */
                    g[0] = q[0]; g[1] = q[1]; g[2] = q[2];
                    if (it < a->burn_in) continue;
                }
                if (!do_splat) continue;
                splat_one(s, a, &pm, q, alive, k, point_rgba8, &n_in, &n_drop);
            }
        }
        if (final_g) { final_g[3 * i] = g[0]; final_g[3 * i + 1] = g[1]; final_g[3 * i + 2] = g[2]; }
        if (final_q) { final_q[3 * i] = q[0]; final_q[3 * i + 1] = q[1]; final_q[3 * i + 2] = q[2]; }
        if (final_alive) final_alive[i] = (uint8_t)alive;
    }
    if (do_splat && a->counters) { a->counters[0] += n_in; a->counters[1] += n_drop; }
    return 0;
}

int orc_render(const orc_system *s, const orc_render_args *a)
{
    if (a && a->n_points && !a->image) return -1;
    return run(s, a, 1, NULL, NULL, NULL, NULL);
}

int orc_trace(const orc_system *s, const orc_render_args *a, uint8_t *picks,
              float *final_g, float *final_q, uint8_t *final_alive)
{
    return run(s, a, 0, picks, final_g, final_q, final_alive);
}

/* ---------------------------------------------------------------- S9: tone map
 * Not in the paper; BJ: "cfs_tonemap does log-density tone mapping" (fractal-flame
 * convention).  DESIGN R10.  Evaluated in double. */
int orc_tonemap(const void *image, int out_mode, int W, int H, float gamma, float colour_scale,
                uint32_t *out)
{
    if (!image || !out || W < 1 || H < 1 || !(gamma > 0.0f)) return -1;
    int64_t n = (int64_t)W * H;
    if (out_mode == ORC_OUT_DEPTH_U64) {          /* no density: resolve = colour, empty -> 0 */
        const uint64_t *b = (const uint64_t *)image;
        for (int64_t i = 0; i < n; ++i)
            out[i] = (b[i] == 0xFFFFFFFFFFFFFFFFull) ? 0u : (uint32_t)(b[i] & 0xFFFFFFFFu);
        return 0;
    }
    double nmax = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        double c = (out_mode == ORC_OUT_HIST_U32) ? (double)((const uint32_t *)image)[i]
                                                  : (double)((const float *)image)[4 * i + 3];
        if (c > nmax) nmax = c;
    }
    double inv_g = 1.0 / (double)gamma;
    for (int64_t i = 0; i < n; ++i) {
        double c = (out_mode == ORC_OUT_HIST_U32) ? (double)((const uint32_t *)image)[i]
                                                  : (double)((const float *)image)[4 * i + 3];
        if (!(c > 0.0)) { out[i] = 0u; continue; }
        double L = log1p(c) / log1p(nmax);
        double Lg = pow(L, inv_g);
        double v[4];
        if (out_mode == ORC_OUT_HIST_U32) {
            v[0] = v[1] = v[2] = Lg;
        } else {
            const float *px = (const float *)image + 4 * i;
            for (int ch = 0; ch < 3; ++ch) v[ch] = (double)colour_scale * (double)px[ch] / c * Lg;
        }
        v[3] = L;
        uint32_t o = 0;
        for (int ch = 0; ch < 4; ++ch) {
            double x = v[ch];
            if (!(x >= 0.0)) x = 0.0;
            if (x > 1.0) x = 1.0;
            o |= (uint32_t)floor(255.0 * x + 0.5) << (8 * ch);
        }
        out[i] = o;
    }
    return 0;
}
