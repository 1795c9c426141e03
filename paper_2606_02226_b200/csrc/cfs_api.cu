// cfs_api.cu -- C ABI of the CFS hot path (include/cfs.h): validation, host-side resolution of
// tables and frame-dependent parameters, kernel selection and launch.  No CPU fallback.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <map>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "../../include/cfs.h"
#include "cfs_bin.cuh"
#include "cfs_cloud.cuh"
#include "cfs_hiz.cuh"
#include "cfs_jit.h"
#include "cfs_device.cuh"
#include "cfs_microbench.cuh"
#include "cfs_registry.h"
#include "cfs_tonemap.cuh"

static_assert((int)CFS_T_AFFINE == (int)cfs::T_AFFINE && (int)CFS_T_SWIRL == (int)cfs::T_SWIRL &&
              (int)CFS_T_SINUSOIDAL == (int)cfs::T_SINUSOIDAL && (int)CFS_T_ROTATE_Z == (int)cfs::T_ROTATE_Z &&
              (int)CFS_T_TWIST_Z == (int)cfs::T_TWIST_Z && (int)CFS_T_BEND == (int)cfs::T_BEND &&
              (int)CFS_T_PINHOLE == (int)cfs::T_PINHOLE && (int)CFS_T_STRETCH_COS == (int)cfs::T_STRETCH_COS &&
              (int)CFS_T_BRANCH == (int)cfs::T_BRANCH && (int)CFS_T_SCATTER == (int)cfs::T_SCATTER,
              "chain type ids");
static_assert(CFS_MAX_FUNCS == cfs::kMaxFuncs && CFS_MAX_CHAIN == cfs::kMaxChain, "limits");
static_assert(sizeof(cfs_cloud_rec) == 16, "cloud record is one 128-bit load");
static_assert(sizeof(cfs::RenderParams) < 16 * 1024, "parameter block");

namespace {

thread_local char g_err[512] = "";
thread_local uint64_t g_launches = 0;

cfs_status fail(cfs_status st, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return st;
}

cfs_status cuda_fail(cudaError_t e, const char *what)
{
    return fail(CFS_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

struct DeviceInfo { int ok = -1; int dev = -1; int sms = 0; int smem_optin = 0; int smem_sm = 0; int cc = 0; };

constexpr int kMaxDevices = 64;
std::mutex g_dev_mutex;
DeviceInfo g_dev[kMaxDevices];          // one entry per device ordinal, filled on first use

// attributes of the CURRENT device of the calling thread (a thread may switch devices between calls)
const DeviceInfo &device_info()
{
    static const DeviceInfo none = [] { DeviceInfo d; d.ok = 0; return d; }();
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return none; }
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    DeviceInfo &di = g_dev[dev];
    if (di.ok < 0) {
        int major = 0, minor = 0;
        cudaDeviceGetAttribute(&di.sms, cudaDevAttrMultiProcessorCount, dev);
        cudaDeviceGetAttribute(&di.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        cudaDeviceGetAttribute(&di.smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
        cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev);
        di.cc = major * 10 + minor;
        di.dev = dev;
        di.ok = (di.sms > 0) ? 1 : 0;
        if (di.ok != 1) cudaGetLastError();
    }
    return di;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is sticky per (function, device): set it once, and again only
// when a render needs more than any before it
std::map<std::pair<const void *, int>, int> g_dyn_smem;

cudaError_t ensure_dyn_smem(const void *fn, size_t bytes)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    int &have = g_dyn_smem[std::make_pair(fn, dev)];
    if ((int)bytes <= have) return cudaSuccess;
    e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) have = (int)bytes;
    return e;
}

}  // namespace

// -------------------------------------------------------------------------------------------------
struct cfs_system {
    int32_t dim = 2, gen = 0, color = 0, reuse = 0;
    std::vector<cfs_func> funcs;
    std::vector<cfs_xform> chain;
    std::vector<float> palette;
    // pick tables (DESIGN R2)
    uint32_t T[cfs::kMaxFuncs];
    uint32_t lut[256][2];
    int32_t n_thr = 0, pick_steps = 0, pick_shift = -1;
    bool pick_mulhi = false;     // T_j == floor((j + 1) 2^32 / n) for every j < n - 1: the pick is one 64-bit multiply (run-time compiled kernels)
    int32_t aff = cfs::AFF_GENERAL;
    bool uscale_ok = false;      // AFF_DIAG and every map has the same scale: AFF_USCALE table available (run-time compiled kernels)
    float coef[cfs::kMaxFuncs * 12];
    uint32_t pal8[cfs::kMaxFuncs];
    // scratch of cfs_render_host (device), cached
    void *d_image = nullptr; size_t image_bytes = 0;
    void *d_cloud = nullptr; size_t cloud_bytes = 0;
    unsigned long long *d_counters = nullptr;
    void *d_scratch = nullptr; size_t scratch_bytes = 0;
    void *d_rgba8 = nullptr; size_t rgba8_bytes = 0;       // cfs_render_rgba8_host
    void *d_tone = nullptr;                                // 16 bytes: scratch of the resolve
};

namespace {

bool bad_float(float v) { return std::isnan(v) || std::isinf(v); }

uint32_t pack_rgba8(const float *c)
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

// thresholds, bucket table and the affine table form
cfs_status build_tables(cfs_system *s)
{
    const int n = (int)s->funcs.size();
    double total = 0.0;
    for (int j = 0; j < n; ++j) {
        const float p = s->funcs[j].prob;
        if (!(p >= 0.0f) || std::isinf(p)) return fail(CFS_ERR_INVALID_ARG, "funcs[%d].prob must be finite and >= 0", j);
        total += (double)p;
    }
    if (!(total > 0.0)) return fail(CFS_ERR_INVALID_ARG, "sum of probabilities must be > 0");
    uint64_t T64[cfs::kMaxFuncs];
    double c = 0.0;
    for (int j = 0; j < n; ++j) {
        c += (double)s->funcs[j].prob;
        T64[j] = (uint64_t)floor(c / total * 4294967296.0);
    }
    s->n_thr = 0;
    for (int j = 0; j < n - 1; ++j)
        if (T64[j] < 4294967296ull) s->n_thr = j + 1;          // T is non-decreasing
    for (int j = 0; j < cfs::kMaxFuncs; ++j) s->T[j] = (j < s->n_thr) ? (uint32_t)T64[j] : 0xFFFFFFFFu;
    s->pick_steps = 0;
    for (int b = 0; b < 256; ++b) {
        const uint64_t lo = (uint64_t)b << 24, hi = lo + 0xFFFFFFull;
        int below = 0, inside = 0;
        uint32_t first_m1 = 0xFFFFFFFFu;                          // none: u > 0xFFFFFFFF never holds
        for (int j = 0; j < s->n_thr; ++j) {
            if (T64[j] <= lo) ++below;
            else if (T64[j] <= hi) { if (!inside) first_m1 = (uint32_t)(T64[j] - 1); ++inside; }    // T > lo >= 0, so T - 1 >= 0
        }
        s->lut[b][0] = ~first_m1;             // complemented: the device adds it to u and takes the carry (pick_index)
        s->lut[b][1] = (uint32_t)below;
        if (inside > s->pick_steps) s->pick_steps = inside;
    }
    // equal thresholds of any n: k = (u n + n - 1) >> 32 (pick_index has the proof; a power-of-two n takes the shift below)
    s->pick_mulhi = (n >= 3 && (n & (n - 1)) != 0 && s->n_thr == n - 1);
    for (int j = 0; j < n - 1 && s->pick_mulhi; ++j)
        if (T64[j] != (((uint64_t)(j + 1)) << 32) / (uint64_t)n) s->pick_mulhi = false;
    // equal power-of-two thresholds: k = u >> shift
    s->pick_shift = -1;
    if (n >= 1 && (n & (n - 1)) == 0 && s->n_thr == n - 1) {
        int lg = 0;
        while ((1 << lg) < n) ++lg;
        bool ok = true;
        for (int j = 0; j < n - 1; ++j) ok = ok && (T64[j] == ((uint64_t)(j + 1) << (32 - lg)));
        if (ok && lg >= 1) s->pick_shift = 32 - lg;
        if (n == 1) { s->pick_shift = -1; }
    }
    // affine form: DIAG when every off-diagonal coefficient is exactly zero
    bool diag = true;
    for (int j = 0; j < n; ++j) {
        const float *m = s->funcs[j].params;
        if (s->dim == 2) diag = diag && m[1] == 0.0f && m[2] == 0.0f;
        else diag = diag && m[1] == 0.0f && m[2] == 0.0f && m[3] == 0.0f && m[5] == 0.0f && m[6] == 0.0f && m[7] == 0.0f;
    }
    const bool circle = n >= 1 && s->funcs[0].type == CFS_F_CIRCLE_HALF;     // all of them are (cfs_create)
    s->aff = circle ? cfs::AFF_CIRCLE : diag ? cfs::AFF_DIAG : cfs::AFF_GENERAL;
    s->uscale_ok = (s->aff == cfs::AFF_DIAG);
    for (int j = 1; j < n && s->uscale_ok; ++j) {
        const float *m = s->funcs[j].params, *m0 = s->funcs[0].params;
        s->uscale_ok = (s->dim == 2) ? (m[0] == m0[0] && m[3] == m0[3]) : (m[0] == m0[0] && m[4] == m0[4] && m[8] == m0[8]);
    }
    memset(s->coef, 0, sizeof(s->coef));
    for (int j = 0; j < n; ++j) {
        const float *m = s->funcs[j].params;
        if (circle) {
            float *r = s->coef + 4 * j;  r[0] = m[0]; r[1] = (m[1] != 0.0f) ? 1.0f : 0.0f;
        } else if (s->dim == 2 && diag) {
            float *r = s->coef + 4 * j;  r[0] = m[0]; r[1] = m[3]; r[2] = m[4]; r[3] = m[5];
        } else if (s->dim == 2) {
            float *r = s->coef + 8 * j;  r[0] = m[0]; r[1] = m[1]; r[2] = m[4]; r[4] = m[2]; r[5] = m[3]; r[6] = m[5];
        } else if (diag) {
            float *r = s->coef + 8 * j;  r[0] = m[0]; r[1] = m[4]; r[2] = m[8]; r[4] = m[9]; r[5] = m[10]; r[6] = m[11];
        } else {
            float *r = s->coef + 12 * j;
            for (int row = 0; row < 3; ++row) {
                r[4 * row + 0] = m[3 * row + 0]; r[4 * row + 1] = m[3 * row + 1];
                r[4 * row + 2] = m[3 * row + 2]; r[4 * row + 3] = m[9 + row];
            }
        }
    }
    return CFS_OK;
}

}  // namespace

extern "C" cfs_status cfs_create(cfs_system **out, int32_t dim, int32_t gen_kind, const cfs_func *funcs,
                                 int32_t n_funcs, const cfs_xform *chain, int32_t n_chain,
                                 int32_t color_rule, const float *palette_rgba, int32_t reuse)
{
    if (!out) return fail(CFS_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (dim != 2 && dim != 3) return fail(CFS_ERR_INVALID_ARG, "dim must be 2 or 3");
    if (gen_kind != CFS_GEN_IFS && gen_kind != CFS_GEN_CLOUD) return fail(CFS_ERR_INVALID_ARG, "unknown generator kind %d", gen_kind);
    if (n_chain < 0 || n_chain > CFS_MAX_CHAIN || (n_chain > 0 && !chain)) return fail(CFS_ERR_INVALID_ARG, "n_chain must be 0..%d", CFS_MAX_CHAIN);
    if (color_rule < CFS_COLOR_NONE || color_rule > CFS_COLOR_POINT) return fail(CFS_ERR_INVALID_ARG, "unknown colour rule %d", color_rule);
    cfs_system *s = new (std::nothrow) cfs_system();
    if (!s) return fail(CFS_ERR_NOMEM, "out of host memory");
    s->dim = dim; s->gen = gen_kind; s->color = color_rule; s->reuse = reuse ? 1 : 0;
    cfs_status st = CFS_OK;
    if (gen_kind == CFS_GEN_IFS) {
        if (n_funcs < 1 || n_funcs > CFS_MAX_FUNCS || !funcs) st = fail(CFS_ERR_INVALID_ARG, "n_funcs must be 1..%d", CFS_MAX_FUNCS);
        if (st == CFS_OK && color_rule == CFS_COLOR_POINT) st = fail(CFS_ERR_INVALID_ARG, "COLOR_POINT needs a CLOUD generator");
        if (st == CFS_OK && color_rule == CFS_COLOR_MAP_INDEX && !palette_rgba) st = fail(CFS_ERR_INVALID_ARG, "COLOR_MAP_INDEX needs a palette");
        for (int j = 0; st == CFS_OK && j < n_funcs; ++j) {
            if (funcs[j].type != CFS_F_AFFINE && funcs[j].type != CFS_F_CIRCLE_HALF) st = fail(CFS_ERR_INVALID_ARG, "funcs[%d]: unknown type %d", j, funcs[j].type);
            if (st == CFS_OK && funcs[j].type != funcs[0].type) st = fail(CFS_ERR_UNSUPPORTED, "funcs[%d]: AFFINE and CIRCLE_HALF maps cannot share a generator", j);
            if (st == CFS_OK && funcs[j].type == CFS_F_CIRCLE_HALF && dim != 2) st = fail(CFS_ERR_INVALID_ARG, "CIRCLE_HALF is a 2-D map");
            if (st == CFS_OK && funcs[j].type == CFS_F_CIRCLE_HALF && funcs[j].params[0] != 0.0f && funcs[j].params[0] != 1.0f)
                st = fail(CFS_ERR_INVALID_ARG, "funcs[%d]: CIRCLE_HALF f_id must be 0 or 1", j);
            const int np = (funcs[j].type == CFS_F_CIRCLE_HALF) ? 2 : (dim == 2) ? 6 : 12;
            for (int i = 0; st == CFS_OK && i < np; ++i)
                if (bad_float(funcs[j].params[i])) st = fail(CFS_ERR_INVALID_ARG, "funcs[%d].params[%d] is not finite", j, i);
        }
        if (st == CFS_OK) {
            s->funcs.assign(funcs, funcs + n_funcs);
            st = build_tables(s);
        }
        if (st == CFS_OK && color_rule == CFS_COLOR_MAP_INDEX) {
            s->palette.assign(palette_rgba, palette_rgba + 4 * n_funcs);
            for (int j = 0; j < n_funcs; ++j) s->pal8[j] = pack_rgba8(palette_rgba + 4 * j);
        }
    } else {
        if (color_rule == CFS_COLOR_MAP_INDEX) st = fail(CFS_ERR_INVALID_ARG, "COLOR_MAP_INDEX needs an IFS generator");
    }
    for (int m = 0; st == CFS_OK && m < n_chain; ++m) {
        if (chain[m].type < CFS_T_AFFINE || chain[m].type > CFS_T_SCATTER) st = fail(CFS_ERR_INVALID_ARG, "chain[%d]: unknown type %d", m, chain[m].type);
        if (st == CFS_OK && chain[m].type == CFS_T_BRANCH && reuse) st = fail(CFS_ERR_INVALID_ARG, "chain[%d]: BRANCH cannot be combined with reuse", m);
        for (int i = 0; st == CFS_OK && i < 12; ++i)
            if (bad_float(chain[m].p0[i]) || bad_float(chain[m].p1[i])) st = fail(CFS_ERR_INVALID_ARG, "chain[%d] parameter %d is not finite", m, i);
    }
    if (st != CFS_OK) { delete s; return st; }
    if (n_chain) s->chain.assign(chain, chain + n_chain);
    *out = s;
    return CFS_OK;
}

extern "C" void cfs_destroy(cfs_system *s)
{
    if (!s) return;
    if (s->d_image) cudaFree(s->d_image);
    if (s->d_cloud) cudaFree(s->d_cloud);
    if (s->d_counters) cudaFree(s->d_counters);
    if (s->d_scratch) cudaFree(s->d_scratch);
    if (s->d_rgba8) cudaFree(s->d_rgba8);
    if (s->d_tone) cudaFree(s->d_tone);
    delete s;
}

// -------------------------------------------------------------------------------------------------
namespace {

using cfs::RenderParams;

// per-render host resolution: validation, chain parameters at t, pixel map, round keys
cfs_status build_params(const cfs_system *s, const cfs_render_args *a, RenderParams *out, bool need_image)
{
    if (!s || !a) return fail(CFS_ERR_INVALID_ARG, "system or args is NULL");
    if (a->flags & ~(CFS_FLAG_FAST_TRIG | CFS_FLAG_INTERPRET_CHAIN | CFS_FLAG_BIN_PASS1_ONLY | CFS_FLAG_JIT | CFS_FLAG_BIN_HYBRID)) return fail(CFS_ERR_INVALID_ARG, "unknown flags 0x%x", a->flags);
    if (a->iterations < 1) return fail(CFS_ERR_INVALID_ARG, "iterations must be >= 1");
    if (a->burn_in < 0 || a->burn_in >= a->iterations) return fail(CFS_ERR_INVALID_ARG, "burn_in must be in [0, iterations)");
    if (s->gen == CFS_GEN_CLOUD && (a->iterations != 1 || a->burn_in != 0)) return fail(CFS_ERR_INVALID_ARG, "CLOUD generator needs iterations = 1, burn_in = 0");
    if (a->width < 1 || a->height < 1 || (int64_t)a->width * a->height > 2147483647ll) return fail(CFS_ERR_INVALID_ARG, "bad image size %d x %d", a->width, a->height);
    if (bad_float(a->xmin) || bad_float(a->xmax) || bad_float(a->ymin) || bad_float(a->ymax) || !(a->xmax > a->xmin) || !(a->ymax > a->ymin))
        return fail(CFS_ERR_INVALID_ARG, "bounds must be finite with max > min");
    if (bad_float(a->t)) return fail(CFS_ERR_INVALID_ARG, "t is not finite");
    if (a->out_mode < CFS_OUT_HIST_U32 || a->out_mode > CFS_OUT_DEPTH_RGBA8_U64) return fail(CFS_ERR_INVALID_ARG, "unknown out_mode %d", a->out_mode);
    if (a->out_mode == CFS_OUT_RGBA_F32 && s->color == CFS_COLOR_NONE) return fail(CFS_ERR_INVALID_ARG, "RGBA output needs a colour rule");
    if (a->out_mode == CFS_OUT_DEPTH_RGBA8_U64) {
        if (s->color == CFS_COLOR_NONE || s->dim != 3) return fail(CFS_ERR_INVALID_ARG, "DEPTH output needs dim 3 and a colour rule");
        if (s->chain.empty()) return fail(CFS_ERR_INVALID_ARG, "DEPTH output needs a chain ending in PINHOLE");
        for (size_t m = 0; m <= s->chain.size(); ++m)       // every branch ends in PINHOLE
            if ((m == s->chain.size() || s->chain[m].type == CFS_T_BRANCH) && (m == 0 || s->chain[m - 1].type != CFS_T_PINHOLE))
                return fail(CFS_ERR_INVALID_ARG, "DEPTH output needs every branch of the chain to end in PINHOLE");
    }
    if (need_image && a->n_points && !a->d_image) return fail(CFS_ERR_INVALID_ARG, "d_image is NULL");
    if (need_image && a->n_points && s->gen == CFS_GEN_CLOUD && !a->d_cloud) return fail(CFS_ERR_INVALID_ARG, "d_cloud is NULL");
    if (a->out_mode == CFS_OUT_RGBA_F32 && ((uintptr_t)a->d_image & 15)) return fail(CFS_ERR_INVALID_ARG, "RGBA image must be 16-byte aligned");
    if (a->out_mode == CFS_OUT_DEPTH_RGBA8_U64 && ((uintptr_t)a->d_image & 7)) return fail(CFS_ERR_INVALID_ARG, "DEPTH image must be 8-byte aligned");
    if (s->gen == CFS_GEN_CLOUD && ((uintptr_t)a->d_cloud & 15)) return fail(CFS_ERR_INVALID_ARG, "cloud must be 16-byte aligned");

    RenderParams &p = *out;
    memset(&p, 0, sizeof(p));
    p.n_points = a->n_points; p.point_offset = a->point_offset;
    uint32_t k0 = (uint32_t)(a->seed & 0xFFFFFFFFu), k1 = (uint32_t)(a->seed >> 32);
    for (int r = 0; r < 10; ++r) { p.rk[r][0] = k0; p.rk[r][1] = k1; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    p.iterations = a->iterations; p.burn_in = a->burn_in;
    p.W = a->width; p.H = a->height;
    p.xmin = a->xmin; p.xmax = a->xmax; p.ymin = a->ymin; p.ymax = a->ymax;
    const double wx = (double)a->xmax - (double)a->xmin, wy = (double)a->ymax - (double)a->ymin;
    p.sx = (float)((double)a->width / wx);  p.ox = (float)(-(double)a->xmin * (double)a->width / wx);
    p.sy = (float)((double)a->height / wy); p.oy = (float)(-(double)a->ymin * (double)a->height / wy);
    p.image = a->d_image; p.cloud = a->d_cloud; p.counters = (unsigned long long *)a->d_counters;
    p.dim = s->dim; p.n_funcs = (int)s->funcs.size(); p.n_chain = (int)s->chain.size();
    // colour rule AS THE OUTPUT USES IT: a histogram ignores colour whatever the system was created with
    // (include/cfs.h, oracle: "colour ignored"), so the kernels see COLOR_NONE there -- the tile bins key
    // their record layout (one counter per pixel against one per pixel and map) on this field
    p.color_rule = (a->out_mode == CFS_OUT_HIST_U32) ? (int)CFS_COLOR_NONE : s->color;
    p.reuse = s->reuse; p.fast_trig = (a->flags & CFS_FLAG_FAST_TRIG) ? 1 : 0;
    p.pick_shift = s->pick_shift; p.n_thr = s->n_thr; p.pick_steps = s->pick_steps;
    p.aff_form = s->aff;
    {   // coefficient rows are replicated in shared memory (up to 8 copies) when more than 8 of them are in
        // use: with fewer, every row already has a bank group of its own
        const uint32_t rows_per_map = (s->aff == cfs::AFF_CIRCLE) ? 1u : (s->aff == cfs::AFF_DIAG) ? (s->dim == 2 ? 1u : 2u) : (s->dim == 2 ? 2u : 3u);
        p.coef_rows = (uint32_t)s->funcs.size() * rows_per_map;
        p.coef_cshift = 0;
        if (p.coef_rows > 8) while (p.coef_cshift < 3 && (p.coef_rows << (p.coef_cshift + 1)) <= (uint32_t)cfs::kCoefSlots) ++p.coef_cshift;
        p.coef_rstride = 16u << p.coef_cshift; p.coef_kstride = rows_per_map * p.coef_rstride;
    }
    memcpy(p.T, s->T, sizeof(p.T)); memcpy(p.lut, s->lut, sizeof(p.lut));
    memcpy(p.coef, s->coef, sizeof(p.coef)); memcpy(p.pal8, s->pal8, sizeof(p.pal8));
    if (!s->palette.empty()) memcpy(p.palette, s->palette.data(), s->palette.size() * sizeof(float));

    // chain parameters at t: (float)((double)p0 + (double)t*(double)p1)
    const double t = (double)a->t;
    p.n_branches = 1;
    for (int m = 0; m < p.n_chain; ++m) if (s->chain[m].type == CFS_T_BRANCH) ++p.n_branches;
    for (int m = 0; m < p.n_chain; ++m) {
        const cfs_xform &x = s->chain[m];
        cfs::ChainStep &st = p.chain[m];
        st.type = x.type;
        auto res = [&](int i) { return (float)((double)x.p0[i] + t * (double)x.p1[i]); };
        switch (x.type) {
        case CFS_T_AFFINE: {
            for (int i = 0; i < 12; ++i) st.p[i] = res(i);
            // zero off-diagonals: the internal SCALE step, bit-identical because fma(0, y, b) == b
            const bool diag = (s->dim == 2) ? (st.p[1] == 0.0f && st.p[2] == 0.0f)
                                            : (st.p[1] == 0.0f && st.p[2] == 0.0f && st.p[3] == 0.0f && st.p[5] == 0.0f &&
                                               st.p[6] == 0.0f && st.p[7] == 0.0f);
            if (diag) st.type = cfs::T_SCALE;
            break;
        }
        case CFS_T_ROTATE_Z: {   // resolved once per render to an AFFINE rotation (DESIGN R5)
            const double th = (double)x.p0[0] + t * (double)x.p1[0];
            const float c = (float)cos(th), sn = (float)sin(th);
            st.type = CFS_T_AFFINE;
            if (s->dim == 2) { st.p[0] = c; st.p[1] = -sn; st.p[2] = sn; st.p[3] = c; }
            else { st.p[0] = c; st.p[1] = -sn; st.p[3] = sn; st.p[4] = c; st.p[8] = 1.0f; }
            break;
        }
        case CFS_T_TWIST_Z:
        case CFS_T_BEND:
            st.p[0] = res(0);
            break;
        case CFS_T_SCATTER:
            for (int i = 0; i < 4; ++i) st.p[i] = res(i);
            if (!(st.p[0] >= 1.0f && st.p[0] <= 1048576.0f) || st.p[0] != (float)(uint32_t)st.p[0])
                return fail(CFS_ERR_INVALID_ARG, "chain[%d]: SCATTER needs a whole number of duplicates in [1, 2^20]", m);
            break;
        case CFS_T_PINHOLE: {
            const double fov = (double)x.p0[0] + t * (double)x.p1[0];
            if (!(fov > 0.0 && fov < 180.0)) return fail(CFS_ERR_INVALID_ARG, "chain[%d]: PINHOLE fov must be in (0, 180) degrees", m);
            const double f = 1.0 / tan(fov * (3.14159265358979323846 / 180.0) * 0.5);
            st.p[0] = (float)(f * (double)a->height / (double)a->width);
            st.p[1] = (float)f;
            st.p[2] = res(1);
            st.p[3] = res(2);
            if (bad_float(st.p[0]) || bad_float(st.p[1]) || !(st.p[0] > 0.0f) || !(st.p[1] > 0.0f))
                return fail(CFS_ERR_INVALID_ARG, "chain[%d]: PINHOLE focal lengths are not finite and positive", m);
            // the depth key orders like the depth only for d > 0 (DESIGN R8): near < 0 would let d <= 0 through
            if (a->out_mode == CFS_OUT_DEPTH_RGBA8_U64 && !(st.p[3] >= 0.0f))
                return fail(CFS_ERR_INVALID_ARG, "chain[%d]: DEPTH output needs PINHOLE near >= 0", m);
            break;
        }
        default:
            break;
        }
    }
    return CFS_OK;
}

using cfs::render_fn;

// chain signature after host resolution (ROTATE_Z is an AFFINE by now)
uint32_t chain_signature(const RenderParams &p)
{
    uint32_t sig = 0;
    for (int m = 0; m < p.n_chain; ++m) sig |= (uint32_t)(p.chain[m].type + 1) << (4 * m);
    return sig;
}

// A kernel to launch: an ahead-of-time instantiation linked into the library, or a run-time-compiled one
// (cfs_jit.h).  Both are instantiations of the same templates.
struct Kernel {
    render_fn aot = nullptr;
    cfs::JitKernel jit;
    bool compiled_chain = false;     // the chain is compiled in (not the interpreter)
};

bool is_cloud_stream(const cfs_system *s, int splat)
{
    return s->gen == CFS_GEN_CLOUD && (splat == cfs::SPLAT_HIST_DIRECT || splat == cfs::SPLAT_RGBA || splat == cfs::SPLAT_DEPTH);
}

// run-time compilation is used when the render asks for it (CFS_FLAG_JIT), or for every render of the process
// when $CFS_FORCE_JIT is set (kernel development) -- never together with CFS_FLAG_INTERPRET_CHAIN
bool wants_jit(int flags)
{
    if (flags & CFS_FLAG_INTERPRET_CHAIN) return false;
    if (flags & CFS_FLAG_JIT) return true;
    static const bool forced = [] { const char *e = getenv("CFS_FORCE_JIT"); return e && *e && *e != '0'; }();
    return forced;
}

// which iterations of a steady-state Philox block splat straight to L2 in the tile-binned variant: 0 = none (pure
// bins); the hybrid stage (CFS_FLAG_BIN_HYBRID, or chosen by AUTO) sends every other one
uint32_t hybrid_mask(const cfs_render_args *a)
{
    if (!((a->flags & CFS_FLAG_BIN_HYBRID) || a->variant == CFS_VARIANT_AUTO)) return 0u;
    static const int forced = [] { const char *e = getenv("CFS_BIN_MASK"); return (e && *e) ? atoi(e) & 15 : -1; }();   // kernel development
    if (forced >= 0) return (uint32_t)forced;
    return 1u;       // one splat in four: measured against 5 (every other), 0 (pure bins) and 7 on configs[1] and [2] (DESIGN "hybrid")
}

// generator table form of a run-time compiled kernel
int jit_aff(const cfs_system *s)
{
    if (s->gen == CFS_GEN_CLOUD) return cfs::AFF_GENERAL;
    return s->uscale_ok ? (int)cfs::AFF_USCALE : s->aff;
}

// rewrite the coefficient table of `p` for AFF_USCALE (translations only, the shared scale in p.uscale)
void apply_uscale(const cfs_system *s, RenderParams &p)
{
    if (s->gen != CFS_GEN_IFS || !s->uscale_ok || p.aff_form == cfs::AFF_USCALE) return;
    const int n = (int)s->funcs.size();
    memset(p.coef, 0, sizeof(p.coef));
    const float *m0 = s->funcs[0].params;
    p.uscale[0] = m0[0]; p.uscale[1] = (s->dim == 2) ? m0[3] : m0[4]; p.uscale[2] = (s->dim == 2) ? 0.0f : m0[8];
    for (int j = 0; j < n; ++j) {
        const float *m = s->funcs[j].params;
        float *r = p.coef + 4 * j;
        if (s->dim == 2) { r[0] = m[4]; r[1] = m[5]; } else { r[0] = m[9]; r[1] = m[10]; r[2] = m[11]; }
    }
    p.aff_form = cfs::AFF_USCALE;
    p.coef_rows = (uint32_t)n;
    p.coef_cshift = 0;
    if (p.coef_rows > 8) while (p.coef_cshift < 3 && (p.coef_rows << (p.coef_cshift + 1)) <= (uint32_t)cfs::kCoefSlots) ++p.coef_cshift;
    p.coef_rstride = 16u << p.coef_cshift; p.coef_kstride = p.coef_rstride;
}

// What the host can PROVE about a render and hand to a run-time compiled kernel as a dropped test.  An IFS of affine
// contractions keeps its points inside the cube of half-width R = max(1, max_k |b_k| / (1 - |A_k|)) (infinity norms;
// the initial point lies in [-1, 1)^3); AFFINE / ROTATE_Z / TWIST_Z / BEND / SWIRL / SINUSOIDAL / STRETCH_COS / SCATTER
// steps change that bound by a computable amount, a PINHOLE turns it into a depth interval [d_min, d_max] and a bound on the projected
// coordinates.  Hence: d in [2^-126, 2^126) at every PINHOLE (near >= 2^-100, |z| < 2^100), where the reciprocal's
// normal-range sequence IS the correctly rounded one (OPT_RCP_NORMAL).  A stored cloud, reuse, the Eq. 1
// generator or any other step: no proof, no option.
// Returns the OPT_* bits proved for this render: OPT_RCP_NORMAL, and OPT_NO_DROP when moreover every splat of every
// branch is alive (d > near at each PINHOLE) and lands strictly inside the image bounds, with a 1e-3 relative margin
// against float rounding (the kernels' own CFS_CHECK re-tests both claims under -DCFS_CHECKS=1).
int proved_options(const cfs_system *s, const RenderParams &p)
{
    if (s->gen != CFS_GEN_IFS || p.reuse || s->aff == cfs::AFF_CIRCLE) return 0;
    const int d = s->dim;
    auto norms = [d](const float *m, double *na, double *nb) {
        *na = 0.0; *nb = 0.0;
        for (int r = 0; r < d; ++r) {
            double row = 0.0;
            for (int c = 0; c < d; ++c) row += std::fabs((double)m[r * d + c]);
            *na = std::max(*na, row);
            *nb = std::max(*nb, std::fabs((double)m[d * d + r]));
        }
    };
    double R = 1.0;                                  // half-width of a cube that holds every generated point
    for (const cfs_func &f : s->funcs) {
        double na, nb;
        norms(f.params, &na, &nb);
        if (!(na < 0.999)) return 0;
        R = std::max(R, nb / (1.0 - na));
    }
    const double margin = 1.001;
    const double bx = std::min(-(double)p.xmin, (double)p.xmax), by = std::min(-(double)p.ymin, (double)p.ymax);
    bool rcp_ok = true, any_pinhole = false, no_drop = true;
    double Rx = R, Ry = R, Rz = R;                   // per-axis bounds inside the current branch
    bool projected = false;
    auto end_branch = [&]() { if (!(Rx * margin < bx && Ry * margin < by)) no_drop = false; };
    for (int m = 0; m < p.n_chain; ++m) {
        const cfs::ChainStep &st = p.chain[m];
        if (projected && st.type != cfs::T_BRANCH) return 0;      // nothing may follow a projection in this proof
        switch (st.type) {
        case cfs::T_BRANCH: end_branch(); Rx = Ry = Rz = R; projected = false; break;
        case cfs::T_AFFINE: case cfs::T_SCALE: {
            double na, nb;
            norms(st.p, &na, &nb);
            const double Rm = std::max(Rx, std::max(Ry, d == 3 ? Rz : 0.0));
            Rx = Ry = na * Rm + nb;
            if (d == 3) Rz = Rx;
            break;
        }
        case cfs::T_TWIST_Z: case cfs::T_BEND: case cfs::T_SWIRL: { const double r2 = std::sqrt(Rx * Rx + Ry * Ry); Rx = Ry = r2; break; }   // (x, y) rotated, z kept
        case cfs::T_SINUSOIDAL: Rx = std::sin(std::min(Rx, 1.5707963267948966)); Ry = std::sin(std::min(Ry, 1.5707963267948966)); break;   // |sin| is increasing up to pi/2
        case cfs::T_STRETCH_COS: Ry += 1.0; Rx *= 2.0; break;
        case cfs::T_SCATTER: Rx += std::fabs((double)st.p[1]); Ry += std::fabs((double)st.p[2]); Rz += std::fabs((double)st.p[3]); break;
        case cfs::T_PINHOLE: {
            if (d != 3) return 0;
            any_pinhole = true;
            const double cam = (double)st.p[2], nearp = (double)st.p[3];
            const double dmin = -Rz - cam, dmax = Rz - cam;
            if (!(nearp >= 0x1p-100 && std::fabs(dmax) < 0x1p100 && std::fabs(dmin) < 0x1p100)) rcp_ok = false;
            if (dmin > nearp * margin && dmin > 0x1p-100) {
                Rx = (double)st.p[0] * Rx / dmin; Ry = (double)st.p[1] * Ry / dmin; Rz = dmax;
            } else {
                no_drop = false;                     // some splats may be behind the near plane
                Rx = Ry = 1e300;
            }
            projected = true;
            break;
        }
        default: return 0;
        }
    }
    end_branch();
    int opt = 0;
    if (any_pinhole && rcp_ok) opt |= cfs::OPT_RCP_NORMAL;
    if (no_drop) opt |= cfs::OPT_NO_DROP;
    return opt;
}

// options compiled into a run-time specialised kernel (cfs_params.h KernelOpt): everything the host knows about
// the system and the render that lets the kernel drop a run-time decision
int jit_options(const cfs_system *s, const RenderParams &p, int splat)
{
    int opt = p.reuse ? cfs::OPT_REUSE : 0;
    if (s->gen == CFS_GEN_IFS) {
        if (p.pick_shift >= 0) opt |= cfs::OPT_PICK_SHIFT;
        else if (p.n_thr == 2) opt |= cfs::OPT_PICK_CMP2;          // exactly two real thresholds (unused slots hold 2^32 - 1)
        else if (s->pick_mulhi) opt |= cfs::OPT_PICK_MULHI;        // configs[4]: 128.4 -> 122.9 ms against the table read below
        else if (p.pick_steps <= 1) opt |= cfs::OPT_PICK_LUT1;
    }
    if (p.xmin == -p.xmax && p.ymin == -p.ymax) opt |= cfs::OPT_SYM_BOUNDS;
    opt |= proved_options(s, p);
    if (splat == cfs::SPLAT_BIN) {
        opt |= cfs::OPT_BIN_FIXED | ((int)(p.bin.hybrid & 15u) << cfs::OPT_BIN_MASK_SHIFT);
        if (p.color_rule != 0) opt |= cfs::OPT_BIN_RGBA;
        // every chunk of this render is a whole number of pass-1 CTAs (bin_layout cuts chunks at multiples of kBinThreads)
        if (p.n_points > 0 && p.n_points % (uint64_t)cfs::kBinThreads == 0) opt |= cfs::OPT_ALL_HAVE;
    }
    return opt;
}

int trig_of(uint32_t sig, int flags)
{
    return ((flags & CFS_FLAG_FAST_TRIG) && cfs::sig_has_trig(sig)) ? cfs::TRIG_FAST : cfs::TRIG_ACCURATE;
}

// The kernel for this render and splat sink.  Order: run-time compiled (when asked for), the kernel compiled
// ahead of time for the chain's signature when there is one, else the chain interpreter; all evaluate the
// same device functions.  UNSUPPORTED + message when CFS_FLAG_JIT was given and compilation is impossible.
cfs_status pick_kernel(const cfs_system *s, RenderParams &p, int splat, int flags, Kernel *out)
{
    *out = Kernel();
    const uint32_t sig = chain_signature(p);
    if (wants_jit(flags) && splat != cfs::SPLAT_HIST_CLUSTER) {
        const int opt = jit_options(s, p, splat);
        const std::string name = is_cloud_stream(s, splat)
            ? cfs::jit_cloud_name(s->dim, splat, sig, trig_of(sig, flags), opt)
            : cfs::jit_render_name(s->dim, s->gen, jit_aff(s), splat, sig, trig_of(sig, flags), opt);
        std::string err;
        if (cfs::jit_get(name, &out->jit, &err)) { apply_uscale(s, p); out->compiled_chain = true; return CFS_OK; }
        if (flags & CFS_FLAG_JIT) return fail(CFS_ERR_UNSUPPORTED, "%s", err.c_str());
        *out = Kernel();                       // $CFS_FORCE_JIT only: fall back to what is linked in
    }
    if (!(flags & CFS_FLAG_INTERPRET_CHAIN) && p.n_chain > 0 && !p.reuse && p.n_branches == 1) {
        const int trig = (flags & CFS_FLAG_FAST_TRIG) ? cfs::TRIG_FAST : cfs::TRIG_ACCURATE;
        out->aot = (s->dim == 2) ? cfs::lookup_render_static2d(s->gen, s->aff, splat, sig, trig)
                                 : cfs::lookup_render_static3d(s->gen, s->aff, splat, sig, trig);
        if (out->aot) { out->compiled_chain = true; return CFS_OK; }
    }
    out->aot = cfs::lookup_render_generic(s->dim, s->gen, s->aff, splat);
    if (!out->aot) return fail(CFS_ERR_UNSUPPORTED, "no kernel for dim %d / generator form %d / splat %d", s->dim, s->aff, splat);
    return CFS_OK;
}

cfs_status pick_trace(const cfs_system *s, RenderParams &p, int flags, Kernel *out)
{
    *out = Kernel();
    const uint32_t sig = chain_signature(p);
    if (wants_jit(flags) && !p.reuse) {
        std::string err;
        const std::string name = cfs::jit_trace_name(s->dim, s->gen, jit_aff(s), sig, trig_of(sig, flags));
        if (cfs::jit_get(name, &out->jit, &err)) { apply_uscale(s, p); out->compiled_chain = true; return CFS_OK; }
        if (flags & CFS_FLAG_JIT) return fail(CFS_ERR_UNSUPPORTED, "%s", err.c_str());
        *out = Kernel();
    }
    if (!(flags & CFS_FLAG_INTERPRET_CHAIN) && p.n_chain > 0 && !p.reuse && p.n_branches == 1) {
        const int trig = (flags & CFS_FLAG_FAST_TRIG) ? cfs::TRIG_FAST : cfs::TRIG_ACCURATE;
        out->aot = (s->dim == 2) ? cfs::lookup_trace_static2d(s->gen, s->aff, sig, trig)
                                 : cfs::lookup_trace_static3d(s->gen, s->aff, sig, trig);
        if (out->aot) { out->compiled_chain = true; return CFS_OK; }
    }
    out->aot = cfs::lookup_trace_generic(s->dim, s->gen, s->aff);
    if (!out->aot) return fail(CFS_ERR_UNSUPPORTED, "no trace kernel for dim %d / generator form %d", s->dim, s->aff);
    return CFS_OK;
}

// one launch of either kind; dynamic shared memory beyond the default is opted into once per kernel
cfs_status launch(const Kernel &k, unsigned grid, unsigned block, size_t dyn, cudaStream_t st, const RenderParams &p, const char *what)
{
    if (k.jit.func) {
        std::string err;
        if (cfs::jit_launch(k.jit, grid, block, dyn, st, p, &err) != cudaSuccess) return fail(CFS_ERR_CUDA, "%s: %s", what, err.c_str());
        ++g_launches;
        return CFS_OK;
    }
    cudaError_t e;
    if (dyn > 32 * 1024 && (e = ensure_dyn_smem((const void *)k.aot, dyn)) != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute");
    k.aot<<<grid, block, dyn, st>>>(p);
    ++g_launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(e, what);
    return CFS_OK;
}

size_t shared_hist_limit(const DeviceInfo &di)
{
    const long lim = (long)di.smem_optin - (long)sizeof(cfs::SharedTables) - 1024;
    return lim > 0 ? (size_t)lim : 0;
}

}  // namespace

// splats one generated point drives per iteration past burn-in: 1 + BRANCH markers of the chain
static uint64_t branches_of(const cfs_system *s)
{
    uint64_t n = 1;
    for (const cfs_xform &x : s->chain) if (x.type == CFS_T_BRANCH) ++n;
    return n;
}

// ---- tile-binned variant: plan (tiles, staging rows, scratch layout, chunking) -------------------
namespace {

struct BinPlan {
    cfs::BinParams bp;         // pointers filled from the scratch buffer
    size_t smem_pass1, smem_pass2;
    uint32_t grid1;            // persistent CTAs of pass 1
    uint64_t chunk_points;     // points per (pass 1, pass 2) pair
    size_t clear_bytes;        // ctrl + tile_n at the start of the scratch: zeroed per chunk
};

constexpr size_t kBinCtrlBytes = 256;
constexpr uint64_t kHostScratchCap = 1ull << 30;     // scratch the host entry points allocate for the tile bins, at most (more chunks beyond)
constexpr size_t kBinBlockBytes = cfs::kBinBlockRecords * 2;      // 16-bit records

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// tiles and staging rows; false when the variant cannot serve this system / image
bool bin_shape_raw(int gen, int out_mode, int color, uint32_t n_funcs, int32_t width, int32_t height, const DeviceInfo &di,
                   uint32_t hybrid, uint32_t branches, BinPlan *pl, const char **why)
{
    if (gen != CFS_GEN_IFS) { *why = "binned variant needs an IFS generator"; return false; }
    if (out_mode == CFS_OUT_DEPTH_RGBA8_U64) { *why = "binned variant serves HIST and RGBA output"; return false; }
    uint32_t nk = 1;                       // colour slots per pixel: 1 = HIST, else one per function
    if (out_mode == CFS_OUT_RGBA_F32) {
        if (color != CFS_COLOR_MAP_INDEX) { *why = "binned RGBA needs COLOR_MAP_INDEX"; return false; }
        if (n_funcs > 16) { *why = "binned RGBA supports at most 16 functions"; return false; }
        nk = n_funcs;
    }
    const uint64_t n_pix = (uint64_t)width * height;
    if (n_pix > (1ull << 28)) { *why = "binned variant serves images up to 2^28 pixels"; return false; }
    // pass 2 keeps (pixels per tile) x nk counters in shared memory: at most 3 * 2^14 (192 KiB), which is also
    // what a 16-bit record can index.  Tiles are INTERLEAVED: with n_tiles = 2^t, pixel p belongs to tile p & (2^t - 1)
    // and is its pixel p >> t -- every tile samples the whole image, so all tiles draw splats at the same rate
    // whatever the attractor looks like (contiguous tiles drew up to 2.4 x the even share on configs[1], whose
    // swirled square covers 41 % of the image, and the staging rows had to be sized and drained for the hottest one),
    // and the tile / record arithmetic of a splat is an AND, a shift and a multiply-add.  The fewest tiles (at least
    // 64) whose counters fit: longer staging rows, fewer drains.
    uint32_t tshift = 6;
    auto tp_for = [&](uint32_t t) { return (n_pix + (1ull << t) - 1) >> t; };
    while (tshift < 10 && tp_for(tshift) * nk > 49152u) ++tshift;
    if (tp_for(tshift) * nk > 49152u) { *why = "image has too many pixels (x colour slots) for 1024 tiles of 49152 counters"; return false; }
    const uint64_t n_tiles = 1ull << tshift;
    // pass 1 staging: cnt + rows of `cap` records per tile, next to the static tables
    // kBinCtasPerSm CTAs of pass 1 share the SM's shared memory (1 KiB per CTA is reserved by the system)
    const long budget = ((long)di.smem_sm / cfs::kBinCtasPerSm < (long)di.smem_optin ? (long)di.smem_sm / cfs::kBinCtasPerSm : (long)di.smem_optin)
                        - (long)sizeof(cfs::SharedTables) - 2048;
    const long row_bytes = (budget - 4 * (long)(n_tiles + cfs::kBinDummy) - 16) / (long)n_tiles;       // u32 cnt[] + u16 rows
    long cap = (row_bytes - (long)cfs::kBinRowPad) / 2 / 64 * 64;
    if (cap > 4096) cap = 4096;
    if (cap < 320) { *why = "image has too many tiles for the binned variant's staging rows"; return false; }
    cfs::BinParams &b = pl->bp;
    memset(&b, 0, sizeof(b));
    b.n_tiles = (uint32_t)n_tiles; b.tile_pixels = (uint32_t)tp_for(tshift);
    b.tshift = tshift; b.tmask = (uint32_t)n_tiles - 1u;
    b.nk = nk; b.cap = (uint32_t)cap;
    // the rows are drained every E iterations (a multiple of 4: whole Philox blocks), E the largest value <= 128 whose
    // expected arrivals per row, times 1.9 for tiles that draw more than the even share, fit what a drained row has
    // free (a row keeps < drain_min records behind) with 16 records of slack.  Hotter rows overflow now and then; an
    // overflowing splat costs one L2 reduction (its pixel is still in registers), which is cheaper than draining all
    // rows more often: measured on configs[1] / [2] at E = 48 / 64 / 80 / 96: 2.70 / 2.66 / 2.64 / 2.80 and 5.57 / 5.54 /
    // 5.65 / 5.86 ms.  The hybrid stage bins three splats in four; one-to-many systems append one record per branch.
    const double per_it = (double)cfs::kBinThreads / (double)n_tiles * (1.0 - 0.25 * __builtin_popcount(hybrid & 15u)) * (double)branches;
    b.drain_min = cfs::kBinDrainMin;
    if (const char *x = getenv("CFS_BIN_DRAIN_MIN")) { const int v = atoi(x); if (v >= 8 && v <= 1024) b.drain_min = (uint32_t)v / 8 * 8; }   // kernel development
    const double room = (double)cap - (double)b.drain_min - 16.0;
    uint32_t every = 128;
    while (every > 4 && 1.25 * every * per_it > room) every -= 4;
    if (const char *x = getenv("CFS_BIN_EVERY")) { const int v = atoi(x); if (v >= 4 && v <= 4096) every = (uint32_t)v / 4 * 4; }   // kernel development
    b.check_every = every / 4;                         // in Philox blocks of 4 iterations
    // pass 2 runs one CTA per SM (the tile fills shared memory) in waves of `sms` CTAs: among the splits
    // that give 2.5 to 8 waves take the one whose last wave is fullest (configs[1]: 86 tiles x 7 = 4.07 waves
    // ran as 5; x 5 = 2.9 waves runs as 3)
    {
        uint32_t best = 1;
        double best_eff = 0.0;
        for (uint32_t sp = 1; sp <= 64; ++sp) {
            const double waves = (double)(n_tiles * sp) / (double)di.sms;
            if (waves < 2.5 && sp < 64) continue;
            const double eff = waves / std::ceil(waves);
            if (eff > best_eff + 1e-9) { best_eff = eff; best = sp; }
            if (waves >= 8.0) break;
        }
        b.split = best;
    }
    pl->smem_pass1 = (n_tiles + cfs::kBinDummy + 3) / 4 * 4 * 4 + n_tiles * ((size_t)cap * 2 + cfs::kBinRowPad);
    pl->smem_pass2 = ((size_t)b.tile_pixels * nk + 32) / 32 * 32 * 4;      // + the dummy counter the padding records of a drained row hit, in whole groups of 32 (bin_slot)
    pl->grid1 = (uint32_t)di.sms * cfs::kBinCtasPerSm;
    return true;
}

// list capacity per (tile, pass-1 CTA): four times the even share of the pool
uint64_t bin_lcap(const BinPlan &pl, uint64_t nb) { return 4 * nb / ((uint64_t)pl.bp.n_tiles * pl.grid1) + 8; }

size_t bin_fixed_bytes(const BinPlan &pl)
{
    return kBinCtrlBytes + align_up((size_t)pl.bp.n_tiles * pl.grid1 * 4, 256) + 1024;
}

bool bin_shape(const cfs_system *s, const cfs_render_args *a, const DeviceInfo &di, BinPlan *pl, const char **why)
{
    const uint32_t hybrid = hybrid_mask(a);
    return bin_shape_raw(s->gen, a->out_mode, s->color, (uint32_t)s->funcs.size(), a->width, a->height, di, hybrid, (uint32_t)branches_of(s), pl, why);
}

// scratch needed to render `points` points in one chunk
uint64_t bin_scratch_for(const BinPlan &pl, uint64_t points, uint64_t splats_per_point)
{
    const uint64_t rec = points * splats_per_point;
    // every (CTA, tile) holds one prefetched and one partial block; 12.5 % head-room for uneven tiles
    const uint64_t nb = rec / cfs::kBinBlockRecords * 9 / 8 + 4 * ((uint64_t)pl.grid1 * pl.bp.n_tiles + 64);
    return bin_fixed_bytes(pl) + align_up((size_t)((uint64_t)pl.bp.n_tiles * pl.grid1 * bin_lcap(pl, nb)) * 4, 256) +
           nb * kBinBlockBytes + 1024;
}

// carve the scratch buffer; false when it is too small for even one wave of points
bool bin_layout(BinPlan *pl, void *scratch, uint64_t bytes, uint64_t n_points, uint64_t splats_per_point, const char **why)
{
    cfs::BinParams &b = pl->bp;
    uint8_t *base = (uint8_t *)align_up((size_t)scratch, 512);
    if ((size_t)(base - (uint8_t *)scratch) >= bytes) { *why = "scratch too small"; return false; }
    bytes -= (size_t)(base - (uint8_t *)scratch);
    const uint64_t pairs = (uint64_t)pl->grid1 * b.n_tiles;
    const size_t fixed = bin_fixed_bytes(*pl) + 32 * pairs + 1024;      // + the "+ 8" list entries of every pair
    if (bytes <= fixed) { *why = "scratch too small"; return false; }
    // per block: 2 KiB of records (1024 x 16 bit) + 16 B of list capacity
    uint64_t nb = (bytes - fixed) / (kBinBlockBytes + 16);
    if (nb > (1u << 22) - 1) nb = (1u << 22) - 1;                 // record positions are 32-bit
    const uint64_t partial = 2 * (pairs + 64);
    if (nb < partial + partial / 2) { *why = "scratch too small for the binned variant (two blocks per CTA and tile)"; return false; }
    const uint64_t lcap = bin_lcap(*pl, nb);
    b.nb = (uint32_t)nb; b.lcap = (uint32_t)lcap; b.grid = pl->grid1;
    b.ctrl = (uint32_t *)base;
    b.tails = (uint32_t *)(base + kBinCtrlBytes);
    uint8_t *q = base + kBinCtrlBytes + align_up((size_t)pairs * 4, 256);
    pl->clear_bytes = (size_t)(q - base);
    b.list = (uint32_t *)q;  q += align_up((size_t)(pairs * lcap) * 4, 256);
    b.pool = (uint16_t *)align_up((size_t)q, 512);
    // records one chunk may produce: the blocks left after the prefetched / partial ones, with head-room
    const uint64_t rec_cap = (nb - partial) * 8 / 9 * cfs::kBinBlockRecords;
    uint64_t cp = rec_cap / splats_per_point;
    const uint64_t wave = (uint64_t)pl->grid1 * cfs::kBinThreads;
    if (cp < cfs::kBinThreads) { *why = "scratch too small for one CTA of points"; return false; }
    if (cp >= n_points) cp = n_points;                          // everything in one chunk
    else if (cp >= wave) cp = cp / wave * wave;                 // whole waves: no ragged trip inside a chunk
    else cp = cp / cfs::kBinThreads * cfs::kBinThreads;         // whole CTAs: only the render's last chunk can be ragged (OPT_ALL_HAVE)
    pl->chunk_points = cp;
    return true;
}

}  // namespace

// host-only view of the plan (no device needed): lets the CPU tests check the tile arithmetic
extern "C" cfs_status cfs_binned_plan(int32_t width, int32_t height, int32_t out_mode, int32_t n_funcs, int32_t sms,
                                      int32_t smem_per_block_optin, uint32_t out[8])
{
    if (!out || width < 1 || height < 1 || sms < 1 || n_funcs < 1) return fail(CFS_ERR_INVALID_ARG, "bad plan arguments");
    DeviceInfo di; di.ok = 1; di.sms = sms; di.smem_optin = smem_per_block_optin; di.smem_sm = smem_per_block_optin + 1024;
    BinPlan pl;
    const char *why = "";
    if (!bin_shape_raw(CFS_GEN_IFS, out_mode, out_mode == CFS_OUT_RGBA_F32 ? CFS_COLOR_MAP_INDEX : CFS_COLOR_NONE, (uint32_t)n_funcs,
                       width, height, di, 0u, 1u, &pl, &why)) return fail(CFS_ERR_UNSUPPORTED, "%s", why);
    out[0] = pl.bp.n_tiles; out[1] = pl.bp.tile_pixels; out[2] = pl.bp.tshift; out[3] = pl.bp.tmask;
    out[4] = pl.bp.nk; out[5] = pl.bp.cap; out[6] = 4u * pl.bp.check_every; out[7] = pl.bp.split;
    return CFS_OK;
}

// records one point sends through the tile bins: its splats minus those the hybrid stage sends straight to L2
// (iterations whose bit is set in the direct mask, in the steady-state Philox blocks only: the blocks touching
// burn-in or the ragged end bin everything)
static uint64_t binned_per_point(const cfs_system *s, const cfs_render_args *a)
{
    const uint64_t br = branches_of(s);
    const int I = a->iterations, B = a->burn_in;
    const int fast0 = std::min((B + 3) & ~3, I & ~3), fast1 = I & ~3;
    const uint64_t direct = (uint64_t)__builtin_popcount(hybrid_mask(a)) * (uint64_t)((fast1 - fast0) / 4) * br;
    return (uint64_t)(I - B) * br - direct;
}

extern "C" uint64_t cfs_binned_scratch_bytes(const cfs_system *s, const cfs_render_args *a)
{
    const DeviceInfo &di = device_info();
    if (!s || !a || di.ok != 1 || a->iterations <= a->burn_in || a->width < 1 || a->height < 1) return 0;
    BinPlan pl;
    const char *why = "";
    if (!bin_shape(s, a, di, &pl, &why)) return 0;
    return bin_scratch_for(pl, a->n_points, binned_per_point(s, a));
}

extern "C" uint64_t cfs_shared_hist_max_bytes(void)
{
    const DeviceInfo &di = device_info();
    return di.ok == 1 ? shared_hist_limit(di) : 0;
}

namespace {

// bins per CTA (log2) of the cluster histogram, or -1 when the image does not fit a cluster
int cluster_slice_shift(size_t hist_bytes, const DeviceInfo &di)
{
    const size_t bins = hist_bytes / 4;
    int shift = 8;
    while (((size_t)cfs::kClusterSize << shift) < bins) ++shift;
    const long lim = (long)di.smem_optin - (long)sizeof(cfs::SharedTables) - 2048;
    return ((long)(4ull << shift) <= lim) ? shift : -1;
}

// histogram distributed over the shared memory of 8-CTA clusters (DSMEM reductions), one CTA per SM
cfs_status render_cluster_hist(const cfs_system *s, const cfs_render_args *a, RenderParams &p, const DeviceInfo &di, cudaStream_t st)
{
    if (a->out_mode != CFS_OUT_HIST_U32 || s->gen != CFS_GEN_IFS) return fail(CFS_ERR_UNSUPPORTED, "cluster histogram needs HIST_U32 output and an IFS generator");
    const size_t hist_bytes = (size_t)a->width * a->height * 4;
    const int shift = cluster_slice_shift(hist_bytes, di);
    if (shift < 0) return fail(CFS_ERR_UNSUPPORTED, "image of %zu bytes does not fit the shared memory of a %d-CTA cluster", hist_bytes, cfs::kClusterSize);
    Kernel kc;
    cfs_status ks = pick_kernel(s, p, cfs::SPLAT_HIST_CLUSTER, a->flags, &kc);
    if (ks != CFS_OK) return ks;
    render_fn fn = kc.aot;
    const size_t dyn = (size_t)4 << shift;
    cudaError_t e = ensure_dyn_smem((const void *)fn, dyn);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute");
    p.hist_bins = (uint32_t)(hist_bytes / 4);
    p.slice_shift = (uint32_t)shift;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cfs::kClusterSize; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(cfs::kClusterThreads); cfg.dynamicSmemBytes = dyn; cfg.stream = st; cfg.attrs = attr; cfg.numAttrs = 1;
    cfg.gridDim = dim3(cfs::kClusterSize);
    int max_clusters = 0;
    e = cudaOccupancyMaxActiveClusters(&max_clusters, (const void *)fn, &cfg);
    if (e != cudaSuccess || max_clusters < 1) { cudaGetLastError(); return fail(CFS_ERR_UNSUPPORTED, "no co-resident %d-CTA cluster with %zu bytes of shared memory", cfs::kClusterSize, dyn); }
    uint64_t clusters = (a->n_points + (uint64_t)cfs::kClusterSize * cfs::kClusterThreads - 1) / ((uint64_t)cfs::kClusterSize * cfs::kClusterThreads);
    if (clusters > (uint64_t)max_clusters) clusters = (uint64_t)max_clusters;     // persistent: grid-stride over points
    cfg.gridDim = dim3((unsigned)(clusters * cfs::kClusterSize));
    e = cudaLaunchKernelEx(&cfg, fn, p);
    ++g_launches;
    if (e != cudaSuccess) return cuda_fail(e, "cluster histogram launch");
    return CFS_OK;
}

// tile-binned render: per chunk of points, clear the bin heads, pass 1 (sample + bin), pass 2
// (accumulate tiles in shared memory, merge).  `force`: the caller asked for this variant, so
// report why it cannot run; otherwise return UNSUPPORTED quietly and let AUTO fall back.
cfs_status render_binned(const cfs_system *s, const cfs_render_args *a, RenderParams &p, const DeviceInfo &di, cudaStream_t st)
{
    BinPlan pl;
    const char *why = "";
    if (!bin_shape(s, a, di, &pl, &why)) return fail(CFS_ERR_UNSUPPORTED, "%s", why);
    if (!a->d_scratch) return fail(CFS_ERR_UNSUPPORTED, "binned variant needs d_scratch (see cfs_binned_scratch_bytes)");
    const uint64_t spp = binned_per_point(s, a);          // records per point that really go through the bins
    if (!bin_layout(&pl, a->d_scratch, a->scratch_bytes, a->n_points, spp, &why)) return fail(CFS_ERR_UNSUPPORTED, "%s", why);
    p.bin = pl.bp;
    p.bin.hybrid = hybrid_mask(a);
    Kernel k1;
    cfs_status ks = pick_kernel(s, p, cfs::SPLAT_BIN, a->flags, &k1);
    if (ks != CFS_OK) return ks;
    Kernel k2;
    k2.aot = (a->out_mode == CFS_OUT_HIST_U32) ? cfs::bin_accumulate_kernel<0> : cfs::bin_accumulate_kernel<1>;
    cudaError_t e;
    const uint64_t total = a->n_points, first = a->point_offset;
    for (uint64_t done = 0; done < total; done += pl.chunk_points) {
        const uint64_t n = (total - done < pl.chunk_points) ? total - done : pl.chunk_points;
        p.n_points = n;
        p.point_offset = first + done;
        if ((e = cudaMemsetAsync(pl.bp.ctrl, 0, pl.clear_bytes, st)) != cudaSuccess) return cuda_fail(e, "clear bin heads");
        // always the full persistent grid: pass 2 reads the tail word of every (tile, CTA)
        if ((ks = launch(k1, pl.grid1, cfs::kBinThreads, pl.smem_pass1, st, p, "binned render, pass 1")) != CFS_OK) return ks;
        if (!(a->flags & CFS_FLAG_BIN_PASS1_ONLY) &&
            (ks = launch(k2, pl.bp.n_tiles * pl.bp.split, cfs::kBinAccThreads, pl.smem_pass2, st, p, "binned render, pass 2")) != CFS_OK) return ks;
    }
    return CFS_OK;
}

}  // namespace

// ---- Hi-Z depth variant: plan + phased render ---------------------------------------------------
namespace {

struct HizPlan { uint32_t shift, nbx, nby, n, n_pad; uint64_t bytes; };

// smallest block (8, 16 or 32 pixels square) whose map fits kHizMaxBytes of shared memory
bool hiz_plan(int32_t width, int32_t height, HizPlan *pl)
{
    if (width < 1 || height < 1) return false;
    for (uint32_t sh = 3; sh <= 5; ++sh) {
        const uint64_t nbx = ((uint64_t)width + (1u << sh) - 1) >> sh, nby = ((uint64_t)height + (1u << sh) - 1) >> sh;
        const uint64_t n = nbx * nby, n_pad = (n + 7) / 8 * 8;
        if (n_pad * 2 <= cfs::kHizMaxBytes) {
            pl->shift = sh; pl->nbx = (uint32_t)nbx; pl->nby = (uint32_t)nby; pl->n = (uint32_t)n; pl->n_pad = (uint32_t)n_pad;
            pl->bytes = n_pad * 2 + 256;         // + alignment slack
            return true;
        }
    }
    return false;
}

}  // namespace

extern "C" uint64_t cfs_hiz_scratch_bytes(int32_t width, int32_t height)
{
    HizPlan pl;
    return hiz_plan(width, height, &pl) ? pl.bytes : 0;
}

namespace {

// Phases over disjoint point ranges (min is order-free, so any split gives the same image):
//   [0, n0)      plain depth splats -- n0 sized so that the image holds ~64 splats per pixel,
//   build Hi-Z,  [n0, 8 n0) behind it,  rebuild (tighter),  the rest behind that.
cfs_status render_depth_hiz(const cfs_system *s, const cfs_render_args *a, RenderParams &p, const DeviceInfo &di, cudaStream_t st)
{
    (void)di;
    if (a->out_mode != CFS_OUT_DEPTH_RGBA8_U64 || s->gen != CFS_GEN_IFS)
        return fail(CFS_ERR_UNSUPPORTED, "Hi-Z variant serves DEPTH output of an IFS generator");
    HizPlan pl;
    if (!hiz_plan(a->width, a->height, &pl)) return fail(CFS_ERR_UNSUPPORTED, "image too large for a shared-memory Hi-Z map");
    if (!a->d_scratch || a->scratch_bytes < pl.bytes)
        return fail(CFS_ERR_UNSUPPORTED, "Hi-Z variant needs d_scratch of cfs_hiz_scratch_bytes() = %llu bytes", (unsigned long long)pl.bytes);
    Kernel k0, k1;
    cfs_status ks;
    if ((ks = pick_kernel(s, p, cfs::SPLAT_DEPTH, a->flags, &k0)) != CFS_OK) return ks;
    if ((ks = pick_kernel(s, p, cfs::SPLAT_DEPTH_HIZ, a->flags, &k1)) != CFS_OK) return ks;
    uint16_t *hz = (uint16_t *)(((uintptr_t)a->d_scratch + 255) & ~(uintptr_t)255);
    const size_t dyn = (size_t)pl.n_pad * 2;
    cudaError_t e;
    p.hiz.hz = hz; p.hiz.shift = pl.shift; p.hiz.nbx = pl.nbx; p.hiz.nby = pl.nby; p.hiz.n_pad = pl.n_pad;
    // the map's padding entries are read into shared memory but never indexed; clear them once
    if ((e = cudaMemsetAsync(hz, 0xFF, dyn, st)) != cudaSuccess) return cuda_fail(e, "clear Hi-Z map");

    const uint64_t P = a->n_points, spp = (uint64_t)(a->iterations - a->burn_in) * branches_of(s);
    uint64_t n0 = (64ull * (uint64_t)a->width * (uint64_t)a->height + spp - 1) / spp;
    n0 = (n0 + cfs::kHizThreads - 1) / cfs::kHizThreads * cfs::kHizThreads;
    const uint64_t cuts[4] = {0, n0 < P ? n0 : P, 8 * n0 < P ? 8 * n0 : P, P};
    const uint64_t off0 = p.point_offset;
    for (int ph = 0; ph < 3; ++ph) {
        const uint64_t lo = cuts[ph], hi = cuts[ph + 1];
        if (hi <= lo) continue;
        p.point_offset = off0 + lo; p.n_points = hi - lo;
        if (ph == 0) {
            uint64_t blocks = (p.n_points + cfs::kRenderThreads - 1) / cfs::kRenderThreads;
            if ((ks = launch(k0, (unsigned)blocks, cfs::kRenderThreads, 0, st, p, "Hi-Z render, plain slice")) != CFS_OK) return ks;
        } else {
            const unsigned side = 1u << pl.shift;
            cfs::hiz_build_kernel<<<pl.n, side * side, 0, st>>>((const unsigned long long *)a->d_image, a->width, a->height,
                                                                  pl.shift, pl.nbx, hz);
            ++g_launches;
            uint64_t blocks = (p.n_points + cfs::kHizThreads - 1) / cfs::kHizThreads;
            if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(e, "Hi-Z build launch");
            if ((ks = launch(k1, (unsigned)blocks, cfs::kHizThreads, dyn, st, p, "Hi-Z render")) != CFS_OK) return ks;
        }
    }
    return CFS_OK;
}

}  // namespace

// cloud_base: index of the record d_cloud[0] in the WHOLE cloud (0 for cfs_render; cfs_render_host uploads
// only the rendered record range)
static cfs_status render_impl(const cfs_system *s, const cfs_render_args *a, void *stream, uint64_t cloud_base)
{
    RenderParams p;
    cfs_status st = build_params(s, a, &p, true);
    if (st != CFS_OK) return st;
    p.cloud_base = cloud_base;
    if (a->variant < CFS_VARIANT_AUTO || a->variant > CFS_VARIANT_DEPTH_HIZ) return fail(CFS_ERR_INVALID_ARG, "unknown variant %d", a->variant);
    const DeviceInfo &di = device_info();
    if (di.ok != 1) return fail(CFS_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    const size_t hist_bytes = (size_t)a->width * a->height * 4;
    const uint64_t n_splats = a->n_points * (uint64_t)(a->iterations - a->burn_in) * branches_of(s);
    int splat;
    if (a->out_mode == CFS_OUT_RGBA_F32) splat = cfs::SPLAT_RGBA;
    else if (a->out_mode == CFS_OUT_DEPTH_RGBA8_U64) splat = cfs::SPLAT_DEPTH;
    else splat = cfs::SPLAT_HIST_DIRECT;
    if (a->variant == CFS_VARIANT_BINNED) {
        if (a->n_points == 0) return CFS_OK;
        return render_binned(s, a, p, di, (cudaStream_t)stream);
    }
    if (a->variant == CFS_VARIANT_CLUSTER_HIST) {
        if (a->n_points == 0) return CFS_OK;
        return render_cluster_hist(s, a, p, di, (cudaStream_t)stream);
    }
    if (a->variant == CFS_VARIANT_DEPTH_HIZ) {
        if (a->n_points == 0) return CFS_OK;
        return render_depth_hiz(s, a, p, di, (cudaStream_t)stream);
    }
    if (a->variant == CFS_VARIANT_SHARED_HIST || a->variant == CFS_VARIANT_WARP_AGG) {
        if (a->out_mode != CFS_OUT_HIST_U32) return fail(CFS_ERR_UNSUPPORTED, "variant %d is for HIST_U32 output only", a->variant);
        if (a->variant == CFS_VARIANT_SHARED_HIST && hist_bytes > shared_hist_limit(di))
            return fail(CFS_ERR_UNSUPPORTED, "image of %zu bytes does not fit the per-CTA shared histogram (%zu)", hist_bytes, shared_hist_limit(di));
        splat = (a->variant == CFS_VARIANT_SHARED_HIST) ? cfs::SPLAT_HIST_SHARED : cfs::SPLAT_HIST_WARPAGG;
    } else if (a->variant == CFS_VARIANT_AUTO) {
        // chosen by image size and work (DESIGN "splat variants"): small histograms are privatised
        // per CTA; big renders with scratch memory go through the tile bins; else direct L2 atomics
        if (a->out_mode == CFS_OUT_HIST_U32 && hist_bytes <= shared_hist_limit(di) && n_splats >= (uint64_t)di.sms * (hist_bytes / 4)) {
            splat = cfs::SPLAT_HIST_SHARED;
        } else if (a->out_mode == CFS_OUT_DEPTH_RGBA8_U64) {
            // direct: ld.cg pre-test + atom.min, measured at the SM-to-L2 request rate (one sector request per clock
            // and SM, l1tex2xbar 98 % busy).  The Hi-Z variant removes that bound and is then bound by instruction
            // issue: level with the direct path as linked ahead of time (227 ms both on configs[4]), ahead of it when
            // compiled for the system (CFS_FLAG_JIT: 178 ms).  AUTO takes it for big renders when the caller provides
            // the scratch for its map.
            if (s->gen == CFS_GEN_IFS && a->d_scratch && cfs_hiz_scratch_bytes(a->width, a->height) != 0 &&
                a->scratch_bytes >= cfs_hiz_scratch_bytes(a->width, a->height) && n_splats >= (1ull << 30)) {
                cfs_status hs = render_depth_hiz(s, a, p, di, (cudaStream_t)stream);
                if (hs != CFS_ERR_UNSUPPORTED) return hs;
                build_params(s, a, &p, true);
                p.cloud_base = cloud_base;
            }
        } else if (a->d_scratch && a->n_points >= (uint64_t)di.sms * cfs::kBinCtasPerSm * cfs::kBinThreads && n_splats >= (1ull << 27)) {
            // the hybrid stage (every other splat direct, the rest through the tile bins) keeps issue slots, the
            // L2 reduction path and HBM busy at once: measured ahead of the direct path with MUFU sin/cos
            // (configs[1] 3.49 against 5.0 ms) and with sincosf (4.06 against 5.21 ms; configs[2] 172 against 197 ms)
            cfs_status bs = render_binned(s, a, p, di, (cudaStream_t)stream);
            if (bs != CFS_ERR_UNSUPPORTED) return bs;
            build_params(s, a, &p, true);      // restore what the attempt changed; fall through to direct
            p.cloud_base = cloud_base;
        }
    }
    if (a->n_points == 0) return CFS_OK;
    Kernel kn;
    if ((st = pick_kernel(s, p, splat, a->flags, &kn)) != CFS_OK) return st;

    const int threads = cfs::kRenderThreads;
    uint64_t blocks = (a->n_points + threads - 1) / threads;
    size_t dyn = 0;
    if (splat == cfs::SPLAT_HIST_SHARED) {
        dyn = hist_bytes;
        p.hist_bins = (uint32_t)(hist_bytes / 4);
    }
    // CLOUD and SHARED_HIST: persistent grid (resident CTAs x SMs), grid-stride over points: one
    // histogram merge per CTA, short per-point work amortises the CTA prologue.  IFS + direct
    // splats: one point per thread, CTAs handed out by the hardware scheduler -- measured faster
    // than a persistent grid (P / resident threads is ~3.5 for configs[1]: the last static trip
    // would run 46 % full; dynamic CTA hand-out has no such tail).
    if (is_cloud_stream(s, splat)) {
        // the streaming cloud kernel (cfs_cloud.cuh): persistent CTAs, chunks of records through a shared-memory ring
        const uint64_t n_chunks = (a->n_points + cfs::kCloudChunk - 1) / cfs::kCloudChunk;
        uint64_t grid = (uint64_t)di.sms * cfs::kCloudCtasPerSm;
        if (grid > n_chunks) grid = n_chunks;
        return launch(kn, (unsigned)grid, cfs::kCloudThreads, cfs::kCloudSmemBytes, (cudaStream_t)stream, p, "cloud kernel launch");
    }
    if (s->gen == CFS_GEN_CLOUD || splat == cfs::SPLAT_HIST_SHARED) {
        // resident CTAs per SM: from the occupancy calculator for a linked kernel; a run-time-compiled one of the
        // same template has the same shape -- the registers allow 8 x 256 threads, shared memory decides
        int per_sm = 1;
        if (kn.aot) {
            if (dyn > 32 * 1024) ensure_dyn_smem((const void *)kn.aot, dyn);
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)kn.aot, threads, dyn);
        } else {
            per_sm = (int)((size_t)di.smem_sm / (dyn + sizeof(cfs::SharedTables) + 2048));
            if (per_sm > 8) per_sm = 8;
        }
        if (per_sm < 1) per_sm = 1;
        const uint64_t cap = (uint64_t)di.sms * per_sm;
        if (blocks > cap) blocks = cap;
    } else if (blocks > (1u << 24)) {
        blocks = 1u << 24;
    }
    return launch(kn, (unsigned)blocks, threads, dyn, (cudaStream_t)stream, p, "render kernel launch");
}

extern "C" cfs_status cfs_render(const cfs_system *s, const cfs_render_args *a, void *stream)
{
    return render_impl(s, a, stream, 0);
}

extern "C" cfs_status cfs_specialize(const cfs_system *s, const cfs_render_args *a, double *out_ms)
{
    if (out_ms) *out_ms = 0.0;
    RenderParams p;
    cfs_render_args r;
    if (a) { r = *a; r.d_image = nullptr; r.d_cloud = nullptr; r.flags = (r.flags | CFS_FLAG_JIT) & ~CFS_FLAG_INTERPRET_CHAIN; }
    cfs_status st = build_params(s, a ? &r : nullptr, &p, false);
    if (st != CFS_OK) return st;
    const DeviceInfo &di = device_info();
    if (di.ok != 1) return fail(CFS_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    int kinds[4], n = 0;
    if (a->out_mode == CFS_OUT_RGBA_F32) kinds[n++] = cfs::SPLAT_RGBA;
    else if (a->out_mode == CFS_OUT_DEPTH_RGBA8_U64) { kinds[n++] = cfs::SPLAT_DEPTH; if (s->gen == CFS_GEN_IFS) kinds[n++] = cfs::SPLAT_DEPTH_HIZ; }
    else kinds[n++] = cfs::SPLAT_HIST_DIRECT;
    BinPlan pl;
    const char *why = "";
    if (bin_shape(s, &r, di, &pl, &why)) kinds[n++] = cfs::SPLAT_BIN;
    double ms = 0.0;
    p.bin.hybrid = hybrid_mask(&r);
    for (int i = 0; i < n; ++i) {
        Kernel k;
        if ((st = pick_kernel(s, p, kinds[i], r.flags, &k)) != CFS_OK) return st;
        ms += k.jit.compile_ms;
    }
    if (out_ms) *out_ms = ms;
    return CFS_OK;
}

// compile-only twin of cfs_specialize: no device needed (the cubin is built and dropped)
extern "C" cfs_status cfs_jit_check(const cfs_system *s, const cfs_render_args *a, int32_t splat_kind, uint64_t *out_cubin_bytes, double *out_ms)
{
    RenderParams p;
    cfs_render_args r;
    if (a) { r = *a; r.d_image = nullptr; r.d_cloud = nullptr; }
    cfs_status st = build_params(s, a ? &r : nullptr, &p, false);
    if (st != CFS_OK) return st;
    int splat = splat_kind;
    if (splat < 0) splat = (a->out_mode == CFS_OUT_RGBA_F32) ? cfs::SPLAT_RGBA : (a->out_mode == CFS_OUT_DEPTH_RGBA8_U64) ? cfs::SPLAT_DEPTH : cfs::SPLAT_HIST_DIRECT;
    const uint32_t sig = chain_signature(p);
    if (splat == cfs::SPLAT_BIN) p.bin.hybrid = hybrid_mask(a);
    const int opt = jit_options(s, p, splat);
    const std::string name = is_cloud_stream(s, splat)
        ? cfs::jit_cloud_name(s->dim, splat, sig, trig_of(sig, a->flags), opt)
        : cfs::jit_render_name(s->dim, s->gen, jit_aff(s), splat, sig, trig_of(sig, a->flags), opt);
    std::string err;
    size_t bytes = 0;
    double ms = 0.0;
    if (!cfs::jit_compile_only(name, &bytes, &ms, &err)) return fail(CFS_ERR_UNSUPPORTED, "%s", err.c_str());
    if (out_cubin_bytes) *out_cubin_bytes = bytes;
    if (out_ms) *out_ms = ms;
    return CFS_OK;
}

extern "C" void cfs_jit_stats(uint64_t *out_n, double *out_ms)
{
    unsigned long long n = 0;
    double ms = 0.0;
    cfs::jit_stats(&n, &ms);
    if (out_n) *out_n = n;
    if (out_ms) *out_ms = ms;
}

// host-only view of what a render resolves before its launch (no device needed): lets the CPU tests pin the
// library's host arithmetic against hand-worked numbers instead of against the oracle's restatement of it
extern "C" cfs_status cfs_host_resolve(const cfs_system *s, const cfs_render_args *a, cfs_resolved *out)
{
    if (!out) return fail(CFS_ERR_INVALID_ARG, "out is NULL");
    RenderParams p;
    cfs_render_args r;
    if (a) { r = *a; r.d_image = nullptr; r.d_cloud = nullptr; }
    cfs_status st = build_params(s, a ? &r : nullptr, &p, false);
    if (st != CFS_OK) return st;
    memset(out, 0, sizeof(*out));
    out->sx = p.sx; out->ox = p.ox; out->sy = p.sy; out->oy = p.oy;
    out->n_chain = p.n_chain;
    for (int m = 0; m < p.n_chain; ++m) {
        out->chain_type[m] = (p.chain[m].type == cfs::T_SCALE) ? (int32_t)CFS_T_AFFINE : p.chain[m].type;
        memcpy(out->chain_p[m], p.chain[m].p, sizeof(out->chain_p[m]));
    }
    out->n_funcs = p.n_funcs;
    out->n_thresholds = p.n_thr;
    { const int po = proved_options(s, p); out->proved = ((po & cfs::OPT_RCP_NORMAL) ? 1 : 0) | ((po & cfs::OPT_NO_DROP) ? 2 : 0); }
    out->pick_form = (s->gen != CFS_GEN_IFS) ? 0 : (p.pick_shift >= 0) ? 1 : (p.n_thr == 2) ? 2 : s->pick_mulhi ? 4 : (p.pick_steps <= 1) ? 3 : 0;
    memcpy(out->thresholds, p.T, sizeof(out->thresholds));
    memcpy(out->pal8, p.pal8, sizeof(out->pal8));
    return CFS_OK;
}

extern "C" cfs_status cfs_trace(const cfs_system *s, const cfs_render_args *a, uint8_t *d_picks, float *d_final_g,
                                float *d_final_q, uint8_t *d_alive, void *stream)
{
    RenderParams p;
    cfs_status st = build_params(s, a, &p, false);
    if (st != CFS_OK) return st;
    if (device_info().ok != 1) return fail(CFS_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    if (a->n_points == 0) return CFS_OK;
    if (p.n_branches > 1) return fail(CFS_ERR_UNSUPPORTED, "cfs_trace does not serve chains with BRANCH markers");
    p.tr_picks = d_picks; p.tr_g = d_final_g; p.tr_q = d_final_q; p.tr_alive = d_alive;
    p.counters = nullptr;
    Kernel kt;
    if ((st = pick_trace(s, p, a->flags, &kt)) != CFS_OK) return st;
    uint64_t blocks = (a->n_points + cfs::kRenderThreads - 1) / cfs::kRenderThreads;
    if (blocks > (1u << 22)) blocks = 1u << 22;
    return launch(kt, (unsigned)blocks, cfs::kRenderThreads, 0, (cudaStream_t)stream, p, "trace kernel launch");
}

// -------------------------------------------------------------------------------------------------
// common body of the host entry points: upload (CLOUD), clear, render; the image stays in s->d_image
static cfs_status render_host_body(cfs_system *s, const cfs_render_args *a, const cfs_cloud_rec *h_cloud, void *stream, size_t *image_bytes)
{
    if (!s || !a) return fail(CFS_ERR_INVALID_ARG, "system or args is NULL");
    if (a->width < 1 || a->height < 1 || (int64_t)a->width * a->height > 2147483647ll) return fail(CFS_ERR_INVALID_ARG, "bad image size");
    if (a->out_mode < CFS_OUT_HIST_U32 || a->out_mode > CFS_OUT_DEPTH_RGBA8_U64) return fail(CFS_ERR_INVALID_ARG, "unknown out_mode %d", a->out_mode);
    if (device_info().ok != 1) return fail(CFS_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t px = (size_t)a->width * a->height;
    const size_t bytes = px * (a->out_mode == CFS_OUT_HIST_U32 ? 4 : a->out_mode == CFS_OUT_RGBA_F32 ? 16 : 8);
    *image_bytes = bytes;
    cudaError_t e;
    if (s->image_bytes < bytes) {
        if (s->d_image) cudaFree(s->d_image);
        s->d_image = nullptr; s->image_bytes = 0;
        if ((e = cudaMalloc(&s->d_image, bytes)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(image)");
        s->image_bytes = bytes;
    }
    if (!s->d_counters && (e = cudaMalloc((void **)&s->d_counters, 16)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(counters)");
    cfs_render_args r = *a;
    r.d_image = s->d_image; r.d_counters = (uint64_t *)s->d_counters; r.d_cloud = nullptr;
    if (s->gen == CFS_GEN_CLOUD && a->n_points) {
        if (!h_cloud) return fail(CFS_ERR_INVALID_ARG, "h_cloud is NULL");
        // only the rendered record range travels; the kernel indexes the WHOLE cloud by p
        const size_t cb = (size_t)a->n_points * sizeof(cfs_cloud_rec);
        if (s->cloud_bytes < cb) {
            if (s->d_cloud) cudaFree(s->d_cloud);
            s->d_cloud = nullptr; s->cloud_bytes = 0;
            if ((e = cudaMalloc(&s->d_cloud, cb)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(cloud)");
            s->cloud_bytes = cb;
        }
        if ((e = cudaMemcpyAsync(s->d_cloud, h_cloud + a->point_offset, cb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e, "H2D cloud");
        r.d_cloud = s->d_cloud;                // holds records [point_offset, point_offset + n_points)
    }
    r.d_scratch = nullptr; r.scratch_bytes = 0;
    if (a->variant == CFS_VARIANT_AUTO || a->variant == CFS_VARIANT_BINNED || a->variant == CFS_VARIANT_DEPTH_HIZ) {
        // scratch of the tile-binned variant (enough for one chunk, capped: more chunks beyond) or of the Hi-Z map
        uint64_t want = cfs_binned_scratch_bytes(s, &r);
        if (want > kHostScratchCap) want = kHostScratchCap;
        if (a->out_mode == CFS_OUT_DEPTH_RGBA8_U64) want = cfs_hiz_scratch_bytes(a->width, a->height);
        if (want > s->scratch_bytes) {
            if (s->d_scratch) cudaFree(s->d_scratch);
            s->d_scratch = nullptr; s->scratch_bytes = 0;
            if (cudaMalloc(&s->d_scratch, want) == cudaSuccess) s->scratch_bytes = want;
            else cudaGetLastError();           // no scratch: AUTO renders directly
        }
        if (want && s->d_scratch) { r.d_scratch = s->d_scratch; r.scratch_bytes = s->scratch_bytes; }
    }
    if ((e = cudaMemsetAsync(s->d_image, a->out_mode == CFS_OUT_DEPTH_RGBA8_U64 ? 0xFF : 0, bytes, st)) != cudaSuccess) return cuda_fail(e, "clear image");
    if ((e = cudaMemsetAsync(s->d_counters, 0, 16, st)) != cudaSuccess) return cuda_fail(e, "clear counters");
    return render_impl(s, &r, stream, s->gen == CFS_GEN_CLOUD ? a->point_offset : 0);
}

extern "C" cfs_status cfs_render_host(cfs_system *s, const cfs_render_args *a, void *h_image,
                                      const cfs_cloud_rec *h_cloud, uint64_t *h_counters, void *stream)
{
    if (!h_image) return fail(CFS_ERR_INVALID_ARG, "h_image is NULL");
    size_t bytes = 0;
    cfs_status rs = render_host_body(s, a, h_cloud, stream, &bytes);
    if (rs != CFS_OK) return rs;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    if ((e = cudaMemcpyAsync(h_image, s->d_image, bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e, "D2H image");
    if (h_counters && (e = cudaMemcpyAsync(h_counters, s->d_counters, 16, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e, "D2H counters");
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e, "stream synchronize");
    return CFS_OK;
}

extern "C" cfs_status cfs_render_rgba8_host(cfs_system *s, const cfs_render_args *a, float gamma, float colour_scale, float n_max,
                                            uint32_t *h_rgba8, const cfs_cloud_rec *h_cloud, uint64_t *h_counters,
                                            float *h_n_max, void *stream)
{
    if (!h_rgba8) return fail(CFS_ERR_INVALID_ARG, "h_rgba8 is NULL");
    size_t bytes = 0;
    cfs_status rs = render_host_body(s, a, h_cloud, stream, &bytes);
    if (rs != CFS_OK) return rs;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    const size_t out_bytes = (size_t)a->width * a->height * 4;
    if (s->rgba8_bytes < out_bytes) {
        if (s->d_rgba8) cudaFree(s->d_rgba8);
        s->d_rgba8 = nullptr; s->rgba8_bytes = 0;
        if ((e = cudaMalloc(&s->d_rgba8, out_bytes)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(rgba8)");
        s->rgba8_bytes = out_bytes;
    }
    if (!s->d_tone && (e = cudaMalloc(&s->d_tone, 16)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(tone scratch)");
    rs = cfs_resolve_rgba8(s->d_image, a->out_mode, a->width, a->height, gamma, colour_scale, n_max, (uint32_t *)s->d_rgba8, s->d_tone, stream);
    if (rs != CFS_OK) return rs;
    if ((e = cudaMemcpyAsync(h_rgba8, s->d_rgba8, out_bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e, "D2H rgba8");
    if (h_counters && (e = cudaMemcpyAsync(h_counters, s->d_counters, 16, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e, "D2H counters");
    if (h_n_max && a->out_mode != CFS_OUT_DEPTH_RGBA8_U64 &&
        (e = cudaMemcpyAsync(h_n_max, s->d_tone, 4, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e, "D2H n_max");
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e, "stream synchronize");
    return CFS_OK;
}

extern "C" cfs_status cfs_resolve_rgba8(const void *d_image, int32_t out_mode, int32_t width, int32_t height, float gamma,
                                        float colour_scale, float n_max, uint32_t *d_out, void *d_scratch, void *stream)
{
    if (!d_image || !d_out) return fail(CFS_ERR_INVALID_ARG, "image or output is NULL");
    if (width < 1 || height < 1 || (int64_t)width * height > 2147483647ll) return fail(CFS_ERR_INVALID_ARG, "bad image size");
    if (out_mode < CFS_OUT_HIST_U32 || out_mode > CFS_OUT_DEPTH_RGBA8_U64) return fail(CFS_ERR_INVALID_ARG, "unknown out_mode %d", out_mode);
    const DeviceInfo &di = device_info();
    if (di.ok != 1) return fail(CFS_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    cudaStream_t st = (cudaStream_t)stream;
    size_t n = (size_t)width * height;
    const int threads = cfs::kToneThreads;
    const size_t want = (n + threads - 1) / threads;
    if (out_mode == CFS_OUT_DEPTH_RGBA8_U64) {
        const unsigned grid = (unsigned)(want < (size_t)di.sms * 32 ? want : (size_t)di.sms * 32);
        cfs::tone_depth_kernel<<<grid, threads, 0, st>>>((const unsigned long long *)d_image, n, d_out);
        ++g_launches;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "resolve kernel launch");
        return CFS_OK;
    }
    if (!(gamma > 0.0f) || bad_float(gamma) || bad_float(colour_scale)) return fail(CFS_ERR_INVALID_ARG, "gamma must be > 0 and finite");
    if (std::isnan(n_max) || std::isinf(n_max)) return fail(CFS_ERR_INVALID_ARG, "n_max is not finite");
    if (!d_scratch) return fail(CFS_ERR_INVALID_ARG, "d_scratch is NULL");
    cudaError_t e;
    // [0] n_max bits (output), [1] barrier arrivals, [2] the previous call's n_max when n_max < 0 asks for it
    if (n_max < 0.0f && (e = cudaMemcpyAsync((char *)d_scratch + 8, d_scratch, 4, cudaMemcpyDeviceToDevice, st)) != cudaSuccess) return cuda_fail(e, "park previous n_max");
    if ((e = cudaMemsetAsync(d_scratch, 0, 8, st)) != cudaSuccess) return cuda_fail(e, "clear scratch");
    float inv_gamma = 1.0f / gamma;
    uint32_t *scratch = (uint32_t *)d_scratch;
    const bool hist = out_mode == CFS_OUT_HIST_U32;
    if (n_max != 0.0f) {         // single pass with the given maximum (> 0) or the previous call's (< 0)
        const unsigned grid = (unsigned)(want < (size_t)di.sms * 16 ? want : (size_t)di.sms * 16);
        if (hist) cfs::resolve_kernel<0, true><<<grid, threads, 0, st>>>(d_image, n, scratch, n_max, inv_gamma, colour_scale, d_out);
        else      cfs::resolve_kernel<1, true><<<grid, threads, 0, st>>>(d_image, n, scratch, n_max, inv_gamma, colour_scale, d_out);
        ++g_launches;
        if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(e, "resolve kernel launch");
        return CFS_OK;
    }
    // maximum + map in one cooperative launch: as many CTAs as are resident at once
    const void *fn = hist ? (const void *)cfs::resolve_kernel<0, false> : (const void *)cfs::resolve_kernel<1, false>;
    int per_sm = 0;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, threads, 0)) != cudaSuccess || per_sm < 1) return cuda_fail(e, "resolve occupancy");
    if (per_sm > 8) per_sm = 8;
    size_t grid = (size_t)di.sms * per_sm;
    if (grid > want) grid = want;
    float zero = 0.0f;
    void *args[] = {(void *)&d_image, (void *)&n, (void *)&scratch, (void *)&zero, (void *)&inv_gamma, (void *)&colour_scale, (void *)&d_out};
    if ((e = cudaLaunchCooperativeKernel(fn, dim3((unsigned)grid), dim3(threads), args, 0, st)) != cudaSuccess) return cuda_fail(e, "resolve kernel launch");
    ++g_launches;
    return CFS_OK;
}

extern "C" cfs_status cfs_tonemap(const void *d_image, int32_t out_mode, int32_t width, int32_t height, float gamma,
                                  float colour_scale, uint32_t *d_out, void *d_scratch, void *stream)
{
    if (out_mode == CFS_OUT_HIST_U32 && ((uintptr_t)d_image & 15)) return fail(CFS_ERR_INVALID_ARG, "HIST image must be 16-byte aligned for the tone map");
    return cfs_resolve_rgba8(d_image, out_mode, width, height, gamma, colour_scale, 0.0f, d_out, d_scratch, stream);
}

extern "C" cfs_status cfs_microbench(int32_t kind, void *d_buf, uint64_t footprint, uint64_t ops, int32_t blocks,
                                     int32_t threads, void *stream)
{
    if (!d_buf || blocks < 1 || threads < 32 || threads > 1024 || (threads & 31)) return fail(CFS_ERR_INVALID_ARG, "bad microbench launch shape");
    const DeviceInfo &di = device_info();
    if (di.ok != 1) return fail(CFS_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    cudaStream_t st = (cudaStream_t)stream;
    auto bins = [&](size_t elem) -> uint32_t { const uint64_t b = footprint / elem; return (uint32_t)(b > 0xFFFFFFFFull ? 0xFFFFFFFFull : b); };
    switch (kind) {
    case CFS_MB_RED_ADD_U32:   if (!bins(4)) return fail(CFS_ERR_INVALID_ARG, "footprint too small");  cfs::mb_mem_kernel<0><<<blocks, threads, 0, st>>>(d_buf, bins(4), ops); break;
    case CFS_MB_RED_ADD_V4F32: if (!bins(16)) return fail(CFS_ERR_INVALID_ARG, "footprint too small"); cfs::mb_mem_kernel<1><<<blocks, threads, 0, st>>>(d_buf, bins(16), ops); break;
    case CFS_MB_ATOM_MIN_U64:  if (!bins(8)) return fail(CFS_ERR_INVALID_ARG, "footprint too small");  cfs::mb_mem_kernel<2><<<blocks, threads, 0, st>>>(d_buf, bins(8), ops); break;
    case CFS_MB_LD_U64:        if (!bins(8)) return fail(CFS_ERR_INVALID_ARG, "footprint too small");  cfs::mb_mem_kernel<3><<<blocks, threads, 0, st>>>(d_buf, bins(8), ops); break;
    case CFS_MB_ATOMS_ADD_U32: {
        if (footprint < 4 || footprint > (uint64_t)di.smem_optin) return fail(CFS_ERR_INVALID_ARG, "shared footprint must be 4..%d bytes", di.smem_optin);
        cudaError_t e = ensure_dyn_smem((const void *)cfs::mb_atoms_kernel, footprint);
        if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute");
        cfs::mb_atoms_kernel<<<blocks, threads, footprint, st>>>(d_buf, (uint32_t)(footprint / 4), ops);
        break;
    }
    case CFS_MB_FFMA:      cfs::mb_alu_kernel<5><<<blocks, threads, 0, st>>>(d_buf, ops); break;
    case CFS_MB_IMAD_WIDE: cfs::mb_alu_kernel<6><<<blocks, threads, 0, st>>>(d_buf, ops); break;
    case CFS_MB_LOP3:      cfs::mb_alu_kernel<7><<<blocks, threads, 0, st>>>(d_buf, ops); break;
    case CFS_MB_MUFU:      cfs::mb_alu_kernel<8><<<blocks, threads, 0, st>>>(d_buf, ops); break;
    case CFS_MB_STREAM_LD128: cfs::mb_stream_kernel<<<blocks, threads, 0, st>>>(d_buf, footprint / 16); break;
    case CFS_MB_STREAM_RED_V4F32: if (!bins(16)) return fail(CFS_ERR_INVALID_ARG, "footprint too small"); cfs::mb_stream_red_kernel<<<blocks, threads, 0, st>>>(d_buf, bins(16), ops); break;
    default: return fail(CFS_ERR_INVALID_ARG, "unknown microbench kind %d", kind);
    }
    ++g_launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "microbench launch");
    return CFS_OK;
}

extern "C" uint64_t cfs_launch_count(int32_t reset)
{
    const uint64_t v = g_launches;
    if (reset) g_launches = 0;
    return v;
}

extern "C" const char *cfs_last_error(void) { return g_err; }
extern "C" const char *cfs_version(void) { return "cfs-b200 0.1 (sm_100a)"; }

// ---- cfs_render_depth_noalloc: the Hi-Z depth render with its scratch inside the library ---------------------------
// For callers that cannot allocate device memory (include/cfs.h has the contract).  The Hi-Z map lives in this
// file-scope device array, which every GPU that loads the library holds until the process exits.  In HOST code the
// name below is a host-side stand-in for the symbol, NOT a device address: a kernel handed `g_noalloc_scratch`
// itself would fault (or, where the GPU can reach host memory, quietly use the wrong bytes).  The device address
// is resolved with cudaGetSymbolAddress, once per device, with that device current, and only that pointer is
// passed on.  Every call on a device shares the array; render_depth_hiz resets the map before it reads it, so the
// last call's contents never reach a render -- but calls that overlap on the GPU race on it.
static __device__ __align__(256) unsigned char g_noalloc_scratch[CFS_NOALLOC_SCRATCH_BYTES];
static_assert(CFS_NOALLOC_SCRATCH_BYTES >= cfs::kHizMaxBytes + 256, "the built-in scratch must hold the largest Hi-Z map plus its alignment slack");

namespace {

std::mutex g_noalloc_mutex;
void *g_noalloc_ptr[kMaxDevices];       // device address of g_noalloc_scratch per device ordinal; nullptr = not resolved yet

cfs_status noalloc_scratch(void **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices) return fail(CFS_ERR_UNSUPPORTED, "device ordinal %d beyond %d", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);      // the address on the CURRENT device
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(built-in scratch)");
        if (!ptr || ((uintptr_t)ptr & 255u) != 0) return fail(CFS_ERR_CUDA, "built-in scratch resolved to a bad address %p", ptr);
        g_noalloc_ptr[dev] = ptr;
    }
    *out = g_noalloc_ptr[dev];
    return CFS_OK;
}

}  // namespace

extern "C" cfs_status cfs_render_depth_noalloc(const cfs_system *s, const cfs_render_args *a, void *stream)
{
    if (!s || !a) return fail(CFS_ERR_INVALID_ARG, "system or args is NULL");
    if (wants_jit(a->flags))
        return fail(CFS_ERR_INVALID_ARG, "cfs_render_depth_noalloc allocates nothing: CFS_FLAG_JIT / $CFS_FORCE_JIT compile and load a module, use cfs_render for that");
    if (a->width >= 1 && a->height >= 1) {          // (a bad size is reported by the render's own validation below)
        const uint64_t need = cfs_hiz_scratch_bytes(a->width, a->height);
        if (need == 0 || need > (uint64_t)CFS_NOALLOC_SCRATCH_BYTES)
            return fail(CFS_ERR_INVALID_ARG, "image %d x %d needs %llu bytes of Hi-Z scratch (0 = more than 49152 blocks of 32 x 32 pixels); the built-in scratch holds %d",
                        a->width, a->height, (unsigned long long)need, (int)CFS_NOALLOC_SCRATCH_BYTES);
    }
    void *scratch = nullptr;
    cfs_status st = noalloc_scratch(&scratch);
    if (st != CFS_OK) return st;
    cfs_render_args r = *a;
    r.variant = CFS_VARIANT_DEPTH_HIZ;              // refuses anything but DEPTH output of an IFS (UNSUPPORTED)
    r.d_scratch = scratch;
    r.scratch_bytes = CFS_NOALLOC_SCRATCH_BYTES;
    return render_impl(s, &r, stream, 0);
}
