// cfs_kernels_static2d.cu -- 2-D render / trace kernels with a chain signature compiled in.
//
// The list below is the set of chains that get a dedicated kernel; any other chain runs on the
// interpreter of cfs_kernels_generic.cu with identical results (same device functions).
#include "cfs_select.cuh"

namespace cfs {

namespace {

#define CFS_STATIC_CHAINS(X) \
    X(chain_sig(T_SWIRL, T_SCALE))           /* BASELINE cfg 1 */ \
    X(chain_sig(T_AFFINE, T_SINUSOIDAL))     /* BASELINE cfg 2 */ \
    X(chain_sig(T_STRETCH_COS, T_AFFINE))    /* PAPER Eq. 2    */

// a signature without sin/cos steps has one kernel: the TRIG axis is collapsed onto TRIG_ACCURATE
template <int TRIG>
render_fn render_static_t(int gen, int aff, int splat, uint32_t sig)
{
#define X(S)                                                                              \
    if constexpr (TRIG == TRIG_ACCURATE || sig_has_trig(S)) {                             \
        if (sig == (S)) return select_render<2, (S), TRIG, kSplatsDirect>(gen, aff, splat); \
    }
    CFS_STATIC_CHAINS(X)
#undef X
    return nullptr;
}

template <int TRIG>
render_fn trace_static_t(int gen, int aff, uint32_t sig)
{
#define X(S)                                                                \
    if constexpr (TRIG == TRIG_ACCURATE || sig_has_trig(S)) {               \
        if (sig == (S)) return select_trace<2, (S), TRIG>(gen, aff);         \
    }
    CFS_STATIC_CHAINS(X)
#undef X
    return nullptr;
}

}  // namespace

render_fn lookup_render_static2d(int gen, int aff, int splat, uint32_t sig, int trig)
{
    if (trig == TRIG_FAST && sig_has_trig(sig)) return render_static_t<TRIG_FAST>(gen, aff, splat, sig);
    return render_static_t<TRIG_ACCURATE>(gen, aff, splat, sig);
}

render_fn lookup_trace_static2d(int gen, int aff, uint32_t sig, int trig)
{
    if (trig == TRIG_FAST && sig_has_trig(sig)) return trace_static_t<TRIG_FAST>(gen, aff, sig);
    return trace_static_t<TRIG_ACCURATE>(gen, aff, sig);
}

}  // namespace cfs
