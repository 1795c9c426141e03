// cfs_kernels_generic.cu -- render / trace kernels with the chain INTERPRETER (any chain).
// sin/cos evaluation is a warp-uniform run-time choice here (TRIG_RUNTIME, prm.fast_trig).
#include "cfs_select.cuh"

namespace cfs {

render_fn lookup_render_generic(int dim, int gen, int aff, int splat)
{
    if (dim == 2) return select_render<2, kChainGeneric, TRIG_RUNTIME, kSplatsAll>(gen, aff, splat);
    return select_render<3, kChainGeneric, TRIG_RUNTIME, kSplatsAll>(gen, aff, splat);
}

render_fn lookup_trace_generic(int dim, int gen, int aff)
{
    if (dim == 2) return select_trace<2, kChainGeneric, TRIG_RUNTIME>(gen, aff);
    return select_trace<3, kChainGeneric, TRIG_RUNTIME>(gen, aff);
}

}  // namespace cfs
