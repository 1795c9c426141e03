// cfs_kernels_generic2d.cu -- 2-D render / trace kernels with the chain INTERPRETER (any chain).
// sin/cos evaluation is a warp-uniform run-time choice here (TRIG_RUNTIME, prm.fast_trig).
#include "cfs_select.cuh"

namespace cfs {

render_fn lookup_render_generic2d(int gen, int aff, int splat)
{
    return select_render<2, kChainGeneric, TRIG_RUNTIME, kSplatsAll>(gen, aff, splat);
}

render_fn lookup_trace_generic2d(int gen, int aff)
{
    return select_trace<2, kChainGeneric, TRIG_RUNTIME>(gen, aff);
}

}  // namespace cfs
