// cfs_kernels_generic3d.cu -- 3-D render / trace kernels with the chain INTERPRETER (any chain).
// sin/cos evaluation is a warp-uniform run-time choice here (TRIG_RUNTIME, prm.fast_trig).
#include "cfs_select.cuh"

namespace cfs {

render_fn lookup_render_generic3d(int gen, int aff, int splat)
{
    return select_render<3, kChainGeneric, TRIG_RUNTIME, kSplatsAll>(gen, aff, splat);
}

render_fn lookup_trace_generic3d(int gen, int aff)
{
    return select_trace<3, kChainGeneric, TRIG_RUNTIME>(gen, aff);
}

}  // namespace cfs
