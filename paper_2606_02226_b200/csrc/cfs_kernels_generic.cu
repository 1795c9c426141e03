// cfs_kernels_generic.cu -- lookup of the kernels: dispatch to the translation units that hold them.
#include "cfs_registry.h"

namespace cfs {

// the interpreter kernels live in one translation unit per dimension (cfs_kernels_generic{2,3}d.cu)
render_fn lookup_render_generic2d(int gen, int aff, int splat);
render_fn lookup_render_generic3d(int gen, int aff, int splat);
render_fn lookup_trace_generic2d(int gen, int aff);
render_fn lookup_trace_generic3d(int gen, int aff);

render_fn lookup_render_generic(int dim, int gen, int aff, int splat)
{
    return (dim == 2) ? lookup_render_generic2d(gen, aff, splat) : lookup_render_generic3d(gen, aff, splat);
}

render_fn lookup_trace_generic(int dim, int gen, int aff)
{
    return (dim == 2) ? lookup_trace_generic2d(gen, aff) : lookup_trace_generic3d(gen, aff);
}

// the 2-D kernels compiled for a chain live in one translation unit per signature
render_fn lookup_render_static2d_a(int, int, int, uint32_t, int);
render_fn lookup_render_static2d_b(int, int, int, uint32_t, int);
render_fn lookup_render_static2d_c(int, int, int, uint32_t, int);
render_fn lookup_trace_static2d_a(int, int, uint32_t, int);
render_fn lookup_trace_static2d_b(int, int, uint32_t, int);
render_fn lookup_trace_static2d_c(int, int, uint32_t, int);

render_fn lookup_render_static2d(int gen, int aff, int splat, uint32_t sig, int trig)
{
    if (render_fn f = lookup_render_static2d_a(gen, aff, splat, sig, trig)) return f;
    if (render_fn f = lookup_render_static2d_b(gen, aff, splat, sig, trig)) return f;
    return lookup_render_static2d_c(gen, aff, splat, sig, trig);
}

render_fn lookup_trace_static2d(int gen, int aff, uint32_t sig, int trig)
{
    if (render_fn f = lookup_trace_static2d_a(gen, aff, sig, trig)) return f;
    if (render_fn f = lookup_trace_static2d_b(gen, aff, sig, trig)) return f;
    return lookup_trace_static2d_c(gen, aff, sig, trig);
}

}  // namespace cfs
