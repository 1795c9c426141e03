// cfs_registry.h -- lookup of the compiled render / trace kernels.
//
// The kernels are template instantiations spread over several translation units (compiled in
// parallel by build.py): the GENERIC ones interpret any chain; the STATIC ones have one chain
// signature compiled in (the role Quibble's run-time code splicing plays in the paper, PAPER L37,
// L182 -- here ahead of time, so a scene costs no compile time, cf. the 0.745 s the paper reports
// for compilation against 0.0215 s of rendering, L200).
#pragma once
#include "cfs_params.h"

namespace cfs {

typedef void (*render_fn)(const RenderParams);

// nullptr when the combination does not exist (e.g. DEPTH in 2-D)
render_fn lookup_render_generic(int dim, int gen, int aff, int splat);
render_fn lookup_trace_generic(int dim, int gen, int aff);
// nullptr when no kernel was compiled for this signature: the caller falls back to the generic one
render_fn lookup_render_static2d(int gen, int aff, int splat, uint32_t sig, int trig);
render_fn lookup_trace_static2d(int gen, int aff, uint32_t sig, int trig);
render_fn lookup_render_static3d(int gen, int aff, int splat, uint32_t sig, int trig);
render_fn lookup_trace_static3d(int gen, int aff, uint32_t sig, int trig);

}  // namespace cfs
