// cfs_jit.h -- run-time specialisation of the render kernels.
//
// The paper's central engineering idea is splicing the user's transforms into ONE fused kernel at run time
// ("staged compilation", L182; its cost is quoted at L200: 0.745 s with compilation against 0.0215 s
// per frame).  Here the same role is played by NVRTC: the render kernel template of cfs_render.cuh /
// cfs_cloud.cuh is instantiated for the system's own (dimension, generator form, splat sink, chain signature,
// sin/cos evaluation, options) -- chain unrolled, every step's type a compile-time constant, BRANCH / SCATTER /
// reuse / the Eq. 1 generator included -- compiled to sm_100a SASS in the process, loaded through the driver
// API and cached.  The ahead-of-time kernels (cfs_kernels_*.cu) are instantiations of the very same templates,
// so the three ways to run a chain (interpreter, ahead-of-time, run-time) evaluate the same device functions.
#pragma once
#include <cuda_runtime.h>

#include <string>

#include "cfs_params.h"

namespace cfs {

struct JitKernel {
    void *func = nullptr;        // CUfunction of the current device's primary context
    double compile_ms = 0.0;     // NVRTC + module load time when this call compiled it, 0 when it came from the cache
    bool cached = false;
};

// true when NVRTC and the driver entry points could be loaded (dlopen; no link-time dependency)
bool jit_available(std::string *why);

// C++ name of a render / cloud / trace kernel instantiation, e.g. "cfs::render_kernel<2, 0, 1, 3, 178u, 1, 0>"
std::string jit_render_name(int dim, int gen, int aff, int splat, uint32_t sig, int trig, int opt);
std::string jit_cloud_name(int dim, int splat, uint32_t sig, int trig, int opt);
std::string jit_trace_name(int dim, int gen, int aff, uint32_t sig, int trig);

// the kernel for `name` on the current device: from the process cache, else from the disk cache
// (directory $CFS_JIT_CACHE, only when set), else compiled now.  false + *err on failure.
bool jit_get(const std::string &name, JitKernel *out, std::string *err);

// compile `name` to sm_100a SASS without loading it (no device needed: test instrument, compile-time measurement)
bool jit_compile_only(const std::string &name, size_t *cubin_bytes, double *ms, std::string *err);

// launch with the kernel's single by-value parameter block; dynamic shared memory is opted into as needed
cudaError_t jit_launch(const JitKernel &k, unsigned grid, unsigned block, size_t dyn_smem, cudaStream_t stream,
                       const RenderParams &prm, std::string *err);

// totals since process start (bench accounting): kernels compiled, milliseconds spent compiling
void jit_stats(unsigned long long *n_compiled, double *total_ms);

}  // namespace cfs
