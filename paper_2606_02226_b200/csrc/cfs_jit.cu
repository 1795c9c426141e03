// cfs_jit.cu -- NVRTC specialiser of the render kernels (see cfs_jit.h).  Host code only.
//
// No link-time dependency on NVRTC or on libcuda: NVRTC is dlopen()ed on first use, the driver entry points come
// from cudaGetDriverEntryPoint.  The device sources are the headers of this directory, embedded into the library
// at build time (build.py writes cfs_embedded_sources.inc); $CFS_JIT_SOURCE_DIR makes the specialiser read them
// from a directory instead (kernel development: edit a header, render, no rebuild of the library).
#include "cfs_jit.h"

#include <cuda.h>
#include <dlfcn.h>
#include <nvrtc.h>
#include <sys/stat.h>
#include <unistd.h>

#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <utility>
#include <vector>

namespace cfs {

namespace {

struct EmbeddedSource { const char *name; const char *text; };
#include "cfs_embedded_sources.inc"      // static const EmbeddedSource kEmbedded[] = { {"cfs_params.h", R"CFS(...)CFS"}, ... };

const char *const kHeaderNames[] = {"cfs_params.h", "cfs_device.cuh", "cfs_bin.cuh", "cfs_render.cuh", "cfs_cloud.cuh", "cfs_hiz.cuh"};
constexpr int kNumHeaders = (int)(sizeof(kHeaderNames) / sizeof(kHeaderNames[0]));
const char *const kProgram = "#include \"cfs_cloud.cuh\"\n#include \"cfs_hiz.cuh\"\n";
const char *const kOptions[] = {"--gpu-architecture=sm_100a", "-std=c++17", "--fmad=false", "--prec-div=true", "--prec-sqrt=true",
                                "-lineinfo", "-default-device"};
constexpr int kNumOptions = (int)(sizeof(kOptions) / sizeof(kOptions[0]));

struct Nvrtc {
    void *lib = nullptr;
    decltype(&nvrtcCreateProgram) CreateProgram = nullptr;
    decltype(&nvrtcDestroyProgram) DestroyProgram = nullptr;
    decltype(&nvrtcCompileProgram) CompileProgram = nullptr;
    decltype(&nvrtcGetCUBINSize) GetCUBINSize = nullptr;
    decltype(&nvrtcGetCUBIN) GetCUBIN = nullptr;
    decltype(&nvrtcGetProgramLogSize) GetProgramLogSize = nullptr;
    decltype(&nvrtcGetProgramLog) GetProgramLog = nullptr;
    decltype(&nvrtcAddNameExpression) AddNameExpression = nullptr;
    decltype(&nvrtcGetLoweredName) GetLoweredName = nullptr;
    decltype(&nvrtcGetErrorString) GetErrorString = nullptr;
    decltype(&nvrtcVersion) Version = nullptr;
};

struct Driver {
    bool ok = false;
    CUresult (*ModuleLoadData)(CUmodule *, const void *) = nullptr;
    CUresult (*ModuleGetFunction)(CUfunction *, CUmodule, const char *) = nullptr;
    CUresult (*FuncSetAttribute)(CUfunction, CUfunction_attribute, int) = nullptr;
    CUresult (*LaunchKernel)(CUfunction, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, CUstream, void **, void **) = nullptr;
    CUresult (*GetErrorString)(CUresult, const char **) = nullptr;
};

struct Entry { CUfunction func = nullptr; int dyn_smem = 0; };

std::mutex g_mutex;
Nvrtc g_nvrtc;
Driver g_driver;
int g_state = 0;                       // 0 = not tried, 1 = available, -1 = unavailable (g_why says why)
std::string g_why;
std::map<std::pair<int, std::string>, Entry> g_cache;
unsigned long long g_n_compiled = 0;
double g_total_ms = 0.0;
std::vector<std::string> g_sources;    // header texts in kHeaderNames order
uint64_t g_source_hash = 0;
std::vector<std::string> g_extra_options;   // $CFS_JIT_OPTIONS

uint64_t fnv1a(const void *data, size_t n, uint64_t h = 1469598103934665603ull)
{
    const unsigned char *p = (const unsigned char *)data;
    for (size_t i = 0; i < n; ++i) { h ^= p[i]; h *= 1099511628211ull; }
    return h;
}

bool read_file(const std::string &path, std::string *out)
{
    FILE *f = fopen(path.c_str(), "rb");
    if (!f) return false;
    out->clear();
    char buf[65536];
    size_t n;
    while ((n = fread(buf, 1, sizeof(buf), f)) > 0) out->append(buf, n);
    fclose(f);
    return true;
}

bool load_sources(std::string *err)
{
    g_sources.assign(kNumHeaders, std::string());
    const char *dir = getenv("CFS_JIT_SOURCE_DIR");
    for (int i = 0; i < kNumHeaders; ++i) {
        if (dir && *dir) {
            if (!read_file(std::string(dir) + "/" + kHeaderNames[i], &g_sources[i])) {
                *err = std::string("cannot read ") + dir + "/" + kHeaderNames[i];
                return false;
            }
        } else {
            bool found = false;
            for (const EmbeddedSource &e : kEmbedded)
                if (strcmp(e.name, kHeaderNames[i]) == 0) { g_sources[i] = e.text; found = true; }
            if (!found) { *err = std::string("source not embedded: ") + kHeaderNames[i]; return false; }
        }
    }
    // kernel development: extra compiler options (e.g. -DNAME=value), separated by blanks
    g_extra_options.clear();
    if (const char *x = getenv("CFS_JIT_OPTIONS")) {
        std::string cur;
        for (const char *c = x;; ++c) {
            if (*c == ' ' || *c == '\0') { if (!cur.empty()) g_extra_options.push_back(cur); cur.clear(); if (!*c) break; }
            else cur.push_back(*c);
        }
    }
    uint64_t h = fnv1a(kProgram, strlen(kProgram));
    for (int i = 0; i < kNumHeaders; ++i) h = fnv1a(g_sources[i].data(), g_sources[i].size(), h);
    for (int i = 0; i < kNumOptions; ++i) h = fnv1a(kOptions[i], strlen(kOptions[i]), h);
    for (const std::string &o : g_extra_options) h = fnv1a(o.data(), o.size(), h);
    g_source_hash = h;
    return true;
}

template <typename F>
bool sym(void *lib, const char *name, F *out)
{
    *out = (F)dlsym(lib, name);
    return *out != nullptr;
}

template <typename F>
bool drv(const char *name, F *out)
{
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult st;
    if (cudaGetDriverEntryPoint(name, &fn, cudaEnableDefault, &st) != cudaSuccess || st != cudaDriverEntryPointSuccess || !fn) {
        cudaGetLastError();
        return false;
    }
    *out = (F)fn;
    return true;
}

// caller holds g_mutex
bool init_locked()
{
    if (g_state != 0) return g_state > 0;
    g_state = -1;
    const char *names[] = {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so"};
    for (const char *n : names)
        if ((g_nvrtc.lib = dlopen(n, RTLD_NOW | RTLD_LOCAL)) != nullptr) break;
    if (!g_nvrtc.lib) { g_why = "libnvrtc.so.12 could not be loaded"; return false; }
    Nvrtc &r = g_nvrtc;
    if (!(sym(r.lib, "nvrtcCreateProgram", &r.CreateProgram) && sym(r.lib, "nvrtcDestroyProgram", &r.DestroyProgram) &&
          sym(r.lib, "nvrtcCompileProgram", &r.CompileProgram) && sym(r.lib, "nvrtcGetCUBINSize", &r.GetCUBINSize) &&
          sym(r.lib, "nvrtcGetCUBIN", &r.GetCUBIN) && sym(r.lib, "nvrtcGetProgramLogSize", &r.GetProgramLogSize) &&
          sym(r.lib, "nvrtcGetProgramLog", &r.GetProgramLog) && sym(r.lib, "nvrtcAddNameExpression", &r.AddNameExpression) &&
          sym(r.lib, "nvrtcGetLoweredName", &r.GetLoweredName) && sym(r.lib, "nvrtcGetErrorString", &r.GetErrorString) &&
          sym(r.lib, "nvrtcVersion", &r.Version))) {
        g_why = "libnvrtc lacks an entry point";
        return false;
    }
    if (!load_sources(&g_why)) return false;
    g_state = 1;
    return true;
}

bool init_driver_locked(std::string *err)
{
    if (g_driver.ok) return true;
    Driver &d = g_driver;
    if (!(drv("cuModuleLoadData", &d.ModuleLoadData) && drv("cuModuleGetFunction", &d.ModuleGetFunction) &&
          drv("cuFuncSetAttribute", &d.FuncSetAttribute) && drv("cuLaunchKernel", &d.LaunchKernel) &&
          drv("cuGetErrorString", &d.GetErrorString))) {
        *err = "CUDA driver entry points unavailable (no device?)";
        return false;
    }
    d.ok = true;
    return true;
}

std::string cu_error(CUresult r)
{
    const char *s = nullptr;
    if (g_driver.GetErrorString && g_driver.GetErrorString(r, &s) == CUDA_SUCCESS && s) return s;
    return "CUDA driver error " + std::to_string((int)r);
}

// NVRTC: program -> (cubin, lowered kernel name); caller holds g_mutex
bool compile_locked(const std::string &name, std::vector<char> *cubin, std::string *lowered, std::string *err)
{
    Nvrtc &r = g_nvrtc;
    const char *hdr_text[kNumHeaders];
    for (int i = 0; i < kNumHeaders; ++i) hdr_text[i] = g_sources[i].c_str();
    nvrtcProgram prog = nullptr;
    nvrtcResult rc = r.CreateProgram(&prog, kProgram, "cfs_jit_unit.cu", kNumHeaders, hdr_text, kHeaderNames);
    if (rc != NVRTC_SUCCESS) { *err = std::string("nvrtcCreateProgram: ") + r.GetErrorString(rc); return false; }
    bool ok = false;
    do {
        if ((rc = r.AddNameExpression(prog, name.c_str())) != NVRTC_SUCCESS) { *err = std::string("nvrtcAddNameExpression: ") + r.GetErrorString(rc); break; }
        std::vector<const char *> opts(kOptions, kOptions + kNumOptions);
        for (const std::string &o : g_extra_options) opts.push_back(o.c_str());
        rc = r.CompileProgram(prog, (int)opts.size(), opts.data());
        if (rc != NVRTC_SUCCESS) {
            size_t n = 0;
            r.GetProgramLogSize(prog, &n);
            std::string log(n, '\0');
            if (n) r.GetProgramLog(prog, &log[0]);
            if (log.size() > 1500) log.resize(1500);
            *err = std::string("nvrtcCompileProgram(") + name + "): " + r.GetErrorString(rc) + "\n" + log;
            break;
        }
        const char *low = nullptr;
        if ((rc = r.GetLoweredName(prog, name.c_str(), &low)) != NVRTC_SUCCESS || !low) { *err = std::string("nvrtcGetLoweredName: ") + r.GetErrorString(rc); break; }
        *lowered = low;
        size_t n = 0;
        if ((rc = r.GetCUBINSize(prog, &n)) != NVRTC_SUCCESS || n == 0) { *err = std::string("nvrtcGetCUBINSize: ") + r.GetErrorString(rc); break; }
        cubin->resize(n);
        if ((rc = r.GetCUBIN(prog, cubin->data())) != NVRTC_SUCCESS) { *err = std::string("nvrtcGetCUBIN: ") + r.GetErrorString(rc); break; }
        ok = true;
    } while (false);
    r.DestroyProgram(&prog);
    return ok;
}

std::string cache_path(const std::string &name)
{
    const char *dir = getenv("CFS_JIT_CACHE");
    if (!dir || !*dir) return std::string();
    int major = 0, minor = 0;
    g_nvrtc.Version(&major, &minor);
    uint64_t h = fnv1a(name.data(), name.size(), g_source_hash);
    h = fnv1a(&major, sizeof(major), h);
    h = fnv1a(&minor, sizeof(minor), h);
    char buf[64];
    snprintf(buf, sizeof(buf), "/cfs_%016llx.cubin", (unsigned long long)h);
    return std::string(dir) + buf;
}

// disk cache file: "CFSJ", u32 length of the lowered name, u64 cubin bytes, u64 FNV-1a of the cubin, the name, the cubin.
// The driver loads a module from memory without a length, so a truncated or damaged image must be caught HERE: a file
// whose sizes or checksum do not match is ignored (and rewritten after the compile).
constexpr uint32_t kDiskMagic = 0x4A534643u;    // "CFSJ"
struct DiskHeader { uint32_t magic, name_len; uint64_t cubin_bytes, cubin_hash; };

bool disk_load(const std::string &path, std::vector<char> *cubin, std::string *lowered)
{
    std::string all;
    if (path.empty() || !read_file(path, &all) || all.size() < sizeof(DiskHeader)) return false;
    DiskHeader h;
    memcpy(&h, all.data(), sizeof(h));
    if (h.magic != kDiskMagic || h.name_len == 0 || h.cubin_bytes == 0) return false;
    if ((uint64_t)all.size() != sizeof(h) + (uint64_t)h.name_len + h.cubin_bytes) return false;
    const char *body = all.data() + sizeof(h) + h.name_len;
    if (fnv1a(body, (size_t)h.cubin_bytes, 0xcbf29ce484222325ull) != h.cubin_hash) return false;
    lowered->assign(all.data() + sizeof(h), h.name_len);
    cubin->assign(body, body + h.cubin_bytes);
    return true;
}

void disk_store(const std::string &path, const std::vector<char> &cubin, const std::string &lowered)
{
    if (path.empty()) return;
    const std::string dir = path.substr(0, path.rfind('/'));
    mkdir(dir.c_str(), 0755);
    const std::string tmp = path + ".tmp" + std::to_string((long)getpid());
    FILE *f = fopen(tmp.c_str(), "wb");
    if (!f) return;
    DiskHeader h;
    h.magic = kDiskMagic; h.name_len = (uint32_t)lowered.size(); h.cubin_bytes = cubin.size();
    h.cubin_hash = fnv1a(cubin.data(), cubin.size(), 0xcbf29ce484222325ull);
    const bool ok = fwrite(&h, sizeof(h), 1, f) == 1 && fwrite(lowered.data(), 1, h.name_len, f) == h.name_len &&
                    fwrite(cubin.data(), 1, cubin.size(), f) == cubin.size();
    fclose(f);
    if (ok) rename(tmp.c_str(), path.c_str());
    else unlink(tmp.c_str());
}

std::string targ(uint32_t sig) { return std::to_string(sig) + "u"; }

}  // namespace

bool jit_available(std::string *why)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    const bool ok = init_locked();
    if (!ok && why) *why = g_why;
    return ok;
}

std::string jit_render_name(int dim, int gen, int aff, int splat, uint32_t sig, int trig, int opt)
{
    return "cfs::render_kernel<" + std::to_string(dim) + ", " + std::to_string(gen) + ", " + std::to_string(aff) + ", " +
           std::to_string(splat) + ", " + targ(sig) + ", " + std::to_string(trig) + ", " + std::to_string(opt) + ">";
}

std::string jit_cloud_name(int dim, int splat, uint32_t sig, int trig, int opt)
{
    return "cfs::cloud_kernel<" + std::to_string(dim) + ", " + std::to_string(splat) + ", " + targ(sig) + ", " +
           std::to_string(trig) + ", " + std::to_string(opt) + ">";
}

std::string jit_trace_name(int dim, int gen, int aff, uint32_t sig, int trig)
{
    return "cfs::trace_kernel<" + std::to_string(dim) + ", " + std::to_string(gen) + ", " + std::to_string(aff) + ", " +
           targ(sig) + ", " + std::to_string(trig) + ">";
}

bool jit_get(const std::string &name, JitKernel *out, std::string *err)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!init_locked()) { *err = "run-time compilation unavailable: " + g_why; return false; }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); *err = "no CUDA device"; return false; }
    const auto key = std::make_pair(dev, name);
    auto it = g_cache.find(key);
    if (it != g_cache.end()) { out->func = it->second.func; out->compile_ms = 0.0; out->cached = true; return true; }
    if (!init_driver_locked(err)) return false;
    cudaFree(nullptr);                                   // the primary context of the device is current from here on
    const auto t0 = std::chrono::steady_clock::now();
    std::vector<char> cubin;
    std::string lowered;
    const std::string path = cache_path(name);
    bool from_disk = disk_load(path, &cubin, &lowered);
    if (!from_disk && !compile_locked(name, &cubin, &lowered, err)) return false;
    CUmodule mod = nullptr;
    CUresult r = g_driver.ModuleLoadData(&mod, cubin.data());
    if (r != CUDA_SUCCESS && from_disk) {                // a stale or damaged cache file: compile afresh
        from_disk = false;
        if (!compile_locked(name, &cubin, &lowered, err)) return false;
        r = g_driver.ModuleLoadData(&mod, cubin.data());
    }
    if (r != CUDA_SUCCESS) { *err = "cuModuleLoadData: " + cu_error(r); return false; }
    CUfunction fn = nullptr;
    if ((r = g_driver.ModuleGetFunction(&fn, mod, lowered.c_str())) != CUDA_SUCCESS) { *err = "cuModuleGetFunction(" + lowered + "): " + cu_error(r); return false; }
    if (!from_disk) disk_store(path, cubin, lowered);
    const double ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    if (!from_disk) { ++g_n_compiled; g_total_ms += ms; }
    Entry e;
    e.func = fn;
    g_cache[key] = e;
    out->func = fn; out->compile_ms = ms; out->cached = false;
    return true;
}

bool jit_compile_only(const std::string &name, size_t *cubin_bytes, double *ms, std::string *err)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!init_locked()) { *err = "run-time compilation unavailable: " + g_why; return false; }
    const auto t0 = std::chrono::steady_clock::now();
    std::vector<char> cubin;
    std::string lowered;
    if (!compile_locked(name, &cubin, &lowered, err)) return false;
    if (cubin_bytes) *cubin_bytes = cubin.size();
    if (ms) *ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    return true;
}

cudaError_t jit_launch(const JitKernel &k, unsigned grid, unsigned block, size_t dyn_smem, cudaStream_t stream,
                       const RenderParams &prm, std::string *err)
{
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        if (!g_driver.ok || !k.func) { *err = "kernel was not compiled"; return cudaErrorInvalidDeviceFunction; }
        if (dyn_smem > 32 * 1024) {          // static + dynamic beyond the 48 KiB default needs the opt-in
            int dev = 0;
            cudaGetDevice(&dev);
            for (auto &kv : g_cache) {
                if (kv.first.first == dev && kv.second.func == (CUfunction)k.func && kv.second.dyn_smem < (int)dyn_smem) {
                    const CUresult r = g_driver.FuncSetAttribute((CUfunction)k.func, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, (int)dyn_smem);
                    if (r != CUDA_SUCCESS) { *err = "cuFuncSetAttribute: " + cu_error(r); return cudaErrorInvalidValue; }
                    kv.second.dyn_smem = (int)dyn_smem;
                }
            }
        }
    }
    void *args[1] = {const_cast<RenderParams *>(&prm)};
    const CUresult r = g_driver.LaunchKernel((CUfunction)k.func, grid, 1, 1, block, 1, 1, (unsigned)dyn_smem, (CUstream)stream, args, nullptr);
    if (r != CUDA_SUCCESS) { *err = "cuLaunchKernel: " + cu_error(r); return cudaErrorLaunchFailure; }
    return cudaSuccess;
}

void jit_stats(unsigned long long *n_compiled, double *total_ms)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    if (n_compiled) *n_compiled = g_n_compiled;
    if (total_ms) *total_ms = g_total_ms;
}

}  // namespace cfs
