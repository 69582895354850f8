// gq_jit.cpp — compiles generated kernel sources to sm_100a cubins with NVRTC, caches them on disk (in-tree) and in
// the process, and loads them through the CUDA runtime's library API (cudaLibraryLoadData; no driver-API link).
// NVRTC is dlopen'ed lazily so libgq.so loads (and cached kernels run) even where libnvrtc is absent. Compilation
// needs no GPU: build() pre-populates the cache for the benchmark plan shapes on the CPU-only build box.
#include <dlfcn.h>
#include <sys/stat.h>

#include <cstdio>
#include <cstdlib>
#include <unistd.h>

#include <fstream>
#include <map>
#include <mutex>
#include <sstream>

#include "gq_internal.h"

namespace {
std::mutex g_mu;
std::string g_cache_dir;
std::map<std::string, GqKernel> g_loaded;   // hash@device -> loaded kernel (the shared-memory attribute is per device)

typedef int (*fn_create)(void**, const char*, const char*, int, const char* const*, const char* const*);
typedef int (*fn_compile)(void*, int, const char* const*);
typedef int (*fn_size)(void*, size_t*);
typedef int (*fn_get)(void*, char*);
typedef int (*fn_destroy)(void**);
struct Nvrtc {
  void* h = nullptr;
  fn_create create; fn_compile compile; fn_size log_size; fn_get log; fn_size cubin_size; fn_get cubin; fn_destroy destroy;
} g_nvrtc;

bool load_nvrtc(std::string* msg) {
  if (g_nvrtc.h) return true;
  const char* names[] = {"/usr/local/cuda/lib64/libnvrtc.so.12", "libnvrtc.so.12", "libnvrtc.so", nullptr};   // the toolkit's own NVRTC first: an older one bundled with a Python package may already be in the process
  for (int i = 0; names[i] && !g_nvrtc.h; ++i) g_nvrtc.h = dlopen(names[i], RTLD_NOW | RTLD_LOCAL);
  if (!g_nvrtc.h) { if (msg) *msg = "cannot dlopen libnvrtc.so.12"; return false; }
  g_nvrtc.create = (fn_create)dlsym(g_nvrtc.h, "nvrtcCreateProgram");
  g_nvrtc.compile = (fn_compile)dlsym(g_nvrtc.h, "nvrtcCompileProgram");
  g_nvrtc.log_size = (fn_size)dlsym(g_nvrtc.h, "nvrtcGetProgramLogSize");
  g_nvrtc.log = (fn_get)dlsym(g_nvrtc.h, "nvrtcGetProgramLog");
  g_nvrtc.cubin_size = (fn_size)dlsym(g_nvrtc.h, "nvrtcGetCUBINSize");
  g_nvrtc.cubin = (fn_get)dlsym(g_nvrtc.h, "nvrtcGetCUBIN");
  g_nvrtc.destroy = (fn_destroy)dlsym(g_nvrtc.h, "nvrtcDestroyProgram");
  if (!g_nvrtc.create || !g_nvrtc.compile || !g_nvrtc.cubin || !g_nvrtc.cubin_size) {
    if (msg) *msg = "libnvrtc lacks expected symbols"; return false; }
  return true;
}

std::string cache_dir() {
  if (!g_cache_dir.empty()) return g_cache_dir;
  if (const char* e = getenv("GQ_KERNEL_CACHE")) return g_cache_dir = e;
  Dl_info info;
  if (dladdr((void*)&gq_jit_set_cache_dir, &info) && info.dli_fname) {
    std::string p = info.dli_fname;
    size_t s = p.find_last_of('/');
    g_cache_dir = (s == std::string::npos ? std::string(".") : p.substr(0, s)) + "/_kcache";
  } else g_cache_dir = "./_kcache";
  return g_cache_dir;
}

bool read_file(const std::string& path, std::string* out) {
  std::ifstream f(path, std::ios::binary);
  if (!f) return false;
  std::ostringstream ss; ss << f.rdbuf(); *out = ss.str();
  return !out->empty();
}
bool write_file(const std::string& path, const std::string& data) {
  std::string tmp = path + ".tmp" + std::to_string((long long)getpid());
  { std::ofstream f(tmp, std::ios::binary); if (!f) return false; f.write(data.data(), (std::streamsize)data.size()); }
  return rename(tmp.c_str(), path.c_str()) == 0;
}

gq_status compile(const GqKernelInfo& info, std::string* cubin, std::string* msg) {
  if (!load_nvrtc(msg)) return GQ_ERR_COMPILE;
  void* prog = nullptr;
  std::string name = cache_dir() + "/" + info.hash + ".cu";   // -lineinfo then points at the cached source
  if (g_nvrtc.create(&prog, info.source.c_str(), name.c_str(), 0, nullptr, nullptr) != 0) {
    if (msg) *msg = "nvrtcCreateProgram failed"; return GQ_ERR_COMPILE; }
  const char* opts[] = {"--gpu-architecture=sm_100a", "-lineinfo", "--std=c++17", "-default-device"};
  int rc = g_nvrtc.compile(prog, 3, opts);
  if (rc != 0) {
    size_t n = 0; g_nvrtc.log_size(prog, &n);
    std::string log(n, '\0'); if (n) g_nvrtc.log(prog, &log[0]);
    if (msg) *msg = "nvrtc: " + log.substr(0, 4000);
    g_nvrtc.destroy(&prog);
    return GQ_ERR_COMPILE;
  }
  size_t n = 0; g_nvrtc.cubin_size(prog, &n);
  cubin->assign(n, '\0'); g_nvrtc.cubin(prog, &(*cubin)[0]);
  g_nvrtc.destroy(&prog);
  return GQ_OK;
}

gq_status get_cubin(const GqKernelInfo& info, std::string* cubin, std::string* path_out, std::string* msg) {
  std::string dir = cache_dir();
  mkdir(dir.c_str(), 0755);
  std::string cpath = dir + "/" + info.hash + ".cubin";
  if (path_out) *path_out = cpath;
  std::string src;
  if (read_file(cpath, cubin) && read_file(dir + "/" + info.hash + ".cu", &src) && src == info.source) return GQ_OK;
  gq_status st = compile(info, cubin, msg);
  if (st != GQ_OK) return st;
  write_file(dir + "/" + info.hash + ".cu", info.source);   // best effort: a read-only tree still works
  write_file(cpath, *cubin);
  return GQ_OK;
}
}  // namespace

void gq_jit_set_cache_dir(const char* path) { std::lock_guard<std::mutex> l(g_mu); g_cache_dir = path ? path : ""; }

gq_status gq_jit_compile_to_cache(const GqKernelInfo& info, std::string* cubin_path, std::string* msg) {
  std::lock_guard<std::mutex> l(g_mu);
  std::string cubin;
  return get_cubin(info, &cubin, cubin_path, msg);
}

gq_status gq_jit_get(const GqKernelInfo& info, int device, GqKernel* out, std::string* msg, int* cuda_err) {
  std::lock_guard<std::mutex> l(g_mu);
  const std::string lkey = info.hash + "@" + std::to_string(device);
  auto it = g_loaded.find(lkey);
  if (it != g_loaded.end()) { *out = it->second; return GQ_OK; }
  std::string cubin;
  gq_status st = get_cubin(info, &cubin, nullptr, msg);
  if (st != GQ_OK) return st;
  cudaLibrary_t lib;
  cudaError_t e = cudaLibraryLoadData(&lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
  cudaKernel_t fn = nullptr;
  if (e == cudaSuccess) e = cudaLibraryGetKernel(&fn, lib, info.entry.c_str());
  if (e == cudaSuccess) e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, info.smem_bytes);
  if (e != cudaSuccess) {
    if (cuda_err) *cuda_err = (int)e;
    if (msg) *msg = std::string("loading generated kernel: ") + cudaGetErrorString(e);
    return GQ_ERR_CUDA;
  }
  GqKernel k; k.fn = fn; k.threads = info.threads; k.smem_bytes = info.smem_bytes; k.tile_rows = info.tile_rows; k.cluster = info.cluster;
  g_loaded[lkey] = k;
  *out = k;
  return GQ_OK;
}
