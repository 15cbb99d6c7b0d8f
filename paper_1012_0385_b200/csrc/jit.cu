// jit.cu — run-time specialisation of the sweep kernels with NVRTC.
//
// The kernel sources (csrc/*.cuh listed in build.py's JIT_SOURCES) are embedded in the library as strings by the
// build (jit_embed.inc).  jit_get() compiles one entry point for sm_100a with a list of -D definitions (ring size,
// thresholds, ...), loads the cubin through the CUDA runtime's library API and caches the kernel handle per
// process.  Compilation needs no GPU; loading does.
#include "jit.h"

#include <cuda_runtime.h>
#include <nvrtc.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "common.cuh"

namespace kpz {

namespace {
struct Embedded {
  const char* name;
  const char* text;
};
#include "jit_embed.inc"  // static const Embedded kEmbedded[] = {{"philox.cuh", R"...(...)..."}, ...};

struct Entry {
  std::vector<char> cubin;
  cudaLibrary_t lib = nullptr;
  cudaKernel_t kernel = nullptr;
};
std::mutex g_mu;
std::map<std::string, Entry> g_cache;

const Embedded* find_source(const char* name) {
  for (const Embedded& e : kEmbedded)
    if (std::strcmp(e.name, name) == 0) return &e;
  return nullptr;
}
}  // namespace

bool jit_enabled() {
  const char* e = std::getenv("KPZ_B200_JIT");
  return !(e && e[0] == '0');
}

int jit_compile(const char* source, const char* entry, const std::vector<std::string>& defines,
                std::vector<char>* cubin, std::string* log) {
  const Embedded* src = find_source(source);
  if (!src) return fail(KPZ_EINVAL, "jit: no embedded source named %s", source);
  std::vector<const char*> hnames, htexts;
  for (const Embedded& e : kEmbedded) {
    hnames.push_back(e.name);
    htexts.push_back(e.text);
  }
  // name the program by its path at build time when that file still exists (ncu --import-source, -lineinfo)
  std::string pname = std::string(kEmbeddedDir) + "/" + src->name;
  if (FILE* f = std::fopen(pname.c_str(), "r")) std::fclose(f);
  else pname = src->name;
  nvrtcProgram prog;
  nvrtcResult r = nvrtcCreateProgram(&prog, src->text, pname.c_str(), (int)hnames.size(), htexts.data(), hnames.data());
  if (r != NVRTC_SUCCESS) return fail(KPZ_ECUDA, "nvrtcCreateProgram: %s", nvrtcGetErrorString(r));
  std::vector<std::string> opts = {"--gpu-architecture=sm_100a", "-std=c++17", "-lineinfo", "-DKPZ_JIT=1"};
  for (const std::string& d : defines) opts.push_back("-D" + d);
  std::vector<const char*> copts;
  for (const std::string& o : opts) copts.push_back(o.c_str());
  r = nvrtcCompileProgram(prog, (int)copts.size(), copts.data());
  size_t logsz = 0;
  nvrtcGetProgramLogSize(prog, &logsz);
  std::string text(logsz, '\0');
  if (logsz > 1) nvrtcGetProgramLog(prog, &text[0]);
  if (log) *log = text;
  if (r != NVRTC_SUCCESS) {
    nvrtcDestroyProgram(&prog);
    return fail(KPZ_ECUDA, "nvrtc compile of %s failed: %s\n%.400s", entry, nvrtcGetErrorString(r), text.c_str());
  }
  size_t n = 0;
  r = nvrtcGetCUBINSize(prog, &n);
  if (r != NVRTC_SUCCESS || n == 0) {
    nvrtcDestroyProgram(&prog);
    return fail(KPZ_ECUDA, "nvrtcGetCUBINSize: %s", nvrtcGetErrorString(r));
  }
  cubin->resize(n);
  r = nvrtcGetCUBIN(prog, cubin->data());
  nvrtcDestroyProgram(&prog);
  if (r != NVRTC_SUCCESS) return fail(KPZ_ECUDA, "nvrtcGetCUBIN: %s", nvrtcGetErrorString(r));
  return KPZ_OK;
}

int jit_get(const char* source, const char* entry, const std::vector<std::string>& defines, void** kernel) {
  std::string key = std::string(source) + "|" + entry;
  for (const std::string& d : defines) key += "|" + d;
  std::lock_guard<std::mutex> lock(g_mu);
  auto it = g_cache.find(key);
  if (it == g_cache.end()) {
    Entry e;
    int rc = jit_compile(source, entry, defines, &e.cubin, nullptr);
    if (rc) return rc;
    cudaError_t ce = cudaLibraryLoadData(&e.lib, e.cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (ce != cudaSuccess) return fail(KPZ_ECUDA, "cudaLibraryLoadData(%s): %s", entry, cudaGetErrorString(ce));
    ce = cudaLibraryGetKernel(&e.kernel, e.lib, entry);
    if (ce != cudaSuccess) return fail(KPZ_ECUDA, "cudaLibraryGetKernel(%s): %s", entry, cudaGetErrorString(ce));
    it = g_cache.emplace(key, std::move(e)).first;
  }
  *kernel = (void*)it->second.kernel;
  return KPZ_OK;
}

}  // namespace kpz
