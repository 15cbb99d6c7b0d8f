// jit.cu — run-time specialisation of the sweep kernels with NVRTC.
//
// The kernel sources (csrc/*.cuh listed in build.py's JIT_SOURCES) are embedded in the library as strings by the
// build (jit_embed.inc).  jit_get() compiles one entry point for sm_100a with a list of -D definitions (ring size,
// thresholds, ...), loads the cubin through the CUDA runtime's library API and caches the kernel handle per
// process.  Compilation needs no GPU; loading does.
#include "jit.h"

#include <cuda_runtime.h>
#include <nvrtc.h>

#include <cctype>
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
// every image compiled by this process, loaded or not (kpz_debug_dump_cubins): entry -> (definitions, cubin)
struct Compiled {
  std::string entry, defines;
  std::vector<char> cubin;
};
std::mutex g_compiled_mu;
std::vector<Compiled> g_compiled;

const Embedded* find_source(const char* name) {
  for (const Embedded& e : kEmbedded)
    if (std::strcmp(e.name, name) == 0) return &e;
  return nullptr;
}
}  // namespace

namespace {
std::mutex g_dbg_mu;
bool g_jit_on = true;
std::vector<std::string> g_dbg_defs;
}  // namespace

bool jit_enabled() {
  std::lock_guard<std::mutex> lock(g_dbg_mu);
  return g_jit_on;
}

int debug_config(const char* spec) {
  std::vector<std::string> defs;
  bool jit_on = true;
  std::string s = spec ? spec : "";
  size_t pos = 0;
  while (pos <= s.size()) {
    size_t end = s.find(';', pos);
    if (end == std::string::npos) end = s.size();
    std::string tok = s.substr(pos, end - pos);
    pos = end + 1;
    while (!tok.empty() && tok.front() == ' ') tok.erase(tok.begin());
    while (!tok.empty() && tok.back() == ' ') tok.pop_back();
    if (tok.empty()) continue;
    const size_t eq = tok.find('=');
    if (eq == std::string::npos || eq == 0 || eq + 1 >= tok.size())
      return fail(KPZ_EINVAL, "debug config: '%s' is not NAME=VALUE", tok.c_str());
    for (char c : tok)
      if (!(std::isalnum((unsigned char)c) || c == '_' || c == '=' || c == '-'))
        return fail(KPZ_EINVAL, "debug config: bad character in '%s'", tok.c_str());
    if (tok.compare(0, eq, "jit") == 0) {
      jit_on = tok[eq + 1] != '0';
    } else if (tok.compare(0, 4, "K1J_") == 0 || tok.compare(0, 4, "K4J_") == 0 || tok.compare(0, 4, "K5J_") == 0) {
      defs.push_back(tok);
    } else {
      return fail(KPZ_EINVAL, "debug config: unknown name in '%s' (jit, K1J_*, K4J_*, K5J_*)", tok.c_str());
    }
  }
  std::lock_guard<std::mutex> lock(g_dbg_mu);
  g_jit_on = jit_on;
  g_dbg_defs.swap(defs);
  return KPZ_OK;
}

void debug_defines(const char* prefix, std::vector<std::string>* out) {
  std::lock_guard<std::mutex> lock(g_dbg_mu);
  const size_t n = std::strlen(prefix);
  for (const std::string& d : g_dbg_defs)
    if (d.compare(0, n, prefix) == 0) out->push_back(d);
}

bool debug_has(const char* name) {
  std::lock_guard<std::mutex> lock(g_dbg_mu);
  const size_t n = std::strlen(name);
  for (const std::string& d : g_dbg_defs)
    if (d.size() > n && d.compare(0, n, name) == 0 && d[n] == '=') return true;
  return false;
}

int debug_int(const char* name, int dflt) {
  std::lock_guard<std::mutex> lock(g_dbg_mu);
  const size_t n = std::strlen(name);
  for (const std::string& d : g_dbg_defs)
    if (d.size() > n && d.compare(0, n, name) == 0 && d[n] == '=') return std::atoi(d.c_str() + n + 1);
  return dflt;
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
  {
    std::string dl;
    for (const std::string& d : defines) dl += "-D" + d + "\n";
    std::lock_guard<std::mutex> lock(g_compiled_mu);
    bool seen = false;
    for (const Compiled& c : g_compiled) seen = seen || (c.entry == entry && c.defines == dl);
    if (!seen) g_compiled.push_back(Compiled{entry, dl, *cubin});
  }
  return KPZ_OK;
}

int dump_cubins(const char* dir, int* count) {
  if (!dir) return fail(KPZ_EINVAL, "dir is NULL");
  std::lock_guard<std::mutex> lock(g_compiled_mu);
  int n = 0;
  for (const Compiled& c : g_compiled) {
    const std::string base = std::string(dir) + "/" + c.entry + "_" + std::to_string(n);
    FILE* f = std::fopen((base + ".cubin").c_str(), "wb");
    if (!f) return fail(KPZ_EINVAL, "cannot write %s.cubin", base.c_str());
    std::fwrite(c.cubin.data(), 1, c.cubin.size(), f);
    std::fclose(f);
    f = std::fopen((base + ".txt").c_str(), "w");
    if (!f) return fail(KPZ_EINVAL, "cannot write %s.txt", base.c_str());
    std::fputs(c.defines.c_str(), f);
    std::fclose(f);
    ++n;
  }
  if (count) *count = n;
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
