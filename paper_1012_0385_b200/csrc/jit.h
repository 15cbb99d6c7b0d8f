// jit.h — run-time kernel specialisation (NVRTC); see jit.cu.
#pragma once
#include <string>
#include <vector>

namespace kpz {

// False after kpz_debug_config("jit=0"): the statically compiled generic kernels are used instead.
bool jit_enabled();

// Process-wide debug configuration (kpz_debug_config in include/kpz_b200.h; tests and tuning only): replaces the
// list of extra definitions; "jit=0|1" switches run-time specialisation.  The run entry points read no environment.
int debug_config(const char* spec);
// The extra NAME=VALUE definitions whose name starts with `prefix` ("K1J_", "K4J_"), appended to a kernel's list.
void debug_defines(const char* prefix, std::vector<std::string>* defs);
// True when the debug configuration defines NAME (whatever its value).
bool debug_has(const char* name);
// Integer value of NAME in the debug configuration, or dflt.
int debug_int(const char* name, int dflt);

// Compile `entry` (an extern "C" __global__ function) of the embedded source file `source` for sm_100a with the
// given NAME=VALUE definitions.  Needs no GPU.  Returns KPZ_OK and the cubin, or an error code (text in
// kpz_last_error()).
int jit_compile(const char* source, const char* entry, const std::vector<std::string>& defines,
                std::vector<char>* cubin, std::string* log);

// Compile (once per process and per definition list), load on the current device, and return a handle that
// cudaLaunchKernel accepts as its function argument.
int jit_get(const char* source, const char* entry, const std::vector<std::string>& defines, void** kernel);

// Write every cubin compiled by this process (loaded or not) to dir; see kpz_debug_dump_cubins.
int dump_cubins(const char* dir, int* count);

}  // namespace kpz
