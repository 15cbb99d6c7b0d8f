// jit.h — run-time kernel specialisation (NVRTC); see jit.cu.
#pragma once
#include <string>
#include <vector>

namespace kpz {

// False when the environment variable KPZ_B200_JIT is "0": the statically compiled kernels are used instead.
bool jit_enabled();

// Compile `entry` (an extern "C" __global__ function) of the embedded source file `source` for sm_100a with the
// given NAME=VALUE definitions.  Needs no GPU.  Returns KPZ_OK and the cubin, or an error code (text in
// kpz_last_error()).
int jit_compile(const char* source, const char* entry, const std::vector<std::string>& defines,
                std::vector<char>* cubin, std::string* log);

// Compile (once per process and per definition list), load on the current device, and return a handle that
// cudaLaunchKernel accepts as its function argument.
int jit_get(const char* source, const char* entry, const std::vector<std::string>& defines, void** kernel);

}  // namespace kpz
