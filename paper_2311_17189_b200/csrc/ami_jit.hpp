// Per-table specialised kernels: interface between the C ABI (ami_api.cu) and ami_jit.cpp.
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "ami_params.h"
#include "ami_table.hpp"

namespace ami {

constexpr int kJitBlockThreadsDefault = 64;
int jit_block_threads();   // kJitBlockThreadsDefault unless AMI_JIT_NT overrides it (tuning knob)

// Tables whose straight-line form is small enough to live in registers and in the instruction
// cache; larger ones are evaluated by the table-driven kernels.
bool jit_eligible(const FlatTable& ft, const HornerPlan& hp);

std::string jit_generate_source(const FlatTable& ft, const HornerPlan& hp, int block_threads);

// NVRTC: CUDA C++ -> sm_100a cubin.  Needs no GPU.  Returns AMI_OK, AMI_EUNSUPPORTED when the
// NVRTC library cannot be loaded, or AMI_EINVAL when compilation fails (`log` has the reason).
int jit_compile(const std::string& src, std::vector<char>& cubin, std::string& log);

// Loads the cubin on the table's device.  Thread-safe, idempotent.
int jit_prepare(ami_table* tab, std::string& err);
cudaError_t jit_launch(const ami_table* tab, bool fused, const AmiBatch& b, cudaStream_t st);
void jit_destroy(ami_table* tab);
int jit_status(const ami_table* tab);   // AMI_OK once loaded, 1 = not tried yet, else the error

}  // namespace ami
