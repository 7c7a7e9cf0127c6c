// Per-table specialised kernels: interface between the C ABI (ami_api.cu) and ami_jit.cpp.
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "ami_params.h"
#include "ami_table.hpp"

namespace ami {

constexpr int kJitBlockThreadsDefault = 64;
constexpr int kJitTilesPerCtaDefault = 1;
constexpr int kJitPrefetchCtasDefault = 0;
int jit_prefetch_ctas();    // L2 prefetch distance of the fused kernel in CTAs, 0 = off (AMI_JIT_PF, tuning knob)
constexpr int kJitStoreModeDefault = 1;
int jit_store_mode();       // result stores: 0 plain, 1 streaming (st.global.cs), 2 write-through (AMI_JIT_STORE, tuning knob)
constexpr int kJitWarpsPerSmTarget = 12;   // occupancy the register cap of the specialised kernels is set for
int jit_min_blocks(int block_threads);   // second argument of __launch_bounds__ (AMI_JIT_MINB overrides; tuning knob)
bool jit_fermi_in_smem();   // Fermi/Bose leaves in shared memory instead of registers (AMI_JIT_SMEM_F=1, tuning knob)
int jit_tiles_per_cta();    // kJitTilesPerCtaDefault unless AMI_JIT_U overrides it (tuning knob)
int jit_block_threads();   // kJitBlockThreadsDefault unless AMI_JIT_NT overrides it (tuning knob)

// Tables whose straight-line form is small enough to live in registers and in the instruction
// cache; larger ones are evaluated by the table-driven kernels.
enum { kJitNone = 0, kJitRegister = 1, kJitScratch = 2 };
// kJitRegister: every value in registers.  kJitScratch (tables beyond that, e.g. order 8): the same
// generated arithmetic with Fermi/Bose leaves in shared memory and the long-lived sums in a
// per-sample column of a global scratch array.  kJitNone: table-driven kernels only.
int jit_mode(const FlatTable& ft, const HornerPlan& hp);
bool jit_eligible(const FlatTable& ft, const HornerPlan& hp);

// *scratch_slots receives the doubles of scratch per sample the generated kernels need (0 in register mode).
std::string jit_generate_source(const FlatTable& ft, const HornerPlan& hp, int block_threads, bool scratch,
                                int* scratch_slots);

// NVRTC: CUDA C++ -> sm_100a cubin.  Needs no GPU.  Returns AMI_OK, AMI_EUNSUPPORTED when the
// NVRTC library cannot be loaded, or AMI_EINVAL when compilation fails (`log` has the reason).
int jit_compile(const std::string& src, std::vector<char>& cubin, std::string& log);

// Loads the cubin on the table's device.  Thread-safe, idempotent.
int jit_prepare(ami_table* tab, std::string& err);
// `launches` (may be NULL) is incremented per kernel launched (the memory-backed variant walks a large
// batch in chunks).
cudaError_t jit_launch(const ami_table* tab, bool fused, const AmiBatch& b, cudaStream_t st, int* launches);
void jit_destroy(ami_table* tab);
int jit_status(const ami_table* tab);   // AMI_OK once loaded, 1 = not tried yet, else the error

}  // namespace ami
