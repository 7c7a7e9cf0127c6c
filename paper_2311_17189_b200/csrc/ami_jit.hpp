// Per-table specialised kernels: interface between the C ABI (ami_api.cu) and ami_jit.cpp.
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "ami_params.h"
#include "ami_table.hpp"

namespace ami {

constexpr int kJitBlockThreads = 64;       // threads per CTA of every specialised kernel
constexpr int kJitWarpsPerSmTarget = 12;   // occupancy the register cap of the specialised kernels is set for
constexpr int kJitTallyTiles = 8;          // samples a thread adds up itself in the single-row fused tally

// How a table is specialised.
//   kJitRegister  the whole table is ONE straight-line kernel, every value a register (orders <= 6-7)
//   kJitSplit     larger tables (order 7-8: 1e4-1e5 terms): a leaf kernel writes the Fermi/Bose values and the
//                 reciprocal denominators of a chunk of samples to an L2-resident array, then the groups of the
//                 Horner plan, partitioned into parts of register-plan size, are evaluated by ONE launch whose
//                 grid.y is the part, and a last kernel adds the parts' partial results in a fixed order
//   kJitNone      table-driven kernels only (AMI_DISABLE_JIT=1, or outside every limit)
enum { kJitNone = 0, kJitRegister = 1, kJitSplit = 2 };
int jit_mode(const FlatTable& ft, const HornerPlan& hp);
bool jit_eligible(const FlatTable& ft, const HornerPlan& hp);

// What the generated text is specialised for besides the table: the lattice of the inline dispersion (the
// momenta have `dim` components, Eq. 14) and its band, and whether the energies are complex.
struct JitVariant {
  int dim = 2;
  int band = AMI_BAND_TIGHT_BINDING;
  bool cplx = false;
  int key() const { return dim + 4 * band + 16 * (cplx ? 1 : 0); }
};

// Layout facts of a generated module that the launcher needs.
struct JitLayout {
  int mode = kJitNone;
  int n_parts = 0;          // split plan: parts of the Horner plan
  int n_real_den = 0;       // split plan: leaf slots per sample = n_real_den + n_b * U_F + 2 * n_f * n_cplx_den
  int n_cplx_den = 0;
  int n_fermi = 0;
  std::vector<int> part0;   // split plan: module j (of the parts) holds parts part0[j] .. part0[j+1]-1
};

// The translation units of one variant: one for the register plan; for the split plan the leaf kernels and the
// combine kernel first, then the parts, a few per unit.
std::vector<std::string> jit_generate_sources(const FlatTable& ft, const HornerPlan& hp, const JitVariant& var,
                                              JitLayout* layout);

// stream-ordered workspace from the library's own memory pool (ami_kernels.cu; free with cudaFreeAsync)
cudaError_t scratch_alloc(void** ptr, size_t bytes, cudaStream_t st);

// NVRTC: CUDA C++ -> sm_100a cubin.  Needs no GPU.  Returns AMI_OK, AMI_EUNSUPPORTED when the
// NVRTC library cannot be loaded, or AMI_EINVAL when compilation fails (`log` has the reason).
// With `use_cache` the cubin is looked up in / added to the on-disk cache (see ami_jit.cpp).
int jit_compile(const std::string& src, std::vector<char>& cubin, std::string& log, bool use_cache = true,
                bool* cache_hit = nullptr);

// Compiles (or fetches) and loads the kernels of one variant on the table's device.  Thread-safe, idempotent.
int jit_prepare(ami_table* tab, const JitVariant& var, std::string& err);
// `launches` (may be NULL) is incremented per kernel launched; *tally_slots (may be NULL) receives the number of
// per-row partial sums the fused tally wrote.
cudaError_t jit_launch(const ami_table* tab, const JitVariant& var, bool fused, const AmiBatch& b, cudaStream_t st,
                       int* launches, long long* tally_slots);
void jit_destroy(ami_table* tab);
int jit_status(const ami_table* tab);   // of the default variant: AMI_OK once loaded, 1 = not tried yet, else the error
bool jit_fused_tally_ok(const ami_table* tab);   // the loaded plan forms the Monte-Carlo tally inside its kernel
double jit_last_compile_ms(const ami_table* tab, int* cache_hit);   // default variant: time spent in jit_prepare

}  // namespace ami
