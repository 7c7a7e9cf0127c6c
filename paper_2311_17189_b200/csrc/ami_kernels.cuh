// Kernel parameter blocks and launcher declarations (internal).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "ami_table.hpp"

namespace ami {

constexpr int kMaxFreqWords = 64;   // n_f * n_ext complex values per launch
constexpr int kMaxBeta = 8;         // inverse temperatures per launch
constexpr int kMaxSumBlocks = 8 * 148;   // partial sums per row of the tally kernels
constexpr int kTermTile = 256;      // terms per shared-memory tile of the flat plan (multiple of 8)

struct EvalParams {
  // table (device pointers)
  const int32_t* leaf_ptr;
  const int8_t* leaf_sym;
  const int8_t* leaf_coef;
  const int8_t* leafF_sig;
  const int8_t* leafF_k;
  const int8_t* leafD_a;
  const uint16_t* term_idx;
  const double* term_coef;
  const double* derivQ;
  // tree plan: programs (padded to whole tiles), constants, value slots
  const uint32_t* tree_beta;
  const uint32_t* tree_freq;
  const double* tree_consts;
  long long n_words_beta, n_words_freq;
  int n_slots, n_consts;
  double* v_scratch;           // global value slots [n_slots][v_stride] when they do not fit in shared memory
  long long v_stride;
  int n_eps, n_ext, U_F, U_D, m_f, n_d;
  long long T;
  // batch
  const double* e;          // [n_eps][n_e] (complex: interleaved)
  double* out;              // complex128, row r = b * n_f_total + f at out + 2 * r * out_row_stride
  long long n_e, e_stride, out_row_stride;
  int n_f, n_b, n_f_total, f0, b0;
  double e_reg, prefactor;
  double beta[kMaxBeta];
  double z[2 * kMaxFreqWords];  // [n_f][n_ext] complex
};

struct DispParams {
  const int8_t* sym_alpha;   // [n_eps][L]
  int n_int, n_ext, n_eps;
  const double* k;
  long long k_stride_sample, k_stride_comp, n;
  int dim, band;             // momentum components (1..3); 0 = hypercubic tight binding, 1 = free particles
  double q[3 * AMI_MAX_EXT]; // [n_ext][dim]
  double t, mu;
  double* e;                 // [n_eps][n]
  long long e_stride;
};

cudaError_t launch_dispersion(const DispParams& p, cudaStream_t st);
cudaError_t launch_eval_flat(const EvalParams& p, bool e_is_complex, cudaStream_t st, int* launches);
cudaError_t launch_eval_tree(const EvalParams& p, cudaStream_t st, int* launches);   // real energies
bool tree_values_fit_smem(const EvalParams& p);
cudaError_t launch_generate_momenta(uint64_t seed, long long first, long long n, int n_comp, double* d_k,
                                    cudaStream_t st);
cudaError_t launch_block_sums(const double* d_vals, long long n_rows, long long n, long long row_stride,
                              double* d_partial, double* d_sum, bool first, cudaStream_t st, int* launches);
cudaError_t launch_warp_partial_sums(const double* d_warp_partials, long long n_rows, long long n_warps,
                                     long long row_stride, double* d_partial, double* d_sum, bool first,
                                     cudaStream_t st, int* launches);
// stream-ordered workspace from the library's own memory pool (free with cudaFreeAsync)
cudaError_t scratch_alloc(void** ptr, size_t bytes, cudaStream_t st);
cudaError_t run_fp64_probe(int distinct_sources, double* dfma_per_s, double* ms);
long long total_launches();
void count_external_launch(int* launches);

}  // namespace ami
