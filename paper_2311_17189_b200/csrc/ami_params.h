// Kernel parameter blocks (plain data).  This header is compiled twice: by nvcc into the library
// and, embedded as text, by NVRTC in front of a specialised kernel (ami_jit.cpp), so it uses
// only builtin types and includes nothing.
#ifndef AMI_PARAMS_H
#define AMI_PARAMS_H

#define AMI_K_MAX_FREQ_WORDS 64   // n_f * n_ext complex values per launch
#define AMI_K_MAX_BETA 8          // inverse temperatures per launch
#define AMI_K_MAX_EXT 4

// Batch description shared by every evaluation kernel.
struct AmiBatch {
  // energies, [n_eps][n] doubles (complex: interleaved), rows e_stride samples apart; NULL when the
  // kernel forms them from momenta (fused S1+S2+S3)
  const double* e;
  long long e_stride;
  // momenta for the fused path: component c of internal momentum l of sample s at
  // k[s * k_stride_sample + (2 l + c) * k_stride_comp]
  const double* k;
  long long k_stride_sample, k_stride_comp;
  double q[2 * AMI_K_MAX_EXT];
  double t, mu;
  // split plan (tables too large for one register-resident kernel): the leaf kernel writes every Fermi/Bose
  // value and reciprocal denominator of sample s to leaves[(s / NT) * leaf_stride + slot * NT + s % NT] (one record
  // of leaf_stride doubles per tile of NT = blockDim.x samples); part kernel p writes its partial result of
  // launch-local row r to partial[(p * n_b * n_f + r) * partial_stride + s] (complex)
  double* leaves;
  long long leaf_stride;
  double* partial;
  long long partial_stride;
  int n_parts;
  int part0;                // split plan: index of the first part of the module being launched
  int tiles;                // fused kernels: consecutive tiles of blockDim.x samples one CTA walks
  int tally_acc;            // fused tally with ONE result row: every thread adds its `tiles` samples before the warp adds up
  int unordered;            // register plan: the caller declared this launch independent of the specialised launches just
                            // before it in the stream (AMI_PLAN_UNORDERED): it waits for them at its END, not its start
  double* e_out;            // optional [n_eps][n] copy of the energies formed by the fused path
  // fused tally (or NULL): per-warp partial sums (re, im, re^2, im^2) of row r at tally[(r * tally_stride + (s >> 5)) * 4]
  double* tally;
  long long tally_stride;
  // results (out may be NULL when only the tally is wanted): complex128, row r = (b0 + b) * n_f_total + (f0 + f) at out + 2 * r * out_row_stride
  double* out;
  long long n, out_row_stride;
  int n_f, n_b, n_f_total, f0, b0;
  int gen;                  // fused path: momenta come from the counter-based generator (P22), k is not read
  unsigned long long seed;  // generator seed and the stream index of sample 0 of this batch
  long long first_sample;
  double e_reg, prefactor;
  double beta[AMI_K_MAX_BETA];
  double ceta[AMI_K_MAX_BETA];          // exp(beta * e_reg), formed on the host (exactly 1 without regulator)
  double z[2 * AMI_K_MAX_FREQ_WORDS];   // [n_f][n_ext] complex
};

#endif
