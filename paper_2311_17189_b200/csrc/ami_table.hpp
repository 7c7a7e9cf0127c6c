// Internal definition of ami_table: the host-side symbolic result, the evaluation plans
// derived from it, and the handles of the device-resident copy.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/ami.h"

namespace ami {

// A distinct Fermi/Bose leaf f_sigma^{(k)}(c . e)   (reading P4, P11)
struct LeafF {
  std::vector<int> c;   // [n_eps]
  int sigma;            // +1 / -1
  int k;                // derivative order
  bool operator<(const LeafF& o) const {
    if (k != o.k) return k < o.k;
    if (sigma != o.sigma) return sigma < o.sigma;
    return c < o.c;
  }
};
// A distinct denominator  a . z_ext + c . e, in the orientation the recursion produced (P10)
struct LeafD {
  std::vector<int> a;   // [n_ext]
  std::vector<int> c;   // [n_eps]
  bool operator<(const LeafD& o) const { return a != o.a ? a < o.a : c < o.c; }
};

struct FlatTerm {
  long long num, den;       // exact coefficient num/den
  std::vector<int> f;       // n_int Fermi leaf ids (sorted)
  std::vector<int> d;       // denominator leaf ids (sorted, repeats = powers)
};

struct FlatTable {
  int n_int = 0, n_ext = 0, n_g = 0, n_eps = 0;
  std::vector<uint8_t> ferm;            // [L]
  std::vector<int> sym_alpha;           // [n_eps][L]: momentum combination of each energy symbol
  double prefactor = 1.0;
  std::vector<LeafF> leafF;
  std::vector<LeafD> leafD;
  std::vector<FlatTerm> terms;
  int max_deriv = 0, max_den = 0;
  long long n_terms_raw = 0, n_multipoles = 0;
};

// ---- Horner plan: terms grouped by denominator product R (Eq. 6: FT * R), the
// Fermi/Bose products of each group as a trie evaluated in Horner form, and the denominator
// products of all groups as one trie whose terminals carry the groups' FT sums:
//   result = S_D(root),  S_D(n) = [FT_g if group g ends at n] + sum_{c in kids(n)} Dinv[c.leaf] * S_D(c)
//   FT_g   = S_F(root_g), S_F(n) = [coef if a term ends at n] + sum_{c in kids(n)} F[c.leaf] * S_F(c)
struct HNode {
  int leaf = -1;             // factor of the edge into this node (Fermi leaf id or denominator leaf id)
  std::vector<int> kids;     // node ids
  int group = -1;            // D-trie: the group whose denominator product ends here
};
// FT sums as a DAG: S-nodes are hash-consed across ALL groups, so a partial sum that occurs under
// several denominator products is evaluated once (the AMI recursion produces many of those).
struct SItem {
  int leaf;                  // Fermi leaf of the factor
  int child;                 // S-node multiplied by it, or -1: the item is coef * F[leaf]
  long long num, den;        // coef when child == -1
};
struct SNode {
  std::vector<SItem> items;  // S = sum of items; inner items first
  int height = 1;
};
struct HGroup {
  std::vector<int> d;        // sorted denominator leaf ids (repeats = powers)
  int root = -1;             // S-node of FT_g, or -1: FT_g is the constant num/den
  long long num = 0, den = 1;
};
struct HornerPlan {
  std::vector<HGroup> groups;
  std::vector<SNode> snodes; // children have smaller ids than their parents
  std::vector<HNode> dn;     // dn[0] = root
  std::vector<char> d_is_real;   // [U_D]: no external-frequency part => purely real denominator
  int f_order = 0;           // which factor ordering won (0 = per-group frequency, 1..4 = global)
  long long n_fnodes = 0, n_dnodes = 0;
  long long ops_f = 0;       // FP64 instructions per (sample, beta) of all FT sums
  long long ops_d = 0;       // FP64 instructions per (sample, beta, frequency) of the R part
  long long ops_d_beta = 0;  // R-part products under purely real denominators: per (sample, beta) only
  long long ops_leaf_f = 0;  // FP64 instructions per (sample, beta) of the Fermi/Bose leaves
  long long ops_leaf_d = 0;  // FP64 instructions per (sample, beta, frequency) of the reciprocals
  long long ops_disp = 0;    // FP64 instructions per sample of the dispersion
  long long ops_combo = 0;   // FP64 instructions done once per sample: the distinct energy combinations
                             // and the reciprocals of the purely real denominators
};

// ---- tree plan: the Horner plan as a program for a table-driven interpreter (ami_kernels.cu) ----
// One 32-bit word per operation: op (4 bits) | a (12 bits) | b (16 bits).  A thread keeps one real
// accumulator `acc` and one complex accumulator `c`; F[] are its Fermi/Bose leaves, D[] its
// reciprocal denominators, V[] its value slots, C[] the table's constants.
enum TreeOp : uint32_t {
  kOpSetF = 0,     // acc = F[a]
  kOpSetNegF,      // acc = -F[a]
  kOpMulFV,        // acc = F[a] * V[b]
  kOpFmaFV,        // acc = fma(F[a], V[b], acc)
  kOpAddF,         // acc += F[a]
  kOpSubF,         // acc -= F[a]
  kOpMulCF,        // acc = C[b] * F[a]
  kOpFmaCF,        // acc = fma(C[b], F[a], acc)
  kOpStore,        // a == 0: V[b] = acc;  a == 1: (V[b], V[b+1]) = c
  kOpSetV,         // acc = V[b]
  kOpSetC,         // acc = C[b]
  kOpMulDV,        // acc = Re D[a] * V[b]            (purely real denominator)
  kOpFmaDV,        // acc = fma(Re D[a], V[b], acc)
  kOpCSetV,        // c = (V[b], 0);  b == 0xffff: c = 0
  kOpCFmaDV,       // c += D[a] * V[b]                (complex denominator, real value)
  kOpCFmaDC        // c += D[a] * (V[b], V[b+1])      (complex denominator, complex value)
};
inline uint32_t tree_word(uint32_t op, uint32_t a, uint32_t b) { return (op << 28) | ((a & 0xfffu) << 16) | (b & 0xffffu); }

struct TreeProgram {
  std::vector<uint32_t> code_beta;   // once per (sample, beta): FT sums and frequency-independent sub-sums
  std::vector<uint32_t> code_freq;   // once per (sample, beta, frequency): the R part; the result is left in c
  std::vector<double> consts;
  int n_slots = 0;                   // doubles of V per sample
  bool ok = false;                   // false: table outside the encoding's limits (4095 leaves, 65534 slots)
};
void build_tree_program(const FlatTable& ft, const HornerPlan& hp, TreeProgram& tp);

// The compiled, per-table specialised kernels (ami_jit.cpp).
struct JitState;

int construct_flat(int n_int, int n_ext, int n_g, int n_eps, const int32_t* alpha, const int32_t* eps,
                   const uint8_t* ferm, const int32_t* sum_order, double prefactor, FlatTable& out);
void build_horner_plan(const FlatTable& ft, HornerPlan& plan);
std::vector<double> deriv_poly(int k);   // Q_k of f^{(k)} = beta^k f g Q_k(f), ascending powers of f

}  // namespace ami

// Device-resident arrays (all plain device pointers, owned by the table).
struct ami_device_copy {
  int device = -1;
  // leaf descriptors, compressed: for each leaf a list of (symbol, coefficient) pairs
  int32_t* leaf_ptr = nullptr;    // [U_F + U_D + 1] offsets into leaf_sym / leaf_coef
  int8_t* leaf_sym = nullptr;     // symbol index of each non-zero coefficient
  int8_t* leaf_coef = nullptr;    // its integer coefficient
  int8_t* leafF_sig = nullptr;    // [U_F]
  int8_t* leafF_k = nullptr;      // [U_F]
  int8_t* leafD_a = nullptr;      // [U_D][n_ext]
  // flat plan
  uint16_t* term_idx = nullptr;   // [T][n_int + n_d]: Fermi ids then denominator ids (U_D = unit leaf)
  double* term_coef = nullptr;    // [T]
  // tree plan
  uint32_t* tree_beta = nullptr;  // code_beta, padded to whole tiles
  uint32_t* tree_freq = nullptr;  // code_freq, padded to whole tiles
  double* tree_consts = nullptr;
  // dispersion
  int8_t* sym_alpha = nullptr;    // [n_eps][L]
  double* derivQ = nullptr;       // [AMI_MAX_DERIV+1][8] polynomials of the Fermi derivatives
  int64_t bytes = 0;
};

struct ami_table {
  ami::FlatTable flat;
  ami::HornerPlan horner;
  ami::TreeProgram tree;
  ami::JitState* jit = nullptr;   // owned; see ami_jit.cpp
  void* run_ws = nullptr;         // owned; workspace of ami_run (ami_api.cu)
  ami_device_copy dev;
  int64_t fp64_ops_flat = 0;
};
