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
  std::vector<std::vector<int>> dseq;   // per group: its denominators in the order of its path through dn
  std::vector<char> d_is_real;   // [U_D]: no external-frequency part => purely real denominator
  int f_order = 0;           // which factor ordering won (0 = per-group frequency, 1..4 = global)
  long long n_fnodes = 0, n_dnodes = 0;
  long long ops_f = 0;       // FP64 instructions per (sample, beta) of all FT sums
  long long ops_d = 0;       // FP64 instructions per (sample, beta, frequency) of the R part
  long long ops_d_beta = 0;  // R-part products under purely real denominators: per (sample, beta) only
  // several-temperature body of the register plan (ami_jit.cpp): R part as Q(root) + sum_n Q(n) P_n
  long long ops_prefix = 0;  // per (sample, frequency): the prefix products P_n, 4 per complex trie node below the first level
  long long ops_qsum = 0;    // per (sample, beta, frequency): 2 per complex trie node that carries a Q, 1 for the root's
  bool mb_prefix = false;    // that form is what the several-temperature body uses: it is the cheaper one from two temperatures on
  long long ops_leaf_f = 0;  // FP64 instructions per (sample, beta) of the Fermi/Bose leaves
  long long ops_leaf_d = 0;  // FP64 instructions per (sample, beta, frequency) of the reciprocals
  long long ops_disp = 0;    // FP64 instructions per sample of the dispersion
  long long ops_combo = 0;   // FP64 instructions done once per sample: the distinct energy combinations
                             // and the reciprocals of the purely real denominators
};

// ---- tree plan: the Horner plan as a program for a table-driven interpreter (ami_kernels.cu) ----
// A program is a list of NODES.  A node is one header word  count << 16 | dst  followed by `count`
// item words  flag << 28 | a << 16 | b.  Executing a node:
//   real node (per-beta program):        acc = sum_i L[a_i] * V[b_i];                V[dst] = acc
//   complex node (per-frequency program): c  = sum_i D[a_i] * (V[b_i], flag_i ? V[b_i+1] : 0);
//                                          (V[dst], V[dst+1]) = c, or c is the result when dst == 0xffff
// L[] is the thread's leaf array: L[u] = Fermi/Bose leaf u for u < U_F, L[U_F + 2u] = Re of reciprocal
// denominator u, L[U_F + 2 U_D] = 1.  D[u] is reciprocal denominator u as a complex number, D[U_D] = 1.
// V[] are the thread's value slots; V[0 .. n_consts) hold the table's constants (1, -1, coefficients).
// Items are uniform (no opcode to branch on), so the interpreter's inner loop is a plain FMA loop.
// A node never straddles a tile of kTreeTileWords words (the builder pads with empty headers).
constexpr int kTreeTileWords = 1024;
constexpr uint32_t kTreeNoDst = 0xffffu;
inline uint32_t tree_header(uint32_t count, uint32_t dst) { return (count << 16) | (dst & 0xffffu); }
inline uint32_t tree_item(uint32_t flag, uint32_t a, uint32_t b) { return (flag << 28) | ((a & 0xfffu) << 16) | (b & 0xffffu); }

struct TreeProgram {
  std::vector<uint32_t> code_beta;   // real nodes, once per (sample, beta): FT sums and frequency-independent sub-sums
  std::vector<uint32_t> code_freq;   // complex nodes, once per (sample, beta, frequency): the R part
  std::vector<double> consts;        // preloaded into V[0 .. consts.size())
  int n_slots = 0;                   // doubles of V per sample, constants included
  bool ok = false;                   // false: table outside the encoding's limits
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
