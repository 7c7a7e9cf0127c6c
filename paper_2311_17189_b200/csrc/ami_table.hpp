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

// ---- tree plan: terms grouped by denominator product, Fermi products in a trie ----------
// Byte-code executed identically by every thread; see ami_plan.cpp for the format.
struct TreePlan {
  std::vector<uint32_t> code;     // program words
  std::vector<double> consts;     // non-unit coefficients referenced by the code
  long long n_groups = 0, n_fnodes = 0, n_dnodes = 0, fp64_ops = 0;
  int max_depth_f = 0, max_depth_d = 0;
};

int construct_flat(int n_int, int n_ext, int n_g, int n_eps, const int32_t* alpha, const int32_t* eps,
                   const uint8_t* ferm, const int32_t* sum_order, double prefactor, FlatTable& out);
void build_tree_plan(const FlatTable& ft, TreePlan& plan);

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
  uint32_t* tree_code = nullptr;
  double* tree_consts = nullptr;
  // dispersion
  int8_t* sym_alpha = nullptr;    // [n_eps][L]
  double* derivQ = nullptr;       // [AMI_MAX_DERIV+1][8] polynomials of the Fermi derivatives
  int64_t bytes = 0;
};

struct ami_table {
  ami::FlatTable flat;
  ami::TreePlan tree;
  ami_device_copy dev;
  int64_t fp64_ops_flat = 0;
};
