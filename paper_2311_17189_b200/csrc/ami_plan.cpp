// Evaluation plans derived from the flat term table (host, one-time).
#include <algorithm>
#include <map>

#include "ami_table.hpp"

namespace ami {

// FP64 instructions of the flat term loop per (sample, frequency, beta), real energies:
// (m-1) real multiplies + first real*complex (2) + 4 per further complex multiply + 2 adds.
long long flat_fp64_ops(const FlatTable& ft) {
  long long ops = 0;
  for (const FlatTerm& t : ft.terms) {
    const long long nf = (long long)t.f.size(), nd = (long long)t.d.size();
    ops += nf;                         // coef * f1 * ... * fm
    ops += nd ? 2 + 4 * (nd - 1) : 0;  // real x complex, then complex x complex
    ops += 2;                          // accumulate
  }
  return ops;
}

void build_tree_plan(const FlatTable& ft, TreePlan& plan) {
  (void)ft;
  plan = TreePlan();
}

}  // namespace ami
