// Per-table specialised evaluation kernels ("register plan").
//
// The table-driven kernels pay an index load, an address computation and a shared-memory load for
// every multiply, which bounds them by instruction issue and shared-memory bandwidth (128 B/clk/SM
// against 64 DFMA/clk/SM) at a fraction of the FP64 pipe (profiles/r01_baseline_flat_cfg3.md).
// Here the symbolic result of ONE diagram is written out as straight-line CUDA C++ -- every
// Fermi/Bose leaf, every denominator and every partial sum a named register, the term table turned
// into the Horner form of ami_table.hpp -- and compiled for sm_100a with NVRTC when the table is
// first evaluated.  The same generated body serves two kernels: ami_jit_eval (energies from
// memory, S2+S3) and ami_jit_fused (momenta from memory, S1+S2+S3 with the dispersion inline).
//
// The source text is produced by this file from the table; the arithmetic helpers it calls are
// the ones in ami_device.cuh, embedded as text at build time (generated/ami_embedded_src.h).
#include <cuda.h>
#include <cuda_runtime.h>
#include <dlfcn.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <sstream>
#include <string>
#include <vector>

#include "ami_jit.hpp"
#include "generated/ami_embedded_src.h"

namespace ami {

namespace {

// ---------------------------------------------------------------------------------------------
// source generation
// ---------------------------------------------------------------------------------------------
std::string dlit(double v) {
  char buf[48];
  snprintf(buf, sizeof buf, "%.17g", v);
  std::string s(buf);
  if (s.find_first_of(".eEn") == std::string::npos) s += ".0";
  return s;
}

// "+ e0 - e3 + 2.0 * e5": integer combination of named doubles, left to right
std::string combo(const std::vector<int>& c, const char* base, const std::string& suffix = "") {
  std::string s;
  for (size_t i = 0; i < c.size(); ++i) {
    if (!c[i]) continue;
    const int a = c[i] < 0 ? -c[i] : c[i];
    const std::string v = std::string(base) + std::to_string(i) + suffix;
    const std::string term = a == 1 ? v : dlit((double)a) + " * " + v;
    if (s.empty()) s = (c[i] < 0 ? "-" : "") + term;
    else s += (c[i] < 0 ? " - " : " + ") + term;
  }
  return s.empty() ? "0.0" : s;
}

// A list of statements that must stay in order; independent lists are interleaved round-robin
// before they are written out, so that the straight-line code offers the FP64 pipe several
// independent dependency chains at any point (ptxas keeps the source order it is given far more
// than it reorders across long chains).
typedef std::vector<std::string> Stmts;

struct Emitter {
  int tmp = 0;
  std::string fresh(const char* p) { return std::string(p) + std::to_string(tmp++); }
};

void interleave(std::vector<Stmts>& lists, size_t ways, std::ostringstream& o, const char* indent) {
  for (size_t base = 0; base < lists.size(); base += ways) {
    const size_t end = std::min(lists.size(), base + ways);
    size_t longest = 0;
    for (size_t i = base; i < end; ++i) longest = std::max(longest, lists[i].size());
    for (size_t k = 0; k < longest; ++k)
      for (size_t i = base; i < end; ++i)
        if (k < lists[i].size()) o << indent << lists[i][k] << "\n";
  }
}

// One S-node of the FT DAG (ami_table.hpp) as a chain of statements defining `S<id>`
void emit_snode(const HornerPlan& hp, int id, Emitter& E, Stmts& out) {
  const SNode& n = hp.snodes[id];
  std::string acc;
  for (size_t i = 0; i < n.items.size(); ++i) {
    const SItem& it = n.items[i];
    const bool last = i + 1 == n.items.size();
    const std::string v = last ? "S" + std::to_string(id) : E.fresh("s");
    const std::string leaf = "F" + std::to_string(it.leaf);
    if (it.child >= 0) {
      const std::string sc = "S" + std::to_string(it.child);
      if (acc.empty()) out.push_back("const double " + v + " = " + leaf + " * " + sc + ";");
      else out.push_back("const double " + v + " = fma(" + leaf + ", " + sc + ", " + acc + ");");
      acc = v;
      continue;
    }
    const bool plus = it.num == 1 && it.den == 1, minus = it.num == -1 && it.den == 1;
    const std::string coef = dlit((double)it.num / (double)it.den);
    if (acc.empty()) {
      if (plus && !last) { acc = leaf; continue; }
      if (minus && !last) { acc = "(-" + leaf + ")"; continue; }
      if (plus) out.push_back("const double " + v + " = " + leaf + ";");
      else if (minus) out.push_back("const double " + v + " = -" + leaf + ";");
      else out.push_back("const double " + v + " = " + coef + " * " + leaf + ";");
    } else if (plus) {
      out.push_back("const double " + v + " = " + acc + " + " + leaf + ";");
    } else if (minus) {
      out.push_back("const double " + v + " = " + acc + " - " + leaf + ";");
    } else {
      out.push_back("const double " + v + " = fma(" + coef + ", " + leaf + ", " + acc + ");");
    }
    acc = v;
  }
}

// Emits the S-nodes that groups [g0, g1) need and that have not been emitted yet, level by level
// (nodes of equal height are independent of one another), kWays chains side by side.
void emit_ft_chunk(const HornerPlan& hp, size_t g0, size_t g1, std::vector<char>& done, size_t ways, Emitter& E,
                   std::ostringstream& o, const char* indent) {
  std::vector<int> need, stack;
  for (size_t g = g0; g < g1; ++g)
    if (hp.groups[g].root >= 0) stack.push_back(hp.groups[g].root);
  while (!stack.empty()) {
    const int id = stack.back();
    stack.pop_back();
    if (done[id]) continue;
    done[id] = 1;
    need.push_back(id);
    for (const SItem& it : hp.snodes[id].items)
      if (it.child >= 0 && !done[it.child]) stack.push_back(it.child);
  }
  std::sort(need.begin(), need.end(), [&](int a, int b) {
    const int ha = hp.snodes[a].height, hb = hp.snodes[b].height;
    return ha != hb ? ha < hb : a < b;
  });
  for (size_t i = 0; i < need.size();) {
    size_t j = i;
    std::vector<Stmts> lists;
    while (j < need.size() && hp.snodes[need[j]].height == hp.snodes[need[i]].height) {
      lists.emplace_back();
      emit_snode(hp, need[j], E, lists.back());
      ++j;
    }
    interleave(lists, ways, o, indent);
    i = j;
  }
  for (size_t g = g0; g < g1; ++g) {
    const HGroup& hg = hp.groups[g];
    o << indent << "const double FT" << g << " = "
      << (hg.root >= 0 ? "S" + std::to_string(hg.root) : dlit((double)hg.num / (double)hg.den)) << ";\n";
  }
}

// ---- memory-backed variant for tables too large for registers ------------------------------------
// Long-lived values live in a per-thread column of a global scratch array (slot i at W(i)); the
// generated text names them through macros, so the emitters below and above are shared.  The FT DAG
// is written depth first: a sum is formed right before its first use, kept in its slot while other
// sums still need it (slots are recycled after the last use), and single-use sums stay in registers.
struct SlotPool {
  std::vector<int> free_list;
  int next = 0, peak = 0;
  int take() {
    if (!free_list.empty()) { const int s = free_list.back(); free_list.pop_back(); return s; }
    peak = std::max(peak, next + 1);
    return next++;
  }
  void give(int s) { free_list.push_back(s); }
};

struct DfsState {
  std::vector<int> uses_left;    // remaining uses of each S-node
  std::vector<int> slot;         // scratch slot of a computed shared node, -1 otherwise
  std::vector<char> done;
  SlotPool pool;
  int base = 0;                  // first scratch slot of the pool
};

// value of S-node `id` as an expression usable once; emits what is needed into `out`
std::string emit_snode_dfs(const HornerPlan& hp, int id, DfsState& st, Emitter& E, Stmts& out) {
  auto consume = [&](int n) {
    if (--st.uses_left[n] == 0 && st.slot[n] >= 0) { st.pool.give(st.slot[n]); st.slot[n] = -1; }
  };
  if (st.done[id]) {             // shared and already computed: read it back
    const std::string v = E.fresh("s");
    out.push_back("const double " + v + " = W(" + std::to_string(st.base + st.slot[id]) + ");");
    consume(id);
    return v;
  }
  const SNode& n = hp.snodes[id];
  std::string acc;
  for (size_t i = 0; i < n.items.size(); ++i) {
    const SItem& it = n.items[i];
    const std::string v = E.fresh("s");
    const std::string leaf = "F" + std::to_string(it.leaf);
    if (it.child >= 0) {
      const std::string sc = emit_snode_dfs(hp, it.child, st, E, out);
      if (acc.empty()) out.push_back("const double " + v + " = " + leaf + " * " + sc + ";");
      else out.push_back("const double " + v + " = fma(" + leaf + ", " + sc + ", " + acc + ");");
    } else {
      const std::string coef = dlit((double)it.num / (double)it.den);
      if (acc.empty()) out.push_back("const double " + v + " = " + coef + " * " + leaf + ";");
      else out.push_back("const double " + v + " = fma(" + coef + ", " + leaf + ", " + acc + ");");
    }
    acc = v;
  }
  st.done[id] = 1;
  if (st.uses_left[id] > 1) {    // needed again later: park it in a slot
    st.slot[id] = st.pool.take();
    out.push_back("W(" + std::to_string(st.base + st.slot[id]) + ") = " + acc + ";");
  }
  consume(id);
  return acc;
}

struct CV {            // a complex value held in named doubles; im empty = purely real
  std::string re, im;
  bool real() const { return im.empty(); }
};

// acc + Dinv[u] * s as new named doubles appended to `out` (acc may be absent)
CV emit_cmul_acc(const HornerPlan& hp, int u, const CV& s, const CV* accp, Emitter& E, Stmts& out) {
  const bool dreal = hp.d_is_real[u] != 0;
  const std::string dr = "Dr" + std::to_string(u), di = "Di" + std::to_string(u);
  CV r;
  r.re = E.fresh("r");
  {   // real part: dr*s.re - di*s.im (+ acc.re)
    std::string inner = accp ? accp->re : "";
    if (!dreal && !s.real()) {
      const std::string t = E.fresh("r");
      if (inner.empty()) out.push_back("const double " + t + " = -" + di + " * " + s.im + ";");
      else out.push_back("const double " + t + " = fma(-" + di + ", " + s.im + ", " + inner + ");");
      inner = t;
    }
    if (inner.empty()) out.push_back("const double " + r.re + " = " + dr + " * " + s.re + ";");
    else out.push_back("const double " + r.re + " = fma(" + dr + ", " + s.re + ", " + inner + ");");
  }
  {   // imaginary part: dr*s.im + di*s.re (+ acc.im)
    std::string inner = (accp && !accp->real()) ? accp->im : "";
    if (!s.real()) {
      const std::string t = E.fresh("r");
      if (inner.empty()) out.push_back("const double " + t + " = " + dr + " * " + s.im + ";");
      else out.push_back("const double " + t + " = fma(" + dr + ", " + s.im + ", " + inner + ");");
      inner = t;
    }
    if (!dreal) {
      const std::string t = E.fresh("r");
      if (inner.empty()) out.push_back("const double " + t + " = " + di + " * " + s.re + ";");
      else out.push_back("const double " + t + " = fma(" + di + ", " + s.re + ", " + inner + ");");
      inner = t;
    }
    r.im = inner;   // stays empty when the product and the running sum are both real
  }
  return r;
}

// Frequency-independent part of S_D(n): Q(n) = [FT_g if group g ends at n] + sum over kids c with a
// purely real denominator of Dr_c * Q(c).  Denominators are ordered complex first (ami_plan.cpp), so
// everything below a real denominator is real.  Returns the name of the value, "" if there is none.
std::string emit_q(const HornerPlan& hp, int n, Emitter& E, Stmts& out) {
  std::string acc;
  if (hp.dn[n].group >= 0) acc = "FT" + std::to_string(hp.dn[n].group);
  for (int c : hp.dn[n].kids) {
    if (!hp.d_is_real[hp.dn[c].leaf]) continue;
    const std::string qc = emit_q(hp, c, E, out);   // never empty: a trie leaf carries a group
    const std::string v = E.fresh("q"), dr = "Dr" + std::to_string(hp.dn[c].leaf);
    if (acc.empty()) out.push_back("const double " + v + " = " + dr + " * " + qc + ";");
    else out.push_back("const double " + v + " = fma(" + dr + ", " + qc + ", " + acc + ");");
    acc = v;
  }
  return acc;
}

// S_D(n) = Q(n) + sum over kids c with a complex denominator of Dinv_c * S_D(c)
CV emit_d_sum(const HornerPlan& hp, const std::vector<std::string>& qname, int n, Emitter& E, Stmts& out) {
  CV acc;
  bool have = false;
  if (!qname[n].empty()) { acc.re = qname[n]; have = true; }
  for (int c : hp.dn[n].kids) {
    if (hp.d_is_real[hp.dn[c].leaf]) continue;
    const CV s = emit_d_sum(hp, qname, c, E, out);
    acc = emit_cmul_acc(hp, hp.dn[c].leaf, s, have ? &acc : nullptr, E, out);
    have = true;
  }
  if (!have) acc.re = "0.0";
  return acc;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// The translation unit handed to NVRTC.
// ---------------------------------------------------------------------------------------------
std::string jit_generate_source(const FlatTable& ft, const HornerPlan& hp, int block_threads, bool scratch,
                                int* scratch_slots) {
  const int L = ft.n_int + ft.n_ext;
  size_t kWays = 16;          // independent chains kept side by side (measured: profiles/r01_batch_sweep.md)
  if (const char* env = getenv("AMI_JIT_WAYS")) {   // tuning knob (profiles/)
    const int w = atoi(env);
    if (w >= 1 && w <= 64) kWays = (size_t)w;
  }
  Emitter E;
  // The body of one sample is generated in four sections that are assembled twice below: once
  // nested beta { ... frequency { ... } } and once with the beta-only work of all temperatures
  // done first (section 1), so that the frequency-only work (section 2) is not repeated per beta.
  //   0: once per sample   1: per beta   2: per frequency   3: per (beta, frequency)
  std::ostringstream sec[4];
  int cur = 0;
#define o sec[cur]
  // every distinct integer combination of the energies, up to sign, once per sample
  std::vector<std::vector<int>> combos;
  auto combo_ref = [&](const std::vector<int>& c) -> std::string {
    std::vector<int> pos = c;
    int sign = 0;
    for (int v : c)
      if (v) { sign = v > 0 ? 1 : -1; break; }
    if (!sign) return "0.0";
    if (sign < 0)
      for (int& v : pos) v = -v;
    size_t j = 0;
    for (; j < combos.size(); ++j)
      if (combos[j] == pos) break;
    if (j == combos.size()) combos.push_back(pos);
    return std::string(sign < 0 ? "-E" : "E") + std::to_string(j);
  };
  for (const LeafD& l : ft.leafD) combo_ref(l.c);
  for (size_t j = 0; j < combos.size(); ++j) o << "  const double E" << j << " = " << combo(combos[j], "e") << ";\n";
  // reciprocals of the denominators, kWays at a time
  auto emit_d_leaves = [&](const std::vector<size_t>& ids, const std::string& ind) {
    if (!scratch)
      for (size_t u : ids) o << ind << "double Dr" << u << (hp.d_is_real[u] ? "" : ", Di" + std::to_string(u)) << ";\n";
    for (size_t i0 = 0; i0 < ids.size(); i0 += kWays) {
      const size_t n = std::min(kWays, ids.size() - i0);
      o << ind << "{\n";
      for (size_t j = 0; j < n; ++j) {
        const size_t u = ids[i0 + j];
        const LeafD& l = ft.leafD[u];
        const std::string en = combo_ref(l.c);
        if (hp.d_is_real[u]) {
          o << ind << "  const double re" << j << " = " << en << " + p.e_reg;\n";
        } else {
          std::string cond;
          for (int x = 0; x < ft.n_ext; ++x)
            if (l.a[x]) cond += (cond.empty() ? "" : " && ") + std::string("zz") + std::to_string(x);
          o << ind << "  const double re" << j << " = ((" << combo(l.a, "zr") << ") + " << en << ") + ((" << cond
            << ") ? p.e_reg : 0.0), im" << j << " = " << combo(l.a, "zi") << ";\n";
        }
      }
      o << ind << "  double d[" << n << "] = {";
      for (size_t j = 0; j < n; ++j) {
        if (hp.d_is_real[ids[i0 + j]]) o << (j ? ", " : "") << "re" << j;
        else o << (j ? ", " : "") << "fma(re" << j << ", re" << j << ", im" << j << " * im" << j << ")";
      }
      o << "};\n" << ind << "  fast_rcp_n<" << n << ">(d);\n";
      for (size_t j = 0; j < n; ++j) {
        const size_t u = ids[i0 + j];
        if (hp.d_is_real[u]) o << ind << "  Dr" << u << " = d[" << j << "];\n";
        else o << ind << "  Dr" << u << " = re" << j << " * d[" << j << "]; Di" << u << " = -im" << j << " * d[" << j << "];\n";
      }
      o << ind << "}\n";
    }
  };
  // denominators without an external frequency are purely real and the same for every beta and
  // frequency: once per sample, regulator always applied (P10(b))
  {
    std::vector<size_t> ids;
    for (size_t u = 0; u < ft.leafD.size(); ++u)
      if (hp.d_is_real[u]) ids.push_back(u);
    emit_d_leaves(ids, "  ");
  }
  cur = 1;
  // Fermi/Bose leaves (independent of the external frequency), kWays at a time
  // Leaves that differ only in the derivative order share one exponential and one reciprocal.
  const size_t UF = ft.leafF.size();
  std::vector<std::vector<size_t>> base;      // base -> leaves with the same (combination, sigma)
  for (size_t u = 0; u < UF; ++u) {
    size_t b = 0;
    for (; b < base.size(); ++b)
      if (ft.leafF[base[b][0]].c == ft.leafF[u].c && ft.leafF[base[b][0]].sigma == ft.leafF[u].sigma) break;
    if (b == base.size()) base.emplace_back();
    base[b].push_back(u);
  }
  const bool smem_f = scratch || jit_fermi_in_smem();
  if (!smem_f)
    for (size_t u = 0; u < UF; ++u) o << "    double F" << u << ";\n";
  // One exponential per ENERGY SYMBOL, e^{beta e_i} = 2^{n_i} m_i; the exponential of a leaf's
  // combination is assembled from them: integer exponents add, mantissas multiply, so nothing can
  // overflow and 17 FP64 instructions per leaf become one or two multiplies.
  std::vector<char> sym_used(ft.n_eps, 0);
  for (const auto& members : base)
    for (int i = 0; i < ft.n_eps; ++i)
      if (ft.leafF[members[0]].c[i]) sym_used[i] = 1;
  std::vector<int> syms;
  for (int i = 0; i < ft.n_eps; ++i)
    if (sym_used[i]) syms.push_back(i);
  for (int i : syms) o << "    int n" << i << "; double m" << i << ";\n";
  for (size_t i0 = 0; i0 < syms.size(); i0 += kWays) {
    const size_t n = std::min(kWays, syms.size() - i0);
    o << "    {\n      const double x[" << n << "] = {";
    for (size_t j = 0; j < n; ++j) o << (j ? ", " : "") << "beta * e" << syms[i0 + j];
    o << "};\n      int nn[" << n << "]; double mm[" << n << "];\n      exp_split_n<" << n << ">(x, nn, mm);\n";
    for (size_t j = 0; j < n; ++j)
      o << "      n" << syms[i0 + j] << " = nn[" << j << "]; m" << syms[i0 + j] << " = mm[" << j << "];\n";
    o << "    }\n";
  }
  // a leaf with x = beta (E [+ eta]) = ln(A/B): f_sigma = 1/(sigma A/B + 1) = B/(sigma A + B), with
  // A (B) the product over the symbols with positive (negative) coefficient; A carries e^{beta eta}
  // for sigma = -1 (P10(a)).  Exponents: A/B = 2^(Na - Nb) Ma/Mb, so d = fma(2^(Na-Nb), sigma Ma, Mb).
  auto product = [&](const std::vector<int>& c, int sign, std::string* mant, std::string* expo) {
    for (int i = 0; i < ft.n_eps; ++i) {
      const int a = c[i] * sign;
      for (int r = 0; r < a; ++r) {
        *mant += (mant->empty() ? "" : " * ") + std::string("m") + std::to_string(i);
        *expo += std::string(sign > 0 ? " + n" : " - n") + std::to_string(i);
      }
    }
  };
  for (size_t b0 = 0; b0 < base.size(); b0 += kWays) {
    const size_t n = std::min(kWays, base.size() - b0);
    o << "    {\n";
    for (size_t j = 0; j < n; ++j) {
      const LeafF& l = ft.leafF[base[b0 + j][0]];
      std::string ma, mb, ex;
      product(l.c, +1, &ma, &ex);
      product(l.c, -1, &mb, &ex);
      if (l.sigma < 0) ma += (ma.empty() ? "" : " * ") + std::string("p.ceta[b]");
      if (ma.empty()) ma = "1.0";
      o << "      const double s" << j << " = pow2_clamped(0" << ex << "), a" << j << " = " << ma << ", b" << j << " = "
        << (mb.empty() ? "1.0" : mb) << ";\n";
    }
    o << "      double d[" << n << "] = {";
    for (size_t j = 0; j < n; ++j)
      o << (j ? ", " : "") << "fma(s" << j << ", " << (ft.leafF[base[b0 + j][0]].sigma > 0 ? "" : "-") << "a" << j << ", b"
        << j << ")";
    o << "};\n      fast_rcp_n<" << n << ">(d);\n";
    for (size_t j = 0; j < n; ++j) {
      const std::vector<size_t>& members = base[b0 + j];
      const LeafF& l0 = ft.leafF[members[0]];
      bool has_b = false, need_g = false;
      for (int v : l0.c) has_b |= v < 0;
      for (size_t u : members) need_g |= ft.leafF[u].k > 0;
      const std::string f = has_b ? "(b" + std::to_string(j) + " * d[" + std::to_string(j) + "])" : "d[" + std::to_string(j) + "]";
      if (need_g)   // g = 1 - f = sigma A / (sigma A + B)  (P11)
        o << "      const double g" << j << " = " << (l0.sigma > 0 ? "" : "-") << "(s" << j << " * a" << j << ") * d[" << j
          << "];\n";
      for (size_t u : members) {
        const LeafF& l = ft.leafF[u];
        if (l.k == 0) {
          o << "      F" << u << " = " << f << ";\n";
          continue;
        }
        // f^{(k)} = beta^k f g Q_k(f)
        o << "      {\n        const double f = " << f << ";\n";
        const std::vector<double> q = deriv_poly(l.k);
        o << "        double q = " << dlit(q.back()) << ";\n";
        for (int i = (int)q.size() - 2; i >= 0; --i) o << "        q = fma(q, f, " << dlit(q[i]) << ");\n";
        o << "        double bk = beta;\n";
        for (int i = 1; i < l.k; ++i) o << "        bk *= beta;\n";
        o << "        F" << u << " = bk * f * g" << j << " * q;\n      }\n";
      }
    }
    o << "    }\n";
  }
  // FT sums of every group (per beta): a DAG shared by all groups, emitted eight groups at a time
  // scratch layout: [Dr/Di of every denominator][FT of every group][Q of every R-trie node][pool of shared sums]
  std::vector<int> slot_dr(ft.leafD.size(), -1), slot_di(ft.leafD.size(), -1), slot_ft(hp.groups.size(), -1);
  int n_slots = 0;
  for (size_t u = 0; u < ft.leafD.size(); ++u) {
    slot_dr[u] = n_slots++;
    if (!hp.d_is_real[u]) slot_di[u] = n_slots++;
  }
  for (size_t g = 0; g < hp.groups.size(); ++g) slot_ft[g] = n_slots++;
  const int slot_q0 = n_slots;
  n_slots += (int)hp.dn.size();
  DfsState dfs;
  if (!scratch) {
    std::vector<char> done(hp.snodes.size(), 0);
    for (size_t g0 = 0; g0 < hp.groups.size(); g0 += 8)
      emit_ft_chunk(hp, g0, std::min(hp.groups.size(), g0 + 8), done, kWays, E, o, "    ");
  } else {
    dfs.uses_left.assign(hp.snodes.size(), 0);
    dfs.slot.assign(hp.snodes.size(), -1);
    dfs.done.assign(hp.snodes.size(), 0);
    dfs.base = n_slots;
    for (const SNode& n : hp.snodes)
      for (const SItem& it : n.items)
        if (it.child >= 0) ++dfs.uses_left[it.child];
    for (const HGroup& g : hp.groups)
      if (g.root >= 0) ++dfs.uses_left[g.root];
    for (size_t g = 0; g < hp.groups.size(); ++g) {
      const HGroup& hg = hp.groups[g];
      Stmts lst;
      const std::string v = hg.root >= 0 ? emit_snode_dfs(hp, hg.root, dfs, E, lst) : dlit((double)hg.num / (double)hg.den);
      o << "    {\n";
      for (const std::string& st : lst) o << "      " << st << "\n";
      o << "      FT" << g << " = " << v << ";\n    }\n";
    }
    n_slots += dfs.pool.peak;
  }
  if (scratch_slots) *scratch_slots = scratch ? n_slots : 0;
  // frequency-independent parts of the R sums (products under purely real denominators), per beta
  std::vector<std::string> qname(hp.dn.size());
  {
    std::vector<Stmts> lists;
    for (size_t n = 0; n < hp.dn.size(); ++n) {
      if (n != 0 && hp.d_is_real[hp.dn[n].leaf]) continue;
      lists.emplace_back();
      qname[n] = emit_q(hp, (int)n, E, lists.back());
      if (scratch && !qname[n].empty() && qname[n][0] == 'q') {     // keep it in memory until the R part reads it
        const std::string w = "W(" + std::to_string(slot_q0 + (int)n) + ")";
        lists.back().push_back(w + " = " + qname[n] + ";");
        qname[n] = w;
      }
    }
    interleave(lists, kWays, o, "    ");
  }
  // frequencies
  cur = 2;
  for (int x = 0; x < ft.n_ext; ++x) {
    o << "      const double zr" << x << " = p.z[2 * (f * " << ft.n_ext << " + " << x << ")], zi" << x
      << " = p.z[2 * (f * " << ft.n_ext << " + " << x << ") + 1];\n";
    o << "      const bool zz" << x << " = (zr" << x << " == 0.0 && zi" << x << " == 0.0);\n";
  }
  // reciprocals of the denominators that carry an external frequency (P10(b) decides at run time
  // whether the regulator applies)
  {
    std::vector<size_t> ids;
    for (size_t u = 0; u < ft.leafD.size(); ++u)
      if (!hp.d_is_real[u]) ids.push_back(u);
    emit_d_leaves(ids, "      ");
  }
  // R part: the subtrees under the root side by side, then the root's own sum
  cur = 3;
  {
    std::vector<int> kids;
    for (int c : hp.dn[0].kids)
      if (!hp.d_is_real[hp.dn[c].leaf]) kids.push_back(c);
    std::vector<Stmts> lists(kids.size());
    std::vector<CV> sub(kids.size());
    for (size_t i = 0; i < kids.size(); ++i) sub[i] = emit_d_sum(hp, qname, kids[i], E, lists[i]);
    interleave(lists, kWays, o, "      ");
    Stmts tail;
    CV acc;
    bool have = false;
    if (!qname[0].empty()) { acc.re = qname[0]; have = true; }
    for (size_t i = 0; i < kids.size(); ++i) {
      acc = emit_cmul_acc(hp, hp.dn[kids[i]].leaf, sub[i], have ? &acc : nullptr, E, tail);
      have = true;
    }
    if (!have) acc.re = "0.0";
    for (const std::string& st : tail) o << "      " << st << "\n";
    o << "      const long long row = (long long)(p.b0 + b) * p.n_f_total + (p.f0 + f);\n";
    o << "      const double2 val = make_double2(p.prefactor * (" << acc.re << "), "
      << (acc.real() ? std::string("0.0") : "p.prefactor * (" + acc.im + ")") << ");\n";
    o << "      if (!AMI_TALLY || p.out) AMI_STORE(reinterpret_cast<double2*>(p.out) + row * p.out_row_stride + s, val);\n";
    o << "      if (AMI_TALLY) ami_tally(reinterpret_cast<double4*>(p.tally) + row * p.tally_stride + (s >> 5), val);\n";
  }
#undef o
  std::ostringstream o;
  o << kAmiParamsSrc << "\n" << kAmiDeviceSrc << "\n";
  int tiles = scratch ? 1 : jit_tiles_per_cta();
  o << "using namespace amidev;\n#define AMI_NT " << block_threads << "\n#define AMI_U " << tiles << "\n#define AMI_PF " << jit_prefetch_ctas() << "\n#define AMI_MINB " << (scratch ? 1 : jit_min_blocks(block_threads)) << "\n"
    << (jit_store_mode() == 1 ? "#define AMI_STORE(p, v) __stcs(p, v)\n"
        : jit_store_mode() == 2 ? "#define AMI_STORE(p, v) __stwt(p, v)\n" : "#define AMI_STORE(p, v) (*(p) = (v))\n");
  // Fused tally (S4, Monte-Carlo sums of PAPER.md:291): the warp adds its samples' (re, im, re^2, im^2) in a fixed
  // order and lane 0 stores one partial per (row, warp).  The lanes of a ragged last warp are the low ones.
  o << "__device__ __forceinline__ void ami_tally(double4* dst, const double2 v) {\n"
       "  const unsigned mask = __activemask();\n"
       "  const int lane = threadIdx.x & 31, cnt = __popc(mask);\n"
       "  double a = v.x, b = v.y, c = v.x * v.x, d = v.y * v.y;\n"
       "#pragma unroll\n"
       "  for (int off = 16; off > 0; off >>= 1) {\n"
       "    const double a2 = __shfl_down_sync(mask, a, off), b2 = __shfl_down_sync(mask, b, off);\n"
       "    const double c2 = __shfl_down_sync(mask, c, off), d2 = __shfl_down_sync(mask, d, off);\n"
       "    if (lane + off < cnt) { a += a2; b += b2; c += c2; d += d2; }\n"
       "  }\n"
       "  if (lane == 0) *dst = make_double4(a, b, c, d);\n"
       "}\n";
  std::string sig = "(const AmiBatch& p, const long long s";
  for (int i = 0; i < ft.n_eps; ++i) sig += ", const double e" + std::to_string(i);
  if (smem_f && !scratch) {
    // Fermi/Bose leaves in shared memory as [leaf][thread] (conflict-free), everything else in registers
    o << "extern __shared__ double sF[];\n";
    for (size_t u = 0; u < ft.leafF.size(); ++u) o << "#define F" << u << " sF[" << u << " * AMI_NT + threadIdx.x]\n";
  }
  if (scratch) {
    sig += ", double* __restrict__ w, const long long ws";
    // volatile: every scratch access happens where it is written.  Without it the compiler hoists
    // thousands of loads to the top of the straight-line body and then spills them again.
    o << "extern __shared__ double sF[];\n#define W(i) ((volatile double*)w)[(long long)(i) * ws]\n";
    for (size_t u = 0; u < ft.leafF.size(); ++u) o << "#define F" << u << " sF[" << u << " * AMI_NT + threadIdx.x]\n";
    for (size_t u = 0; u < ft.leafD.size(); ++u) {
      o << "#define Dr" << u << " W(" << slot_dr[u] << ")\n";
      if (slot_di[u] >= 0) o << "#define Di" << u << " W(" << slot_di[u] << ")\n";
    }
    for (size_t g = 0; g < hp.groups.size(); ++g) o << "#define FT" << g << " W(" << slot_ft[g] << ")\n";
  }
  sig += ") {\n";
  // ---- body for one temperature per launch: beta { frequency { } } ----------------------------
  o << "template <bool AMI_TALLY> __device__ __forceinline__ void ami_body" << sig << sec[0].str()
    << "#pragma unroll 1\n  for (int b = 0; b < p.n_b; ++b) {\n    const double beta = p.beta[b];\n" << sec[1].str()
    << "#pragma unroll 1\n    for (int f = 0; f < p.n_f; ++f) {\n" << sec[2].str() << sec[3].str() << "    }\n  }\n}\n\n";
  // ---- body for several temperatures: the per-beta values the R part needs are kept in a small
  // per-thread array, then frequency { reciprocals once; beta { R part } } --------------------------
  std::vector<std::string> keep;
  if (!scratch)
  for (const std::string& q : qname)
    if (!q.empty() && std::find(keep.begin(), keep.end(), q) == keep.end()) keep.push_back(q);
  if (!scratch) {
  o << "template <bool AMI_TALLY> __device__ __forceinline__ void ami_body_mb" << sig << sec[0].str();
  o << "  double kept[AMI_K_MAX_BETA][" << std::max<size_t>(keep.size(), 1) << "];\n";
  o << "#pragma unroll 1\n  for (int b = 0; b < p.n_b; ++b) {\n    const double beta = p.beta[b];\n" << sec[1].str();
  for (size_t i = 0; i < keep.size(); ++i) o << "    kept[b][" << i << "] = " << keep[i] << ";\n";
  o << "  }\n#pragma unroll 1\n  for (int f = 0; f < p.n_f; ++f) {\n" << sec[2].str()
    << "#pragma unroll 1\n    for (int b = 0; b < p.n_b; ++b) {\n";
  for (size_t i = 0; i < keep.size(); ++i) o << "      const double " << keep[i] << " = kept[b][" << i << "];\n";
  o << sec[3].str() << "    }\n  }\n}\n\n";
  }
  // ---- kernel 1: energies from memory ---------------------------------------------------------
  o << "extern \"C\" __global__ void __launch_bounds__(AMI_NT, AMI_MINB) ami_jit_eval(const __grid_constant__ AmiBatch p) {\n"
       "  asm volatile(\"griddepcontrol.launch_dependents;\");\n"
       "  asm volatile(\"griddepcontrol.wait;\" ::: \"memory\");\n"
       "  const long long stride = (long long)gridDim.x * AMI_NT;\n"
       "#pragma unroll 1\n"
       "  for (long long s = blockIdx.x * (long long)AMI_NT + threadIdx.x; s < p.n; s += stride) {\n";
  for (int i = 0; i < ft.n_eps; ++i) o << "  const double e" << i << " = p.e[" << i << " * p.e_stride + s];\n";
  std::string call_args = "(p, s";
  for (int i = 0; i < ft.n_eps; ++i) call_args += ", e" + std::to_string(i);
  call_args += scratch ? ", p.scratch + s, p.scratch_stride);\n" : ");\n";
  // @T@ = <false> / <true>: without / with the fused tally (a compile-time switch: the reductions cost the kernels
  // that do not tally nothing); @K2@ = name of the fused kernel
  const std::string call = scratch ? "  ami_body@T@" + call_args
                                   : "  if (p.n_b == 1) ami_body@T@" + call_args + "  else ami_body_mb@T@" + call_args;
  o << call << "  }\n}\n\n";
  const size_t k2_begin = o.str().size();
  // ---- kernel 2: momenta from memory, dispersion inline (Eqs. 8-18) ----------
  o << "extern \"C\" __global__ void __launch_bounds__(AMI_NT, AMI_MINB) @K2@(const __grid_constant__ AmiBatch p) {\n"
       "  asm volatile(\"griddepcontrol.launch_dependents;\");\n"
       "  asm volatile(\"griddepcontrol.wait;\" ::: \"memory\");\n"
       "  // A CTA walks AMI_U consecutive tiles of AMI_NT samples; the momenta of the next tile are loaded into\n"
       "  // registers before the current one is evaluated, so only the first load of a CTA is exposed.\n"
       "  const long long base = blockIdx.x * (long long)(AMI_NT * AMI_U) + threadIdx.x;\n"
       "#if AMI_PF > 0\n"
       "  // The CTA that will take this one's place on the SM (AMI_PF CTAs further on) finds its momenta in L2:\n"
       "  // with a few warps per SM the DRAM latency of the first loads is otherwise exposed once per CTA.\n"
       "  {\n    const long long pb = base + (long long)AMI_PF * (AMI_NT * AMI_U);\n"
       "    if (pb < p.n && !p.gen) {\n      const double* kp = p.k + pb * p.k_stride_sample;\n"
       "      if (p.k_stride_comp == 1) {\n";
  for (int c = 0; c < 2 * ft.n_int; c += 4) o << "        asm volatile(\"prefetch.global.L2 [%0];\" ::\"l\"(kp + " << c << "));\n";
  o << "      } else {\n";
  for (int c = 0; c < 2 * ft.n_int; ++c)
    o << "        asm volatile(\"prefetch.global.L2 [%0];\" ::\"l\"(kp + " << c << " * p.k_stride_comp));\n";
  o << "      }\n    }\n  }\n#endif\n";
  for (int c = 0; c < 2 * ft.n_int; ++c) o << "  double nk" << c << " = 0.0;\n";
  // momenta of sample `at`: from memory, or drawn in place by the counter-based generator (S4 with a seed:
  // the momenta never exist in memory)
  auto emit_momenta = [&](const std::string& at, const std::string& ind) {
    // counter of component c = sample * 2m + c; the generator's state is seed + GOLDEN (counter + 1), so one 64-bit
    // multiply per sample and an addition per component (arithmetic modulo 2^64: same bits as momentum_of)
    o << ind << "if (p.gen) {\n" << ind << "  const unsigned long long z0 = p.seed + 0x9E3779B97F4A7C15ull * ((unsigned long long)"
      << "(p.first_sample + (" << at << ")) * " << 2 * ft.n_int << "ull + 1ull);\n";
    for (int c = 0; c < 2 * ft.n_int; ++c) {
      char lit[32];
      snprintf(lit, sizeof lit, "0x%016llXull", (unsigned long long)(0x9E3779B97F4A7C15ull * (unsigned long long)c));
      o << ind << "  nk" << c << " = momentum_from_state(z0 + " << lit << ");\n";
    }
    o << ind << "} else {\n" << ind << "  const double* kn = p.k + (" << at << ") * p.k_stride_sample;\n";
    for (int c = 0; c < 2 * ft.n_int; ++c) o << ind << "  nk" << c << " = kn[" << c << " * p.k_stride_comp];\n";
    o << ind << "}\n";
  };
  o << "  if (base < p.n) {\n";
  emit_momenta("base", "    ");
  o << "  }\n#pragma unroll 1\n  for (int u = 0; u < AMI_U; ++u) {\n"
       "  const long long s = base + (long long)u * AMI_NT;\n  if (s >= p.n) break;\n";
  for (int l = 0; l < ft.n_int; ++l)
    o << "  const double kx" << l << " = nk" << 2 * l << ", ky" << l << " = nk" << 2 * l + 1 << ";\n";
  o << "  if (u + 1 < AMI_U && s + AMI_NT < p.n) {\n";
  emit_momenta("s + AMI_NT", "    ");
  o << "  }\n";
  for (int x = 0; x < ft.n_ext; ++x)
    o << "  const double kx" << ft.n_int + x << " = p.q[" << 2 * x << "], ky" << ft.n_int + x << " = p.q[" << 2 * x + 1
      << "];\n";
  for (int i = 0; i < ft.n_eps; ++i) o << "  double e" << i << ";\n";
  const int sym_batch = std::max(1, (int)kWays / 2);   // kWays cosines side by side
  for (int i0 = 0; i0 < ft.n_eps; i0 += sym_batch) {
    const int n = std::min(sym_batch, ft.n_eps - i0);
    o << "  {\n    double c[" << 2 * n << "] = {";
    for (int j = 0; j < n; ++j) {
      std::vector<int> a(ft.sym_alpha.begin() + (size_t)(i0 + j) * L, ft.sym_alpha.begin() + (size_t)(i0 + j + 1) * L);
      o << (j ? ", " : "") << combo(a, "kx") << ", " << combo(a, "ky");
    }
    o << "};\n    cos_bounded_n<" << 2 * n << ">(c);\n";
    for (int j = 0; j < n; ++j)
      o << "    e" << i0 + j << " = fma(2.0 * p.t, c[" << 2 * j << "] + c[" << 2 * j + 1 << "], p.mu);\n";
    o << "  }\n";
  }
  o << "  if (p.e_out) {\n";
  for (int i = 0; i < ft.n_eps; ++i) o << "    p.e_out[" << i << " * p.e_stride + s] = e" << i << ";\n";
  o << "  }\n" << call << "  }\n}\n";
  auto subst = [](std::string t, const std::string& targ, const std::string& k2) {
    for (const auto& kv : {std::make_pair(std::string("@T@"), targ), std::make_pair(std::string("@K2@"), k2)})
      for (size_t at = 0; (at = t.find(kv.first, at)) != std::string::npos; at += kv.second.size())
        t.replace(at, kv.first.size(), kv.second);
    return t;
  };
  const std::string all = o.str();
  std::string src = subst(all, "<false>", "ami_jit_fused");
  src += "\n" + subst(all.substr(k2_begin), "<true>", "ami_jit_fused_tally");
  return src;
}

int jit_tiles_per_cta() {
  static const int u = [] {
    const char* e = getenv("AMI_JIT_U");
    const int v = e ? atoi(e) : 0;
    return (v >= 1 && v <= 16) ? v : kJitTilesPerCtaDefault;
  }();
  return u;
}

int jit_prefetch_ctas() {
  static const int pf = [] {
    const char* e = getenv("AMI_JIT_PF");
    const int v = e ? atoi(e) : kJitPrefetchCtasDefault;
    return (v >= 0 && v <= 1 << 20) ? v : kJitPrefetchCtasDefault;
  }();
  return pf;
}

int jit_min_blocks(int block_threads) {
  // __launch_bounds__(AMI_NT, AMI_MINB): the register cap that lets AMI_MINB CTAs share an SM.  (--maxrregcount is
  // ignored for kernels that carry launch bounds, so this is the knob that changes occupancy.)  Default: 12 warps
  // per SM = at most 168 registers per thread.  Measured on B200 (profiles/r01_batch_sweep.md): the order-6 kernel
  // wants 248 registers and runs at 0.77 of the DFMA peak with 8 warps per SM; capped at 168 it spills 80 bytes
  // and reaches 0.87; at 128 registers the spills cost more than the occupancy gives.
  static const int env = [] {
    const char* e = getenv("AMI_JIT_MINB");
    const int m = e ? atoi(e) : 0;
    return (m >= 1 && m <= 32) ? m : 0;
  }();
  return env ? env : std::max(1, kJitWarpsPerSmTarget * 32 / block_threads);
}

bool jit_fermi_in_smem() {
  static const bool v = [] { const char* e = getenv("AMI_JIT_SMEM_F"); return e && e[0] == '1'; }();
  return v;
}

int jit_store_mode() {
  static const int m = [] {
    const char* e = getenv("AMI_JIT_STORE");
    const int v = e ? atoi(e) : kJitStoreModeDefault;
    return (v >= 0 && v <= 2) ? v : kJitStoreModeDefault;
  }();
  return m;
}

int jit_block_threads() {
  static const int nt = [] {
    const char* e = getenv("AMI_JIT_NT");
    const int v = e ? atoi(e) : 0;
    return (v == 32 || v == 64 || v == 128 || v == 256) ? v : kJitBlockThreadsDefault;
  }();
  return nt;
}

int jit_mode(const FlatTable& ft, const HornerPlan& hp) {
  if (const char* off = getenv("AMI_DISABLE_JIT"))
    if (off[0] == '1') return kJitNone;
  long long leaf_doubles = (long long)ft.leafF.size();
  for (size_t u = 0; u < ft.leafD.size(); ++u) leaf_doubles += hp.d_is_real[u] ? 1 : 2;
  long long max_leaf = 160, max_edges = 24000, max_scratch_edges = 400000;
  if (const char* env = getenv("AMI_JIT_MAX_LEAF_DOUBLES")) max_leaf = atoll(env);   // tuning knobs
  if (const char* env = getenv("AMI_JIT_MAX_EDGES")) max_edges = atoll(env);
  if (const char* env = getenv("AMI_JIT_MAX_SCRATCH_EDGES")) max_scratch_edges = atoll(env);
  const long long edges = hp.n_fnodes + 4 * hp.n_dnodes;
  if (leaf_doubles <= max_leaf && edges <= max_edges) return kJitRegister;
  // memory-backed variant: Fermi/Bose leaves in shared memory (64 threads per CTA), the rest in scratch.
  // Opt-in (AMI_JIT_SCRATCH=1): NVRTC needs minutes for bodies of this size (order 7: 90 s, order 8: 270 s).
  const char* opt_in = getenv("AMI_JIT_SCRATCH");
  if (opt_in && opt_in[0] == '1' && (long long)ft.leafF.size() * 64 * 8 <= 200 * 1024 && edges <= max_scratch_edges)
    return kJitScratch;
  return kJitNone;
}

bool jit_eligible(const FlatTable& ft, const HornerPlan& hp) { return jit_mode(ft, hp) != kJitNone; }

// ---------------------------------------------------------------------------------------------
// NVRTC, loaded on demand (the library itself does not link against it)
// ---------------------------------------------------------------------------------------------
namespace {

struct Nvrtc {
  void* h = nullptr;
  int (*CreateProgram)(void**, const char*, const char*, int, const char* const*, const char* const*) = nullptr;
  int (*CompileProgram)(void*, int, const char* const*) = nullptr;
  int (*GetProgramLogSize)(void*, size_t*) = nullptr;
  int (*GetProgramLog)(void*, char*) = nullptr;
  int (*GetCUBINSize)(void*, size_t*) = nullptr;
  int (*GetCUBIN)(void*, char*) = nullptr;
  int (*DestroyProgram)(void**) = nullptr;
  const char* (*GetErrorString)(int) = nullptr;
  bool ok = false;
};

Nvrtc& nvrtc() {
  static Nvrtc n;
  static std::once_flag once;
  std::call_once(once, [] {
    const char* names[] = {"/usr/local/cuda/lib64/libnvrtc.so.12", "libnvrtc.so.12", "libnvrtc.so",
                           "/usr/local/cuda/lib64/libnvrtc.so"};
    if (const char* env = getenv("AMI_NVRTC_PATH")) n.h = dlopen(env, RTLD_NOW | RTLD_LOCAL);
    for (const char* nm : names)
      if (!n.h) n.h = dlopen(nm, RTLD_NOW | RTLD_LOCAL);
    if (!n.h) return;
#define AMI_SYM(f) *(void**)(&n.f) = dlsym(n.h, "nvrtc" #f)
    AMI_SYM(CreateProgram); AMI_SYM(CompileProgram); AMI_SYM(GetProgramLogSize); AMI_SYM(GetProgramLog);
    AMI_SYM(GetCUBINSize); AMI_SYM(GetCUBIN); AMI_SYM(DestroyProgram); AMI_SYM(GetErrorString);
#undef AMI_SYM
    n.ok = n.CreateProgram && n.CompileProgram && n.GetProgramLogSize && n.GetProgramLog && n.GetCUBINSize &&
           n.GetCUBIN && n.DestroyProgram;
  });
  return n;
}

}  // namespace

int jit_compile(const std::string& src, std::vector<char>& cubin, std::string& log) {
  Nvrtc& n = nvrtc();
  if (!n.ok) { log = "NVRTC library not found (set AMI_NVRTC_PATH)"; return AMI_EUNSUPPORTED; }
  void* prog = nullptr;
  if (n.CreateProgram(&prog, src.c_str(), "ami_jit.cu", 0, nullptr, nullptr) != 0) {
    log = "nvrtcCreateProgram failed";
    return AMI_EINVAL;
  }
  std::vector<const char*> opts = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo", "--ptxas-options=-v",
                                   "-default-device"};
  std::string popt;
  if (const char* env = getenv("AMI_JIT_PTXAS_OPT")) {   // tuning knob: e.g. -O1
    popt = std::string("--ptxas-options=") + env;
    opts.push_back(popt.c_str());
  }
  // (no --maxrregcount: it is ignored for kernels with __launch_bounds__; the register cap is AMI_MINB)
  const int rc = n.CompileProgram(prog, (int)opts.size(), opts.data());
  size_t ls = 0;
  n.GetProgramLogSize(prog, &ls);
  if (ls > 1) {
    log.resize(ls);
    n.GetProgramLog(prog, &log[0]);
  }
  if (rc != 0) {
    log = std::string("NVRTC: ") + (n.GetErrorString ? n.GetErrorString(rc) : "error") + "\n" + log;
    n.DestroyProgram(&prog);
    return AMI_EINVAL;
  }
  size_t cs = 0;
  n.GetCUBINSize(prog, &cs);
  cubin.resize(cs);
  n.GetCUBIN(prog, cubin.data());
  n.DestroyProgram(&prog);
  return cs ? AMI_OK : AMI_EINVAL;
}

// ---------------------------------------------------------------------------------------------
// module loading and launch through driver entry points obtained from the runtime (the library
// does not link against libcuda, so that it loads on a machine without a driver)
// ---------------------------------------------------------------------------------------------
struct JitState {
  std::mutex mu;
  bool tried = false;
  int status = AMI_EUNSUPPORTED;
  std::string log;
  CUmodule mod = nullptr;
  CUfunction fn_eval = nullptr, fn_fused = nullptr, fn_fused_tally = nullptr;
  int mode = kJitNone;
  int block = 0;            // threads per CTA the kernels were generated for
  int tiles = 1;            // tiles of `block` samples one CTA of the fused kernel walks
  int scratch_slots = 0;    // doubles of global scratch per sample (memory-backed variant)
  unsigned smem_bytes = 0;  // dynamic shared memory per CTA (memory-backed variant)
};

namespace {

struct Driver {
  CUresult (*ModuleLoadData)(CUmodule*, const void*) = nullptr;
  CUresult (*ModuleGetFunction)(CUfunction*, CUmodule, const char*) = nullptr;
  CUresult (*ModuleUnload)(CUmodule) = nullptr;
  CUresult (*LaunchKernel)(CUfunction, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, CUstream,
                           void**, void**) = nullptr;
  CUresult (*GetErrorString)(CUresult, const char**) = nullptr;
  CUresult (*LaunchKernelEx)(const CUlaunchConfig*, CUfunction, void**, void**) = nullptr;   // optional
  CUresult (*FuncSetAttribute)(CUfunction, CUfunction_attribute, int) = nullptr;
  bool ok = false;
};

Driver& driver() {
  static Driver d;
  static std::once_flag once;
  std::call_once(once, [] {
    auto get = [](const char* name, void** fn) {
      cudaDriverEntryPointQueryResult st;
      return cudaGetDriverEntryPoint(name, fn, cudaEnableDefault, &st) == cudaSuccess &&
             st == cudaDriverEntryPointSuccess && *fn;
    };
    d.ok = get("cuModuleLoadData", (void**)&d.ModuleLoadData) &&
           get("cuModuleGetFunction", (void**)&d.ModuleGetFunction) &&
           get("cuModuleUnload", (void**)&d.ModuleUnload) && get("cuLaunchKernel", (void**)&d.LaunchKernel) &&
           get("cuGetErrorString", (void**)&d.GetErrorString);
    get("cuLaunchKernelEx", (void**)&d.LaunchKernelEx);
    d.ok = d.ok && get("cuFuncSetAttribute", (void**)&d.FuncSetAttribute);
  });
  return d;
}

std::mutex g_state_mu;   // guards creation of tab->jit

}  // namespace

int jit_prepare(ami_table* tab, std::string& err) {
  {
    std::lock_guard<std::mutex> lk(g_state_mu);
    if (!tab->jit) tab->jit = new JitState;
  }
  JitState& js = *tab->jit;
  std::lock_guard<std::mutex> lk(js.mu);
  if (js.tried) { err = js.log; return js.status; }
  js.tried = true;
  if (tab->dev.device < 0) { js.log = "table has no device copy"; js.status = AMI_ECUDA; err = js.log; return js.status; }
  if (!jit_eligible(tab->flat, tab->horner)) {
    js.log = "table too large for the register plan";
    js.status = AMI_EUNSUPPORTED;
    err = js.log;
    return js.status;
  }
  std::vector<char> cubin;
  js.mode = jit_mode(tab->flat, tab->horner);
  js.block = js.mode == kJitScratch ? 64 : jit_block_threads();
  js.tiles = js.mode == kJitScratch ? 1 : jit_tiles_per_cta();
  const std::string src = jit_generate_source(tab->flat, tab->horner, js.block, js.mode == kJitScratch, &js.scratch_slots);
  js.smem_bytes = (js.mode == kJitScratch || jit_fermi_in_smem())
                      ? (unsigned)(tab->flat.leafF.size() * js.block * sizeof(double)) : 0u;
  js.status = jit_compile(src, cubin, js.log);
  if (js.status != AMI_OK) { err = js.log; return js.status; }
  Driver& d = driver();
  if (!d.ok) { js.log = "CUDA driver entry points unavailable"; js.status = AMI_ECUDA; err = js.log; return js.status; }
  cudaSetDevice(tab->dev.device);
  cudaFree(nullptr);   // makes the primary context current
  CUresult rc = d.ModuleLoadData(&js.mod, cubin.data());
  if (rc == CUDA_SUCCESS) rc = d.ModuleGetFunction(&js.fn_eval, js.mod, "ami_jit_eval");
  if (rc == CUDA_SUCCESS) rc = d.ModuleGetFunction(&js.fn_fused, js.mod, "ami_jit_fused");
  if (rc == CUDA_SUCCESS) rc = d.ModuleGetFunction(&js.fn_fused_tally, js.mod, "ami_jit_fused_tally");
  if (rc == CUDA_SUCCESS && js.fn_fused_tally && js.smem_bytes > 48 * 1024)
    rc = d.FuncSetAttribute(js.fn_fused_tally, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, (int)js.smem_bytes);
  if (rc == CUDA_SUCCESS && js.smem_bytes > 48 * 1024) {
    rc = d.FuncSetAttribute(js.fn_eval, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, (int)js.smem_bytes);
    if (rc == CUDA_SUCCESS) rc = d.FuncSetAttribute(js.fn_fused, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, (int)js.smem_bytes);
  }
  if (rc != CUDA_SUCCESS) {
    const char* msg = nullptr;
    d.GetErrorString(rc, &msg);
    js.log = std::string("loading the specialised kernels failed: ") + (msg ? msg : "?");
    js.status = AMI_ECUDA;
    err = js.log;
    return js.status;
  }
  js.status = AMI_OK;
  return AMI_OK;
}

namespace {

CUresult launch_one(const JitState* js, bool fused, AmiBatch& batch, cudaStream_t st) {
  void* args[] = {&batch};
  // One CTA per `block` samples: the hardware CTA scheduler balances the SMs better than a
  // persistent grid with a static stride does (measured: persistent + L2 prefetch of the next sample
  // was 12 % slower on cfg3 and 5 % slower on cfg4, profiles/r01_register_plan.md).  The kernels keep
  // their grid-stride loop, so any grid size is correct.
  const unsigned block = (unsigned)js->block;
  const long long per_cta = (long long)block * (fused ? js->tiles : 1);   // the unfused kernel strides over the grid
  const unsigned grid = (unsigned)((batch.n + per_cta - 1) / per_cta);
  // Programmatic dependent launch: the kernels begin with griddepcontrol.launch_dependents + .wait, so
  // the NEXT specialised kernel in the stream may be scheduled while this one drains and starts the
  // moment it has completed (stream order is kept: nothing is read or written before the wait).
  static const bool pdl = [] { const char* e = getenv("AMI_JIT_PDL"); return !(e && e[0] == '0'); }();
  CUfunction fn = fused ? (batch.tally ? js->fn_fused_tally : js->fn_fused) : js->fn_eval;
  if (!fn) return CUDA_ERROR_INVALID_VALUE;
  if (pdl && driver().LaunchKernelEx) {
    CUlaunchAttribute attr;
    memset(&attr, 0, sizeof attr);
    attr.id = CU_LAUNCH_ATTRIBUTE_PROGRAMMATIC_STREAM_SERIALIZATION;
    attr.value.programmaticStreamSerializationAllowed = 1;
    CUlaunchConfig cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDimX = grid; cfg.gridDimY = 1; cfg.gridDimZ = 1;
    cfg.blockDimX = block; cfg.blockDimY = 1; cfg.blockDimZ = 1;
    cfg.sharedMemBytes = js->smem_bytes; cfg.hStream = (CUstream)st; cfg.attrs = &attr; cfg.numAttrs = 1;
    return driver().LaunchKernelEx(&cfg, fn, args, nullptr);
  }
  return driver().LaunchKernel(fn, grid, 1, 1, block, 1, 1, js->smem_bytes, (CUstream)st, args, nullptr);
}

}  // namespace

cudaError_t jit_launch(const ami_table* tab, bool fused, const AmiBatch& b, cudaStream_t st, int* launches) {
  const JitState* js = tab->jit;
  if (!js || js->status != AMI_OK) return cudaErrorInvalidDeviceFunction;
  if (b.n == 0) return cudaSuccess;
  if (js->mode != kJitScratch) {
    AmiBatch copy = b;
    if (launch_one(js, fused, copy, st) != CUDA_SUCCESS) return cudaErrorLaunchFailure;
    if (launches) ++*launches;
    return cudaSuccess;
  }
  // memory-backed variant: a stream-ordered scratch of [slots][chunk] doubles, at most ~512 MiB at a
  // time, so the batch is walked in chunks of samples
  const long long per_sample = (long long)js->scratch_slots * 8;
  long long chunk = std::max<long long>(js->block, ((512LL << 20) / std::max<long long>(per_sample, 1)) / js->block * js->block);
  chunk = std::min(chunk, (b.n + js->block - 1) / js->block * js->block);
  double* scratch = nullptr;
  cudaError_t crc = cudaMallocAsync((void**)&scratch, (size_t)(per_sample * chunk), st);
  if (crc != cudaSuccess) return crc;
  for (long long c0 = 0; c0 < b.n; c0 += chunk) {
    AmiBatch part = b;
    part.n = std::min(chunk, b.n - c0);
    if (part.e) part.e += c0;                       // SoA rows keep their stride
    if (part.e_out) part.e_out += c0;
    if (part.k) part.k += c0 * b.k_stride_sample;
    part.first_sample += c0;
    if (part.out) part.out += 2 * c0;
    if (part.tally) part.tally += 4 * (c0 >> 5);   // chunks are multiples of the block size
    part.scratch = scratch;
    part.scratch_stride = chunk;
    if (launch_one(js, fused, part, st) != CUDA_SUCCESS) { cudaFreeAsync(scratch, st); return cudaErrorLaunchFailure; }
    if (launches) ++*launches;
  }
  return cudaFreeAsync(scratch, st);
}

int jit_status(const ami_table* tab) {
  if (!tab->jit || !tab->jit->tried) return 1;
  return tab->jit->status;
}

void jit_destroy(ami_table* tab) {
  if (!tab->jit) return;
  if (tab->jit->mod && driver().ok) driver().ModuleUnload(tab->jit->mod);
  delete tab->jit;
  tab->jit = nullptr;
}

}  // namespace ami
