// Per-table specialised evaluation kernels ("register plan" and, for large tables, "split plan").
//
// The table-driven kernels pay an index load, an address computation and a shared-memory load for
// every multiply, which bounds them by instruction issue and shared-memory bandwidth (128 B/clk/SM
// against 64 DFMA/clk/SM) at a fraction of the FP64 pipe (profiles/r01_baseline_flat_cfg3.md).
// Here the symbolic result of ONE diagram is written out as straight-line CUDA C++ -- every
// Fermi/Bose leaf, every denominator and every partial sum a named register, the term table turned
// into the Horner form of ami_table.hpp -- and compiled for sm_100a with NVRTC when the table is
// first evaluated (cubins are cached on disk).
//
// Register plan (orders <= 6-7): the whole table is one body; ami_jit_eval (energies from memory,
// S2+S3), ami_jit_fused (momenta from memory or drawn in place, S1+S2+S3) and ami_jit_fused_tally
// (the same with the Monte-Carlo tally of S4 folded in) are generated from it.  Each kernel holds two bodies: one
// temperature per launch (beta { frequency { R part in Horner form } }), and several (per-beta values kept in a
// per-thread array, then frequency { reciprocals, R part for all temperatures }; where it is cheaper the R part
// is the sum over prefix products of Sections::secP / qrefs, four temperatures side by side).  A launch flagged
// AMI_PLAN_UNORDERED waits for its predecessor at its end instead of its start (kUnorderedEnd).
//
// Split plan (orders 7-8: 1e4-1e5 flat terms, hundreds of leaves, thousands of shared sums -- more
// than one thread's registers hold): the groups of the Horner plan are partitioned, in the order of
// the denominator trie, into PARTS of register-plan size; sums that several parts need are formed in
// each of them.  Per chunk of samples (sized so that what follows stays in L2):
//   ami_split_leaves_{eval,fused}  every Fermi/Bose value and reciprocal denominator -> leaves[slot][sample]
//   ami_split_parts                grid.y = part: its FT sums and its slice of the R part from those
//                                  leaves -> partial[part][row][sample]
//   ami_split_combine              adds the parts in a fixed order -> results
//
// The source text is produced by this file from the table; the arithmetic helpers it calls are
// the ones in ami_device.cuh, embedded as text at build time (generated/ami_embedded_src.h).
#include <cuda.h>
#include <cuda_runtime.h>
#include <dlfcn.h>
#include <sys/stat.h>
#include <unistd.h>

#include <algorithm>
#include <atomic>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <map>
#include <mutex>
#include <set>
#include <sstream>
#include <string>
#include <thread>
#include <vector>

#include "ami_jit.hpp"
#include "generated/ami_embedded_src.h"

namespace ami {

namespace {

constexpr size_t kWays = 16;            // independent chains kept side by side (measured: profiles/r01_batch_sweep.md)
constexpr size_t kGroupsPerChunk = 8;   // FT sums are emitted this many groups at a time

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

// One S-node of the FT DAG (ami_table.hpp) as a chain of statements defining `S<id>`; Fermi/Bose leaf u
// is named F<u><fsuffix>
void emit_snode(const HornerPlan& hp, int id, const std::string& fsuffix, Emitter& E, Stmts& out) {
  const SNode& n = hp.snodes[id];
  std::string acc;
  for (size_t i = 0; i < n.items.size(); ++i) {
    const SItem& it = n.items[i];
    const bool last = i + 1 == n.items.size();
    const std::string v = last ? "S" + std::to_string(id) : E.fresh("s");
    const std::string leaf = "F" + std::to_string(it.leaf) + fsuffix;
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
// (nodes of equal height are independent of one another), kWays chains side by side.  With
// `leaf_load` (split plan) the Fermi/Bose leaves these nodes use are first loaded into names private
// to this chunk, so that a leaf occupies a register only while a chunk that uses it is being formed.
void emit_ft_chunk(const HornerPlan& hp, size_t g0, size_t g1, std::vector<char>& done, Emitter& E,
                   std::ostringstream& o, const char* indent, const std::string* leaf_load,
                   std::ostringstream* loads = nullptr) {
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
  std::string fsuffix;
  if (leaf_load) {
    fsuffix = "_" + std::to_string(g0);
    std::set<int> used;
    for (int id : need)
      for (const SItem& it : hp.snodes[id].items) used.insert(it.leaf);
    for (int u : used)
      (loads ? *loads : o) << indent << "const double F" << u << fsuffix << " = " << *leaf_load << "(" << u << ");\n";
  }
  for (size_t i = 0; i < need.size();) {
    size_t j = i;
    std::vector<Stmts> lists;
    while (j < need.size() && hp.snodes[need[j]].height == hp.snodes[need[i]].height) {
      lists.emplace_back();
      emit_snode(hp, need[j], fsuffix, E, lists.back());
      ++j;
    }
    interleave(lists, kWays, o, indent);
    i = j;
  }
  for (size_t g = g0; g < g1; ++g) {
    const HGroup& hg = hp.groups[g];
    o << indent << "const double FT" << g << " = "
      << (hg.root >= 0 ? "S" + std::to_string(hg.root) : dlit((double)hg.num / (double)hg.den)) << ";\n";
  }
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

// ---- complex energies (energy_t is complex128 in the paper; reading P19 variant 5b) ----------
// The same plan with every value a pair of doubles.  acc + a * b for values that may be purely real:
CV emit_cv_fma(const CV& a, const CV& b, const CV* accp, Emitter& E, Stmts& out) {
  CV r;
  {   // real part: a.re*b.re - a.im*b.im (+ acc.re)
    std::string inner = accp ? accp->re : "";
    if (!a.real() && !b.real()) {
      const std::string t = E.fresh("c");
      if (inner.empty()) out.push_back("const double " + t + " = -" + a.im + " * " + b.im + ";");
      else out.push_back("const double " + t + " = fma(-" + a.im + ", " + b.im + ", " + inner + ");");
      inner = t;
    }
    r.re = E.fresh("c");
    if (inner.empty()) out.push_back("const double " + r.re + " = " + a.re + " * " + b.re + ";");
    else out.push_back("const double " + r.re + " = fma(" + a.re + ", " + b.re + ", " + inner + ");");
  }
  {   // imaginary part: a.re*b.im + a.im*b.re (+ acc.im)
    std::string inner = (accp && !accp->real()) ? accp->im : "";
    if (!b.real()) {
      const std::string t = E.fresh("c");
      if (inner.empty()) out.push_back("const double " + t + " = " + a.re + " * " + b.im + ";");
      else out.push_back("const double " + t + " = fma(" + a.re + ", " + b.im + ", " + inner + ");");
      inner = t;
    }
    if (!a.real()) {
      const std::string t = E.fresh("c");
      if (inner.empty()) out.push_back("const double " + t + " = " + a.im + " * " + b.re + ";");
      else out.push_back("const double " + t + " = fma(" + a.im + ", " + b.re + ", " + inner + ");");
      inner = t;
    }
    r.im = inner;
  }
  return r;
}

CV cv_leaf_f(int u) { return CV{"Fr" + std::to_string(u), "Fi" + std::to_string(u)}; }
CV cv_leaf_d(int u) { return CV{"Dr" + std::to_string(u), "Di" + std::to_string(u)}; }
CV cv_snode(int id) { return CV{"Sr" + std::to_string(id), "Si" + std::to_string(id)}; }

// S-node `id` with complex leaves: defines Sr<id>, Si<id>
void emit_snode_cplx(const HornerPlan& hp, int id, Emitter& E, Stmts& out) {
  const SNode& n = hp.snodes[id];
  CV acc;
  bool have = false;
  for (const SItem& it : n.items) {
    if (it.child >= 0) {
      acc = emit_cv_fma(cv_leaf_f(it.leaf), cv_snode(it.child), have ? &acc : nullptr, E, out);
    } else {
      const CV coef{dlit((double)it.num / (double)it.den), ""};
      acc = emit_cv_fma(coef, cv_leaf_f(it.leaf), have ? &acc : nullptr, E, out);
    }
    have = true;
  }
  const CV s = cv_snode(id);
  out.push_back("const double " + s.re + " = " + acc.re + ", " + s.im + " = " + (acc.real() ? std::string("0.0") : acc.im) + ";");
}

// Q(n) as in emit_q; with complex energies the frequency-independent denominators are complex too
CV emit_q_cplx(const HornerPlan& hp, int n, Emitter& E, Stmts& out, bool* have_out) {
  CV acc;
  bool have = false;
  if (hp.dn[n].group >= 0) {
    const std::string g = std::to_string(hp.dn[n].group);
    acc = CV{"FTr" + g, "FTi" + g};
    have = true;
  }
  for (int c : hp.dn[n].kids) {
    if (!hp.d_is_real[hp.dn[c].leaf]) continue;
    bool sub_have = false;
    const CV qc = emit_q_cplx(hp, c, E, out, &sub_have);   // never empty: a trie leaf carries a group
    acc = emit_cv_fma(cv_leaf_d(hp.dn[c].leaf), qc, have ? &acc : nullptr, E, out);
    have = true;
  }
  *have_out = have;
  return acc;
}

CV emit_d_sum_cplx(const HornerPlan& hp, const std::vector<CV>& q, const std::vector<char>& q_have, int n, Emitter& E,
                   Stmts& out) {
  CV acc;
  bool have = false;
  if (q_have[n]) { acc = q[n]; have = true; }
  for (int c : hp.dn[n].kids) {
    if (hp.d_is_real[hp.dn[c].leaf]) continue;
    const CV s = emit_d_sum_cplx(hp, q, q_have, c, E, out);
    acc = emit_cv_fma(cv_leaf_d(hp.dn[c].leaf), s, have ? &acc : nullptr, E, out);
    have = true;
  }
  if (!have) { acc.re = "0.0"; acc.im = ""; }
  return acc;
}

// ---- split plan: partition of the groups and the Horner plan of one part -----------------------
// FP64 instructions of the FT sums reachable from S-node `root` that are not in `seen` yet
long long mark_reachable(const HornerPlan& hp, int root, std::vector<char>& seen) {
  long long ops = 0;
  std::vector<int> stack(1, root);
  while (!stack.empty()) {
    const int id = stack.back();
    stack.pop_back();
    if (seen[id]) continue;
    seen[id] = 1;
    ops += (long long)hp.snodes[id].items.size();
    for (const SItem& it : hp.snodes[id].items)
      if (it.child >= 0 && !seen[it.child]) stack.push_back(it.child);
  }
  return ops;
}

// Groups in the order in which a depth-first walk of the denominator trie meets them: consecutive groups
// share denominator prefixes, and the recursion that produced them makes them share Fermi/Bose sums.
void groups_in_trie_order(const HornerPlan& hp, int n, std::vector<int>& out) {
  if (hp.dn[n].group >= 0) out.push_back(hp.dn[n].group);
  for (int c : hp.dn[n].kids) groups_in_trie_order(hp, c, out);
}

// Cuts an order of the groups into parts of about `budget` FP64 instructions each: the FT sums a part reaches (sums
// it shares with an earlier part are counted, and formed, again) plus its slice of the denominator trie.  Returns the
// total work of all parts in *total.
std::vector<std::vector<int>> cut_into_parts(const HornerPlan& hp, const std::vector<int>& order,
                                             const std::vector<std::vector<int>>& path, long long budget, long long* total) {
  std::vector<std::vector<int>> parts(1);
  std::vector<char> seen(hp.snodes.size(), 0), dseen(hp.dn.size(), 0);
  long long cur = 0;
  *total = 0;
  auto cost_of = [&](int g, bool commit) {
    const HGroup& hg = hp.groups[g];
    long long add = 0;
    if (hg.root >= 0) {
      if (commit) {
        add += mark_reachable(hp, hg.root, seen);
      } else {
        std::vector<int> stack(1, hg.root), touched;
        while (!stack.empty()) {
          const int id = stack.back();
          stack.pop_back();
          if (seen[id]) continue;
          seen[id] = 1;
          touched.push_back(id);
          add += (long long)hp.snodes[id].items.size();
          for (const SItem& it : hp.snodes[id].items)
            if (it.child >= 0 && !seen[it.child]) stack.push_back(it.child);
        }
        for (int id : touched) seen[id] = 0;
      }
    }
    for (int n : path[g])
      if (!dseen[n]) {
        add += hp.d_is_real[hp.dn[n].leaf] ? 1 : 4;
        if (commit) dseen[n] = 1;
      }
    return add;
  };
  for (int g : order) {
    long long add = cost_of(g, false);
    if (cur > 0 && cur + add > budget) {
      parts.emplace_back();
      std::fill(seen.begin(), seen.end(), 0);
      std::fill(dseen.begin(), dseen.end(), 0);
      cur = 0;
    }
    add = cost_of(g, true);
    cur += add;
    *total += add;
    parts.back().push_back(g);
  }
  return parts;
}

// Two orders of the groups are tried and the cheaper partition is kept: the depth-first order of the denominator
// trie (neighbours share denominator prefixes) and the order of the groups' top-level Fermi/Bose sums (neighbours share
// FT sums).  Which one wins depends on the diagram: order 8 (seed 0) 1.5x / 1.4x the work of the undivided plan,
// order 9 (seed 0) 3.6x / 1.5x.
std::vector<std::vector<int>> partition_groups(const HornerPlan& hp, long long budget) {
  const int G = (int)hp.groups.size();
  std::vector<std::vector<int>> path(G);          // trie nodes on the way to each group
  for (int g = 0; g < G; ++g) {
    int cur = 0;
    for (int leaf : hp.dseq[g])
      for (int c : hp.dn[cur].kids)
        if (hp.dn[c].leaf == leaf) { cur = c; path[g].push_back(c); break; }
  }
  std::vector<int> by_trie;
  groups_in_trie_order(hp, 0, by_trie);
  std::vector<int> pos(G, 0);
  for (int i = 0; i < G; ++i) pos[by_trie[i]] = i;
  std::vector<std::vector<int>> sig(G);           // children of the group's top-level sum
  for (int g = 0; g < G; ++g)
    if (hp.groups[g].root >= 0) {
      for (const SItem& it : hp.snodes[hp.groups[g].root].items)
        if (it.child >= 0) sig[g].push_back(it.child);
      std::sort(sig[g].begin(), sig[g].end());
    }
  std::vector<int> by_sum = by_trie;
  std::stable_sort(by_sum.begin(), by_sum.end(), [&](int a, int b) { return sig[a] != sig[b] ? sig[a] < sig[b] : pos[a] < pos[b]; });
  long long cost_trie = 0, cost_sum = 0;
  std::vector<std::vector<int>> p_trie = cut_into_parts(hp, by_trie, path, budget, &cost_trie);
  std::vector<std::vector<int>> p_sum = cut_into_parts(hp, by_sum, path, budget, &cost_sum);
  return cost_sum < cost_trie ? p_sum : p_trie;
}

// The Horner plan restricted to `groups`: their FT sums (renumbered, children still before parents) and the
// denominator trie of their products.  Leaf ids stay those of the whole table.
HornerPlan make_sub_plan(const HornerPlan& hp, const std::vector<int>& groups) {
  HornerPlan sub;
  sub.d_is_real = hp.d_is_real;
  std::vector<char> seen(hp.snodes.size(), 0);
  for (int g : groups)
    if (hp.groups[g].root >= 0) mark_reachable(hp, hp.groups[g].root, seen);
  std::vector<int> new_id(hp.snodes.size(), -1);
  for (size_t id = 0; id < hp.snodes.size(); ++id) {
    if (!seen[id]) continue;
    new_id[id] = (int)sub.snodes.size();
    SNode n = hp.snodes[id];
    for (SItem& it : n.items)
      if (it.child >= 0) it.child = new_id[it.child];
    sub.snodes.push_back(std::move(n));
  }
  sub.dn.assign(1, HNode());
  for (int g : groups) {
    HGroup hg = hp.groups[g];
    if (hg.root >= 0) hg.root = new_id[hg.root];
    const int gi = (int)sub.groups.size();
    sub.groups.push_back(hg);
    sub.dseq.push_back(hp.dseq[g]);
    int cur = 0;
    for (int leaf : hp.dseq[g]) {
      int nxt = -1;
      for (int c : sub.dn[cur].kids)
        if (sub.dn[c].leaf == leaf) { nxt = c; break; }
      if (nxt < 0) {
        nxt = (int)sub.dn.size();
        HNode nn;
        nn.leaf = leaf;
        sub.dn.push_back(nn);
        sub.dn[cur].kids.push_back(nxt);
      }
      cur = nxt;
    }
    sub.dn[cur].group = gi;
  }
  return sub;
}

long long split_budget() {
  static const long long b = [] {
    const char* e = getenv("AMI_JIT_SPLIT_BUDGET");   // tuning knob: FP64 instructions per part
    const long long v = e ? atoll(e) : 0;
    return v >= 100 ? v : 1500LL;
  }();
  return b;
}

// ---------------------------------------------------------------------------------------------
// The body of one sample in four sections that the kernels assemble:
//   0: once per sample   1: per beta   2: per frequency   3: per (beta, frequency)
// Leaves (Fermi/Bose values, reciprocal denominators) are, depending on the kernel,
//   kLeafInline  computed and kept in registers (register plan)
//   kLeafStore   computed and written to the leaf array, nothing else is emitted (split plan, leaf kernel)
//   kLeafLoad    read from the leaf array where they are used (split plan, a part)
// ---------------------------------------------------------------------------------------------
enum LeafMode { kLeafInline, kLeafStore, kLeafLoad };

struct Sections {
  std::ostringstream sec[4];
  std::vector<std::string> keep;   // per-beta values the R part reads (for the several-temperature body)
  // several-temperature body, R part as a sum over prefix products: S_D(root) = Q(root) + sum_n Q(n) P_n with
  // P_n = the product of the complex reciprocals on the way from the root to trie node n.  The P_n depend on the
  // frequency only (secP: once per frequency, 4 instructions per node below the first level), the Q(n) on the
  // temperature only (keep), so a (frequency, temperature) pair costs 2 instructions per node that carries a Q
  // instead of the 2-4 per trie edge of the Horner form in sec[3].
  std::ostringstream secP;
  struct QRef { int keep, keep_im; std::string pr, pi; };   // keep_im < 0: Q is real; pr empty: the root's own Q (no product)
  std::vector<QRef> qrefs;
};

struct LeafSlots {                 // layout of the split plan's leaf array
  std::vector<int> ridx, cidx;     // position of denominator u among the purely real / the complex ones
  int n_real = 0, n_cplx = 0, n_fermi = 0;
};

LeafSlots leaf_slots(const FlatTable& ft, const HornerPlan& hp) {
  LeafSlots ls;
  ls.ridx.assign(ft.leafD.size(), -1);
  ls.cidx.assign(ft.leafD.size(), -1);
  for (size_t u = 0; u < ft.leafD.size(); ++u) {
    if (hp.d_is_real[u]) ls.ridx[u] = ls.n_real++;
    else ls.cidx[u] = ls.n_cplx++;
  }
  ls.n_fermi = (int)ft.leafF.size();
  return ls;
}

// The R part as Q(root) + sum_n Q(n) P_n (several-temperature body of the register plan; see Sections): the
// statements that form the prefix products P_n (S.secP) and, in depth-first order, which kept value meets which P_n
// (S.qrefs).  q[n] names Q(n) (re empty: there is none; im empty: it is real).
void build_prefix_form(const HornerPlan& hp, const std::vector<CV>& q, Emitter& E, Sections& S) {
  auto keep_index = [&](const std::string& name) {
    if (name.empty() || name == "0.0") return -1;
    return (int)(std::find(S.keep.begin(), S.keep.end(), name) - S.keep.begin());
  };
  if (!q[0].re.empty()) S.qrefs.push_back({keep_index(q[0].re), keep_index(q[0].im), "", ""});
  std::vector<Stmts> lists;
  // P of a node on the first level is its reciprocal itself; below, (P.re + i P.im)(Dr + i Di): 4 instructions
  std::function<void(int, const CV&)> below = [&](int n, const CV& P) {
    if (!q[n].re.empty()) S.qrefs.push_back({keep_index(q[n].re), keep_index(q[n].im), P.re, P.im});
    for (int c : hp.dn[n].kids) {
      const int u = hp.dn[c].leaf;
      if (hp.d_is_real[u]) continue;
      const std::string dr = "Dr" + std::to_string(u), di = "Di" + std::to_string(u);
      const CV Pc{E.fresh("P"), E.fresh("P")};
      const std::string t0 = E.fresh("P"), t1 = E.fresh("P");
      Stmts& out = lists.back();
      out.push_back("const double " + t0 + " = -" + P.im + " * " + di + ";");
      out.push_back("const double " + t1 + " = " + P.re + " * " + di + ";");
      out.push_back("const double " + Pc.re + " = fma(" + P.re + ", " + dr + ", " + t0 + ");");
      out.push_back("const double " + Pc.im + " = fma(" + P.im + ", " + dr + ", " + t1 + ");");
      below(c, Pc);
    }
  };
  for (int c : hp.dn[0].kids) {
    const int u = hp.dn[c].leaf;
    if (hp.d_is_real[u]) continue;
    lists.emplace_back();
    below(c, CV{"Dr" + std::to_string(u), "Di" + std::to_string(u)});
  }
  interleave(lists, kWays, S.secP, "      ");
}

// `hp` may be the plan of one part; leaf ids and `ls` are those of the whole table
void gen_sections(const FlatTable& ft, const HornerPlan& hp, const LeafSlots& ls, LeafMode mode, Emitter& E,
                  Sections& S) {
  int cur = 0;
#define o S.sec[cur]
  auto slot_c = [&](size_t u) {
    return "(CB + 2 * (f * " + std::to_string(ls.n_cplx) + " + " + std::to_string(ls.cidx[u]) + "))";
  };
  // which leaves this plan uses
  std::vector<char> useF(ft.leafF.size(), 0), useD(ft.leafD.size(), 0);
  if (mode == kLeafLoad) {
    for (const SNode& n : hp.snodes)
      for (const SItem& it : n.items) useF[it.leaf] = 1;
    for (size_t n = 1; n < hp.dn.size(); ++n) useD[hp.dn[n].leaf] = 1;
  } else {
    std::fill(useF.begin(), useF.end(), 1);
    std::fill(useD.begin(), useD.end(), 1);
  }
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
  if (mode != kLeafLoad) {
    for (const LeafD& l : ft.leafD) combo_ref(l.c);
    for (size_t j = 0; j < combos.size(); ++j) o << "  const double E" << j << " = " << combo(combos[j], "e") << ";\n";
  }
  // reciprocals of the denominators, kWays at a time
  auto emit_d_leaves = [&](const std::vector<size_t>& ids, const std::string& ind) {
    if (mode == kLeafLoad) {
      // read where they are used: a denominator enters one product per trie node that carries it
      for (size_t u : ids) {
        if (!useD[u]) continue;
        if (hp.d_is_real[u]) {
          o << "#define Dr" << u << " AMI_L(" << ls.ridx[u] << ")\n";
        } else {
          o << "#define Dr" << u << " AMI_LC(" << 2 * ls.cidx[u] << ")\n#define Di" << u << " AMI_LC(" << 2 * ls.cidx[u] + 1 << ")\n";
        }
      }
      return;
    }
    if (mode == kLeafInline)
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
        if (mode == kLeafInline) {
          if (hp.d_is_real[u]) o << ind << "  Dr" << u << " = d[" << j << "];\n";
          else o << ind << "  Dr" << u << " = re" << j << " * d[" << j << "]; Di" << u << " = -im" << j << " * d[" << j << "];\n";
        } else if (hp.d_is_real[u]) {
          o << ind << "  AMI_LS(" << ls.ridx[u] << ", d[" << j << "]);\n";
        } else {
          o << ind << "  AMI_LSC(" << 2 * ls.cidx[u] << ", re" << j << " * d[" << j << "]); AMI_LSC(" << 2 * ls.cidx[u] + 1
            << ", -im" << j << " * d[" << j << "]);\n";
        }
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
  if (mode != kLeafLoad) {
    std::vector<std::vector<size_t>> base;      // base -> leaves with the same (combination, sigma)
    for (size_t u = 0; u < UF; ++u) {
      size_t b = 0;
      for (; b < base.size(); ++b)
        if (ft.leafF[base[b][0]].c == ft.leafF[u].c && ft.leafF[base[b][0]].sigma == ft.leafF[u].sigma) break;
      if (b == base.size()) base.emplace_back();
      base[b].push_back(u);
    }
    if (mode == kLeafInline)
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
    auto assign = [&](size_t u, const std::string& value, const std::string& ind) {
      if (mode == kLeafInline) o << ind << "F" << u << " = " << value << ";\n";
      else o << ind << "AMI_LSF(" << u << ", " << value << ");\n";
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
            assign(u, f, "      ");
            continue;
          }
          // f^{(k)} = beta^k f g Q_k(f)
          o << "      {\n        const double f = " << f << ";\n";
          const std::vector<double> q = deriv_poly(l.k);
          o << "        double q = " << dlit(q.back()) << ";\n";
          for (int i = (int)q.size() - 2; i >= 0; --i) o << "        q = fma(q, f, " << dlit(q[i]) << ");\n";
          o << "        double bk = beta;\n";
          for (int i = 1; i < l.k; ++i) o << "        bk *= beta;\n";
          assign(u, "bk * f * g" + std::to_string(j) + " * q", "        ");
          o << "      }\n";
        }
      }
      o << "    }\n";
    }
  }
  std::vector<std::string> qname(hp.dn.size());
  if (mode != kLeafStore) {
    // FT sums of every group (per beta): a DAG shared by all groups, emitted a few groups at a time
    std::vector<char> done(hp.snodes.size(), 0);
    const std::string loader = "AMI_LF";
    if (mode != kLeafLoad) {
      for (size_t g0 = 0; g0 < hp.groups.size(); g0 += kGroupsPerChunk)
        emit_ft_chunk(hp, g0, std::min(hp.groups.size(), g0 + kGroupsPerChunk), done, E, o, "    ", nullptr);
    } else {
      // split plan: the leaves of chunk c+1 are requested before the sums of chunk c are formed, so that their
      // way from L2 (ncu: half of the stall samples were waits for these loads) overlaps arithmetic
      std::vector<std::string> loads, bodies;
      for (size_t g0 = 0; g0 < hp.groups.size(); g0 += kGroupsPerChunk) {
        std::ostringstream l, b;
        emit_ft_chunk(hp, g0, std::min(hp.groups.size(), g0 + kGroupsPerChunk), done, E, b, "    ", &loader, &l);
        loads.push_back(l.str());
        bodies.push_back(b.str());
      }
      if (!loads.empty()) o << loads[0];
      for (size_t c = 0; c < bodies.size(); ++c) {
        if (c + 1 < loads.size()) o << loads[c + 1];
        o << bodies[c];
      }
    }
    // frequency-independent parts of the R sums (products under purely real denominators), per beta
    std::vector<Stmts> lists;
    for (size_t n = 0; n < hp.dn.size(); ++n) {
      if (n != 0 && hp.d_is_real[hp.dn[n].leaf]) continue;
      lists.emplace_back();
      qname[n] = emit_q(hp, (int)n, E, lists.back());
    }
    interleave(lists, kWays, o, "    ");
    for (const std::string& q : qname)
      if (!q.empty() && std::find(S.keep.begin(), S.keep.end(), q) == S.keep.end()) S.keep.push_back(q);
  }
  // frequencies
  cur = 2;
  if (mode != kLeafLoad)
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
  if (mode != kLeafStore) {
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
    o << "      AMI_EMIT(" << acc.re << ", " << (acc.real() ? std::string("0.0") : acc.im) << ");\n";
  }
#undef o
  if (mode == kLeafInline) {
    std::vector<CV> q(hp.dn.size());
    for (size_t n = 0; n < hp.dn.size(); ++n) q[n].re = qname[n];
    build_prefix_form(hp, q, E, S);
  }
}

// The four sections of the body for complex energies e<i>r + i e<i>i (register plan only).
// `ls` (split plan only): the leaf slots of the whole table, every value two doubles (re at the slot, im at the next).
void gen_sections_cplx(const FlatTable& ft, const HornerPlan& hp, const LeafSlots& ls, LeafMode mode, Emitter& E,
                       Sections& S) {
  int cur = 0;
#define o S.sec[cur]
  // which leaves this plan uses (a part of the split plan: those its sums and its slice of the trie reach)
  std::vector<char> useF(ft.leafF.size(), 1), useD(ft.leafD.size(), 1);
  if (mode == kLeafLoad) {
    std::fill(useF.begin(), useF.end(), 0);
    std::fill(useD.begin(), useD.end(), 0);
    for (const SNode& n : hp.snodes)
      for (const SItem& it : n.items) useF[it.leaf] = 1;
    for (size_t n = 1; n < hp.dn.size(); ++n) useD[hp.dn[n].leaf] = 1;
  }
  std::vector<std::vector<int>> combos;
  auto combo_ref = [&](const std::vector<int>& c, std::string* sign) -> int {
    std::vector<int> pos = c;
    int sg = 0;
    for (int v : c)
      if (v) { sg = v > 0 ? 1 : -1; break; }
    *sign = sg < 0 ? "-" : "";
    if (!sg) return -1;
    if (sg < 0)
      for (int& v : pos) v = -v;
    size_t j = 0;
    for (; j < combos.size(); ++j)
      if (combos[j] == pos) break;
    if (j == combos.size()) combos.push_back(pos);
    return (int)j;
  };
  if (mode != kLeafLoad) {
    for (const LeafD& l : ft.leafD) { std::string sg; combo_ref(l.c, &sg); }
    for (size_t j = 0; j < combos.size(); ++j)
      o << "  const double E" << j << "r = " << combo(combos[j], "e", "r") << ", E" << j << "i = " << combo(combos[j], "e", "i") << ";\n";
  }
  auto emit_d_leaves = [&](bool freq_independent, const std::string& ind) {
    for (size_t u = 0; u < ft.leafD.size(); ++u) {
      if ((hp.d_is_real[u] != 0) != freq_independent) continue;
      if (mode == kLeafLoad) {     // read where it is used
        if (!useD[u]) continue;
        if (freq_independent) o << "#define Dr" << u << " AMI_L(" << ls.ridx[u] << ")\n#define Di" << u << " AMI_L(" << ls.ridx[u] + 1 << ")\n";
        else o << "#define Dr" << u << " AMI_LC(" << 2 * ls.cidx[u] << ")\n#define Di" << u << " AMI_LC(" << 2 * ls.cidx[u] + 1 << ")\n";
        continue;
      }
      const LeafD& l = ft.leafD[u];
      std::string sg;
      const int j = combo_ref(l.c, &sg);
      const std::string er = j < 0 ? "0.0" : sg + "E" + std::to_string(j) + "r", ei = j < 0 ? "0.0" : sg + "E" + std::to_string(j) + "i";
      o << ind << "double Dr" << u << ", Di" << u << ";\n" << ind << "{\n";
      if (freq_independent) {
        o << ind << "  const double re = " << er << " + p.e_reg, im = " << ei << ";\n";      // P10(b): always regulated
      } else {
        std::string cond;
        for (int x = 0; x < ft.n_ext; ++x)
          if (l.a[x]) cond += (cond.empty() ? "" : " && ") + std::string("zz") + std::to_string(x);
        o << ind << "  const double re = ((" << combo(l.a, "zr") << ") + " << er << ") + ((" << cond << ") ? p.e_reg : 0.0), im = ("
          << combo(l.a, "zi") << ") + " << ei << ";\n";
      }
      o << ind << "  const double r = fast_rcp(fma(re, re, im * im));\n" << ind << "  Dr" << u << " = re * r; Di" << u << " = -im * r;\n"
        << ind << "}\n";
      if (mode == kLeafStore) {
        if (freq_independent) o << ind << "AMI_LS(" << ls.ridx[u] << ", Dr" << u << "); AMI_LS(" << ls.ridx[u] + 1 << ", Di" << u << ");\n";
        else o << ind << "AMI_LSC(" << 2 * ls.cidx[u] << ", Dr" << u << "); AMI_LSC(" << 2 * ls.cidx[u] + 1 << ", Di" << u << ");\n";
      }
    }
  };
  emit_d_leaves(true, "  ");
  cur = 1;
  if (mode == kLeafLoad) {
    for (size_t u = 0; u < ft.leafF.size(); ++u)
      if (useF[u]) o << "#define Fr" << u << " AMI_LF(" << 2 * u << ")\n#define Fi" << u << " AMI_LF(" << 2 * u + 1 << ")\n";
  } else {
  // one exponential per energy symbol: e^{beta e_i} = 2^{n_i} (m_i r + i m_i i), |m_i| in [0.70, 1.42]
  std::vector<char> sym_used(ft.n_eps, 0);
  for (const LeafF& l : ft.leafF)
    for (int i = 0; i < ft.n_eps; ++i)
      if (l.c[i]) sym_used[i] = 1;
  for (int i = 0; i < ft.n_eps; ++i) {
    if (!sym_used[i]) continue;
    o << "    int n" << i << "; double m" << i << "r, m" << i << "i;\n    {\n      const double x[1] = {beta * e" << i
      << "r};\n      int nn[1]; double mm[1];\n      exp_split_n<1>(x, nn, mm);\n      double sn, cs;\n      sincos(beta * e" << i
      << "i, &sn, &cs);\n      n" << i << " = nn[0]; m" << i << "r = mm[0] * cs; m" << i << "i = mm[0] * sn;\n    }\n";
  }
  // leaves: f_sigma = B / (sigma 2^N A + B) with A, B complex mantissa products (P12); derivatives by Q_k (P11)
  std::vector<std::vector<size_t>> base;
  for (size_t u = 0; u < ft.leafF.size(); ++u) {
    size_t b = 0;
    for (; b < base.size(); ++b)
      if (ft.leafF[base[b][0]].c == ft.leafF[u].c && ft.leafF[base[b][0]].sigma == ft.leafF[u].sigma) break;
    if (b == base.size()) base.emplace_back();
    base[b].push_back(u);
  }
  for (size_t u = 0; u < ft.leafF.size(); ++u) o << "    double Fr" << u << ", Fi" << u << ";\n";
  for (const auto& members : base) {
    const LeafF& l = ft.leafF[members[0]];
    o << "    {\n";
    Stmts st;
    std::string ex;
    auto product = [&](int sign) -> CV {
      CV acc;
      bool have = false;
      for (int i = 0; i < ft.n_eps; ++i)
        for (int r = 0; r < l.c[i] * sign; ++r) {
          const CV m{"m" + std::to_string(i) + "r", "m" + std::to_string(i) + "i"};
          ex += std::string(sign > 0 ? " + n" : " - n") + std::to_string(i);
          if (!have) { acc = m; have = true; }
          else acc = emit_cv_fma(acc, m, nullptr, E, st);
        }
      if (!have) acc = CV{"1.0", ""};
      return acc;
    };
    CV A = product(+1);
    const CV B = product(-1);
    if (l.sigma < 0) A = emit_cv_fma(CV{"p.ceta[b]", ""}, A, nullptr, E, st);      // e^{beta eta} (P10(a))
    for (const std::string& s : st) o << "      " << s << "\n";
    // d = sigma 2^N A + B is formed as d' = A' + B' with A' = sigma 2^min(N,0) A and B' = 2^-max(N,0) B, i.e. divided by
    // 2^N when that is large: |d'| stays of order one, so |d'|^2 cannot overflow for any beta (P12), and
    // f = B' conj(d') / |d'|^2,  g = 1 - f = A' conj(d') / |d'|^2  hold in both cases.
    const std::string sg = l.sigma > 0 ? "" : "-";
    o << "      const int N = 0" << ex << ";\n"
      << "      const double s1 = pow2_clamped(min(N, 0)), s2 = pow2_clamped(-max(N, 0));\n"
      << "      const double ar = s1 * " << sg << A.re << ", ai = " << (A.real() ? std::string("0.0") : "s1 * " + sg + A.im) << ";\n"
      << "      const double br = s2 * " << B.re << ", bi = " << (B.real() ? std::string("0.0") : "s2 * " + B.im) << ";\n"
      << "      const double dr = ar + br, di = ai + bi;\n"
      << "      const double rn = fast_rcp(fma(dr, dr, di * di));\n"
      << "      const double fr = fma(br, dr, bi * di) * rn, fi = fma(bi, dr, -br * di) * rn;\n";
    bool need_g = false;
    for (size_t u : members) need_g |= ft.leafF[u].k > 0;
    if (need_g) o << "      const double gr = fma(ar, dr, ai * di) * rn, gi = fma(ai, dr, -ar * di) * rn;\n";
    for (size_t u : members) {
      const int k = ft.leafF[u].k;
      if (k == 0) { o << "      Fr" << u << " = fr; Fi" << u << " = fi;\n"; continue; }
      const std::vector<double> q = deriv_poly(k);
      o << "      {\n        double qr = " << dlit(q.back()) << ", qi = 0.0;\n";
      for (int i = (int)q.size() - 2; i >= 0; --i)
        o << "        { const double t = fma(qr, fr, -qi * fi) + " << dlit(q[i]) << "; qi = fma(qr, fi, qi * fr); qr = t; }\n";
      o << "        double bk = beta;\n";
      for (int i = 1; i < k; ++i) o << "        bk *= beta;\n";
      o << "        const double hr = fma(fr, gr, -fi * gi), hi = fma(fr, gi, fi * gr);\n"
           "        Fr" << u << " = bk * fma(hr, qr, -hi * qi); Fi" << u << " = bk * fma(hr, qi, hi * qr);\n      }\n";
    }
    o << "    }\n";
  }
  if (mode == kLeafStore)
    for (size_t u = 0; u < ft.leafF.size(); ++u) o << "    AMI_LSF(" << 2 * u << ", Fr" << u << "); AMI_LSF(" << 2 * u + 1 << ", Fi" << u << ");\n";
  }   // leaves computed here
  std::vector<CV> q(hp.dn.size());
  std::vector<char> q_have(hp.dn.size(), 0);
  // FT sums, level by level
  if (mode != kLeafStore) {
    std::vector<int> order(hp.snodes.size());
    for (size_t i = 0; i < order.size(); ++i) order[i] = (int)i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return hp.snodes[a].height < hp.snodes[b].height; });
    for (size_t i = 0; i < order.size();) {
      size_t j = i;
      std::vector<Stmts> lists;
      while (j < order.size() && hp.snodes[order[j]].height == hp.snodes[order[i]].height) {
        lists.emplace_back();
        emit_snode_cplx(hp, order[j], E, lists.back());
        ++j;
      }
      interleave(lists, kWays, o, "    ");
      i = j;
    }
    for (size_t g = 0; g < hp.groups.size(); ++g) {
      const HGroup& hg = hp.groups[g];
      if (hg.root >= 0) o << "    const double FTr" << g << " = Sr" << hg.root << ", FTi" << g << " = Si" << hg.root << ";\n";
      else o << "    const double FTr" << g << " = " << dlit((double)hg.num / (double)hg.den) << ", FTi" << g << " = 0.0;\n";
    }
  }
  if (mode != kLeafStore) {
    std::vector<Stmts> lists;
    for (size_t n = 0; n < hp.dn.size(); ++n) {
      if (n != 0 && hp.d_is_real[hp.dn[n].leaf]) continue;
      lists.emplace_back();
      bool have = false;
      q[n] = emit_q_cplx(hp, (int)n, E, lists.back(), &have);
      q_have[n] = have;
      if (have && q[n].im.empty()) q[n].im = "0.0";
      if (have)
        for (const std::string& nm : {q[n].re, q[n].im})
          if (nm != "0.0" && std::find(S.keep.begin(), S.keep.end(), nm) == S.keep.end()) S.keep.push_back(nm);
    }
    interleave(lists, kWays, o, "    ");
  }
  cur = 2;
  if (mode != kLeafLoad)
    for (int x = 0; x < ft.n_ext; ++x) {
      o << "      const double zr" << x << " = p.z[2 * (f * " << ft.n_ext << " + " << x << ")], zi" << x
        << " = p.z[2 * (f * " << ft.n_ext << " + " << x << ") + 1];\n";
      o << "      const bool zz" << x << " = (zr" << x << " == 0.0 && zi" << x << " == 0.0);\n";
    }
  emit_d_leaves(false, "      ");
  cur = 3;
  if (mode != kLeafStore) {
    Stmts st;
    const CV acc = emit_d_sum_cplx(hp, q, q_have, 0, E, st);
    for (const std::string& s : st) o << "      " << s << "\n";
    o << "      AMI_EMIT(" << acc.re << ", " << (acc.real() ? std::string("0.0") : acc.im) << ");\n";
  }
#undef o
  if (mode == kLeafInline) {
    std::vector<CV> qq(hp.dn.size());
    for (size_t n = 0; n < hp.dn.size(); ++n)
      if (q_have[n]) qq[n] = q[n];
    build_prefix_form(hp, qq, E, S);
  }
}

// Momenta of sample `at` into nk0..: from memory, or drawn in place by the counter-based generator (S4 with a
// seed: the momenta never exist in memory).  Counter of component c = sample * n_comp + c; the generator's
// state is seed + GOLDEN (counter + 1), so one 64-bit multiply per sample and an addition per component
// (arithmetic modulo 2^64: same bits as momentum_of).
void emit_momenta(std::ostringstream& o, int n_comp, const std::string& at, const std::string& ind) {
  o << ind << "if (p.gen) {\n" << ind << "  const unsigned long long z0 = p.seed + 0x9E3779B97F4A7C15ull * ((unsigned long long)"
    << "(p.first_sample + (" << at << ")) * " << n_comp << "ull + 1ull);\n";
  for (int c = 0; c < n_comp; ++c) {
    char lit[32];
    snprintf(lit, sizeof lit, "0x%016llXull", (unsigned long long)(0x9E3779B97F4A7C15ull * (unsigned long long)c));
    o << ind << "  nk" << c << " = momentum_from_state(z0 + " << lit << ");\n";
  }
  o << ind << "} else {\n" << ind << "  const double* kn = p.k + (" << at << ") * p.k_stride_sample;\n";
  for (int c = 0; c < n_comp; ++c) o << ind << "  nk" << c << " = kn[" << c << " * p.k_stride_comp];\n";
  o << ind << "}\n";
}

// Inline dispersion (Eqs. 8-18; Eq. 14 for `dim` components): e_i from the momenta kx<l>, ky<l>, ...
// and the external ones.  Same operations in the same order as dispersion_kernel (ami_kernels.cu): bit-identical.
void emit_dispersion(std::ostringstream& o, const FlatTable& ft, const JitVariant& var) {
  static const char* comp[3] = {"kx", "ky", "kz"};
  const int L = ft.n_int + ft.n_ext, dim = var.dim;
  for (int l = 0; l < ft.n_int; ++l) {
    o << "  const double ";
    for (int c = 0; c < dim; ++c) o << (c ? ", " : "") << comp[c] << l << " = nk" << dim * l + c;
    o << ";\n";
  }
  for (int x = 0; x < ft.n_ext; ++x) {
    o << "  const double ";
    for (int c = 0; c < dim; ++c) o << (c ? ", " : "") << comp[c] << ft.n_int + x << " = p.q[" << dim * x + c << "]";
    o << ";\n";
  }
  for (int i = 0; i < ft.n_eps; ++i) o << "  double e" << i << ";\n";
  const int sym_batch = std::max(1, (int)kWays / dim);   // kWays cosines side by side
  for (int i0 = 0; i0 < ft.n_eps; i0 += sym_batch) {
    const int n = std::min(sym_batch, ft.n_eps - i0);
    o << "  {\n    double c[" << dim * n << "] = {";
    for (int j = 0; j < n; ++j) {
      std::vector<int> a(ft.sym_alpha.begin() + (size_t)(i0 + j) * L, ft.sym_alpha.begin() + (size_t)(i0 + j + 1) * L);
      for (int c = 0; c < dim; ++c) o << (j || c ? ", " : "") << combo(a, comp[c]);
    }
    o << "};\n";
    if (var.band == AMI_BAND_TIGHT_BINDING) {
      o << "    cos_bounded_n<" << dim * n << ">(c);\n";
      for (int j = 0; j < n; ++j) {
        std::string sum = "c[" + std::to_string(dim * j) + "]";
        for (int c = 1; c < dim; ++c) sum = "(" + sum + " + c[" + std::to_string(dim * j + c) + "])";
        o << "    e" << i0 + j << " = fma(2.0 * p.t, " << sum << ", p.mu);\n";
      }
    } else {   // free particles: e = mu - t |K|^2
      for (int j = 0; j < n; ++j) {
        std::string sq = "c[" + std::to_string(dim * j) + "] * c[" + std::to_string(dim * j) + "]";
        for (int c = 1; c < dim; ++c) {
          const std::string k = "c[" + std::to_string(dim * j + c) + "]";
          sq = "fma(" + k + ", " + k + ", " + sq + ")";
        }
        o << "    e" << i0 + j << " = fma(-p.t, " << sq << ", p.mu);\n";
      }
    }
    o << "  }\n";
  }
}

const char* kTallySrc =
    // Fused tally (S4, Monte-Carlo sums of PAPER.md:291): the warp adds its lanes' (re, im, re^2, im^2) in a fixed
    // tree and leaves one partial per (row, warp).  All 32 lanes take part (lanes without a sample pass zeros).  The
    // four values are reduced together: after the first exchange a lane carries two of them, after the second one,
    // so six double shuffles do the work of twenty.  Lanes 0, 8, 16, 24 end up with the four totals.
    "__device__ __forceinline__ void ami_tally(double4* dst, const double a, const double b, const double c, const double d) {\n"
    "  const unsigned full = 0xffffffffu;\n"
    "  const int lane = threadIdx.x & 31;\n"
    "  const bool h4 = lane & 16, h3 = lane & 8;\n"
    "  const double ra = __shfl_xor_sync(full, h4 ? a : c, 16), rb = __shfl_xor_sync(full, h4 ? b : d, 16);\n"
    "  const double x = (h4 ? c : a) + ra, y = (h4 ? d : b) + rb;\n"
    "  double z = (h3 ? y : x) + __shfl_xor_sync(full, h3 ? x : y, 8);\n"
    "  z += __shfl_xor_sync(full, z, 4);\n"
    "  z += __shfl_xor_sync(full, z, 2);\n"
    "  z += __shfl_xor_sync(full, z, 1);\n"
    "  if ((lane & 7) == 0) reinterpret_cast<double*>(dst)[lane >> 3] = z;\n"
    "}\n";

}  // namespace

// ---------------------------------------------------------------------------------------------
// The translation unit handed to NVRTC.
// ---------------------------------------------------------------------------------------------
static int jit_min_blocks() {
  // __launch_bounds__(AMI_NT, AMI_MINB): the register cap that lets AMI_MINB CTAs share an SM.  (--maxrregcount is
  // ignored for kernels that carry launch bounds, so this is the knob that changes occupancy.)  Default: 12 warps
  // per SM = at most 168 registers per thread.  Measured on B200 (profiles/): the order-6 kernel wants 248
  // registers and runs at 0.77 of the DFMA peak with 8 warps per SM; capped at 168 it reaches 0.92-0.95; at 128
  // registers the spills cost more than the occupancy gives.  At the configured N = 1e5 every cap from 128 to 255
  // registers and 32-, 64- and 128-thread CTAs give the same 11.6-13.4 us (profiles/r02_cfg4_small_batch.md).
  return std::max(1, kJitWarpsPerSmTarget * 32 / kJitBlockThreads);
}

// Split plan: tables whose parts want the full register file and a larger L2 budget for the leaf array
static bool big_table(const FlatTable& ft, const HornerPlan& hp) {
  long long leaf_doubles = (long long)ft.leafF.size();
  for (size_t u = 0; u < ft.leafD.size(); ++u) leaf_doubles += hp.d_is_real[u] ? 1 : 2;
  return leaf_doubles > 250;
}

// Last statement of the register-plan kernels.  An ordered launch (the default) waited for its predecessor before
// touching memory.  An unordered one (AMI_PLAN_UNORDERED: the caller states that it shares no buffer with the
// specialised launches right before it) ran beside them and waits HERE instead, every thread before it exits: the grid
// then completes only after its predecessor has, so whatever is ordered after it in the stream -- an ordered launch,
// a copy, an event -- still comes after everything before it.
static const char* const kUnorderedEnd = "  if (p.unordered) asm volatile(\"griddepcontrol.wait;\" ::: \"memory\");\n";

std::vector<std::string> jit_generate_sources(const FlatTable& ft, const HornerPlan& hp, const JitVariant& var,
                                              JitLayout* layout) {
  const int mode = jit_mode(ft, hp);
  const int n_comp = var.dim * ft.n_int;
  Emitter E;
  const LeafSlots ls = leaf_slots(ft, hp);
  if (layout) {
    *layout = JitLayout();
    layout->mode = mode;
    layout->n_real_den = ls.n_real;
    layout->n_cplx_den = ls.n_cplx;
    layout->n_fermi = ls.n_fermi;
  }
  std::ostringstream head;
  head << kAmiParamsSrc << "\n" << kAmiDeviceSrc << "\n";
  head << "using namespace amidev;\n#define AMI_NT " << kJitBlockThreads << "\n#define AMI_MINB " << jit_min_blocks() << "\n";
  std::ostringstream o;
  o << head.str();
  std::string esig, eargs;
  for (int i = 0; i < ft.n_eps; ++i) {
    if (var.cplx) {
      esig += ", const double e" + std::to_string(i) + "r, const double e" + std::to_string(i) + "i";
      eargs += ", e" + std::to_string(i) + "r, e" + std::to_string(i) + "i";
    } else {
      esig += ", const double e" + std::to_string(i);
      eargs += ", e" + std::to_string(i);
    }
  }
  // A fused kernel: a CTA walks `tiles` consecutive tiles of AMI_NT samples -- one, known at compile time, in
  // ami_jit_fused (the loop disappears); p.tiles in the tally kernel, where a thread adds up its own samples.
  // A warp leaves only as a whole: lanes past the end of the batch stay, compute on zero momenta and store
  // nothing, so that the tally's shuffles always see 32 lanes.
  auto fused_open = [&](const char* name, const char* tiles) {
    o << "extern \"C\" __global__ void __launch_bounds__(AMI_NT, AMI_MINB) " << name << "(const __grid_constant__ AmiBatch p) {\n"
         "  asm volatile(\"griddepcontrol.launch_dependents;\");\n"
         "  if (!p.unordered) asm volatile(\"griddepcontrol.wait;\" ::: \"memory\");\n"
         "  const long long base = blockIdx.x * (long long)AMI_NT * (" << tiles << ") + threadIdx.x;\n"
         "  double4 t4 = make_double4(0.0, 0.0, 0.0, 0.0);\n"
         "#pragma unroll 1\n  for (int u = 0; u < (" << tiles << "); ++u) {\n"
         "  const long long s = base + (long long)u * AMI_NT;\n";
    // a warp past the end of the batch leaves; where the loop has one trip it EXITS there, so that the compiler keeps
    // treating what follows as converged code (uniform datapath, no reconvergence stack: 40 instructions less).  It may
    // skip the end-of-kernel wait of an unordered launch: the grid completes when its LAST thread has left, and the
    // threads that hold a sample (there is at least one) wait
    if (std::string(tiles) == "1") o << "  if (s - (threadIdx.x & 31) >= p.n) return;\n";
    else o << "  if (s - (threadIdx.x & 31) >= p.n) break;\n";
    o << "  const bool valid = s < p.n;\n";
    for (int c = 0; c < n_comp; ++c) o << "  double nk" << c << " = 0.0;\n";
    o << "  if (valid) {\n";
    emit_momenta(o, n_comp, "s", "    ");
    o << "  }\n";
    emit_dispersion(o, ft, var);
    o << "  if (p.e_out && valid) {\n";
    for (int i = 0; i < ft.n_eps; ++i) o << "    p.e_out[" << i << " * p.e_stride + s] = e" << i << ";\n";
    o << "  }\n";
  };
  if (mode == kJitRegister) {
    Sections S;
    if (var.cplx) gen_sections_cplx(ft, hp, ls, kLeafInline, E, S);
    else gen_sections(ft, hp, ls, kLeafInline, E, S);
    o << kTallySrc;
    // what a finished row does with its value: store it, and/or add it to the tally
    o << "#define AMI_EMIT(VR, VI) { \\\n"
         "    const long long row = (long long)(p.b0 + b) * p.n_f_total + (p.f0 + f); \\\n"
         "    const double vr = p.prefactor * (VR), vi = p.prefactor * (VI); \\\n"
         "    if ((!AMI_TALLY || p.out) && valid) __stcs(reinterpret_cast<double2*>(p.out) + row * p.out_row_stride + s, make_double2(vr, vi)); \\\n"
         "    if (AMI_TALLY) { \\\n"
         "      const double wr = valid ? vr : 0.0, wi = valid ? vi : 0.0; \\\n"
         "      if (p.tally_acc) { t4.x += wr; t4.y += wi; t4.z = fma(wr, wr, t4.z); t4.w = fma(wi, wi, t4.w); } \\\n"
         "      else ami_tally(reinterpret_cast<double4*>(p.tally) + row * p.tally_stride + (s >> 5), wr, wi, wr * wr, wi * wi); \\\n"
         "    } }\n";
    const std::string sig = "(const AmiBatch& p, const long long s, const bool valid, double4& t4" + esig + ") {\n";
    // ---- body for one temperature per launch: beta { frequency { } } ----------------------------
    o << "template <bool AMI_TALLY> __device__ __forceinline__ void ami_body" << sig << S.sec[0].str()
      << "#pragma unroll 1\n  for (int b = 0; b < p.n_b; ++b) {\n    const double beta = p.beta[b];\n" << S.sec[1].str()
      << "#pragma unroll 1\n    for (int f = 0; f < p.n_f; ++f) {\n" << S.sec[2].str() << S.sec[3].str() << "    }\n  }\n}\n\n";
    // ---- body for several temperatures: the per-beta values the R part needs are kept in a small
    // per-thread array, then frequency { reciprocals once; beta { R part } } --------------------------
    // R part: per frequency the prefix products P_n of the complex reciprocals (secP), then per temperature
    // Q(root) + sum_n Q(n) P_n: two instructions per term, W temperatures side by side so that consecutive DFMAs share
    // the P_n operand (a DFMA with three changing register operands runs at 2/3 of the rate) and each
    // temperature's sum is a chain of its own.
    if (!hp.mb_prefix) {   // the Horner form of the single-temperature body (small R parts: the prefix products would
                           // cost more than they save)
      o << "template <bool AMI_TALLY> __device__ __forceinline__ void ami_body_mb" << sig << S.sec[0].str();
      o << "  double kept[AMI_K_MAX_BETA][" << std::max<size_t>(S.keep.size(), 1) << "];\n";
      o << "#pragma unroll 1\n  for (int b = 0; b < p.n_b; ++b) {\n    const double beta = p.beta[b];\n" << S.sec[1].str();
      for (size_t i = 0; i < S.keep.size(); ++i) o << "    kept[b][" << i << "] = " << S.keep[i] << ";\n";
      o << "  }\n#pragma unroll 1\n  for (int f = 0; f < p.n_f; ++f) {\n" << S.sec[2].str()
        << "#pragma unroll 1\n    for (int b = 0; b < p.n_b; ++b) {\n";
      for (size_t i = 0; i < S.keep.size(); ++i) o << "      const double " << S.keep[i] << " = kept[b][" << i << "];\n";
      o << S.sec[3].str() << "    }\n  }\n}\n\n";
    } else {
    o << "template <bool AMI_TALLY> __device__ __forceinline__ void ami_body_mb" << sig << S.sec[0].str();
    o << "  double kept[" << std::max<size_t>(S.keep.size(), 1) << "][AMI_K_MAX_BETA];\n";
    o << "#pragma unroll 1\n  for (int b = 0; b < p.n_b; ++b) {\n    const double beta = p.beta[b];\n" << S.sec[1].str();
    for (size_t i = 0; i < S.keep.size(); ++i) o << "    kept[" << i << "][b] = " << S.keep[i] << ";\n";
    o << "  }\n#pragma unroll 1\n  for (int f = 0; f < p.n_f; ++f) {\n" << S.sec[2].str() << S.secP.str();
    auto block = [&](int W) {
      const int A = std::max(1, 4 / W);       // partial sums per temperature: at least 8 chains in flight
      std::ostringstream q;
      q << "      {\n";
      auto kname = [](int w, int keep) { return "k" + std::to_string(w) + "_" + std::to_string(keep); };
      for (int w = 0; w < W; ++w) {
        std::set<int> loaded;
        for (const Sections::QRef& r : S.qrefs)
          for (int keep : {r.keep, r.keep_im})
            if (keep >= 0 && loaded.insert(keep).second)
              q << "        const double " << kname(w, keep) << " = kept[" << keep << "][b0 + " << w << "];\n";
      }
      std::vector<std::vector<char>> init(W, std::vector<char>(A, 0));
      for (int w = 0; w < W; ++w)
        for (int a = 0; a < A; ++a) q << "        double vr" << w << "_" << a << ", vi" << w << "_" << a << ";\n";
      int j = 0;
      for (const Sections::QRef& r : S.qrefs) {
        if (r.pr.empty()) continue;
        const int a = j++ % A;
        for (int w = 0; w < W; ++w) {
          const std::string kr = kname(w, r.keep), ki = r.keep_im >= 0 ? kname(w, r.keep_im) : "";
          const std::string vr = "vr" + std::to_string(w) + "_" + std::to_string(a), vi = "vi" + std::to_string(w) + "_" + std::to_string(a);
          if (!init[w][a]) {
            q << "        " << vr << " = " << kr << " * " << r.pr << "; " << vi << " = " << kr << " * " << r.pi << ";\n";
            init[w][a] = 1;
          } else {
            q << "        " << vr << " = fma(" << kr << ", " << r.pr << ", " << vr << "); " << vi << " = fma(" << kr << ", " << r.pi
              << ", " << vi << ");\n";
          }
          if (!ki.empty())   // complex Q: (kr + i ki)(Pr + i Pi)
            q << "        " << vr << " = fma(-" << ki << ", " << r.pi << ", " << vr << "); " << vi << " = fma(" << ki << ", " << r.pr
              << ", " << vi << ");\n";
        }
      }
      for (int w = 0; w < W; ++w) {
        std::string re, im;
        for (int a = 0; a < A; ++a) {
          if (!init[w][a]) continue;
          re += (re.empty() ? "" : " + ") + std::string("vr") + std::to_string(w) + "_" + std::to_string(a);
          im += (im.empty() ? "" : " + ") + std::string("vi") + std::to_string(w) + "_" + std::to_string(a);
        }
        if (A == 4 && init[0][3]) {   // pairwise
          re = "(vr" + std::to_string(w) + "_0 + vr" + std::to_string(w) + "_1) + (vr" + std::to_string(w) + "_2 + vr" + std::to_string(w) + "_3)";
          im = "(vi" + std::to_string(w) + "_0 + vi" + std::to_string(w) + "_1) + (vi" + std::to_string(w) + "_2 + vi" + std::to_string(w) + "_3)";
        }
        for (const Sections::QRef& r : S.qrefs) {
          if (!r.pr.empty()) continue;      // the root's own Q
          re = re.empty() ? kname(w, r.keep) : "(" + re + ") + " + kname(w, r.keep);
          if (r.keep_im >= 0) im = im.empty() ? kname(w, r.keep_im) : "(" + im + ") + " + kname(w, r.keep_im);
        }
        if (re.empty()) re = "0.0";
        if (im.empty()) im = "0.0";
        q << "        { const int b = b0 + " << w << "; AMI_EMIT(" << re << ", " << im << "); }\n";
      }
      q << "      }\n";
      return q.str();
    };
    o << "    int b0 = 0;\n#pragma unroll 1\n    for (; b0 + 4 <= p.n_b; b0 += 4)\n" << block(4)
      << "    if (b0 + 2 <= p.n_b) {\n" << block(2) << "      b0 += 2;\n    }\n"
      << "    if (b0 < p.n_b)\n" << block(1) << "  }\n}\n\n";
    }
    const std::string call_args = "(p, s, valid, t4" + eargs + ");\n";
    // @T@ = <false> / <true>: without / with the fused tally (a compile-time switch: the reductions cost the kernels
    // that do not tally nothing)
    const std::string call = "  if (p.n_b == 1) ami_body@T@" + call_args + "  else ami_body_mb@T@" + call_args;
    auto subst = [](std::string t, const std::string& targ) {
      for (size_t at = 0; (at = t.find("@T@", at)) != std::string::npos; at += targ.size()) t.replace(at, 3, targ);
      return t;
    };
    // ---- kernel 1: energies from memory ---------------------------------------------------------
    o << "extern \"C\" __global__ void __launch_bounds__(AMI_NT, AMI_MINB) ami_jit_eval(const __grid_constant__ AmiBatch p) {\n"
         "  asm volatile(\"griddepcontrol.launch_dependents;\");\n"
         "  if (!p.unordered) asm volatile(\"griddepcontrol.wait;\" ::: \"memory\");\n"
         "  const long long s = blockIdx.x * (long long)AMI_NT + threadIdx.x;   // the grid covers the batch\n"
         "  if (s >= p.n) return;       // (an unordered launch: the threads that hold a sample wait at the end)\n"
         "  const bool valid = true;\n"
         "  double4 t4 = make_double4(0.0, 0.0, 0.0, 0.0);\n"
         "  {\n";
    for (int i = 0; i < ft.n_eps; ++i) {
      if (var.cplx)
        o << "  const double e" << i << "r = p.e[2 * (" << i << " * p.e_stride + s)], e" << i << "i = p.e[2 * (" << i
          << " * p.e_stride + s) + 1];\n";
      else
        o << "  const double e" << i << " = p.e[" << i << " * p.e_stride + s];\n";
    }
    o << subst(call, "<false>") << "  }\n" << kUnorderedEnd << "}\n\n";
    if (var.cplx) return std::vector<std::string>(1, o.str());   // momenta give real energies: no fused kernels
    // ---- kernels 2, 3: momenta from memory or drawn in place, dispersion inline; without / with the tally ----
    for (int tally = 0; tally < 2; ++tally) {
      fused_open(tally ? "ami_jit_fused_tally" : "ami_jit_fused", tally ? "p.tiles" : "1");
      o << subst(call, tally ? "<true>" : "<false>") << "  }\n";
      if (tally)   // single-row tally: one partial per warp of the grid, formed from the threads' own sums
        o << "  if (p.tally_acc) ami_tally(reinterpret_cast<double4*>(p.tally) + (long long)(p.b0 * p.n_f_total + p.f0) * "
             "p.tally_stride + blockIdx.x * (AMI_NT / 32) + (threadIdx.x >> 5), t4.x, t4.y, t4.z, t4.w);\n";
      o << kUnorderedEnd << "}\n\n";
    }
    return std::vector<std::string>(1, o.str());
  }
  // ---- split plan ----------------------------------------------------------------------------------
  // Module 0: the leaf kernels and the kernel that adds the parts.  Modules 1..M: the parts, a few per module, so
  // that NVRTC compiles them side by side on the host's cores (a part is 1-2 k statements; one translation unit
  // with all of an order-8 table's parts takes 20 s, eight of them 3-5 s).
  // complex energies: every leaf is two doubles (re at its slot, im at the next), and a complex sum costs three to
  // four times the instructions of a real one, so the parts are cut smaller
  LeafSlots lsc = ls;
  if (var.cplx) {
    for (int& r : lsc.ridx)
      if (r >= 0) r *= 2;
    lsc.n_real = 2 * ls.n_real;
    lsc.n_fermi = 2 * ls.n_fermi;
    if (layout) { layout->n_real_den = lsc.n_real; layout->n_fermi = lsc.n_fermi; }
  }
  const std::vector<std::vector<int>> parts = partition_groups(hp, var.cplx ? std::max(100LL, split_budget() / 3) : split_budget());
  const int n_parts = (int)parts.size();
  const int n_mod = std::min(n_parts, 8);
  if (layout) {
    layout->n_parts = n_parts;
    layout->part0.clear();
    for (int j = 0; j <= n_mod; ++j) layout->part0.push_back((int)((long long)n_parts * j / n_mod));
  }
  std::vector<std::string> sources;
  // Layout of the leaf array: one record per tile of AMI_NT samples, [tile][slot][AMI_NT] (p.leaf_stride = doubles
  // per record), so that inside a part every leaf of a thread sits at a COMPILE-TIME offset from one of three bases
  // (sample; + temperature; + frequency): every leaf load is LDG [R + imm], no address arithmetic at all.
  o << "#define AMI_LS(i, v) Ls[(i) * AMI_NT] = (v)\n#define AMI_LSF(u, v) LsF[(u) * AMI_NT] = (v)\n"
       "#define AMI_LSC(j, v) LsC[(j) * AMI_NT] = (v)\n";
  {   // leaf kernels: everything that depends on one energy combination, written once per sample
    Sections S;
    if (var.cplx) gen_sections_cplx(ft, hp, lsc, kLeafStore, E, S);
    else gen_sections(ft, hp, ls, kLeafStore, E, S);
    o << "__device__ __forceinline__ void ami_leaf_body(const AmiBatch& p, const long long s" << esig << ") {\n"
      << "  const int CB = " << lsc.n_real << " + p.n_b * " << lsc.n_fermi << ";\n"
      << "  double* __restrict__ Ls = p.leaves + (s / AMI_NT) * p.leaf_stride + (s % AMI_NT);\n" << S.sec[0].str()
      << "#pragma unroll 1\n  for (int b = 0; b < p.n_b; ++b) {\n    const double beta = p.beta[b];\n"
      << "    double* __restrict__ LsF = Ls + (" << lsc.n_real << " + b * " << lsc.n_fermi << ") * AMI_NT;\n" << S.sec[1].str() << "  }\n"
      << "#pragma unroll 1\n  for (int f = 0; f < p.n_f; ++f) {\n"
      << "    double* __restrict__ LsC = Ls + (CB + 2 * f * " << ls.n_cplx << ") * AMI_NT;\n" << S.sec[2].str() << "  }\n}\n\n";
    o << "extern \"C\" __global__ void __launch_bounds__(AMI_NT, AMI_MINB) ami_split_leaves_eval(const __grid_constant__ AmiBatch p) {\n"
         "  const long long s = blockIdx.x * (long long)AMI_NT + threadIdx.x;\n  if (s >= p.n) return;\n";
    for (int i = 0; i < ft.n_eps; ++i) {
      if (var.cplx)
        o << "  const double e" << i << "r = p.e[2 * (" << i << " * p.e_stride + s)], e" << i << "i = p.e[2 * (" << i
          << " * p.e_stride + s) + 1];\n";
      else
        o << "  const double e" << i << " = p.e[" << i << " * p.e_stride + s];\n";
    }
    o << "  ami_leaf_body(p, s" << eargs << ");\n}\n\n";
    if (!var.cplx) {   // momenta give real energies: no fused leaf kernel for complex ones
    o << "extern \"C\" __global__ void __launch_bounds__(AMI_NT, AMI_MINB) ami_split_leaves_fused(const __grid_constant__ AmiBatch p) {\n"
         "  const long long s = blockIdx.x * (long long)AMI_NT + threadIdx.x;\n  if (s >= p.n) return;\n";
    for (int c = 0; c < n_comp; ++c) o << "  double nk" << c << ";\n";
    emit_momenta(o, n_comp, "s", "  ");
    emit_dispersion(o, ft, var);
    o << "  if (p.e_out) {\n";
    for (int i = 0; i < ft.n_eps; ++i) o << "    p.e_out[" << i << " * p.e_stride + s] = e" << i << ";\n";
    o << "  }\n  ami_leaf_body(p, s" << eargs << ");\n}\n\n";
    }
  }
  // the parts' partial results, added in the order of the parts (fixed: deterministic), times the prefactor
  // (launched as a programmatic dependent of the last parts kernel: see ami_split_parts)
  o << "extern \"C\" __global__ void __launch_bounds__(256) ami_split_combine(const __grid_constant__ AmiBatch p) {\n"
       "  asm volatile(\"griddepcontrol.wait;\" ::: \"memory\");\n"
       "  const long long s = blockIdx.x * 256ll + threadIdx.x;\n  if (s >= p.n) return;\n"
       "  const int lr = blockIdx.y, b = lr / p.n_f, f = lr - b * p.n_f;\n"
       "  const double2* P = reinterpret_cast<const double2*>(p.partial) + (long long)lr * p.partial_stride + s;\n"
       "  double vr = 0.0, vi = 0.0;\n"
       "  for (int k = 0; k < p.n_parts; ++k) {\n"
       "    const double2 v = P[(long long)k * p.n_b * p.n_f * p.partial_stride];\n    vr += v.x; vi += v.y;\n  }\n"
       "  const long long row = (long long)(p.b0 + b) * p.n_f_total + (p.f0 + f);\n"
       "  __stcs(reinterpret_cast<double2*>(p.out) + row * p.out_row_stride + s, make_double2(p.prefactor * vr, p.prefactor * vi));\n"
       "}\n";
  sources.push_back(o.str());
  // parts: leaves are read where they are used (AMI_L: reciprocal denominators, one product each; AMI_LF: Fermi/Bose
  // values, loaded once per chunk of groups); the prefactor is applied when the parts are added up
  for (int mj = 0; mj < n_mod; ++mj) {
  const int pa = (int)((long long)n_parts * mj / n_mod), pb = (int)((long long)n_parts * (mj + 1) / n_mod);
  o.str("");
  o << head.str();
  // Register cap of the parts: the larger the table, the more leaves a part keeps alive.  Measured (B200, N = 2e5,
  // ms per step at 168 / 255 registers): order 8 (303 leaf doubles) 1.05 / 0.95, order 7 (205) 0.286 / 0.310.
  if (big_table(ft, hp)) o << "#undef AMI_MINB\n#define AMI_MINB 4\n";
  o << "#define AMI_L(i) __ldg(Lp + (i) * AMI_NT)\n#define AMI_LF(u) __ldg(LpF + (u) * AMI_NT)\n"
       "#define AMI_LC(j) __ldg(LpC + (j) * AMI_NT)\n"
       "#define AMI_EMIT(VR, VI) Pp[(long long)(b * n_f + f) * ps] = make_double2((VR), (VI))\n";
  for (int pi = pa; pi < pb; ++pi) {
    const HornerPlan sub = make_sub_plan(hp, parts[pi]);
    Sections S;
    if (var.cplx) gen_sections_cplx(ft, sub, lsc, kLeafLoad, E, S);
    else gen_sections(ft, sub, ls, kLeafLoad, E, S);
    o << "__device__ __noinline__ void ami_part_" << pi
      << "(const double* __restrict__ Lp, double2* __restrict__ Pp, const long long ps, const int n_b, const int n_f) {\n"
      << "  const int CB = " << lsc.n_real << " + n_b * " << lsc.n_fermi << ";\n" << S.sec[0].str()
      << "#pragma unroll 1\n  for (int b = 0; b < n_b; ++b) {\n"
      << "    const double* __restrict__ LpF = Lp + (" << lsc.n_real << " + b * " << lsc.n_fermi << ") * AMI_NT;\n" << S.sec[1].str()
      << "#pragma unroll 1\n    for (int f = 0; f < n_f; ++f) {\n"
      << "      const double* __restrict__ LpC = Lp + (CB + 2 * f * " << ls.n_cplx << ") * AMI_NT;\n"
      << S.sec[2].str() << S.sec[3].str() << "    }\n  }\n";
    // the macros that name this part's denominators end with it
    for (size_t u = 0; u < ft.leafD.size(); ++u) o << "#undef Dr" << u << "\n#undef Di" << u << "\n";
    if (var.cplx)
      for (size_t u = 0; u < ft.leafF.size(); ++u) o << "#undef Fr" << u << "\n#undef Fi" << u << "\n";
    o << "}\n\n";
  }
  // grid.y = part within this module; p.part0 = index of the module's first part.
  // The parts kernels of a chunk are independent of one another (each reads the leaf array and writes its own
  // partial results), so they are launched as a chain of programmatic dependents: launch_dependents at the top lets
  // the next kernel of the chain start as soon as every CTA of this one is running -- the tail of one launch
  // overlaps the head of the next instead of leaving the SMs half empty between them.  The leaf kernel never
  // triggers early, so the first parts kernel (and with it every later one) starts after the leaves are complete.
  // The wait at the END makes this grid complete only after its predecessor has: when the combine kernel's wait
  // returns, every parts kernel of the chunk is done.
  o << "extern \"C\" __global__ void __launch_bounds__(AMI_NT, AMI_MINB) ami_split_parts(const __grid_constant__ AmiBatch p) {\n"
       "  asm volatile(\"griddepcontrol.launch_dependents;\");\n"
       "  const long long s = blockIdx.x * (long long)AMI_NT + threadIdx.x;\n"
       "  if (s >= p.n) { asm volatile(\"griddepcontrol.wait;\" ::: \"memory\"); return; }\n"
       "  const double* Lp = p.leaves + blockIdx.x * p.leaf_stride + threadIdx.x;\n"
       "  double2* Pp = reinterpret_cast<double2*>(p.partial) + (long long)(p.part0 + blockIdx.y) * p.n_b * p.n_f * p.partial_stride + s;\n"
       "  switch (blockIdx.y) {\n";
  for (int pi = pa; pi < pb; ++pi)
    o << "    case " << pi - pa << ": ami_part_" << pi << "(Lp, Pp, p.partial_stride, p.n_b, p.n_f); break;\n";
  o << "  }\n  asm volatile(\"griddepcontrol.wait;\" ::: \"memory\");\n}\n";
  sources.push_back(o.str());
  }
  return sources;
}

int jit_mode(const FlatTable& ft, const HornerPlan& hp) {
  if (const char* off = getenv("AMI_DISABLE_JIT"))
    if (off[0] == '1') return kJitNone;
  long long leaf_doubles = (long long)ft.leafF.size();
  for (size_t u = 0; u < ft.leafD.size(); ++u) leaf_doubles += hp.d_is_real[u] ? 1 : 2;
  const long long edges = hp.n_fnodes + 4 * hp.n_dnodes;
  if (leaf_doubles <= 160 && edges <= 4000) return kJitRegister;
  if (edges <= 2000000) return kJitSplit;
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
  int (*Version)(int*, int*) = nullptr;
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
    AMI_SYM(GetCUBINSize); AMI_SYM(GetCUBIN); AMI_SYM(DestroyProgram); AMI_SYM(GetErrorString); AMI_SYM(Version);
#undef AMI_SYM
    n.ok = n.CreateProgram && n.CompileProgram && n.GetProgramLogSize && n.GetProgramLog && n.GetCUBINSize &&
           n.GetCUBIN && n.DestroyProgram;
  });
  return n;
}

// ---- on-disk cache of compiled kernels -------------------------------------------------------------
// A diagrammatic Monte-Carlo user evaluates thousands of diagrams; NVRTC needs 0.6-1 s per diagram, the
// paper's construct "microseconds".  The cubin of a generated source is therefore kept in
//   $AMI_JIT_CACHE, else $XDG_CACHE_HOME/ami_b200, else $HOME/.cache/ami_b200
// under the 128-bit FNV-1a hash of (source text, NVRTC version, target architecture); AMI_JIT_CACHE=0 turns
// the cache off.  Files are written to a temporary name and renamed, so concurrent processes are safe.
const char* kJitArch = "sm_100a";

std::string cache_dir() {
  if (const char* e = getenv("AMI_JIT_CACHE")) {
    if (!strcmp(e, "0") || !*e) return "";
    return e;
  }
  if (const char* x = getenv("XDG_CACHE_HOME"))
    if (*x) return std::string(x) + "/ami_b200";
  if (const char* h = getenv("HOME"))
    if (*h) return std::string(h) + "/.cache/ami_b200";
  return "";
}

std::string cache_key(const std::string& src) {
  int major = 0, minor = 0;
  if (nvrtc().Version) nvrtc().Version(&major, &minor);
  const std::string salt = std::string("|nvrtc ") + std::to_string(major) + "." + std::to_string(minor) + "|" + kJitArch;
  unsigned long long h1 = 0xcbf29ce484222325ull, h2 = 0x84222325cbf29ce4ull;
  auto feed = [&](const std::string& t) {
    for (unsigned char c : t) {
      h1 = (h1 ^ c) * 0x100000001b3ull;
      h2 = (h2 ^ (unsigned char)(c + 0x5b)) * 0x100000001b3ull;
      h2 ^= h2 >> 29;
    }
  };
  feed(src);
  feed(salt);
  char buf[40];
  snprintf(buf, sizeof buf, "%016llx%016llx", h1, h2);
  return buf;
}

void make_dirs(const std::string& path) {
  for (size_t i = 1; i <= path.size(); ++i)
    if (i == path.size() || path[i] == '/') mkdir(path.substr(0, i).c_str(), 0755);
}

bool cache_read(const std::string& file, std::vector<char>& cubin) {
  FILE* f = fopen(file.c_str(), "rb");
  if (!f) return false;
  fseek(f, 0, SEEK_END);
  const long n = ftell(f);
  fseek(f, 0, SEEK_SET);
  bool ok = n > 4;
  if (ok) {
    cubin.resize((size_t)n);
    ok = fread(cubin.data(), 1, (size_t)n, f) == (size_t)n && !memcmp(cubin.data(), "\x7f" "ELF", 4);
  }
  fclose(f);
  return ok;
}

void cache_write(const std::string& dir, const std::string& file, const std::vector<char>& cubin) {
  make_dirs(dir);
  const std::string tmp = file + ".tmp" + std::to_string((long)getpid());
  FILE* f = fopen(tmp.c_str(), "wb");
  if (!f) return;
  const bool ok = fwrite(cubin.data(), 1, cubin.size(), f) == cubin.size();
  fclose(f);
  if (!ok || rename(tmp.c_str(), file.c_str()) != 0) remove(tmp.c_str());
}

}  // namespace

int jit_compile(const std::string& src, std::vector<char>& cubin, std::string& log, bool use_cache, bool* cache_hit) {
  Nvrtc& n = nvrtc();
  if (cache_hit) *cache_hit = false;
  if (!n.ok) { log = "NVRTC library not found (set AMI_NVRTC_PATH)"; return AMI_EUNSUPPORTED; }
  const std::string dir = use_cache ? cache_dir() : "";
  const std::string file = dir.empty() ? "" : dir + "/" + cache_key(src) + ".cubin";
  if (!file.empty() && cache_read(file, cubin)) {
    if (cache_hit) *cache_hit = true;
    log = "cubin from " + file;
    return AMI_OK;
  }
  void* prog = nullptr;
  if (n.CreateProgram(&prog, src.c_str(), "ami_jit.cu", 0, nullptr, nullptr) != 0) {
    log = "nvrtcCreateProgram failed";
    return AMI_EINVAL;
  }
  const std::string arch = std::string("--gpu-architecture=") + kJitArch;
  std::vector<const char*> opts = {arch.c_str(), "--std=c++17", "-lineinfo", "--ptxas-options=-v", "-default-device"};
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
  if (cs && !file.empty()) cache_write(dir, file, cubin);
  return cs ? AMI_OK : AMI_EINVAL;
}

// ---------------------------------------------------------------------------------------------
// module loading and launch through driver entry points obtained from the runtime (the library
// does not link against libcuda, so that it loads on a machine without a driver)
// ---------------------------------------------------------------------------------------------
struct JitModule {
  bool tried = false;
  int status = AMI_EUNSUPPORTED;
  std::string log;
  std::vector<CUmodule> mods;
  CUfunction fn_eval = nullptr, fn_fused = nullptr, fn_fused_tally = nullptr;                 // register plan
  CUfunction fn_leaves_eval = nullptr, fn_leaves_fused = nullptr, fn_combine = nullptr;       // split plan, module 0
  std::vector<CUfunction> fn_parts;                                                           // split plan, modules 1..M
  JitLayout layout;
  double compile_ms = 0.0;
  int cache_hit = 0;
};

struct JitState {
  std::mutex mu;
  std::map<int, JitModule> variants;   // by JitVariant::key()
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
  });
  return d;
}

std::mutex g_state_mu;   // guards creation of tab->jit

const JitModule* module_of(const ami_table* tab, const JitVariant& var) {
  JitState* js = tab->jit;
  if (!js) return nullptr;
  std::lock_guard<std::mutex> lk(js->mu);
  auto it = js->variants.find(var.key());
  return it == js->variants.end() ? nullptr : &it->second;   // map nodes are stable
}

}  // namespace

int jit_prepare(ami_table* tab, const JitVariant& var, std::string& err) {
  {
    std::lock_guard<std::mutex> lk(g_state_mu);
    if (!tab->jit) tab->jit = new JitState;
  }
  JitState& js = *tab->jit;
  std::lock_guard<std::mutex> lk(js.mu);
  JitModule& m = js.variants[var.key()];
  if (m.tried) { err = m.log; return m.status; }
  m.tried = true;
  auto fail = [&](int code, const std::string& why) {
    m.log = why;
    m.status = code;
    err = why;
    return code;
  };
  if (tab->dev.device < 0) return fail(AMI_ECUDA, "table has no device copy");
  if (var.dim < 1 || var.dim > 3 || (var.band != AMI_BAND_TIGHT_BINDING && var.band != AMI_BAND_FREE))
    return fail(AMI_EINVAL, "bad lattice for the specialised kernels");
  if (!jit_eligible(tab->flat, tab->horner)) return fail(AMI_EUNSUPPORTED, "table outside the limits of the specialised kernels");
  const auto t0 = std::chrono::steady_clock::now();
  const std::vector<std::string> srcs = jit_generate_sources(tab->flat, tab->horner, var, &m.layout);
  // the modules of a split plan are compiled side by side (NVRTC is thread safe across programs)
  std::vector<std::vector<char>> cubins(srcs.size());
  std::vector<std::string> logs(srcs.size());
  std::vector<int> codes(srcs.size(), AMI_OK);
  std::vector<char> hits(srcs.size(), 0);
  {
    const size_t n_thr = std::max<size_t>(1, std::min<size_t>(srcs.size(), std::thread::hardware_concurrency()));
    std::atomic<size_t> next{0};
    auto work = [&] {
      for (size_t i; (i = next.fetch_add(1)) < srcs.size();) {
        bool hit = false;
        codes[i] = jit_compile(srcs[i], cubins[i], logs[i], true, &hit);
        hits[i] = hit;
      }
    };
    std::vector<std::thread> pool;
    for (size_t t = 1; t < n_thr; ++t) pool.emplace_back(work);
    work();
    for (std::thread& t : pool) t.join();
  }
  m.cache_hit = 1;
  for (size_t i = 0; i < srcs.size(); ++i) {
    m.log += logs[i] + "\n";
    if (!hits[i]) m.cache_hit = 0;
  }
  for (size_t i = 0; i < srcs.size(); ++i)
    if (codes[i] != AMI_OK) { m.status = codes[i]; err = m.log; return m.status; }
  Driver& d = driver();
  if (!d.ok) return fail(AMI_ECUDA, "CUDA driver entry points unavailable");
  cudaSetDevice(tab->dev.device);
  cudaFree(nullptr);   // makes the primary context current
  CUresult rc = CUDA_SUCCESS;
  m.mods.assign(srcs.size(), nullptr);
  for (size_t i = 0; i < srcs.size() && rc == CUDA_SUCCESS; ++i) rc = d.ModuleLoadData(&m.mods[i], cubins[i].data());
  auto get = [&](CUfunction* fn, size_t mod, const char* name) {
    if (rc == CUDA_SUCCESS) rc = d.ModuleGetFunction(fn, m.mods[mod], name);
  };
  if (m.layout.mode == kJitRegister) {
    get(&m.fn_eval, 0, "ami_jit_eval");
    if (!var.cplx) {
      get(&m.fn_fused, 0, "ami_jit_fused");
      get(&m.fn_fused_tally, 0, "ami_jit_fused_tally");
    }
  } else {
    get(&m.fn_leaves_eval, 0, "ami_split_leaves_eval");
    if (!var.cplx) get(&m.fn_leaves_fused, 0, "ami_split_leaves_fused");
    get(&m.fn_combine, 0, "ami_split_combine");
    m.fn_parts.assign(srcs.size() - 1, nullptr);
    for (size_t i = 1; i < srcs.size(); ++i) get(&m.fn_parts[i - 1], i, "ami_split_parts");
  }
  if (rc != CUDA_SUCCESS) {
    const char* msg = nullptr;
    d.GetErrorString(rc, &msg);
    return fail(AMI_ECUDA, std::string("loading the specialised kernels failed: ") + (msg ? msg : "?"));
  }
  m.compile_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  m.status = AMI_OK;
  return AMI_OK;
}

namespace {

// Programmatic dependent launch: the register-plan kernels begin with griddepcontrol.launch_dependents + .wait,
// so the NEXT specialised kernel in the stream may be scheduled while this one drains and starts the moment it
// has completed (stream order is kept: nothing is read or written before the wait).
CUresult launch(CUfunction fn, unsigned gx, unsigned gy, unsigned block, AmiBatch& batch, cudaStream_t st, bool pdl) {
  void* args[] = {&batch};
  if (!fn) return CUDA_ERROR_INVALID_VALUE;
  if (pdl && driver().LaunchKernelEx) {
    CUlaunchAttribute attr;
    memset(&attr, 0, sizeof attr);
    attr.id = CU_LAUNCH_ATTRIBUTE_PROGRAMMATIC_STREAM_SERIALIZATION;
    attr.value.programmaticStreamSerializationAllowed = 1;
    CUlaunchConfig cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDimX = gx; cfg.gridDimY = gy; cfg.gridDimZ = 1;
    cfg.blockDimX = block; cfg.blockDimY = 1; cfg.blockDimZ = 1;
    cfg.sharedMemBytes = 0; cfg.hStream = (CUstream)st; cfg.attrs = &attr; cfg.numAttrs = 1;
    return driver().LaunchKernelEx(&cfg, fn, args, nullptr);
  }
  return driver().LaunchKernel(fn, gx, gy, 1, block, 1, 1, 0, (CUstream)st, args, nullptr);
}

}  // namespace

cudaError_t jit_launch(const ami_table* tab, const JitVariant& var, bool fused, const AmiBatch& b, cudaStream_t st,
                       int* launches, long long* tally_slots) {
  const JitModule* m = module_of(tab, var);
  if (tally_slots) *tally_slots = 0;
  if (!m || m->status != AMI_OK) return cudaErrorInvalidDeviceFunction;
  if (b.n == 0) return cudaSuccess;
  const unsigned block = kJitBlockThreads;
  if (m->layout.mode == kJitRegister) {
    // One CTA per `block` samples: the hardware CTA scheduler balances the SMs better than a persistent grid
    // with a static stride does (measured: persistent + L2 prefetch of the next sample was 12 % slower on cfg3
    // and 5 % slower on cfg4, profiles/r01_final_kernels.md).
    AmiBatch copy = b;
    copy.tiles = 1;
    copy.tally_acc = 0;
    if (fused && b.tally && (long long)b.n_b * b.n_f == 1 && b.n >= (long long)kJitTallyTiles * block * 148 * 8) {
      copy.tiles = kJitTallyTiles;     // every thread adds kJitTallyTiles samples itself, then one warp sum
      copy.tally_acc = 1;
    }
    const long long per_cta = (long long)block * copy.tiles;
    const unsigned grid = (unsigned)((b.n + per_cta - 1) / per_cta);
    if (tally_slots && b.tally) *tally_slots = copy.tally_acc ? (long long)grid * (block / 32) : (b.n + 31) / 32;
    CUfunction fn = fused ? (b.tally ? m->fn_fused_tally : m->fn_fused) : m->fn_eval;
    if (launch(fn, grid, 1, block, copy, st, true) != CUDA_SUCCESS) return cudaErrorLaunchFailure;
    if (launches) ++*launches;
    return cudaSuccess;
  }
  // split plan: leaves -> parts -> combine per chunk of samples; the chunk is sized so that the leaf array and the
  // parts' partial results (stream-ordered allocations) stay in L2 between the kernels
  if (b.tally || !b.out || (var.cplx && fused)) return cudaErrorInvalidValue;
  const JitLayout& lay = m->layout;
  const long long rows = (long long)b.n_b * b.n_f;
  const long long slots = lay.n_real_den + (long long)b.n_b * lay.n_fermi + 2LL * b.n_f * lay.n_cplx_den;
  const long long per_sample = slots * 8 + rows * lay.n_parts * 16;
  // 64 MB of leaves + partials per chunk (96 MB for the largest tables: fewer, fuller launches; measured 1.05 -> 0.97 ms
  // per 2e5 order-8 samples, while order 7 loses 3 %): L2 holds 126 MB
  const long long budget = (big_table(tab->flat, tab->horner) ? 96LL : 64LL) << 20;
  long long chunk = std::max<long long>(block, (budget / std::max<long long>(per_sample, 1)) / 256 * 256);
  chunk = std::min(chunk, (b.n + 255) / 256 * 256);
  double *leaves = nullptr, *partial = nullptr;
  cudaError_t crc = scratch_alloc((void**)&leaves, (size_t)(slots * 8 * chunk), st);
  if (crc != cudaSuccess) return crc;
  crc = scratch_alloc((void**)&partial, (size_t)(rows * lay.n_parts * 16 * chunk), st);
  if (crc != cudaSuccess) { cudaFreeAsync(leaves, st); return crc; }
  bool ok = true;
  for (long long c0 = 0; c0 < b.n && ok; c0 += chunk) {
    AmiBatch part = b;
    part.n = std::min(chunk, b.n - c0);
    if (part.e) part.e += var.cplx ? 2 * c0 : c0;   // SoA rows keep their stride (complex: two doubles per sample)
    if (part.e_out) part.e_out += c0;
    if (part.k) part.k += c0 * b.k_stride_sample;
    part.first_sample += c0;
    part.out += 2 * c0;
    part.leaves = leaves; part.leaf_stride = slots * block;      // doubles per tile record [slot][block]
    part.partial = partial; part.partial_stride = chunk;
    part.n_parts = lay.n_parts;
    const unsigned gx = (unsigned)((part.n + block - 1) / block);
    ok = launch(fused ? m->fn_leaves_fused : m->fn_leaves_eval, gx, 1, block, part, st, false) == CUDA_SUCCESS;
    for (size_t j = 0; j < m->fn_parts.size() && ok; ++j) {
      part.part0 = lay.part0[j];
      ok = launch(m->fn_parts[j], gx, (unsigned)(lay.part0[j + 1] - lay.part0[j]), block, part, st, true) == CUDA_SUCCESS;
    }
    ok = ok && launch(m->fn_combine, (unsigned)((part.n + 255) / 256), (unsigned)rows, 256, part, st, true) == CUDA_SUCCESS;
    if (ok && launches) *launches += 2 + (int)m->fn_parts.size();
  }
  cudaFreeAsync(partial, st);
  crc = cudaFreeAsync(leaves, st);
  return ok ? crc : cudaErrorLaunchFailure;
}

int jit_status(const ami_table* tab) {
  const JitModule* m = module_of(tab, JitVariant());
  if (!m || !m->tried) return 1;
  return m->status;
}

bool jit_fused_tally_ok(const ami_table* tab) {
  const JitModule* m = module_of(tab, JitVariant());
  return m && m->status == AMI_OK && m->layout.mode == kJitRegister;
}

double jit_last_compile_ms(const ami_table* tab, int* cache_hit) {
  const JitModule* m = module_of(tab, JitVariant());
  if (cache_hit) *cache_hit = m ? m->cache_hit : 0;
  return m ? m->compile_ms : 0.0;
}

void jit_destroy(ami_table* tab) {
  if (!tab->jit) return;
  for (auto& kv : tab->jit->variants)
    for (CUmodule mod : kv.second.mods)
      if (mod && driver().ok) driver().ModuleUnload(mod);
  delete tab->jit;
  tab->jit = nullptr;
}

}  // namespace ami
