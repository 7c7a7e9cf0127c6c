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

// Q_k polynomials of f^{(k)} = beta^k f g Q_k(f):  Q_1 = -1, Q_{k+1} = (2f-1) Q_k - (f - f^2) Q_k'
// (from f' = -beta f g, g' = beta f g, g = 1 - f; reading P11).  Ascending powers of f.
std::vector<double> deriv_poly(int k) {
  std::vector<double> q(1, -1.0);
  for (int j = 1; j < k; ++j) {
    std::vector<double> r(q.size() + 1, 0.0);
    for (size_t i = 0; i < q.size(); ++i) {
      r[i + 1] += 2.0 * q[i];
      r[i] -= q[i];
      if (i >= 1) {
        r[i] -= (double)i * q[i];        // -f   * (i q_i f^{i-1})
        r[i + 1] += (double)i * q[i];    // +f^2 * (i q_i f^{i-1})
      }
    }
    q.swap(r);
  }
  return q;
}

namespace {

// Inserts `seq` into the trie `nodes` (nodes[0] = root) and returns the node it ends at.
int trie_insert(std::vector<HNode>& nodes, const std::vector<int>& seq) {
  int cur = 0;
  for (int leaf : seq) {
    int nxt = -1;
    for (int c : nodes[cur].kids)
      if (nodes[c].leaf == leaf) { nxt = c; break; }
    if (nxt < 0) {
      nxt = (int)nodes.size();
      HNode n;
      n.leaf = leaf;
      nodes.push_back(n);
      nodes[cur].kids.push_back(nxt);
    }
    cur = nxt;
  }
  return cur;
}

// Reorders every sequence so that ids occurring in more sequences come first (ties: lower id):
// frequent factors sit near the root, which is what makes prefixes shared.
void order_by_frequency(std::vector<std::vector<int>>& seqs) {
  std::map<int, int> cnt;
  for (const auto& q : seqs) {
    int last = -1;
    for (int x : q) {            // q is sorted: count each id once per sequence
      if (x != last) ++cnt[x];
      last = x;
    }
  }
  for (auto& q : seqs)
    std::stable_sort(q.begin(), q.end(), [&](int a, int b) {
      const int ca = cnt[a], cb = cnt[b];
      return ca != cb ? ca > cb : a < b;
    });
}

// FP64 instruction counts of the Horner evaluation, mirroring the emission rules of ami_jit.cpp.
long long count_f_ops(const std::vector<HNode>& f, int n) {
  long long ops = 0;
  bool have = false;
  for (int c : f[n].kids)
    if (!f[c].kids.empty()) {
      ops += count_f_ops(f, c) + 1;     // multiply, or fma into the running sum
      have = true;
    }
  for (int c : f[n].kids)
    if (f[c].kids.empty()) {
      const bool unit = (f[c].num == 1 || f[c].num == -1) && f[c].den == 1;
      if (have || !unit) ++ops;         // add / fma; a leading +-F is free
      have = true;
    }
  return ops;
}

// returns ops; *is_real tells whether S_D(n) has no imaginary part
long long count_d_ops(const HornerPlan& hp, int n, bool* is_real) {
  long long ops = 0;
  bool have = hp.dn[n].group >= 0, acc_real = true;
  for (int c : hp.dn[n].kids) {
    bool sreal = true;
    ops += count_d_ops(hp, c, &sreal);
    const bool dreal = hp.d_is_real[hp.dn[c].leaf] != 0;
    const bool preal = dreal && sreal;
    // product D * S: real*real 1, real*complex or complex*real 2, complex*complex 4; when a
    // running sum exists the adds fuse into the multiplies (fma), except that a real product
    // leaves the imaginary accumulator alone
    long long pops = dreal ? (sreal ? 1 : 2) : (sreal ? 2 : 4);
    (void)have;
    ops += pops;
    acc_real = acc_real && preal;
    have = true;
  }
  *is_real = acc_real;
  return ops;
}

}  // namespace

void build_horner_plan(const FlatTable& ft, HornerPlan& hp) {
  hp = HornerPlan();
  hp.d_is_real.assign(ft.leafD.size(), 0);
  for (size_t u = 0; u < ft.leafD.size(); ++u) {
    bool any = false;
    for (int a : ft.leafD[u].a) any |= (a != 0);
    hp.d_is_real[u] = any ? 0 : 1;
  }
  // group the terms by denominator product
  std::map<std::vector<int>, int> gid;
  std::vector<std::vector<int>> gd;                       // group -> d
  std::vector<std::vector<const FlatTerm*>> members;
  for (const FlatTerm& t : ft.terms) {
    auto it = gid.find(t.d);
    if (it == gid.end()) {
      it = gid.emplace(t.d, (int)gd.size()).first;
      gd.push_back(t.d);
      members.emplace_back();
    }
    members[it->second].push_back(&t);
  }
  const int G = (int)gd.size();
  hp.groups.resize(G);
  for (int g = 0; g < G; ++g) {
    HGroup& hg = hp.groups[g];
    hg.d = gd[g];
    std::vector<std::vector<int>> seqs;
    for (const FlatTerm* t : members[g]) seqs.push_back(t->f);
    order_by_frequency(seqs);
    hg.f.assign(1, HNode());
    for (size_t i = 0; i < seqs.size(); ++i) {
      const int n = trie_insert(hg.f, seqs[i]);
      hg.f[n].terminal = true;
      hg.f[n].num = members[g][i]->num;
      hg.f[n].den = members[g][i]->den;
    }
    hp.n_fnodes += (long long)hg.f.size() - 1;
    hp.ops_f += count_f_ops(hg.f, 0);
  }
  // one trie over the groups' denominator products
  std::vector<std::vector<int>> dseq = gd;
  order_by_frequency(dseq);
  hp.dn.assign(1, HNode());
  for (int g = 0; g < G; ++g) hp.dn[trie_insert(hp.dn, dseq[g])].group = g;
  hp.n_dnodes = (long long)hp.dn.size() - 1;
  bool r = true;
  hp.ops_d = count_d_ops(hp, 0, &r);
}

}  // namespace ami
