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

// ---- tries -----------------------------------------------------------------------------------
struct TrieNode {
  int leaf = -1;
  std::vector<int> kids;
  bool terminal = false;
  long long num = 0, den = 1;
};

template <class Node>
int trie_insert(std::vector<Node>& nodes, const std::vector<int>& seq) {
  int cur = 0;
  for (int leaf : seq) {
    int nxt = -1;
    for (int c : nodes[cur].kids)
      if (nodes[c].leaf == leaf) { nxt = c; break; }
    if (nxt < 0) {
      nxt = (int)nodes.size();
      Node n;
      n.leaf = leaf;
      nodes.push_back(n);
      nodes[cur].kids.push_back(nxt);
    }
    cur = nxt;
  }
  return cur;
}

// number of sequences each id occurs in (sequences are sorted: count an id once per sequence)
std::map<int, int> occurrence(const std::vector<std::vector<int>>& seqs) {
  std::map<int, int> cnt;
  for (const auto& q : seqs) {
    int last = -1;
    for (int x : q) {
      if (x != last) ++cnt[x];
      last = x;
    }
  }
  return cnt;
}

// Factor orderings tried for the FT sums.  0: inside each group, ids in more of the group's terms
// first (shares prefixes within the group).  1-4: one ordering for the whole table, which lines the
// tails of different groups up so that hash-consing finds them equal.
enum { kOrderLocalFreq = 0, kOrderGlobalRareFirst, kOrderGlobalFreqFirst, kOrderIdAsc, kOrderIdDesc, kNumOrders };

void apply_order(std::vector<std::vector<int>>& seqs, int order, const std::map<int, int>& global_cnt) {
  std::map<int, int> local;
  if (order == kOrderLocalFreq) local = occurrence(seqs);
  auto cnt = [&](int x) {
    const std::map<int, int>& m = order == kOrderLocalFreq ? local : global_cnt;
    auto it = m.find(x);
    return it == m.end() ? 0 : it->second;
  };
  for (auto& q : seqs)
    std::stable_sort(q.begin(), q.end(), [&](int a, int b) {
      switch (order) {
        case kOrderLocalFreq:
        case kOrderGlobalFreqFirst: { const int ca = cnt(a), cb = cnt(b); return ca != cb ? ca > cb : a < b; }
        case kOrderGlobalRareFirst: { const int ca = cnt(a), cb = cnt(b); return ca != cb ? ca < cb : a < b; }
        case kOrderIdAsc: return a < b;
        default: return a > b;
      }
    });
}

// FP64 instructions of one S-node as emitted by ami_jit.cpp: one multiply / fma / add per item,
// except that a leading +-F costs nothing.
long long snode_ops(const SNode& n) {
  long long ops = (long long)n.items.size();
  const SItem& first = n.items[0];
  if (first.child < 0 && (first.num == 1 || first.num == -1) && first.den == 1) --ops;
  return ops;
}

typedef std::vector<long long> SKey;

// hash-conses the sub-trie under `t` into `snodes`; returns the S-node id
int intern(const std::vector<TrieNode>& trie, int t, std::vector<SNode>& snodes, std::map<SKey, int>& memo) {
  SNode n;
  for (int c : trie[t].kids)
    if (!trie[c].kids.empty()) {
      const int ch = intern(trie, c, snodes, memo);
      n.items.push_back(SItem{trie[c].leaf, ch, 0, 1});
      n.height = std::max(n.height, snodes[ch].height + 1);
    }
  const size_t n_inner = n.items.size();
  for (int c : trie[t].kids)
    if (trie[c].kids.empty()) n.items.push_back(SItem{trie[c].leaf, -1, trie[c].num, trie[c].den});
  auto less = [](const SItem& a, const SItem& b) {
    if (a.leaf != b.leaf) return a.leaf < b.leaf;
    if (a.child != b.child) return a.child < b.child;
    if (a.num != b.num) return a.num < b.num;
    return a.den < b.den;
  };
  std::sort(n.items.begin(), n.items.begin() + n_inner, less);
  std::sort(n.items.begin() + n_inner, n.items.end(), less);
  SKey key;
  for (const SItem& it : n.items) { key.push_back(it.leaf); key.push_back(it.child); key.push_back(it.num); key.push_back(it.den); }
  auto f = memo.find(key);
  if (f != memo.end()) return f->second;
  const int id = (int)snodes.size();
  snodes.push_back(std::move(n));
  memo.emplace(std::move(key), id);
  return id;
}

// FP64 instructions of the R part as emitted by ami_jit.cpp.  Denominators are ordered complex
// first, so the subtree under a real denominator is real and independent of the frequency: its
// products (one instruction each) are done once per (sample, beta) [*per_beta]; an edge with a complex
// denominator costs 2 when the sum below it is real (no complex kids), else 4 [*per_freq].
void count_d_ops(const HornerPlan& hp, int n, long long* per_beta, long long* per_freq) {
  for (int c : hp.dn[n].kids) {
    count_d_ops(hp, c, per_beta, per_freq);
    if (hp.d_is_real[hp.dn[c].leaf]) {
      *per_beta += 1;
    } else {
      bool sub_complex = false;
      for (int cc : hp.dn[c].kids) sub_complex |= !hp.d_is_real[hp.dn[cc].leaf];
      *per_freq += sub_complex ? 4 : 2;
    }
  }
}

int nnz(const std::vector<int>& v) {
  int n = 0;
  for (int x : v) n += (x != 0);
  return n;
}

}  // namespace

void build_horner_plan(const FlatTable& ft, HornerPlan& hp) {
  hp = HornerPlan();
  hp.d_is_real.assign(ft.leafD.size(), 0);
  for (size_t u = 0; u < ft.leafD.size(); ++u) hp.d_is_real[u] = nnz(ft.leafD[u].a) ? 0 : 1;
  // group the terms by denominator product
  std::map<std::vector<int>, int> gid;
  std::vector<std::vector<int>> gd;                       // group -> d
  std::vector<std::vector<const FlatTerm*>> members;
  std::vector<std::vector<int>> all_f;
  for (const FlatTerm& t : ft.terms) {
    auto it = gid.find(t.d);
    if (it == gid.end()) {
      it = gid.emplace(t.d, (int)gd.size()).first;
      gd.push_back(t.d);
      members.emplace_back();
    }
    members[it->second].push_back(&t);
    all_f.push_back(t.f);
  }
  const int G = (int)gd.size();
  const std::map<int, int> global_cnt = occurrence(all_f);
  // FT sums: try every ordering, keep the cheapest DAG
  long long best = -1;
  for (int order = 0; order < kNumOrders; ++order) {
    std::vector<SNode> snodes;
    std::map<SKey, int> memo;
    std::vector<HGroup> groups(G);
    for (int g = 0; g < G; ++g) {
      groups[g].d = gd[g];
      std::vector<std::vector<int>> seqs;
      for (const FlatTerm* t : members[g]) seqs.push_back(t->f);
      apply_order(seqs, order, global_cnt);
      std::vector<TrieNode> trie(1);
      for (size_t i = 0; i < seqs.size(); ++i) {
        const int n = trie_insert(trie, seqs[i]);
        trie[n].terminal = true;
        trie[n].num = members[g][i]->num;
        trie[n].den = members[g][i]->den;
      }
      if (trie[0].kids.empty()) {       // no Fermi factors at all (n_int = 0)
        groups[g].root = -1;
        groups[g].num = trie[0].terminal ? trie[0].num : 0;
        groups[g].den = trie[0].terminal ? trie[0].den : 1;
      } else {
        groups[g].root = intern(trie, 0, snodes, memo);
      }
    }
    long long ops = 0;
    for (const SNode& n : snodes) ops += snode_ops(n);
    if (best < 0 || ops < best) {
      best = ops;
      hp.groups.swap(groups);
      hp.snodes.swap(snodes);
      hp.f_order = order;
    }
  }
  hp.ops_f = best < 0 ? 0 : best;
  hp.n_fnodes = 0;
  for (const SNode& n : hp.snodes) hp.n_fnodes += (long long)n.items.size();
  // one trie over the groups' denominator products, frequent factors first
  // complex denominators (those with an external frequency) first, then frequent ones first
  std::vector<std::vector<int>> dseq = gd;
  {
    const std::map<int, int> cnt = occurrence(dseq);
    for (auto& q : dseq)
      std::stable_sort(q.begin(), q.end(), [&](int a, int b) {
        const int ra = hp.d_is_real[a], rb = hp.d_is_real[b];
        if (ra != rb) return ra < rb;
        const int ca = cnt.at(a), cb = cnt.at(b);
        return ca != cb ? ca > cb : a < b;
      });
  }
  hp.dn.assign(1, HNode());
  for (int g = 0; g < G; ++g) hp.dn[trie_insert(hp.dn, dseq[g])].group = g;
  hp.dseq = dseq;
  hp.n_dnodes = (long long)hp.dn.size() - 1;
  count_d_ops(hp, 0, &hp.ops_d_beta, &hp.ops_d);
  {   // the same R part as a sum over prefix products (several temperatures per launch)
    auto has_q = [&](int n) {
      if (hp.dn[n].group >= 0) return true;
      for (int c : hp.dn[n].kids)
        if (hp.d_is_real[hp.dn[c].leaf]) return true;
      return false;
    };
    if (has_q(0)) hp.ops_qsum += 1;
    std::vector<std::pair<int, int>> stack;   // (node, depth among the complex denominators)
    for (int c : hp.dn[0].kids)
      if (!hp.d_is_real[hp.dn[c].leaf]) stack.emplace_back(c, 1);
    while (!stack.empty()) {
      const auto [n, depth] = stack.back();
      stack.pop_back();
      if (depth >= 2) hp.ops_prefix += 4;
      if (has_q(n)) hp.ops_qsum += 2;
      for (int c : hp.dn[n].kids)
        if (!hp.d_is_real[hp.dn[c].leaf]) stack.emplace_back(c, depth + 1);
    }
    hp.mb_prefix = hp.ops_prefix + 2 * hp.ops_qsum <= 2 * hp.ops_d;   // fewer instructions at n_b = 2 already
  }
  // leaf costs on the common path of the routines in ami_device.cuh
  const int kExpCore = 15;   // magic fma, subtract, 2 reduction fma, 10 polynomial fma, final fma
  const int kNewton = 3, kCos = 15;   // one third-order reciprocal step = 3 fma
  // every distinct integer combination of the energies (up to sign) that a denominator needs is
  // formed once per sample
  {
    std::map<std::vector<int>, int> seen;
    for (const LeafD& l : ft.leafD) {
      std::vector<int> c = l.c;
      int sign = 0;
      for (int v : c)
        if (v) { sign = v > 0 ? 1 : -1; break; }
      if (!sign) continue;
      if (sign < 0)
        for (int& v : c) v = -v;
      if (seen.emplace(c, 1).second) hp.ops_combo += std::max(0, nnz(c) - 1);
    }
  }
  // Fermi/Bose leaves (ami_jit.cpp): one exponential per energy symbol in use, beta*e + exp_split
  // (17); per distinct (combination, sigma): the mantissa products, one fma, the reciprocal, and one
  // multiply when the combination has negative coefficients; leaves that differ only in the
  // derivative order share all of that
  {
    std::vector<char> used(ft.n_eps, 0);
    std::map<std::pair<std::vector<int>, int>, int> bases;   // (combination, sigma) -> highest k
    for (const LeafF& l : ft.leafF) {
      auto key = std::make_pair(l.c, l.sigma);
      auto it = bases.find(key);
      if (it == bases.end()) {
        bases.emplace(key, l.k);
        int npos = 0, nneg = 0;
        for (int i = 0; i < ft.n_eps; ++i) {
          if (l.c[i]) used[i] = 1;
          if (l.c[i] > 0) npos += l.c[i];
          if (l.c[i] < 0) nneg -= l.c[i];
        }
        if (l.sigma < 0) npos += 1;                     // e^{beta eta}
        hp.ops_leaf_f += std::max(0, npos - 1) + std::max(0, nneg - 1) + 1 /*fma*/ + kNewton + (nneg ? 1 : 0);
        if (l.k > 0) hp.ops_leaf_f += 2;                // g
      } else if (l.k > 0 && it->second == 0) {
        it->second = l.k;
        hp.ops_leaf_f += 2;
      }
      if (l.k > 0) hp.ops_leaf_f += (l.k - 1) /*Q_k*/ + (l.k - 1) /*beta^k*/ + 3;
    }
    for (int i = 0; i < ft.n_eps; ++i)
      if (used[i]) hp.ops_leaf_f += 1 + kExpCore;
  }
  for (size_t u = 0; u < ft.leafD.size(); ++u) {
    const LeafD& l = ft.leafD[u];
    if (hp.d_is_real[u]) hp.ops_combo += 1 /*regulator*/ + kNewton;   // once per sample
    else hp.ops_leaf_d += nnz(l.a) /*a.z + E*/ + 1 /*regulator*/ + std::max(0, nnz(l.a) - 1) + 2 /*|D|^2*/ + kNewton + 2;
  }
  const int L = ft.n_int + ft.n_ext;
  for (int i = 0; i < ft.n_eps; ++i) {
    std::vector<int> a(ft.sym_alpha.begin() + (size_t)i * L, ft.sym_alpha.begin() + (size_t)(i + 1) * L);
    hp.ops_disp += 2 * (std::max(0, nnz(a) - 1) + kCos) + 2;
  }
}


// ---------------------------------------------------------------------------------------------
// Tree program: the Horner plan written as node lists for the table-driven interpreter
// (format in ami_table.hpp).
// ---------------------------------------------------------------------------------------------
namespace {

struct TreeBuilder {
  const FlatTable& ft;
  const HornerPlan& hp;
  TreeProgram& tp;
  std::vector<int> uses_left, slot_of;       // S-nodes
  std::vector<char> keep;                     // S-nodes that are some group's FT: never recycled
  std::vector<int> free_slots;
  std::map<std::pair<long long, long long>, int> const_slot;
  std::vector<int> q_slot;                    // D-trie node -> slot of Q(n), -1 = none
  std::vector<int> s_slot;                    // D-trie node -> first slot of its complex S pair
  bool overflow = false;
  const uint32_t UF, UD;

  TreeBuilder(const FlatTable& f, const HornerPlan& h, TreeProgram& t)
      : ft(f), hp(h), tp(t), UF((uint32_t)f.leafF.size()), UD((uint32_t)f.leafD.size()) {}

  uint32_t leaf_re_d(int u) const { return UF + 2u * (uint32_t)u; }   // index of Re D[u] in L[]
  uint32_t leaf_one() const { return UF + 2u * UD; }                  // L[...] = 1

  int take() {
    if (!free_slots.empty()) { const int s = free_slots.back(); free_slots.pop_back(); return s; }
    if (tp.n_slots >= 65533) { overflow = true; return 0; }
    return tp.n_slots++;
  }
  int take_pair() {                // two consecutive slots, never recycled
    if (tp.n_slots >= 65532) { overflow = true; return 0; }
    const int s = tp.n_slots;
    tp.n_slots += 2;
    return s;
  }
  int constant(long long num, long long den) {     // constants were collected up front: V[slot] = num/den
    auto it = const_slot.find({num, den});
    if (it == const_slot.end()) { overflow = true; return 0; }
    return it->second;
  }
  void add_constant(long long num, long long den) {
    if (const_slot.count({num, den})) return;
    const_slot.emplace(std::make_pair(num, den), (int)tp.consts.size());
    tp.consts.push_back((double)num / (double)den);
  }
  // appends one node; a node never straddles a tile
  void emit(std::vector<uint32_t>& code, uint32_t dst, const std::vector<uint32_t>& items) {
    if (items.size() + 1 > (size_t)kTreeTileWords) { overflow = true; return; }
    while (code.size() % kTreeTileWords + 1 + items.size() > (size_t)kTreeTileWords)
      code.push_back(tree_header(0, kTreeNoDst));
    code.push_back(tree_header((uint32_t)items.size(), dst));
    code.insert(code.end(), items.begin(), items.end());
  }
  void consume(int n) {
    if (--uses_left[n] == 0 && !keep[n] && slot_of[n] >= 0) { free_slots.push_back(slot_of[n]); slot_of[n] = -1; }
  }
  // makes sure S-node `id` is in a slot (depth first) and returns the slot
  int snode(int id, std::vector<uint32_t>& code) {
    if (slot_of[id] >= 0) return slot_of[id];
    const SNode& n = hp.snodes[id];
    std::vector<uint32_t> items;
    std::vector<int> child_slot(n.items.size(), -1);
    for (size_t i = 0; i < n.items.size(); ++i)
      if (n.items[i].child >= 0) child_slot[i] = snode(n.items[i].child, code);
    for (size_t i = 0; i < n.items.size(); ++i) {
      const SItem& it = n.items[i];
      items.push_back(tree_item(0, (uint32_t)it.leaf, (uint32_t)(it.child >= 0 ? child_slot[i] : constant(it.num, it.den))));
    }
    for (const SItem& it : n.items)
      if (it.child >= 0) consume(it.child);
    slot_of[id] = take();
    emit(code, (uint32_t)slot_of[id], items);
    return slot_of[id];
  }
  // Q(n) = [FT of the group ending at n] + sum over kids with a real denominator of Dr * Q(kid);
  // returns its slot or -1 when there is nothing
  int qnode(int n, const std::vector<int>& ft_slot, std::vector<uint32_t>& code) {
    const HNode& nd = hp.dn[n];
    std::vector<uint32_t> items;
    const int ftq = nd.group >= 0 ? ft_slot[nd.group] : -1;
    if (ftq >= 0) items.push_back(tree_item(0, leaf_one(), (uint32_t)ftq));
    bool any = false;
    for (int c : nd.kids)
      if (hp.d_is_real[hp.dn[c].leaf]) {
        items.push_back(tree_item(0, leaf_re_d(hp.dn[c].leaf), (uint32_t)qnode(c, ft_slot, code)));
        any = true;
      }
    if (!any) return ftq;                           // alias of the FT slot (or nothing)
    const int s = take();
    emit(code, (uint32_t)s, items);
    return s;
  }
  bool has_complex_kids(int n) const {
    for (int c : hp.dn[n].kids)
      if (!hp.d_is_real[hp.dn[c].leaf]) return true;
    return false;
  }
  // S(n) = Q(n) + sum over kids with a complex denominator of D * S(kid): the result for the root,
  // stored as a pair otherwise
  void rnode(int n, std::vector<uint32_t>& code) {
    for (int c : hp.dn[n].kids)
      if (!hp.d_is_real[hp.dn[c].leaf] && has_complex_kids(c)) rnode(c, code);
    std::vector<uint32_t> items;
    if (q_slot[n] >= 0) items.push_back(tree_item(0, UD, (uint32_t)q_slot[n]));        // D[U_D] = 1
    for (int c : hp.dn[n].kids) {
      const int u = hp.dn[c].leaf;
      if (hp.d_is_real[u]) continue;
      if (has_complex_kids(c)) items.push_back(tree_item(1, (uint32_t)u, (uint32_t)s_slot[c]));
      else if (q_slot[c] >= 0) items.push_back(tree_item(0, (uint32_t)u, (uint32_t)q_slot[c]));
    }
    if (n != 0) s_slot[n] = take_pair();
    emit(code, n != 0 ? (uint32_t)s_slot[n] : kTreeNoDst, items);
  }
};

}  // namespace

void build_tree_program(const FlatTable& ft, const HornerPlan& hp, TreeProgram& tp) {
  tp = TreeProgram();
  if (ft.leafF.size() + 2 * ft.leafD.size() + 1 > 4095) return;
  TreeBuilder b(ft, hp, tp);
  // constants first: they occupy V[0 .. n_consts)
  for (const SNode& n : hp.snodes)
    for (const SItem& it : n.items)
      if (it.child < 0) b.add_constant(it.num, it.den);
  for (const HGroup& g : hp.groups)
    if (g.root < 0) b.add_constant(g.num, g.den);
  tp.n_slots = (int)tp.consts.size();
  b.uses_left.assign(hp.snodes.size(), 0);
  b.slot_of.assign(hp.snodes.size(), -1);
  b.keep.assign(hp.snodes.size(), 0);
  for (const SNode& n : hp.snodes)
    for (const SItem& it : n.items)
      if (it.child >= 0) ++b.uses_left[it.child];
  for (const HGroup& g : hp.groups)
    if (g.root >= 0) { ++b.uses_left[g.root]; b.keep[g.root] = 1; }
  // FT of every group (a group without Fermi factors IS its constant)
  std::vector<int> ft_slot(hp.groups.size(), -1);
  for (size_t g = 0; g < hp.groups.size(); ++g) {
    const HGroup& hg = hp.groups[g];
    ft_slot[g] = hg.root >= 0 ? b.snode(hg.root, tp.code_beta) : b.constant(hg.num, hg.den);
  }
  b.free_slots.clear();          // what follows lives until the frequency loop has run: no recycling
  // frequency-independent sub-sums of the nodes the R part visits
  b.q_slot.assign(hp.dn.size(), -1);
  b.s_slot.assign(hp.dn.size(), -1);
  for (size_t n = 0; n < hp.dn.size(); ++n)
    if (n == 0 || !hp.d_is_real[hp.dn[n].leaf]) b.q_slot[n] = b.qnode((int)n, ft_slot, tp.code_beta);
  b.rnode(0, tp.code_freq);
  tp.ok = !b.overflow;
}

}  // namespace ami
