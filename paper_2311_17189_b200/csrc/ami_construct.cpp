// ami_construct: the symbolic AMI recursion (host, one-time).
//
// Eqs. 1-5 of arXiv 2311.17189: the n nested Matsubara sums of
//   I = beta^-n sum prod_j 1/(X^j + E^j)
// are resolved one at a time with the residue theorem.  A pole of multiplicity M (Eq. 5) is
// expanded here with the closed Leibniz form
//   Res = s_Q * sum_{k + sum r_j = M-1} (1/k!) prod_j (-alpha_p^j)^{r_j} f^{(k)}(z0)
//         prod_{j in Z} G_j(z0)^{1+r_j} prod_{j in C} G_j
// (Q: the lines sharing the pole, s_Q = prod alpha_p over Q; Z: other lines that depend on nu_p;
// C: lines that do not), using d^r/dz^r G = (-alpha)^r r! G^{r+1}.  The result is the
// unfactorised term list of PAPER.md:100 (Eq. 6 with FT a plain product), merged and stored with
// dictionaries of distinct Fermi/Bose leaves and distinct denominators.  Denominators keep the
// orientation in which the recursion produced them (D and -D are different leaves): the regulator
// of reading P10 is added to D as it arises, and 1/(D+eta) != -1/(-D+eta).
#include <algorithm>
#include <map>
#include <numeric>

#include "ami_table.hpp"

namespace ami {
namespace {

struct SymG { std::vector<int> a, e; };               // 1/(a . i nu + e . eps)
struct SymF { std::vector<int> pe; int sigma, k; };   // f_sigma^{(k)}(pe . eps)
struct SymTerm {
  long long num = 1, den = 1;
  std::vector<SymF> f;
  std::vector<SymG> g;
};

long long gcd_ll(long long a, long long b) {
  a = a < 0 ? -a : a;
  b = b < 0 ? -b : b;
  while (b) { long long t = a % b; a = b; b = t; }
  return a ? a : 1;
}
void reduce(long long& n, long long& d) {
  if (d < 0) { n = -n; d = -d; }
  long long g = gcd_ll(n, d);
  n /= g; d /= g;
}
long long factorial(int k) { long long f = 1; for (int i = 2; i <= k; ++i) f *= i; return f; }

// all (r_0..r_{parts-1}) >= 0 with sum == total, appended to `out`
void compositions(int total, int parts, std::vector<int>& cur, std::vector<std::vector<int>>& out) {
  if ((int)cur.size() == parts - 1) {
    cur.push_back(total);
    out.push_back(cur);
    cur.pop_back();
    return;
  }
  for (int v = 0; v <= total; ++v) {
    cur.push_back(v);
    compositions(total - v, parts, cur, out);
    cur.pop_back();
  }
}

int sum_one(const FlatTable& ft, int p, const std::vector<SymTerm>& in, std::vector<SymTerm>& out,
            long long& n_multipoles, int& max_deriv) {
  const int L = ft.n_int + ft.n_ext, ne = ft.n_eps;
  for (const SymTerm& t : in) {
    std::vector<int> dep;
    for (int j = 0; j < (int)t.g.size(); ++j) {
      int a = t.g[j].a[p];
      if (!a) continue;
      if (a != 1 && a != -1) return AMI_EUNSUPPORTED_ALPHA;
      dep.push_back(j);
    }
    if (dep.empty()) return AMI_ENOPOLE;
    // pole of each dependent line (Eq. 4) as the integer vector (pa | pe)
    std::map<std::vector<int>, std::vector<int>> groups;   // pole -> lines
    std::vector<std::vector<int>> order;                    // first-appearance order of poles
    for (int j : dep) {
      std::vector<int> pole(L + ne);
      const int s = -t.g[j].a[p];
      for (int l = 0; l < L; ++l) pole[l] = (l == p) ? 0 : s * t.g[j].a[l];
      for (int i = 0; i < ne; ++i) pole[L + i] = s * t.g[j].e[i];
      if (!groups.count(pole)) order.push_back(pole);
      groups[pole].push_back(j);
    }
    for (const auto& pole : order) {
      const std::vector<int>& Q = groups[pole];
      const int M = (int)Q.size();
      if (M > 1) ++n_multipoles;
      if (M - 1 > AMI_MAX_DERIV) return AMI_EUNSUPPORTED;
      long long sQ = 1;
      for (int j : Q) sQ *= t.g[j].a[p];
      std::vector<int> Z;
      for (int j : dep)
        if (std::find(Q.begin(), Q.end(), j) == Q.end()) Z.push_back(j);
      // statistics of the pole: odd number of fermionic frequencies -> sigma = -1 (P4)
      int nferm = 0;
      for (int l = 0; l < L; ++l) nferm += std::abs(pole[l]) * (ft.ferm[l] ? 1 : 0);
      const int sigma = (nferm & 1) ? -1 : 1;
      std::vector<int> pe(pole.begin() + L, pole.end());
      // substituted copies of the Z lines: i nu_p -> z0
      std::vector<SymG> zsub;
      for (int j : Z) {
        SymG g = t.g[j];
        const int ap = g.a[p];
        for (int l = 0; l < L; ++l) g.a[l] = (l == p) ? 0 : g.a[l] + ap * pole[l];
        for (int i = 0; i < ne; ++i) g.e[i] += ap * pole[L + i];
        zsub.push_back(g);
      }
      // Leibniz expansion: index 0 of the composition is k (derivatives on f), the rest r_j
      std::vector<std::vector<int>> comps;
      std::vector<int> cur;
      compositions(M - 1, 1 + (int)Z.size(), cur, comps);
      for (const auto& kr : comps) {
        SymTerm nt;
        nt.num = t.num * sQ;
        nt.den = t.den * factorial(kr[0]);
        for (size_t z = 0; z < Z.size(); ++z)
          if ((kr[1 + z] & 1) && t.g[Z[z]].a[p] == 1) nt.num = -nt.num;   // (-alpha)^r
        reduce(nt.num, nt.den);
        nt.f = t.f;
        nt.f.push_back(SymF{pe, sigma, kr[0]});
        max_deriv = std::max(max_deriv, kr[0]);
        for (size_t z = 0; z < Z.size(); ++z)
          for (int rep = 0; rep <= kr[1 + z]; ++rep) nt.g.push_back(zsub[z]);
        for (int j = 0; j < (int)t.g.size(); ++j)
          if (!t.g[j].a[p]) nt.g.push_back(t.g[j]);
        out.push_back(std::move(nt));
      }
    }
  }
  return AMI_OK;
}

}  // namespace

int construct_flat(int n_int, int n_ext, int n_g, int n_eps, const int32_t* alpha, const int32_t* eps,
                   const uint8_t* ferm, const int32_t* sum_order, double prefactor, FlatTable& ft) {
  if (n_int < 0 || n_ext < 0 || n_g < 1 || n_eps < 1 || !alpha || !eps || !ferm) return AMI_EINVAL;
  if (n_int > AMI_MAX_INT || n_ext > AMI_MAX_EXT || n_eps > AMI_MAX_EPS) return AMI_EUNSUPPORTED;
  const int L = n_int + n_ext;
  ft.n_int = n_int; ft.n_ext = n_ext; ft.n_g = n_g; ft.n_eps = n_eps;
  ft.prefactor = prefactor;
  ft.ferm.assign(ferm, ferm + L);
  for (int l = 0; l < n_int; ++l)
    if (!ferm[l]) return AMI_EINVAL;          // Eq. 3 is the fermionic sum
  std::vector<char> seen(n_int, 0);
  for (int s = 0; s < n_int; ++s) {
    int p = sum_order ? sum_order[s] : s;
    if (p < 0 || p >= n_int || seen[p]) return AMI_EINVAL;
    seen[p] = 1;
  }
  // momentum combination of each energy symbol = alpha of the R0 line that carries it
  ft.sym_alpha.assign((size_t)n_eps * L, 0);
  std::vector<char> have(n_eps, 0);
  SymTerm t0;
  for (int j = 0; j < n_g; ++j) {
    SymG g;
    g.a.assign(alpha + (size_t)j * L, alpha + (size_t)(j + 1) * L);
    g.e.assign(eps + (size_t)j * n_eps, eps + (size_t)(j + 1) * n_eps);
    int nnz = 0, sym = -1;
    for (int i = 0; i < n_eps; ++i)
      if (g.e[i]) { ++nnz; sym = i; }
    if (nnz == 1 && g.e[sym] == 1 && !have[sym]) {
      have[sym] = 1;
      for (int l = 0; l < L; ++l) ft.sym_alpha[(size_t)sym * L + l] = g.a[l];
    }
    t0.g.push_back(std::move(g));
  }
  std::vector<SymTerm> cur(1, t0), nxt;
  for (int s = 0; s < n_int; ++s) {
    nxt.clear();
    int rc = sum_one(ft, sum_order ? sum_order[s] : s, cur, nxt, ft.n_multipoles, ft.max_deriv);
    if (rc != AMI_OK) return rc;
    cur.swap(nxt);
  }
  ft.n_terms_raw = (long long)cur.size();

  // ---- canonicalise, build leaf dictionaries, merge identical terms ----------------------
  std::map<LeafF, int> fmap;
  std::map<LeafD, int> dmap;
  std::map<std::pair<std::vector<int>, std::vector<int>>, std::pair<long long, long long>> merged;
  std::vector<std::pair<std::vector<int>, std::vector<int>>> first_seen;
  for (const SymTerm& t : cur) {
    long long num = t.num, den = t.den;
    std::vector<int> fi, di;
    for (const SymF& f : t.f) {
      LeafF key{f.pe, f.sigma, f.k};
      auto it = fmap.find(key);
      if (it == fmap.end()) {
        it = fmap.emplace(key, (int)ft.leafF.size()).first;
        ft.leafF.push_back(key);
      }
      fi.push_back(it->second);
    }
    for (const SymG& g : t.g) {
      for (int l = 0; l < n_int; ++l)
        if (g.a[l]) return AMI_EINVAL;        // cannot happen: every internal slot was summed
      LeafD key{std::vector<int>(g.a.begin() + n_int, g.a.end()), g.e};
      auto it = dmap.find(key);
      if (it == dmap.end()) {
        it = dmap.emplace(key, (int)ft.leafD.size()).first;
        ft.leafD.push_back(key);
      }
      di.push_back(it->second);
    }
    std::sort(fi.begin(), fi.end());
    std::sort(di.begin(), di.end());
    auto key = std::make_pair(fi, di);
    auto it = merged.find(key);
    if (it == merged.end()) {
      merged.emplace(key, std::make_pair(num, den));
      first_seen.push_back(key);
    } else {
      long long n2 = it->second.first * den + num * it->second.second, d2 = it->second.second * den;
      reduce(n2, d2);
      it->second = {n2, d2};
    }
  }
  for (const auto& key : first_seen) {
    auto c = merged[key];
    if (c.first == 0) continue;
    FlatTerm ftm;
    ftm.num = c.first; ftm.den = c.second;
    ftm.f = key.first; ftm.d = key.second;
    ft.max_den = std::max(ft.max_den, (int)ftm.d.size());
    ft.terms.push_back(std::move(ftm));
  }
  if (ft.leafF.size() > 60000 || ft.leafD.size() > 60000) return AMI_EUNSUPPORTED;
  return AMI_OK;
}

}  // namespace ami
