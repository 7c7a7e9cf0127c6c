// oracle/ami_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// A plain, slow CPU implementation of algorithmic Matsubara integration as stated in
// arXiv 2311.17189 (TorchAmi), written from /root/reference/PAPER.md only.  It is the
// oracle the CUDA path is checked against.  It shares no code with
// paper_2311_17189_b200/ and may be used only by tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs.
//
// What it computes (Eqs. 1-5; DESIGN.md "Readings" P1-P23):
//   I = beta^-n sum_{nu_1..nu_n} prod_j G^j,  G^j = 1/(X^j + E^j)            (Eqs. 1-2)
//   X^j = sum_l alpha^j_l * i nu_l,  E^j = sum_i eps^j_i * e_i, where the supplied
//   energies e_i are the NEGATIVE of the dispersion.
// The nested sums are done one at a time with the residue theorem (Eq. 3), poles from
// Eq. 4, multipoles from Eq. 5 by differentiating M-1 times symbolically, one d/dz at a
// time (the CUDA path's construct uses a closed Leibniz form instead; the two are
// independent).  The result is a list of terms (Eq. 6, unfactorised form of PAPER.md:100)
//   coef * prod_a f_sigma^(k_a)(pe_a . e) * prod_b 1/(a_b . z_ext + c_b . e).
// Evaluation is term by term, factor by factor, left to right, with no caching.
//
// Two arithmetic types from one source: double (the timed CPU baseline) and __float128
// (the truth for parity).  Parity pins: tests/test_oracle_pins.py.  Nothing in this file
// is "parity unpinned"; the regulator convention (P10) and the parity norm (P20) are
// DESIGN.md readings, not the paper's.
#include <quadmath.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <map>
#include <string>
#include <thread>
#include <utility>
#include <vector>

namespace {

enum { OR_OK = 0, OR_EINVAL = -1, OR_EALPHA = -2, OR_ENOPOLE = -3 };

// ---- exact rational coefficient -------------------------------------------------------
long long gcdll(long long a, long long b) {
  if (a < 0) a = -a;
  if (b < 0) b = -b;
  while (b) { long long t = a % b; a = b; b = t; }
  return a ? a : 1;
}
struct Rat {
  long long n = 1, d = 1;
  Rat() {}
  Rat(long long n_, long long d_) : n(n_), d(d_) {
    if (d < 0) { n = -n; d = -d; }
    long long g = gcdll(n, d);
    n /= g; d /= g;
  }
  Rat operator*(const Rat& o) const { return Rat(n * o.n, d * o.d); }
};

// ---- symbolic objects -----------------------------------------
struct GFac {                 // G = 1 / (alpha . (i nu) + eps . e)          (Eq. 2)
  std::vector<int> alpha, eps;
};
struct FFac {                 // f_sigma^{(k)}(pe . e), f_sigma(E) = 1/(sigma e^{beta E} + 1)
  std::vector<int> pe;
  int sigma, k;
};
struct Term {
  Rat c;
  std::vector<FFac> F;
  std::vector<GFac> G;
};
// bivariate polynomial in (f, g = 1 - f): sum coef * f^a g^b
typedef std::map<std::pair<int, int>, long long> FGPoly;

struct Table {
  int n_int = 0, n_ext = 0, n_g = 0, n_eps = 0;
  std::vector<unsigned char> ferm;   // [L]
  std::vector<int> sym_alpha;        // [n_eps][L] alpha row of each energy symbol
  double prefactor = 1.0;
  std::vector<Term> terms;
  int max_k = 0;
  long n_multipoles = 0;             // pole groups with M > 1 met during construction
  std::vector<FGPoly> dpoly;         // dpoly[k]: f^{(k)} = beta^k * dpoly[k](f, g)
};

// d/dE of a polynomial in (f,g) using f' = -beta f g, g' = +beta f g (one factor of beta
// is pulled out per derivative):  d(f^a g^b) = -a f^a g^{b+1} + b f^{a+1} g^b.
FGPoly fg_derivative(const FGPoly& p) {
  FGPoly q;
  for (const auto& kv : p) {
    int a = kv.first.first, b = kv.first.second;
    long long c = kv.second;
    if (a) q[{a, b + 1}] += -a * c;
    if (b) q[{a + 1, b}] += b * c;
  }
  return q;
}

// ---- construction: one Matsubara sum (Eqs. 3-5) ------------------------------------------
struct ZProd {                // coef * f^{(kf)}(z) * prod_{i in zl} G_i(z); repeats = powers
  Rat c;
  int kf;
  std::vector<int> zl;
};

int sum_over_nu(Table& tb, int p, const std::vector<Term>& in, std::vector<Term>& out) {
  const int L = tb.n_int + tb.n_ext;
  for (const Term& t : in) {
    std::vector<int> P;       // lines that depend on nu_p
    for (int j = 0; j < (int)t.G.size(); ++j) {
      int a = t.G[j].alpha[p];
      if (a == 0) continue;
      if (a != 1 && a != -1) return OR_EALPHA;   // Eq. 4 is written for |alpha_p| = 1 (P8)
      P.push_back(j);
    }
    if (P.empty()) return OR_ENOPOLE;            // P9
    std::vector<char> used(P.size(), 0);
    for (size_t ia = 0; ia < P.size(); ++ia) {
      if (used[ia]) continue;
      // Eq. 4: z0 = -alpha_p^j (E^j + sum_{l != p} alpha^j_l i nu_l)  ->  integer vectors
      const GFac& ga = t.G[P[ia]];
      std::vector<int> pa(L), pe(tb.n_eps);
      for (int l = 0; l < L; ++l) pa[l] = (l == p) ? 0 : -ga.alpha[p] * ga.alpha[l];
      for (int i = 0; i < tb.n_eps; ++i) pe[i] = -ga.alpha[p] * ga.eps[i];
      // all lines with the same pole: multiplicity M (Eq. 5, P7: exact integer equality)
      std::vector<int> Q;
      for (size_t ib = ia; ib < P.size(); ++ib) {
        if (used[ib]) continue;
        const GFac& gb = t.G[P[ib]];
        bool same = true;
        for (int l = 0; l < L && same; ++l) same = ((l == p) ? 0 : -gb.alpha[p] * gb.alpha[l]) == pa[l];
        for (int i = 0; i < tb.n_eps && same; ++i) same = (-gb.alpha[p] * gb.eps[i]) == pe[i];
        if (same) { Q.push_back(P[ib]); used[ib] = 1; }
      }
      const int M = (int)Q.size();
      if (M > 1) tb.n_multipoles++;
      // prod_{j in Q} G_j(z) = s_Q (z - z0)^-M with s_Q = prod alpha_p^j (alpha = +-1)
      long long sQ = 1, fact = 1;
      for (int j : Q) sQ *= t.G[j].alpha[p];
      for (int i = 2; i <= M - 1; ++i) fact *= i;
      ZProd z0;
      z0.c = t.c * Rat(sQ, fact);
      z0.kf = 0;
      for (int j : P) {
        bool inQ = false;
        for (int q : Q) inQ |= (q == j);
        if (!inQ) z0.zl.push_back(j);
      }
      // Eq. 5: differentiate f(z) prod G_i(z)  M-1 times, one derivative at a time
      std::vector<ZProd> cur(1, z0);
      for (int r = 0; r < M - 1; ++r) {
        std::vector<ZProd> nxt;
        for (const ZProd& w : cur) {
          ZProd df = w;                     // derivative lands on the Fermi function
          df.kf += 1;
          nxt.push_back(df);
          for (size_t i = 0; i < w.zl.size(); ++i) {   // d/dz G = -alpha_p G^2
            ZProd dg = w;
            dg.c = w.c * Rat(-t.G[w.zl[i]].alpha[p], 1);
            dg.zl.push_back(w.zl[i]);
            nxt.push_back(dg);
          }
        }
        cur.swap(nxt);
      }
      // statistics of the pole (P4/P5): e^{beta i Omega} = -1 for an odd number of
      // fermionic frequencies in the pole, so f(z0) = 1/(sigma e^{beta E} + 1)
      int nf = 0;
      for (int l = 0; l < L; ++l) nf += (pa[l] < 0 ? -pa[l] : pa[l]) * (tb.ferm[l] ? 1 : 0);
      const int sigma = (nf & 1) ? -1 : 1;
      // substitute i nu_p -> z0 in the z-dependent lines, keep the constants
      for (const ZProd& w : cur) {
        Term nt;
        nt.c = w.c;
        nt.F = t.F;
        FFac ff;
        ff.pe = pe; ff.sigma = sigma; ff.k = w.kf;
        nt.F.push_back(ff);
        if (w.kf > tb.max_k) tb.max_k = w.kf;
        for (int j : w.zl) {
          GFac g = t.G[j];
          const int ap = g.alpha[p];
          for (int l = 0; l < L; ++l) g.alpha[l] = (l == p) ? 0 : g.alpha[l] + ap * pa[l];
          for (int i = 0; i < tb.n_eps; ++i) g.eps[i] += ap * pe[i];
          nt.G.push_back(g);
        }
        for (int j = 0; j < (int)t.G.size(); ++j)
          if (t.G[j].alpha[p] == 0) nt.G.push_back(t.G[j]);
        out.push_back(nt);
      }
    }
  }
  return OR_OK;
}

// ---- arithmetic in T = double or __float128 ------------------------------------------------
inline double t_exp(double x) { return std::exp(x); }
inline double t_expm1(double x) { return std::expm1(x); }
inline double t_sin(double x) { return std::sin(x); }
inline double t_cos(double x) { return std::cos(x); }
inline double t_sqrt(double x) { return std::sqrt(x); }
inline double t_log2(double x) { return std::log2(x); }
inline __float128 t_log2(__float128 x) { return log2q(x); }
inline __float128 t_exp(__float128 x) { return expq(x); }
inline __float128 t_expm1(__float128 x) { return expm1q(x); }
inline __float128 t_sin(__float128 x) { return sinq(x); }
inline __float128 t_cos(__float128 x) { return cosq(x); }
inline __float128 t_sqrt(__float128 x) { return sqrtq(x); }

template <class T>
struct Cx {
  T re, im;
  Cx() : re(0), im(0) {}
  Cx(T r, T i) : re(r), im(i) {}
};
template <class T> Cx<T> operator+(Cx<T> a, Cx<T> b) { return Cx<T>(a.re + b.re, a.im + b.im); }
template <class T> Cx<T> operator-(Cx<T> a, Cx<T> b) { return Cx<T>(a.re - b.re, a.im - b.im); }
template <class T> Cx<T> operator*(Cx<T> a, Cx<T> b) {
  return Cx<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <class T> Cx<T> operator/(Cx<T> a, Cx<T> b) {
  T den = b.re * b.re + b.im * b.im;
  return Cx<T>((a.re * b.re + a.im * b.im) / den, (a.im * b.re - a.re * b.im) / den);
}
template <class T> T cabs_(Cx<T> a) { return t_sqrt(a.re * a.re + a.im * a.im); }
template <class T> Cx<T> cexp_(Cx<T> x) {
  T m = t_exp(x.re);
  return Cx<T>(m * t_cos(x.im), m * t_sin(x.im));
}
// expm1 of a complex number (P12): expm1(a) cos b - 2 sin^2(b/2) + i e^a sin b
template <class T> Cx<T> cexpm1_(Cx<T> x) {
  T s = t_sin(x.im / 2);
  return Cx<T>(t_expm1(x.re) * t_cos(x.im) - 2 * s * s, t_exp(x.re) * t_sin(x.im));
}

// f_sigma(E) = 1/(sigma e^{beta E} + 1) and g = 1 - f, both without overflow or
// cancellation (P12): the exponential is always taken of the argument with Re <= 0, and
// for sigma = -1 the difference 1 - e^{x} is formed with expm1.
template <class T>
void fermi_fg(Cx<T> E, T beta, int sigma, Cx<T>& f, Cx<T>& g) {
  Cx<T> x(beta * E.re, beta * E.im);
  const Cx<T> one(1, 0);
  if (sigma > 0) {
    if (x.re <= 0) {
      Cx<T> u = cexp_(x);
      f = one / (one + u);
      g = u / (one + u);
    } else {
      Cx<T> u = cexp_(Cx<T>(-x.re, -x.im));
      f = u / (one + u);
      g = one / (one + u);
    }
  } else {
    if (x.re <= 0) {
      Cx<T> u = cexp_(x);
      Cx<T> d = Cx<T>(0, 0) - cexpm1_(x);        // 1 - e^x
      f = one / d;
      g = Cx<T>(0, 0) - u / d;
    } else {
      Cx<T> mx(-x.re, -x.im);
      Cx<T> u = cexp_(mx);
      Cx<T> d = Cx<T>(0, 0) - cexpm1_(mx);       // 1 - e^{-x}
      f = Cx<T>(0, 0) - u / d;
      g = one / d;
    }
  }
}

// k-th derivative with respect to E: beta^k * sum c_ab f^a g^b  (P11)
template <class T>
Cx<T> fermi_deriv(const Table& tb, Cx<T> E, T beta, int sigma, int k) {
  Cx<T> f, g;
  fermi_fg(E, beta, sigma, f, g);
  if (k == 0) return f;
  Cx<T> sum(0, 0);
  for (const auto& kv : tb.dpoly[k]) {
    Cx<T> mono((T)kv.second, 0);
    for (int a = 0; a < kv.first.first; ++a) mono = mono * f;
    for (int b = 0; b < kv.first.second; ++b) mono = mono * g;
    sum = sum + mono;
  }
  T bk = 1;
  for (int i = 0; i < k; ++i) bk = bk * beta;
  return Cx<T>(bk * sum.re, bk * sum.im);
}

// One sample, one external frequency set: sum of the terms, and S = sum |term| (P20).
template <class T>
void eval_one(const Table& tb, const Cx<T>* e, const Cx<T>* zext, const char* zext_is_zero, T beta,
              T eta, Cx<T>& value, T& S) {
  const int L = tb.n_int + tb.n_ext;
  Cx<T> acc(0, 0);
  T sabs = 0;
  for (const Term& t : tb.terms) {
    Cx<T> prod((T)t.c.n / (T)t.c.d, 0);
    for (const FFac& ff : t.F) {
      Cx<T> E(0, 0);
      for (int i = 0; i < tb.n_eps; ++i)
        if (ff.pe[i]) E = E + Cx<T>((T)ff.pe[i] * e[i].re, (T)ff.pe[i] * e[i].im);
      if (ff.sigma < 0) E.re = E.re + eta;                       // P10(a)
      prod = prod * fermi_deriv(tb, E, beta, ff.sigma, ff.k);
    }
    for (const GFac& gf : t.G) {
      Cx<T> D(0, 0);
      bool freq_zero = true;
      for (int l = tb.n_int; l < L; ++l) {
        if (!gf.alpha[l]) continue;
        if (!zext_is_zero[l - tb.n_int]) freq_zero = false;
        D = D + Cx<T>((T)gf.alpha[l] * zext[l - tb.n_int].re, (T)gf.alpha[l] * zext[l - tb.n_int].im);
      }
      for (int i = 0; i < tb.n_eps; ++i)
        if (gf.eps[i]) D = D + Cx<T>((T)gf.eps[i] * e[i].re, (T)gf.eps[i] * e[i].im);
      if (freq_zero) D.re = D.re + eta;                          // P10(b)
      prod = prod / D;
    }
    acc = acc + prod;
    sabs = sabs + cabs_(prod);
  }
  T A = (T)tb.prefactor;
  value = Cx<T>(A * acc.re, A * acc.im);
  S = (A < 0 ? -A : A) * sabs;
}

template <class T>
void eval_range(const Table& tb, const double* e, int e_is_complex, long s0, long s1, long n_e,
                const double* z_ext, int n_f, double beta, double e_reg, double* out, double* S_out,
                double* log2S_out, double* log2abs_out) {
  std::vector<Cx<T>> E(tb.n_eps), Z(tb.n_ext);
  std::vector<char> zz(tb.n_ext);
  for (long s = s0; s < s1; ++s) {
    for (int i = 0; i < tb.n_eps; ++i)
      E[i] = e_is_complex ? Cx<T>((T)e[2 * (s * tb.n_eps + i)], (T)e[2 * (s * tb.n_eps + i) + 1])
                          : Cx<T>((T)e[s * tb.n_eps + i], 0);
    for (int f = 0; f < n_f; ++f) {
      for (int x = 0; x < tb.n_ext; ++x) {
        double zr = z_ext[2 * (f * tb.n_ext + x)], zi = z_ext[2 * (f * tb.n_ext + x) + 1];
        Z[x] = Cx<T>((T)zr, (T)zi);
        zz[x] = (zr == 0.0 && zi == 0.0);
      }
      Cx<T> v;
      T S;
      eval_one<T>(tb, E.data(), Z.data(), zz.data(), (T)beta, (T)e_reg, v, S);
      out[2 * ((long)f * n_e + s)] = (double)v.re;
      out[2 * ((long)f * n_e + s) + 1] = (double)v.im;
      if (S_out) S_out[(long)f * n_e + s] = (double)S;
      // base-2 logarithms taken in T before the cast: they survive where S and |value| underflow a double
      if (log2S_out) log2S_out[(long)f * n_e + s] = (double)t_log2(S);
      if (log2abs_out) log2abs_out[(long)f * n_e + s] = (double)t_log2(cabs_(v));
    }
  }
}

// e_i = -eps(K_i) with K_i = sum_l alpha_l k_l + alpha_ext q, momenta of `dim` components
// (Eqs. 9-18; Eq. 14 is written for any d).  band 0: tight binding on the hypercubic
// lattice, eps(K) = -2t sum_c cos K_c - mu (dim = 2: the square lattice of SURVEY.md 8(d));
// band 1: free particles, eps(K) = t |K|^2 - mu (the paper leaves eps_k to the
// user).
template <class T>
void dispersion_range(const Table& tb, const double* k, const double* q, double t, double mu, int dim, int band,
                      long s0, long s1, double* e_out) {
  const int L = tb.n_int + tb.n_ext;
  for (long s = s0; s < s1; ++s)
    for (int i = 0; i < tb.n_eps; ++i) {
      T K[3] = {0, 0, 0};
      for (int l = 0; l < tb.n_int; ++l)
        for (int c = 0; c < dim; ++c) K[c] = K[c] + (T)tb.sym_alpha[i * L + l] * (T)k[(s * tb.n_int + l) * dim + c];
      for (int x = 0; x < tb.n_ext; ++x)
        for (int c = 0; c < dim; ++c) K[c] = K[c] + (T)tb.sym_alpha[i * L + tb.n_int + x] * (T)q[dim * x + c];
      T acc = 0;
      if (band == 0) {
        for (int c = 0; c < dim; ++c) acc = acc + t_cos(K[c]);
        e_out[s * tb.n_eps + i] = (double)(2 * (T)t * acc + (T)mu);
      } else {
        for (int c = 0; c < dim; ++c) acc = acc + K[c] * K[c];
        e_out[s * tb.n_eps + i] = (double)((T)mu - (T)t * acc);
      }
    }
}

template <class F>
void parallel_for(long n, int n_threads, F fn) {
  if (n_threads <= 1 || n < 2 * n_threads) { fn(0, n); return; }
  std::vector<std::thread> th;
  for (int i = 0; i < n_threads; ++i) {
    long a = n * i / n_threads, b = n * (i + 1) / n_threads;
    th.emplace_back([=] { fn(a, b); });
  }
  for (auto& x : th) x.join();
}

}  // namespace

// ---- C interface (loaded with ctypes by oracle/__init__.py) ---------------------------------
extern "C" {

// alpha [n_g][n_int+n_ext] (external last), eps [n_g][n_eps], slot_is_fermionic [n_int+n_ext],
// sum_order [n_int] or NULL for 0..n_int-1.  Returns a handle or NULL (*err set).
void* oracle_construct(int n_int, int n_ext, int n_g, int n_eps, const int* alpha, const int* eps,
                       const unsigned char* slot_is_fermionic, const int* sum_order, double prefactor,
                       int* err) {
  *err = OR_OK;
  if (n_int < 0 || n_ext < 0 || n_g < 1 || n_eps < 1) { *err = OR_EINVAL; return nullptr; }
  const int L = n_int + n_ext;
  Table* tb = new Table;
  tb->n_int = n_int; tb->n_ext = n_ext; tb->n_g = n_g; tb->n_eps = n_eps;
  tb->prefactor = prefactor;
  tb->ferm.assign(slot_is_fermionic, slot_is_fermionic + L);
  for (int l = 0; l < n_int; ++l)
    if (!tb->ferm[l]) { *err = OR_EINVAL; delete tb; return nullptr; }  // Eq. 3 is for fermionic nu_p
  Term t0;
  for (int j = 0; j < n_g; ++j) {
    GFac g;
    g.alpha.assign(alpha + j * L, alpha + (j + 1) * L);
    g.eps.assign(eps + j * n_eps, eps + (j + 1) * n_eps);
    t0.G.push_back(g);
  }
  // alpha row of each energy symbol (for the dispersion): first R0 line that is that unit vector
  tb->sym_alpha.assign((size_t)n_eps * L, 0);
  for (int i = 0; i < n_eps; ++i)
    for (int j = 0; j < n_g; ++j) {
      bool unit = true;
      for (int c = 0; c < n_eps; ++c) unit &= (eps[j * n_eps + c] == (c == i ? 1 : 0));
      if (unit) { for (int l = 0; l < L; ++l) tb->sym_alpha[i * L + l] = alpha[j * L + l]; break; }
    }
  std::vector<Term> cur(1, t0), nxt;
  for (int step = 0; step < n_int; ++step) {
    int p = sum_order ? sum_order[step] : step;
    if (p < 0 || p >= n_int) { *err = OR_EINVAL; delete tb; return nullptr; }
    nxt.clear();
    int rc = sum_over_nu(*tb, p, cur, nxt);
    if (rc != OR_OK) { *err = rc; delete tb; return nullptr; }
    cur.swap(nxt);
  }
  tb->terms.swap(cur);
  FGPoly p0;
  p0[{1, 0}] = 1;              // f itself
  tb->dpoly.push_back(p0);
  for (int k = 1; k <= tb->max_k; ++k) tb->dpoly.push_back(fg_derivative(tb->dpoly[k - 1]));
  return tb;
}

void oracle_destroy(void* h) { delete (Table*)h; }

// info[0]=T, [1]=max derivative order, [2]=multipole events, [3]=terms with a derivative factor
void oracle_info(void* h, long* info) {
  Table* tb = (Table*)h;
  info[0] = (long)tb->terms.size();
  info[1] = tb->max_k;
  info[2] = tb->n_multipoles;
  long nd = 0;
  for (const Term& t : tb->terms) {
    bool d = false;
    for (const FFac& f : t.F) d |= (f.k > 0);
    nd += d;
  }
  info[3] = nd;
}

// Text dump of the terms, one per line (debugging / inspection).  Returns bytes needed.
long oracle_describe(void* h, char* buf, long cap) {
  Table* tb = (Table*)h;
  std::string s;
  char tmp[64];
  for (const Term& t : tb->terms) {
    snprintf(tmp, sizeof tmp, "%lld/%lld", t.c.n, t.c.d);
    s += tmp;
    for (const FFac& f : t.F) {
      snprintf(tmp, sizeof tmp, " F[s=%d k=%d e=", f.sigma, f.k);
      s += tmp;
      for (int v : f.pe) { snprintf(tmp, sizeof tmp, "%d,", v); s += tmp; }
      s += "]";
    }
    for (const GFac& g : t.G) {
      s += " G[a=";
      for (int v : g.alpha) { snprintf(tmp, sizeof tmp, "%d,", v); s += tmp; }
      s += " e=";
      for (int v : g.eps) { snprintf(tmp, sizeof tmp, "%d,", v); s += tmp; }
      s += "]";
    }
    s += "\n";
  }
  if (buf && cap > 0) {
    long n = (long)s.size() < cap - 1 ? (long)s.size() : cap - 1;
    memcpy(buf, s.data(), n);
    buf[n] = 0;
  }
  return (long)s.size() + 1;
}

// e: [n_e][n_eps] (paper's energy_t; complex interleaved if e_is_complex);
// z_ext: [n_f][n_ext] complex interleaved; out: [n_f][n_e] complex interleaved;
// S_out: [n_f][n_e] = sum over terms of |term| (may be NULL).  precision 0 = double, 1 = quad.
// log2S_out / log2abs_out (may be NULL): log2 S and log2 |value|, taken in the working precision
// before the cast to double, so that the scale of a sample whose terms all underflow a double
// (beta |E| of several hundred) is still known to the parity norm (-inf for an exact zero).
int oracle_evaluate_ex(void* h, const double* e, int e_is_complex, long n_e, const double* z_ext, int n_f,
                       double beta, double e_reg, int precision, int n_threads, double* out, double* S_out,
                       double* log2S_out, double* log2abs_out) {
  Table* tb = (Table*)h;
  if (!tb || n_e < 0 || n_f < 0) return OR_EINVAL;
  parallel_for(n_e, n_threads, [=](long a, long b) {
    if (precision == 0)
      eval_range<double>(*tb, e, e_is_complex, a, b, n_e, z_ext, n_f, beta, e_reg, out, S_out, log2S_out, log2abs_out);
    else
      eval_range<__float128>(*tb, e, e_is_complex, a, b, n_e, z_ext, n_f, beta, e_reg, out, S_out, log2S_out,
                             log2abs_out);
  });
  return OR_OK;
}

int oracle_evaluate(void* h, const double* e, int e_is_complex, long n_e, const double* z_ext, int n_f,
                    double beta, double e_reg, int precision, int n_threads, double* out, double* S_out) {
  return oracle_evaluate_ex(h, e, e_is_complex, n_e, z_ext, n_f, beta, e_reg, precision, n_threads, out, S_out,
                            nullptr, nullptr);
}

// k: [n_e][n_int][dim] (Eq. 8), q: [n_ext][dim]; e_out: [n_e][n_eps]
int oracle_dispersion_lattice(void* h, const double* k, const double* q, double t, double mu, long n_e, int dim,
                              int band, int precision, int n_threads, double* e_out) {
  Table* tb = (Table*)h;
  if (!tb || n_e < 0 || dim < 1 || dim > 3 || band < 0 || band > 1) return OR_EINVAL;
  parallel_for(n_e, n_threads, [=](long a, long b) {
    if (precision == 0) dispersion_range<double>(*tb, k, q, t, mu, dim, band, a, b, e_out);
    else dispersion_range<__float128>(*tb, k, q, t, mu, dim, band, a, b, e_out);
  });
  return OR_OK;
}

// the 2D square-lattice band of the configurations
int oracle_dispersion(void* h, const double* k, const double* q, double t, double mu, long n_e,
                      int precision, int n_threads, double* e_out) {
  return oracle_dispersion_lattice(h, k, q, t, mu, n_e, 2, 0, precision, n_threads, e_out);
}

// f_sigma^{(k)}(E) for one complex argument; out2 = (re, im).  Used by the pins.
int oracle_fermi(double e_re, double e_im, double beta, int sigma, int k, int precision, double* out2) {
  Table tb;
  FGPoly p0;
  p0[{1, 0}] = 1;
  tb.dpoly.push_back(p0);
  for (int i = 1; i <= k; ++i) tb.dpoly.push_back(fg_derivative(tb.dpoly[i - 1]));
  if (precision == 0) {
    Cx<double> v = fermi_deriv<double>(tb, Cx<double>(e_re, e_im), beta, sigma, k);
    out2[0] = v.re; out2[1] = v.im;
  } else {
    Cx<__float128> v = fermi_deriv<__float128>(tb, Cx<__float128>(e_re, e_im), (__float128)beta, sigma, k);
    out2[0] = (double)v.re; out2[1] = (double)v.im;
  }
  return OR_OK;
}

int oracle_hardware_threads(void) { return (int)std::thread::hardware_concurrency(); }

}  // extern "C"
