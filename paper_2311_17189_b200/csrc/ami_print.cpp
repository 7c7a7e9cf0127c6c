// LaTeX output of the term table ("Feature: Pretty printing and latex output";
// the analogue of pretty_print_ft_terms).  Host only.  Notation (include/ami.h, ami_table_latex).
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "ami_table.hpp"

namespace {

void put_linear(std::string& s, const std::vector<int>& a, const char* a_name, const std::vector<int>& c,
                const char* c_name) {
  bool first = true;
  auto one = [&](int coef, const char* name, size_t idx) {
    if (!coef) return;
    if (coef < 0) s += "-";
    else if (!first) s += "+";
    const int mag = coef < 0 ? -coef : coef;
    if (mag != 1) s += std::to_string(mag);
    s += name;
    s += "_{" + std::to_string(idx) + "}";
    first = false;
  };
  for (size_t i = 0; i < a.size(); ++i) one(a[i], a_name, i);
  for (size_t i = 0; i < c.size(); ++i) one(c[i], c_name, i);
  if (first) s += "0";
}

void put_coef(std::string& s, long long num, long long den, bool alone) {
  const long long mag = num < 0 ? -num : num;
  s += num < 0 ? "-" : "+";
  if (den != 1) s += "\\frac{" + std::to_string(mag) + "}{" + std::to_string(den) + "}";
  else if (mag != 1 || alone) s += std::to_string(mag);
}

void put_fermi(std::string& s, const ami::LeafF& l) {
  const std::vector<int> none;
  s += std::string(" f_{") + (l.sigma > 0 ? "+" : "-") + "}";
  if (l.k > 0) s += "^{(" + std::to_string(l.k) + ")}";
  s += "(";
  put_linear(s, none, "", l.c, "\\epsilon");
  s += ")";
}

void put_denominators(std::string& s, const ami::FlatTable& ft, const std::vector<int>& d) {
  for (size_t j = 0; j < d.size();) {
    size_t p = 1;
    while (j + p < d.size() && d[j + p] == d[j]) ++p;
    const ami::LeafD& l = ft.leafD[d[j]];
    s += " \\frac{1}{(";
    put_linear(s, l.a, "z", l.c, "\\epsilon");
    s += ")";
    if (p > 1) s += "^{" + std::to_string(p) + "}";
    s += "}";
    j += p;
  }
}

int give(const std::string& s, char* buf, size_t* bytes) {
  const size_t need = s.size() + 1;
  if (!buf) { *bytes = need; return AMI_OK; }
  if (*bytes < need) return AMI_EINVAL;
  memcpy(buf, s.c_str(), need);
  *bytes = need;
  return AMI_OK;
}

}  // namespace

// The factorised form the paper prints (PAPER.md:100-104 Eq. 6, :115-132: FT * R): the terms grouped by their
// denominator product R_g, the Fermi/Bose sums FT_g in Horner form.  Sums that several groups share are named once,
//   S_{n} = sum_items [coef] f(..) [S_{child}],      I = [A x] sum_g S_{root(g)} R_g.
extern "C" int ami_table_latex_factorized(const ami_table* tab, char* buf, size_t* bytes) {
  if (!tab || !bytes) return AMI_EINVAL;
  try {
    const ami::FlatTable& ft = tab->flat;
    const ami::HornerPlan& hp = tab->horner;
    std::string s = "\\begin{aligned}\n";
    for (size_t id = 0; id < hp.snodes.size(); ++id) {
      s += "S_{" + std::to_string(id) + "} ={}&";
      for (const ami::SItem& it : hp.snodes[id].items) {
        s += " ";
        if (it.child >= 0) put_coef(s, 1, 1, false);
        else put_coef(s, it.num, it.den, false);
        put_fermi(s, ft.leafF[it.leaf]);
        if (it.child >= 0) s += " S_{" + std::to_string(it.child) + "}";
      }
      s += " \\\\\n";
    }
    s += "I ={}& ";
    char num[64];
    if (ft.prefactor != 1.0) {
      snprintf(num, sizeof num, "%.17g", ft.prefactor);
      s += std::string(num) + " \\times \\Big[ \\\\\n& ";
    }
    for (size_t g = 0; g < hp.groups.size(); ++g) {
      const ami::HGroup& hg = hp.groups[g];
      if (g) s += " \\\\\n& ";
      if (hg.root >= 0) s += "+ S_{" + std::to_string(hg.root) + "}";
      else put_coef(s, hg.num, hg.den, true);
      put_denominators(s, ft, hg.d);
    }
    if (hp.groups.empty()) s += "0";
    if (ft.prefactor != 1.0) s += " \\Big]";
    s += "\n\\end{aligned}\n";
    return give(s, buf, bytes);
  } catch (const std::bad_alloc&) {
    return AMI_ENOMEM;
  } catch (...) {
    return AMI_EINVAL;
  }
}

extern "C" int ami_table_latex(const ami_table* tab, char* buf, size_t* bytes) {
  if (!tab || !bytes) return AMI_EINVAL;
  try {
    const ami::FlatTable& ft = tab->flat;
    std::string s = "\\begin{aligned}\nI ={}& ";
    char num[64];
    if (ft.prefactor != 1.0) {
      snprintf(num, sizeof num, "%.17g", ft.prefactor);
      s += std::string(num) + " \\times \\Big[ \\\\\n& ";
    }
    const std::vector<int> none;
    bool first_term = true;
    for (const ami::FlatTerm& t : ft.terms) {
      if (!first_term) s += " \\\\\n& ";
      first_term = false;
      const long long mag = t.num < 0 ? -t.num : t.num;
      s += t.num < 0 ? "-" : "+";
      if (t.den != 1) s += "\\frac{" + std::to_string(mag) + "}{" + std::to_string(t.den) + "}";
      else if (mag != 1 || (t.f.empty() && t.d.empty())) s += std::to_string(mag);
      for (int id : t.f) {
        const ami::LeafF& l = ft.leafF[id];
        s += std::string(" f_{") + (l.sigma > 0 ? "+" : "-") + "}";
        if (l.k > 0) s += "^{(" + std::to_string(l.k) + ")}";
        s += "(";
        put_linear(s, none, "", l.c, "\\epsilon");
        s += ")";
      }
      for (size_t j = 0; j < t.d.size();) {
        size_t p = 1;
        while (j + p < t.d.size() && t.d[j + p] == t.d[j]) ++p;
        const ami::LeafD& l = ft.leafD[t.d[j]];
        s += " \\frac{1}{(";
        put_linear(s, l.a, "z", l.c, "\\epsilon");
        s += ")";
        if (p > 1) s += "^{" + std::to_string(p) + "}";
        s += "}";
        j += p;
      }
    }
    if (ft.terms.empty()) s += "0";
    if (ft.prefactor != 1.0) s += " \\Big]";
    s += "\n\\end{aligned}\n";
    const size_t need = s.size() + 1;
    if (!buf) { *bytes = need; return AMI_OK; }
    if (*bytes < need) return AMI_EINVAL;
    memcpy(buf, s.c_str(), need);
    *bytes = need;
    return AMI_OK;
  } catch (const std::bad_alloc&) {
    return AMI_ENOMEM;
  } catch (...) {
    return AMI_EINVAL;
  }
}
