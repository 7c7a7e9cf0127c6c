// Diagram files -> labelled R0 (Fig. 2): read_graph, label_graph, graph_to_R0.
// Host only, integers only.  See include/ami.h for the file format and the labelling rule.
#include <algorithm>
#include <cctype>
#include <cstdlib>
#include <cstring>
#include <map>
#include <new>
#include <numeric>
#include <vector>

#include "../../include/ami.h"

extern "C" {

int ami_graph_parse(const char* text, ami_graph_edge* edges, int32_t capacity, int32_t* n_edges) {
  if (!text || !n_edges) return AMI_EINVAL;
  int32_t rows = 0;
  const char* p = text;
  while (*p) {
    // one row: up to the newline, cut at '#'
    const char* eol = strchr(p, '\n');
    const char* end = eol ? eol : p + strlen(p);
    const char* hash = (const char*)memchr(p, '#', (size_t)(end - p));
    const char* stop = hash ? hash : end;
    long v[4];
    int got = 0;
    const char* q = p;
    while (q < stop) {
      while (q < stop && isspace((unsigned char)*q)) ++q;
      if (q >= stop) break;
      char* after = nullptr;
      const long x = strtol(q, &after, 10);
      if (after == q || after > stop || got == 4) return AMI_EINVAL;   // not a number, or a fifth column
      if (after < stop && !isspace((unsigned char)*after)) return AMI_EINVAL;
      v[got++] = x;
      q = after;
    }
    if (got != 0) {
      if (got != 4 || v[0] < 0 || v[1] < 0 || v[0] > 1000000 || v[1] > 1000000 || (v[2] != 0 && v[2] != 1))
        return AMI_EINVAL;
      if (edges) {
        if (rows >= capacity) return AMI_EINVAL;
        edges[rows].source = (int32_t)v[0];
        edges[rows].target = (int32_t)v[1];
        edges[rows].is_fermion = (int32_t)v[2];
        edges[rows].spin = (int32_t)v[3];
      }
      ++rows;
    }
    p = eol ? eol + 1 : end;
  }
  *n_edges = rows;
  return AMI_OK;
}

int ami_graph_label(const ami_graph_edge* edges, int32_t n_edges, int32_t* n_int_out, int32_t* n_ext_out,
                    int32_t* n_g_out, int32_t* n_eps_out, int32_t* alpha_all, int32_t* row_of_g, int32_t* alpha,
                    int32_t* eps, uint8_t* slot_is_fermionic, int64_t cap_words) {
  if (!edges || n_edges < 1) return AMI_EINVAL;
  try {
    int V = 0;
    for (int i = 0; i < n_edges; ++i) {
      if (edges[i].source < 0 || edges[i].target < 0 || (edges[i].is_fermion != 0 && edges[i].is_fermion != 1))
        return AMI_EINVAL;
      V = std::max(V, std::max(edges[i].source, edges[i].target) + 1);
    }
    std::vector<int> degree(V, 0);
    for (int i = 0; i < n_edges; ++i) { ++degree[edges[i].source]; ++degree[edges[i].target]; }

    // legs: rows with an end that nothing else touches
    int leg_in = -1, leg_out = -1;
    std::vector<char> is_leg(n_edges, 0);
    for (int i = 0; i < n_edges; ++i) {
      const bool s1 = degree[edges[i].source] == 1, t1 = degree[edges[i].target] == 1;
      if (edges[i].source == edges[i].target) continue;      // a tadpole, not a leg
      if (s1 && t1) return AMI_EINVAL;                        // a line that touches nothing else
      if (s1) { if (leg_in >= 0) return AMI_EINVAL; leg_in = i; is_leg[i] = 1; }
      if (t1) { if (leg_out >= 0) return AMI_EINVAL; leg_out = i; is_leg[i] = 1; }
    }
    if ((leg_in >= 0) != (leg_out >= 0)) return AMI_EINVAL;
    const int n_ext = leg_in >= 0 ? 1 : 0;
    if (n_ext && edges[leg_in].is_fermion != edges[leg_out].is_fermion) return AMI_EINVAL;

    // spanning tree over the internal vertices: bosonic lines first, then fermionic, file order
    std::vector<int> parent(V);
    std::iota(parent.begin(), parent.end(), 0);
    auto find = [&](int x) {
      while (parent[x] != x) { parent[x] = parent[parent[x]]; x = parent[x]; }
      return x;
    };
    std::vector<char> in_tree(n_edges, 0);
    for (int pass = 0; pass < 2; ++pass)
      for (int i = 0; i < n_edges; ++i) {
        if (is_leg[i] || edges[i].is_fermion != pass) continue;
        const int a = find(edges[i].source), b = find(edges[i].target);
        if (a != b) { parent[a] = b; in_tree[i] = 1; }
      }
    int root = -1;
    for (int i = 0; i < n_edges; ++i) {
      if (is_leg[i]) continue;
      const int a = find(edges[i].source);
      if (root < 0) root = a;
      if (a != root || find(edges[i].target) != root) return AMI_EINVAL;   // disconnected
    }
    if (n_ext && (root < 0 || find(edges[leg_in].target) != root || find(edges[leg_out].source) != root))
      return AMI_EINVAL;
    std::vector<int> chords;
    for (int i = 0; i < n_edges; ++i)
      if (!is_leg[i] && !in_tree[i]) {
        if (!edges[i].is_fermion) return AMI_EUNSUPPORTED;    // a bosonic internal sum
        chords.push_back(i);
      }
    const int m = (int)chords.size();
    if (m > AMI_MAX_INT) return AMI_EUNSUPPORTED;
    const int L = m + n_ext;

    std::vector<std::vector<int32_t>> lab(n_edges, std::vector<int32_t>(L, 0));
    std::vector<char> solved(n_edges, 0);
    for (int l = 0; l < m; ++l) { lab[chords[l]][l] = 1; solved[chords[l]] = 1; }
    if (n_ext) {
      lab[leg_in][m] = 1; solved[leg_in] = 1;
      lab[leg_out][m] = 1; solved[leg_out] = 1;
    }
    // leaf stripping: a vertex with one unsolved line fixes it
    std::vector<int> unsolved_at(V, 0);
    for (int i = 0; i < n_edges; ++i)
      if (!solved[i]) { ++unsolved_at[edges[i].source]; ++unsolved_at[edges[i].target]; }
    std::vector<int> queue;
    for (int v = 0; v < V; ++v) if (unsolved_at[v] == 1) queue.push_back(v);
    while (!queue.empty()) {
      const int v = queue.back();
      queue.pop_back();
      if (unsolved_at[v] != 1) continue;
      int line = -1;
      std::vector<int32_t> tot(L, 0);            // sum_in - sum_out over the solved lines at v
      for (int i = 0; i < n_edges; ++i) {
        if (edges[i].source != v && edges[i].target != v) continue;
        if (!solved[i]) { line = i; continue; }
        if (edges[i].source == edges[i].target) continue;     // a tadpole enters and leaves
        const int sgn = edges[i].target == v ? 1 : -1;
        for (int l = 0; l < L; ++l) tot[l] += sgn * lab[i][l];
      }
      if (line < 0) return AMI_EINVAL;
      // the line enters v: +label, leaves v: -label
      const int sgn = edges[line].target == v ? -1 : 1;
      for (int l = 0; l < L; ++l) lab[line][l] = sgn * tot[l];
      solved[line] = 1;
      const int w = edges[line].source == v ? edges[line].target : edges[line].source;
      --unsolved_at[v];
      if (--unsolved_at[w] == 1) queue.push_back(w);
    }
    for (int i = 0; i < n_edges; ++i) if (!solved[i]) return AMI_EINVAL;
    // conservation at every internal vertex (the last vertex of the stripping is not used above)
    for (int v = 0; v < V; ++v) {
      if (degree[v] <= 1) continue;
      std::vector<int32_t> tot(L, 0);
      for (int i = 0; i < n_edges; ++i) {
        if (edges[i].source == edges[i].target) continue;
        if (edges[i].target == v) for (int l = 0; l < L; ++l) tot[l] += lab[i][l];
        if (edges[i].source == v) for (int l = 0; l < L; ++l) tot[l] -= lab[i][l];
      }
      for (int l = 0; l < L; ++l) if (tot[l]) return AMI_EINVAL;
    }

    // R0: fermionic lines that are not legs; equal labels share a symbol
    std::vector<int> rows;
    for (int i = 0; i < n_edges; ++i) if (!is_leg[i] && edges[i].is_fermion) rows.push_back(i);
    const int n_g = (int)rows.size();
    if (n_g < 1) return AMI_EINVAL;
    std::map<std::vector<int32_t>, int> symbol_of;
    std::vector<int> sym(n_g);
    for (int g = 0; g < n_g; ++g) {
      auto it = symbol_of.find(lab[rows[g]]);
      if (it == symbol_of.end()) it = symbol_of.emplace(lab[rows[g]], (int)symbol_of.size()).first;
      sym[g] = it->second;
    }
    const int n_eps = (int)symbol_of.size();
    if (n_eps > AMI_MAX_EPS) return AMI_EUNSUPPORTED;

    if (n_int_out) *n_int_out = m;
    if (n_ext_out) *n_ext_out = n_ext;
    if (n_g_out) *n_g_out = n_g;
    if (n_eps_out) *n_eps_out = n_eps;
    if (alpha_all) {
      if ((int64_t)n_edges * L > cap_words) return AMI_EINVAL;
      for (int i = 0; i < n_edges; ++i) for (int l = 0; l < L; ++l) alpha_all[(size_t)i * L + l] = lab[i][l];
    }
    if (row_of_g) for (int g = 0; g < n_g; ++g) row_of_g[g] = rows[g];
    if (alpha) {
      if ((int64_t)n_g * L > cap_words) return AMI_EINVAL;
      for (int g = 0; g < n_g; ++g) for (int l = 0; l < L; ++l) alpha[(size_t)g * L + l] = lab[rows[g]][l];
    }
    if (eps) {
      if ((int64_t)n_g * n_eps > cap_words) return AMI_EINVAL;
      for (int g = 0; g < n_g; ++g) for (int s = 0; s < n_eps; ++s) eps[(size_t)g * n_eps + s] = sym[g] == s;
    }
    if (slot_is_fermionic) {
      for (int l = 0; l < m; ++l) slot_is_fermionic[l] = 1;
      if (n_ext) slot_is_fermionic[m] = (uint8_t)edges[leg_in].is_fermion;
    }
    return AMI_OK;
  } catch (const std::bad_alloc&) {
    return AMI_ENOMEM;
  } catch (...) {
    return AMI_EINVAL;
  }
}

}  // extern "C"
