// The C ABI of include/ami.h: argument checking, device residency, launches, streamed driver.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "ami_jit.hpp"
#include "ami_kernels.cuh"

namespace ami {
long long flat_fp64_ops(const FlatTable& ft);
}
static void free_run_workspace(ami_table* tab);   // defined next to ami_run

namespace {

thread_local std::string g_cuda_err;

int cuda_fail(cudaError_t rc) {
  g_cuda_err = std::string(cudaGetErrorName(rc)) + ": " + cudaGetErrorString(rc);
  return rc == cudaErrorMemoryAllocation ? AMI_ENOMEM : AMI_ECUDA;
}
#define CU(x)                                   \
  do {                                          \
    cudaError_t rc_ = (x);                      \
    if (rc_ != cudaSuccess) return cuda_fail(rc_); \
  } while (0)

template <class T>
int upload(const std::vector<T>& h, T** d, int64_t& bytes) {
  *d = nullptr;
  const size_t n = std::max<size_t>(h.size(), 1) * sizeof(T);
  CU(cudaMalloc((void**)d, n));
  if (!h.empty()) CU(cudaMemcpy(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
  bytes += (int64_t)n;
  return AMI_OK;
}

// Q_k polynomials of f^{(k)} = beta^k f g Q_k(f):  Q_1 = -1, Q_{k+1} = (2f-1) Q_k - (f - f^2) Q_k'
std::vector<double> deriv_polys() {
  const int S = 8;
  std::vector<double> Q((AMI_MAX_DERIV + 1) * S, 0.0);
  Q[1 * S + 0] = -1.0;
  for (int k = 1; k < AMI_MAX_DERIV; ++k) {
    const double* q = &Q[k * S];
    double* r = &Q[(k + 1) * S];
    for (int i = 0; i < S - 2; ++i) {
      r[i + 1] += 2.0 * q[i];
      r[i] -= q[i];
      if (i >= 1) {
        r[i] -= i * q[i];         // -f * (i q_i f^{i-1})
        r[i + 1] += i * q[i];     // +f^2 * (i q_i f^{i-1})
      }
    }
  }
  return Q;
}

int make_device_copy(ami_table* tab, int device) {
  using namespace ami;
  const FlatTable& ft = tab->flat;
  ami_device_copy& dc = tab->dev;
  CU(cudaSetDevice(device));
  dc.device = device;
  const int UF = (int)ft.leafF.size(), UD = (int)ft.leafD.size();
  std::vector<int32_t> ptr;
  std::vector<int8_t> sym, coef, sig, kk, da, sa;
  ptr.push_back(0);
  for (const LeafF& l : ft.leafF) {
    for (int i = 0; i < ft.n_eps; ++i)
      if (l.c[i]) { sym.push_back((int8_t)i); coef.push_back((int8_t)l.c[i]); }
    ptr.push_back((int32_t)sym.size());
    sig.push_back((int8_t)l.sigma);
    kk.push_back((int8_t)l.k);
  }
  for (const LeafD& l : ft.leafD) {
    for (int i = 0; i < ft.n_eps; ++i)
      if (l.c[i]) { sym.push_back((int8_t)i); coef.push_back((int8_t)l.c[i]); }
    ptr.push_back((int32_t)sym.size());
    for (int x = 0; x < ft.n_ext; ++x) da.push_back((int8_t)l.a[x]);
  }
  const int nd = ft.max_den;
  std::vector<uint16_t> tix;
  std::vector<double> tco;
  for (const FlatTerm& t : ft.terms) {
    for (int f : t.f) tix.push_back((uint16_t)f);
    for (int j = 0; j < nd; ++j) tix.push_back((uint16_t)(j < (int)t.d.size() ? t.d[j] : UD));
    tco.push_back((double)t.num / (double)t.den);
  }
  // pad to whole tiles: the flat kernel stages the table through shared memory with bulk copies
  // whose size must be a multiple of 16 bytes (padded terms are copied, never evaluated)
  while (tco.size() % ami::kTermTile) {
    for (int j = 0; j < ft.n_int + nd; ++j) tix.push_back(0);
    tco.push_back(0.0);
  }
  for (int v : ft.sym_alpha) sa.push_back((int8_t)v);
  (void)UF;
  int rc;
  if ((rc = upload(ptr, &dc.leaf_ptr, dc.bytes))) return rc;
  if ((rc = upload(sym, &dc.leaf_sym, dc.bytes))) return rc;
  if ((rc = upload(coef, &dc.leaf_coef, dc.bytes))) return rc;
  if ((rc = upload(sig, &dc.leafF_sig, dc.bytes))) return rc;
  if ((rc = upload(kk, &dc.leafF_k, dc.bytes))) return rc;
  if ((rc = upload(da, &dc.leafD_a, dc.bytes))) return rc;
  if ((rc = upload(tix, &dc.term_idx, dc.bytes))) return rc;
  if ((rc = upload(tco, &dc.term_coef, dc.bytes))) return rc;
  if ((rc = upload(sa, &dc.sym_alpha, dc.bytes))) return rc;
  {   // tree programs, padded to whole tiles (bulk copies move whole tiles; padding is never executed)
    std::vector<uint32_t> cb = tab->tree.code_beta, cf = tab->tree.code_freq;
    while (cb.size() % ami::kTreeTileWords) cb.push_back(0);
    while (cf.size() % ami::kTreeTileWords) cf.push_back(0);
    if ((rc = upload(cb, &dc.tree_beta, dc.bytes))) return rc;
    if ((rc = upload(cf, &dc.tree_freq, dc.bytes))) return rc;
    if ((rc = upload(tab->tree.consts, &dc.tree_consts, dc.bytes))) return rc;
  }
  if ((rc = upload(deriv_polys(), &dc.derivQ, dc.bytes))) return rc;
  return AMI_OK;
}

void free_device_copy(ami_device_copy& dc) {
  if (dc.device < 0) return;
  cudaSetDevice(dc.device);
  cudaFree(dc.leaf_ptr); cudaFree(dc.leaf_sym); cudaFree(dc.leaf_coef); cudaFree(dc.leafF_sig);
  cudaFree(dc.leafF_k); cudaFree(dc.leafD_a); cudaFree(dc.term_idx); cudaFree(dc.term_coef);
  cudaFree(dc.sym_alpha); cudaFree(dc.derivQ);
  cudaFree(dc.tree_beta); cudaFree(dc.tree_freq); cudaFree(dc.tree_consts);
  dc = ami_device_copy();
}

}  // namespace

extern "C" {

int ami_version(void) { return 1; }

int64_t ami_kernel_launches(void) { return (int64_t)ami::total_launches(); }

const char* ami_strerror(int code) {
  switch (code) {
    case AMI_OK: return "ok";
    case AMI_EINVAL: return "invalid argument";
    case AMI_EUNSUPPORTED_ALPHA: return "|alpha_p| != 1 met at a summation (unsupported)";
    case AMI_ENOPOLE: return "a term has no pole in the summed frequency";
    case AMI_ECUDA: return "CUDA error, or the table has no device copy";
    case AMI_ENOMEM: return "out of memory";
    case AMI_EUNSUPPORTED: return "outside the built limits";
    default: return "unknown error";
  }
}

const char* ami_last_cuda_error(void) { return g_cuda_err.c_str(); }

int ami_construct(int n_int, int n_ext, int n_g, int n_eps, const int32_t* alpha, const int32_t* eps,
                  const uint8_t* slot_is_fermionic, const int32_t* sum_order, double prefactor, int device,
                  ami_table** out) {
  if (!out) return AMI_EINVAL;
  *out = nullptr;
  ami_table* tab = new (std::nothrow) ami_table;
  if (!tab) return AMI_ENOMEM;
  int rc;
  try {
    rc = ami::construct_flat(n_int, n_ext, n_g, n_eps, alpha, eps, slot_is_fermionic, sum_order, prefactor,
                             tab->flat);
    if (rc == AMI_OK) {
      ami::build_horner_plan(tab->flat, tab->horner);
      ami::build_tree_program(tab->flat, tab->horner, tab->tree);
      tab->fp64_ops_flat = ami::flat_fp64_ops(tab->flat);
    }
  } catch (const std::bad_alloc&) {
    rc = AMI_ENOMEM;
  } catch (...) {
    rc = AMI_EINVAL;
  }
  if (rc == AMI_OK && device >= 0) {
    rc = make_device_copy(tab, device);
    if (rc != AMI_OK) free_device_copy(tab->dev);
  }
  if (rc != AMI_OK) { delete tab; return rc; }
  *out = tab;
  return AMI_OK;
}

int ami_search_sum_order(int n_int, int n_ext, int n_g, int n_eps, const int32_t* alpha, const int32_t* eps,
                         const uint8_t* slot_is_fermionic, int criterion, int64_t max_orders,
                         int32_t* best_order, int64_t* best_cost, int64_t* default_cost, int64_t* n_tried) {
  if (!best_order || n_int < 1 || (criterion != AMI_ORDER_FEWEST_TERMS && criterion != AMI_ORDER_FEWEST_OPS))
    return AMI_EINVAL;
  std::vector<int32_t> order(n_int);
  for (int i = 0; i < n_int; ++i) order[i] = i;
  int64_t best = -1, dflt = -1, tried = 0, seen = 0;
  int last_rc = AMI_ENOPOLE;
  try {
    do {
      ami::FlatTable ft;
      const int rc = ami::construct_flat(n_int, n_ext, n_g, n_eps, alpha, eps, slot_is_fermionic, order.data(),
                                         1.0, ft);
      if (rc == AMI_EINVAL || rc == AMI_ENOMEM) return rc;
      if (rc != AMI_OK) last_rc = rc;
      if (rc == AMI_OK) {
        int64_t cost = (int64_t)ft.terms.size();
        if (criterion == AMI_ORDER_FEWEST_OPS) {
          ami::HornerPlan hp;
          ami::build_horner_plan(ft, hp);
          cost = hp.ops_f + hp.ops_d_beta + hp.ops_d + hp.ops_leaf_f + hp.ops_leaf_d + hp.ops_combo;
        }
        if (seen == 0) dflt = cost;
        if (best < 0 || cost < best) {
          best = cost;
          for (int i = 0; i < n_int; ++i) best_order[i] = order[i];
        }
        ++tried;
      }
      ++seen;
    } while ((max_orders <= 0 || seen < max_orders) && std::next_permutation(order.begin(), order.end()));
  } catch (const std::bad_alloc&) {
    return AMI_ENOMEM;
  } catch (...) {
    return AMI_EINVAL;
  }
  if (best_cost) *best_cost = best;
  if (default_cost) *default_cost = dflt;
  if (n_tried) *n_tried = tried;
  return best < 0 ? last_rc : AMI_OK;
}

void ami_table_destroy(ami_table* tab) {
  if (!tab) return;
  if (tab->dev.device >= 0 && cudaSetDevice(tab->dev.device) == cudaSuccess)
    cudaDeviceSynchronize();   // kernels of this table may still run (launches are asynchronous): wait before unloading them
  ami::jit_destroy(tab);
  free_run_workspace(tab);
  free_device_copy(tab->dev);
  delete tab;
}

int ami_table_info(const ami_table* tab, ami_info* info) {
  if (!tab || !info) return AMI_EINVAL;
  const ami::FlatTable& ft = tab->flat;
  memset(info, 0, sizeof *info);
  info->n_int = ft.n_int; info->n_ext = ft.n_ext; info->n_g = ft.n_g; info->n_eps = ft.n_eps;
  info->n_fermi_leaves = (int32_t)ft.leafF.size();
  info->n_den_leaves = (int32_t)ft.leafD.size();
  info->max_deriv = ft.max_deriv;
  info->max_den_per_term = ft.max_den;
  info->n_terms = (int64_t)ft.terms.size();
  info->n_terms_raw = ft.n_terms_raw;
  info->n_multipoles = ft.n_multipoles;
  info->n_groups = (int64_t)tab->horner.groups.size();
  info->n_tree_nodes = tab->horner.n_fnodes;
  info->n_den_nodes = tab->horner.n_dnodes;
  info->table_bytes = tab->dev.bytes;
  info->fp64_ops_flat = tab->fp64_ops_flat;
  info->fp64_ops_tree = tab->horner.ops_f + tab->horner.ops_d_beta + tab->horner.ops_d;
  info->fp64_ops_tree_fermi = tab->horner.ops_f + tab->horner.ops_d_beta;
  info->fp64_ops_leaf_fermi = tab->horner.ops_leaf_f;
  info->fp64_ops_leaf_den = tab->horner.ops_leaf_d;
  info->fp64_ops_dispersion = tab->horner.ops_disp;
  info->fp64_ops_combos = tab->horner.ops_combo;
  info->fp64_ops_mb_prefix = tab->horner.mb_prefix ? tab->horner.ops_prefix : 0;
  info->fp64_ops_mb_sum = tab->horner.mb_prefix ? tab->horner.ops_qsum : tab->horner.ops_d;
  info->tree_plan_words = tab->tree.ok ? (int64_t)(tab->tree.code_beta.size() + tab->tree.code_freq.size()) : -1;
  info->tree_plan_slots = tab->tree.n_slots;
  info->has_device_copy = tab->dev.device >= 0;
  info->reg_plan_status = !ami::jit_eligible(ft, tab->horner) ? AMI_EUNSUPPORTED
                          : (tab->jit ? ami::jit_status(tab) : 1);
  info->plan_kind = ami::jit_mode(ft, tab->horner);
  {
    int hit = 0;
    info->specialize_ms = tab->jit ? ami::jit_last_compile_ms(tab, &hit) : 0.0;
    info->specialize_cached = hit;
  }
  return AMI_OK;
}

int ami_table_export(const ami_table* tab, void* host_buf, size_t* bytes) {
  if (!tab || !bytes) return AMI_EINVAL;
  const ami::FlatTable& ft = tab->flat;
  const size_t UF = ft.leafF.size(), UD = ft.leafD.size(), T = ft.terms.size();
  const size_t mf = ft.n_int, nd = ft.max_den;
  const size_t n_i32 = 9 + UF * ft.n_eps + 2 * UF + UD * ft.n_eps + UD * ft.n_ext + T * mf + T * nd;
  size_t need = n_i32 * 4;
  need = (need + 7) / 8 * 8 + T * 8;
  if (!host_buf) { *bytes = need; return AMI_OK; }
  if (*bytes < need) return AMI_EINVAL;
  int32_t* w = (int32_t*)host_buf;
  *w++ = 0x31494D41;  // 'AMI1'
  *w++ = ft.n_int; *w++ = ft.n_ext; *w++ = ft.n_eps; *w++ = (int32_t)UF; *w++ = (int32_t)UD;
  *w++ = (int32_t)T; *w++ = (int32_t)mf; *w++ = (int32_t)nd;
  for (const auto& l : ft.leafF) for (int v : l.c) *w++ = v;
  for (const auto& l : ft.leafF) *w++ = l.sigma;
  for (const auto& l : ft.leafF) *w++ = l.k;
  for (const auto& l : ft.leafD) for (int v : l.c) *w++ = v;
  for (const auto& l : ft.leafD) for (int v : l.a) *w++ = v;
  for (const auto& t : ft.terms) for (int v : t.f) *w++ = v;
  for (const auto& t : ft.terms)
    for (size_t j = 0; j < nd; ++j) *w++ = j < t.d.size() ? t.d[j] : -1;
  char* p = (char*)host_buf + (n_i32 * 4 + 7) / 8 * 8;
  for (const auto& t : ft.terms) {
    double c = (double)t.num / (double)t.den;
    memcpy(p, &c, 8);
    p += 8;
  }
  *bytes = need;
  return AMI_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// kernel entry points
// ---------------------------------------------------------------------------------------------
namespace {

void fill_table_params(const ami_table* tab, ami::EvalParams& p) {
  const ami::FlatTable& ft = tab->flat;
  const ami_device_copy& dc = tab->dev;
  p.leaf_ptr = dc.leaf_ptr; p.leaf_sym = dc.leaf_sym; p.leaf_coef = dc.leaf_coef;
  p.leafF_sig = dc.leafF_sig; p.leafF_k = dc.leafF_k; p.leafD_a = dc.leafD_a;
  p.term_idx = dc.term_idx; p.term_coef = dc.term_coef;
  p.derivQ = dc.derivQ;
  p.tree_beta = dc.tree_beta; p.tree_freq = dc.tree_freq; p.tree_consts = dc.tree_consts;
  p.n_words_beta = (long long)tab->tree.code_beta.size(); p.n_words_freq = (long long)tab->tree.code_freq.size();
  p.n_slots = tab->tree.n_slots; p.n_consts = (int)tab->tree.consts.size();
  p.n_eps = ft.n_eps; p.n_ext = ft.n_ext;
  p.U_F = (int)ft.leafF.size(); p.U_D = (int)ft.leafD.size();
  p.m_f = ft.n_int; p.n_d = ft.max_den;
  p.T = (long long)ft.terms.size();
  p.prefactor = ft.prefactor;
}

// Decides which representation runs.  Returns AMI_OK and sets *use_reg, or an error when the
// register plan was asked for explicitly and cannot be had.
int choose_plan(const ami_table* tab, int plan, bool e_is_complex, bool* use_reg, bool* use_tree = nullptr,
                const ami::JitVariant& var = ami::JitVariant()) {
  *use_reg = false;
  if (use_tree) *use_tree = false;
  if (plan == AMI_PLAN_FLAT) return AMI_OK;
  const bool tree_ok = tab->tree.ok && !e_is_complex;
  // AUTO prefers the interpreted Horner program to the flat table only where it pays: per word the
  // interpreter costs several times a flat factor, but large tables have 50-70x fewer words than
  // flat factors (measured: order 4 0.86 vs 0.57 ms, order 6 0.95 vs 1.29 ms, order 8 15.9 vs 49.5 ms)
  const bool tree_auto = tree_ok && tab->flat.terms.size() >= 500;
  if (plan == AMI_PLAN_TREE) {
    if (!tree_ok) { g_cuda_err = "tree plan unavailable for this table / energy type"; return AMI_EUNSUPPORTED; }
    if (use_tree) *use_tree = true;
    return AMI_OK;
  }
  if (!ami::jit_eligible(tab->flat, tab->horner)) {
    if (plan == AMI_PLAN_REG) { g_cuda_err = "register plan unavailable for this table / energy type"; return AMI_EUNSUPPORTED; }
    if (use_tree) *use_tree = tree_auto;        // AUTO: the table-driven Horner program for large tables
    return AMI_OK;
  }
  std::string err;
  const int rc = ami::jit_prepare(const_cast<ami_table*>(tab), var, err);   // lazily compiled, cached in the table
  if (rc == AMI_OK) { *use_reg = true; return AMI_OK; }
  g_cuda_err = err;
  if (plan == AMI_PLAN_REG) return rc;
  if (use_tree) *use_tree = tree_auto;          // AUTO falls back to the table-driven kernels
  return AMI_OK;
}

// The tally is formed inside the evaluation kernel up to this many result rows: a warp reduction per (row, 32 samples)
// costs a sixth of the kernel's instructions at 256 rows, storing the results and reading them back a third of its time
// (cfg5, 64 frequencies x 4 temperatures, 1e6 samples: 4.1 -> 3.2 ms).  The limit only bounds the partial-sum workspace.
constexpr int64_t kFusedTallyMaxRows = 1024;

struct MomentaSrc {
  const double* d_k = nullptr;
  int64_t stride_sample = 0, stride_comp = 0;
  const double* q = nullptr;
  double t = 0, mu = 0;
  double* tally = nullptr;      // register plan only: per-warp partial sums [rows][tally_stride] double4, or NULL
  int64_t tally_stride = 0;
  bool gen = false;             // register plan only: draw the momenta inside the kernel (d_k unused)
  uint64_t seed = 0;
  int64_t first_sample = 0;
  int dim = 2, band = AMI_BAND_TIGHT_BINDING;   // lattice of the dispersion (Eq. 14)
  int64_t* tally_slots = nullptr;               // out: per-row partial sums the fused tally wrote
};

// Launches the evaluation for all (beta, frequency) pairs, split so that one launch carries at
// most kMaxBeta temperatures and kMaxFreqWords frequency words.  `out` points at sample 0 of
// row (b=0,f=0); rows are out_row_stride samples apart.  With `mom` the energies are formed from
// momenta first: inline by the register plan (and stored to d_e only when d_e is given), by the
// dispersion kernel into d_e otherwise.
int evaluate_impl(const ami_table* tab, const MomentaSrc* mom, const void* d_e, int e_is_complex, int64_t n_e,
                  int64_t e_stride, const double* z_ext, int n_f, const double* beta, int n_b, double e_reg, int plan,
                  void* d_out, int64_t out_row_stride, cudaStream_t st, int* launches) {
  using namespace ami;
  bool use_reg = false, use_tree = false;
  const bool unordered = (plan & AMI_PLAN_UNORDERED) != 0;   // honoured by the register plan, ignored by the others
  plan &= ~AMI_PLAN_UNORDERED;
  ami::JitVariant var;
  if (mom) { var.dim = mom->dim; var.band = mom->band; }
  var.cplx = e_is_complex != 0;
  int rc = choose_plan(tab, plan, e_is_complex != 0, &use_reg, &use_tree, var);
  if (rc != AMI_OK) return rc;
  const int dim = var.dim;
  const int n_ext = tab->flat.n_ext;
  const int f_chunk = n_ext ? std::max(1, kMaxFreqWords / n_ext) : kMaxFreqWords;
  if (mom && !use_reg) {
    if (!d_e || mom->gen) return AMI_EINVAL;   // the table-driven kernels need the energies in memory
    DispParams dp;
    memset(&dp, 0, sizeof dp);
    dp.sym_alpha = tab->dev.sym_alpha;
    dp.n_int = tab->flat.n_int; dp.n_ext = n_ext; dp.n_eps = tab->flat.n_eps;
    dp.k = mom->d_k; dp.k_stride_sample = mom->stride_sample; dp.k_stride_comp = mom->stride_comp; dp.n = n_e;
    dp.dim = dim; dp.band = var.band;
    for (int i = 0; i < dim * n_ext; ++i) dp.q[i] = mom->q[i];
    dp.t = mom->t; dp.mu = mom->mu; dp.e = (double*)d_e; dp.e_stride = e_stride;
    cudaError_t crc = launch_dispersion(dp, st);
    if (crc != cudaSuccess) return cuda_fail(crc);
    if (launches) ++*launches;
  }
  EvalParams p;
  AmiBatch jb;
  memset(&p, 0, sizeof p);
  memset(&jb, 0, sizeof jb);
  if (use_reg) {
    jb.e = (const double*)d_e; jb.e_stride = e_stride;
    if (mom) {
      jb.k = mom->d_k; jb.k_stride_sample = mom->stride_sample; jb.k_stride_comp = mom->stride_comp;
      jb.gen = mom->gen ? 1 : 0; jb.seed = mom->seed; jb.first_sample = mom->first_sample;
      jb.tally = mom->tally; jb.tally_stride = mom->tally_stride;
      for (int i = 0; i < dim * n_ext; ++i) jb.q[i] = mom->q[i];
      jb.t = mom->t; jb.mu = mom->mu;
      jb.e_out = (double*)d_e;
    }
    jb.out = (double*)d_out; jb.n = n_e; jb.out_row_stride = out_row_stride;
    jb.n_f_total = n_f; jb.e_reg = e_reg; jb.prefactor = tab->flat.prefactor;
  } else {
    fill_table_params(tab, p);
    p.e = (const double*)d_e; p.out = (double*)d_out;
    p.n_e = n_e; p.e_stride = e_stride; p.out_row_stride = out_row_stride;
    p.n_f_total = n_f; p.e_reg = e_reg;
  }
  double* v_scratch = nullptr;
  if (use_tree && !tree_values_fit_smem(p)) {     // value slots in a stream-ordered global scratch
    // at most ~1 GiB of scratch at a time: larger batches are walked in chunks of samples
    const int64_t chunk = std::max<int64_t>(256, ((int64_t)1 << 30) / ((int64_t)p.n_slots * 8) / 256 * 256);
    if (n_e > chunk) {
      for (int64_t c0 = 0; c0 < n_e; c0 += chunk) {
        const int64_t nc = std::min(chunk, n_e - c0);
        MomentaSrc part;
        if (mom) { part = *mom; part.d_k = mom->d_k + c0 * mom->stride_sample; part.first_sample += c0; }
        rc = evaluate_impl(tab, mom ? &part : nullptr, d_e ? (const double*)d_e + c0 : nullptr, e_is_complex, nc, e_stride,
                           z_ext, n_f, beta, n_b, e_reg, plan, (double*)d_out + 2 * c0, out_row_stride, st, launches);
        if (rc != AMI_OK) return rc;
      }
      return AMI_OK;
    }
    p.v_stride = (n_e + 255) / 256 * 256;
    const cudaError_t arc = ami::scratch_alloc((void**)&v_scratch, (size_t)p.n_slots * p.v_stride * sizeof(double), st);
    if (arc != cudaSuccess) return cuda_fail(arc);
    p.v_scratch = v_scratch;
  }
  bool first = true;
  for (int b0 = 0; b0 < n_b; b0 += kMaxBeta) {
    const int nb = std::min(kMaxBeta, n_b - b0);
    for (int f0 = 0; f0 < n_f; f0 += f_chunk) {
      const int nf = std::min(f_chunk, n_f - f0);
      cudaError_t crc;
      if (use_reg) {
        jb.b0 = b0; jb.n_b = nb; jb.f0 = f0; jb.n_f = nf;
        for (int i = 0; i < nb; ++i) { jb.beta[i] = beta[b0 + i]; jb.ceta[i] = std::exp(beta[b0 + i] * e_reg); }
        for (int i = 0; i < nf * n_ext * 2; ++i) jb.z[i] = z_ext[(size_t)f0 * n_ext * 2 + i];
        // later launches of a split grid read the energies the first one stored
        const bool fused = mom && (first || !d_e);
        if (!fused) { jb.e_out = nullptr; }
        jb.unordered = unordered && first ? 1 : 0;   // later launches of the same call stay ordered after the first
        int n_launched = 0;
        long long slots = 0;
        crc = jit_launch(tab, var, fused, jb, st, &n_launched, &slots);
        if (mom && mom->tally_slots) *mom->tally_slots = slots;
        for (int i = 0; i < n_launched; ++i) count_external_launch(launches);
      } else {
        p.b0 = b0; p.n_b = nb; p.f0 = f0; p.n_f = nf;
        for (int i = 0; i < nb; ++i) p.beta[i] = beta[b0 + i];
        for (int i = 0; i < nf * n_ext * 2; ++i) p.z[i] = z_ext[(size_t)f0 * n_ext * 2 + i];
        crc = use_tree ? launch_eval_tree(p, st, launches) : launch_eval_flat(p, e_is_complex != 0, st, launches);
      }
      if (crc != cudaSuccess) { if (v_scratch) cudaFreeAsync(v_scratch, st); return cuda_fail(crc); }
      first = false;
    }
  }
  if (v_scratch) CU(cudaFreeAsync(v_scratch, st));
  return AMI_OK;
}

int check_device(const ami_table* tab) {
  if (!tab) return AMI_EINVAL;
  if (tab->dev.device < 0) { g_cuda_err = "table has no device copy"; return AMI_ECUDA; }
  CU(cudaSetDevice(tab->dev.device));
  return AMI_OK;
}

}  // namespace

extern "C" {

int ami_dispersion_lattice(const ami_table* tab, const double* d_k, int64_t k_stride_sample, int64_t k_stride_comp,
                           const double* q, double t, double mu, int dim, int band, int64_t n, double* d_e,
                           void* stream) {
  int rc = check_device(tab);
  if (rc) return rc;
  if (n < 0 || (n > 0 && (!d_k || !d_e)) || (tab->flat.n_ext > 0 && !q) || dim < 1 || dim > 3 ||
      (band != AMI_BAND_TIGHT_BINDING && band != AMI_BAND_FREE))
    return AMI_EINVAL;
  ami::DispParams p;
  memset(&p, 0, sizeof p);
  p.sym_alpha = tab->dev.sym_alpha;
  p.n_int = tab->flat.n_int; p.n_ext = tab->flat.n_ext; p.n_eps = tab->flat.n_eps;
  p.k = d_k; p.k_stride_sample = k_stride_sample; p.k_stride_comp = k_stride_comp; p.n = n;
  p.dim = dim; p.band = band;
  for (int i = 0; i < dim * p.n_ext; ++i) p.q[i] = q[i];
  p.t = t; p.mu = mu; p.e = d_e; p.e_stride = n;
  CU(ami::launch_dispersion(p, (cudaStream_t)stream));
  return AMI_OK;
}

int ami_dispersion(const ami_table* tab, const double* d_k, int64_t k_stride_sample, int64_t k_stride_comp,
                   const double* q, double t, double mu, int64_t n, double* d_e, void* stream) {
  return ami_dispersion_lattice(tab, d_k, k_stride_sample, k_stride_comp, q, t, mu, 2, AMI_BAND_TIGHT_BINDING, n, d_e,
                                stream);
}

int ami_evaluate(const ami_table* tab, const void* d_e, int e_is_complex, int64_t n_e, const double* z_ext,
                 int n_f, const double* beta, int n_b, double e_reg, int plan, void* d_out, void* stream) {
  int rc = check_device(tab);
  if (rc) return rc;
  const int base_plan = plan & ~AMI_PLAN_UNORDERED;
  if (n_e < 0 || n_f < 0 || n_b < 0 || (n_f > 0 && tab->flat.n_ext > 0 && !z_ext) || (n_b > 0 && !beta) ||
      base_plan < AMI_PLAN_AUTO || base_plan > AMI_PLAN_TREE)
    return AMI_EINVAL;
  if (n_e == 0 || n_f == 0 || n_b == 0) return AMI_OK;
  if (!d_e || !d_out) return AMI_EINVAL;
  return evaluate_impl(tab, nullptr, d_e, e_is_complex, n_e, n_e, z_ext, n_f, beta, n_b, e_reg, plan, d_out, n_e,
                       (cudaStream_t)stream, nullptr);
}

int ami_evaluate_momenta_lattice(const ami_table* tab, const double* d_k, int64_t k_stride_sample,
                                 int64_t k_stride_comp, const double* q, double t, double mu, int dim, int band,
                                 int64_t n, const double* z_ext, int n_f, const double* beta, int n_b, double e_reg,
                                 int plan, double* d_e, void* d_out, void* stream) {
  int rc = check_device(tab);
  if (rc) return rc;
  if (n < 0 || n_f < 0 || n_b < 0 || (n_f > 0 && tab->flat.n_ext > 0 && !z_ext) || (n_b > 0 && !beta) ||
      (tab->flat.n_ext > 0 && !q) || (plan & ~AMI_PLAN_UNORDERED) < AMI_PLAN_AUTO ||
      (plan & ~AMI_PLAN_UNORDERED) > AMI_PLAN_TREE || dim < 1 || dim > 3 ||
      (band != AMI_BAND_TIGHT_BINDING && band != AMI_BAND_FREE))
    return AMI_EINVAL;
  if (n == 0) return AMI_OK;
  if (!d_k || (!d_out && n_f > 0 && n_b > 0)) return AMI_EINVAL;
  MomentaSrc ms;
  ms.d_k = d_k; ms.stride_sample = k_stride_sample; ms.stride_comp = k_stride_comp;
  ms.q = q; ms.t = t; ms.mu = mu; ms.dim = dim; ms.band = band;
  if (n_f == 0 || n_b == 0) {
    if (!d_e) return AMI_OK;
    return ami_dispersion_lattice(tab, d_k, k_stride_sample, k_stride_comp, q, t, mu, dim, band, n, d_e, stream);
  }
  // the table-driven plans need the energies in memory: a stream-ordered workspace when the caller gave none
  double* ws = nullptr;
  bool use_reg = false;
  ami::JitVariant var;
  var.dim = dim; var.band = band;
  if (!d_e) {
    rc = choose_plan(tab, plan & ~AMI_PLAN_UNORDERED, false, &use_reg, nullptr, var);
    if (rc) return rc;
    if (!use_reg) {
      CU(ami::scratch_alloc((void**)&ws, (size_t)tab->flat.n_eps * (size_t)n * sizeof(double), (cudaStream_t)stream));
      d_e = ws;
    }
  }
  rc = evaluate_impl(tab, &ms, d_e, 0, n, n, z_ext, n_f, beta, n_b, e_reg, plan, d_out, n, (cudaStream_t)stream, nullptr);
  if (ws) cudaFreeAsync(ws, (cudaStream_t)stream);
  return rc;
}

int ami_evaluate_momenta(const ami_table* tab, const double* d_k, int64_t k_stride_sample, int64_t k_stride_comp,
                         const double* q, double t, double mu, int64_t n, const double* z_ext, int n_f,
                         const double* beta, int n_b, double e_reg, int plan, double* d_e, void* d_out, void* stream) {
  return ami_evaluate_momenta_lattice(tab, d_k, k_stride_sample, k_stride_comp, q, t, mu, 2, AMI_BAND_TIGHT_BINDING, n,
                                      z_ext, n_f, beta, n_b, e_reg, plan, d_e, d_out, stream);
}

int ami_table_export_tree(const ami_table* tab, void* host_buf, size_t* bytes) {
  if (!tab || !bytes) return AMI_EINVAL;
  if (!tab->tree.ok) return AMI_EUNSUPPORTED;
  const ami::TreeProgram& tp = tab->tree;
  size_t need = (5 + tp.code_beta.size() + tp.code_freq.size()) * 4;
  need = (need + 7) / 8 * 8 + tp.consts.size() * 8;
  if (!host_buf) { *bytes = need; return AMI_OK; }
  if (*bytes < need) return AMI_EINVAL;
  uint32_t* w = (uint32_t*)host_buf;
  *w++ = 0x31544D41;  // 'AMT1'
  *w++ = (uint32_t)tp.code_beta.size(); *w++ = (uint32_t)tp.code_freq.size(); *w++ = (uint32_t)tp.consts.size();
  *w++ = (uint32_t)tp.n_slots;
  for (uint32_t x : tp.code_beta) *w++ = x;
  for (uint32_t x : tp.code_freq) *w++ = x;
  char* c = (char*)host_buf + ((5 + tp.code_beta.size() + tp.code_freq.size()) * 4 + 7) / 8 * 8;
  if (!tp.consts.empty()) memcpy(c, tp.consts.data(), tp.consts.size() * 8);
  *bytes = need;
  return AMI_OK;
}

int ami_table_specialize(ami_table* tab) {
  int rc = check_device(tab);
  if (rc) return rc;
  std::string err;
  rc = ami::jit_prepare(tab, ami::JitVariant(), err);
  if (rc != AMI_OK) g_cuda_err = err;
  return rc;
}

namespace {
int variant_of(int dim, int band, int complex_energies, ami::JitVariant* var) {
  if (dim < 1 || dim > 3 || (band != AMI_BAND_TIGHT_BINDING && band != AMI_BAND_FREE)) return AMI_EINVAL;
  var->dim = dim; var->band = band; var->cplx = complex_energies != 0;
  return AMI_OK;
}
}  // namespace

int ami_table_kernel_source_variant(const ami_table* tab, int dim, int band, int complex_energies, char* buf,
                                    size_t* bytes) {
  if (!tab || !bytes) return AMI_EINVAL;
  ami::JitVariant var;
  if (variant_of(dim, band, complex_energies, &var)) return AMI_EINVAL;
  if (!ami::jit_eligible(tab->flat, tab->horner)) return AMI_EUNSUPPORTED;
  const std::vector<std::string> srcs = ami::jit_generate_sources(tab->flat, tab->horner, var, nullptr);
  std::string src;
  for (size_t i = 0; i < srcs.size(); ++i) {
    if (srcs.size() > 1) src += "// ======== translation unit " + std::to_string(i) + " of " + std::to_string(srcs.size()) + " ========\n";
    src += srcs[i];
  }
  if (!buf) { *bytes = src.size() + 1; return AMI_OK; }
  if (*bytes < src.size() + 1) return AMI_EINVAL;
  memcpy(buf, src.c_str(), src.size() + 1);
  *bytes = src.size() + 1;
  return AMI_OK;
}

int ami_table_kernel_source(const ami_table* tab, char* buf, size_t* bytes) {
  return ami_table_kernel_source_variant(tab, 2, AMI_BAND_TIGHT_BINDING, 0, buf, bytes);
}

int ami_table_kernel_units(const ami_table* tab, int* n_units) {
  if (!tab || !n_units) return AMI_EINVAL;
  if (!ami::jit_eligible(tab->flat, tab->horner)) return AMI_EUNSUPPORTED;
  *n_units = (int)ami::jit_generate_sources(tab->flat, tab->horner, ami::JitVariant(), nullptr).size();
  return AMI_OK;
}

int ami_table_kernel_cubin_variant(const ami_table* tab, int dim, int band, int complex_energies, int unit, void* buf,
                                   size_t* bytes, char* log, size_t log_cap) {
  if (!tab || !bytes) return AMI_EINVAL;
  ami::JitVariant var;
  if (variant_of(dim, band, complex_energies, &var)) return AMI_EINVAL;
  if (!ami::jit_eligible(tab->flat, tab->horner)) return AMI_EUNSUPPORTED;
  const std::vector<std::string> srcs = ami::jit_generate_sources(tab->flat, tab->horner, var, nullptr);
  if (unit < 0 || unit >= (int)srcs.size()) return AMI_EINVAL;
  std::vector<char> cubin;
  std::string lg;
  const int rc = ami::jit_compile(srcs[unit], cubin, lg, /*use_cache=*/false);
  if (log && log_cap) {
    const size_t nlog = std::min(log_cap - 1, lg.size());
    memcpy(log, lg.data(), nlog);
    log[nlog] = 0;
  }
  if (rc != AMI_OK) { g_cuda_err = lg; return rc; }
  if (buf) {
    if (*bytes < cubin.size()) return AMI_EINVAL;
    memcpy(buf, cubin.data(), cubin.size());
  }
  *bytes = cubin.size();
  return AMI_OK;
}

int ami_table_kernel_cubin_unit(const ami_table* tab, int unit, void* buf, size_t* bytes, char* log, size_t log_cap) {
  return ami_table_kernel_cubin_variant(tab, 2, AMI_BAND_TIGHT_BINDING, 0, unit, buf, bytes, log, log_cap);
}

int ami_table_kernel_cubin(const ami_table* tab, void* buf, size_t* bytes, char* log, size_t log_cap) {
  return ami_table_kernel_cubin_unit(tab, 0, buf, bytes, log, log_cap);
}

int ami_generate_momenta_lattice(const ami_table* tab, uint64_t seed, int64_t first_sample, int64_t n, int dim,
                                 double* d_k, void* stream) {
  int rc = check_device(tab);
  if (rc) return rc;
  if (n < 0 || first_sample < 0 || (n > 0 && !d_k) || dim < 1 || dim > 3) return AMI_EINVAL;
  CU(ami::launch_generate_momenta(seed, first_sample, n, dim * tab->flat.n_int, d_k, (cudaStream_t)stream));
  return AMI_OK;
}

int ami_generate_momenta(const ami_table* tab, uint64_t seed, int64_t first_sample, int64_t n, double* d_k,
                         void* stream) {
  return ami_generate_momenta_lattice(tab, seed, first_sample, n, 2, d_k, stream);
}

int ami_fp64_peak_probe(int device, int distinct_sources, double* dfma_per_s, double* elapsed_ms) {
  if (!dfma_per_s || !elapsed_ms || device < 0 || distinct_sources < 2 || distinct_sources > 7) return AMI_EINVAL;
  CU(cudaSetDevice(device));
  CU(ami::run_fp64_probe(distinct_sources, dfma_per_s, elapsed_ms));
  return AMI_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// S4: streamed driver (PAPER.md:113: repeated calls over energy batches; :291 tally).  With host
// buffers the chunks run through a three-stage pipeline on three internal streams -- host-to-device
// copy of chunk c+1 | kernels of chunk c | device-to-host copy of chunk c-1 -- so that the two copy
// engines (PCIe is full duplex) and the SMs work at the same time; each stage has two buffers and
// waits, through events, for the stage that last used the buffer it is about to overwrite.  Without
// host buffers there is nothing to overlap and everything runs on the caller's stream.
// ---------------------------------------------------------------------------------------------
namespace {

// Workspace of the streamed driver, cached in the table between calls: streams, events and device
// buffers that only ever grow (allocation costs more than a chunk's kernels).
struct RunBuffers {
  std::mutex mu;           // one ami_run at a time per table
  cudaStream_t s_in = nullptr, s_k = nullptr, s_out = nullptr;   // H2D copies, kernels, D2H copies
  cudaEvent_t ev_start = nullptr, ev_stop = nullptr;
  cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_k[2] = {nullptr, nullptr}, ev_out[2] = {nullptr, nullptr};
  double* k[2] = {nullptr, nullptr};      // momenta of a chunk
  double* out[2] = {nullptr, nullptr};    // results of a chunk
  double* e = nullptr;                    // energies of a chunk (table-driven plans only)
  double* wp = nullptr;                   // per-warp partial sums of the fused tally
  double* partial = nullptr;
  double* sum = nullptr;
  double* h_tally = nullptr;              // pinned host copy of `sum` (a pageable destination would stage the copy)
  size_t cap_h_tally = 0;
  size_t cap_k = 0, cap_out = 0, cap_e = 0, cap_wp = 0, cap_partial = 0, cap_sum = 0;
  int init() {
    if (ev_start) return AMI_OK;
    CU(cudaEventCreate(&ev_start));
    CU(cudaEventCreate(&ev_stop));
    CU(cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking));
    CU(cudaStreamCreateWithFlags(&s_k, cudaStreamNonBlocking));
    CU(cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      CU(cudaEventCreateWithFlags(&ev_in[i], cudaEventDisableTiming));
      CU(cudaEventCreateWithFlags(&ev_k[i], cudaEventDisableTiming));
      CU(cudaEventCreateWithFlags(&ev_out[i], cudaEventDisableTiming));
    }
    return AMI_OK;
  }
  static int grow(double** p, size_t* cap, size_t bytes) {
    if (bytes <= *cap) return AMI_OK;
    cudaFree(*p);
    *p = nullptr;
    *cap = 0;
    CU(cudaMalloc((void**)p, bytes));
    *cap = bytes;
    return AMI_OK;
  }
  int reserve(size_t bk, size_t be, size_t bo, size_t bs, size_t bw) {
    int rc;
    for (int i = 0; i < 2; ++i) {
      size_t ck = cap_k, co = cap_out;
      if ((rc = grow(&k[i], &ck, bk)) || (rc = grow(&out[i], &co, bo))) return rc;
      if (i == 1) { cap_k = ck; cap_out = co; }
    }
    if ((rc = grow(&e, &cap_e, be)) || (rc = grow(&wp, &cap_wp, bw)) ||
        (rc = grow(&partial, &cap_partial, bs * ami::kMaxSumBlocks)) || (rc = grow(&sum, &cap_sum, bs)))
      return rc;
    if (bs > cap_h_tally) {
      if (h_tally) cudaFreeHost(h_tally);
      h_tally = nullptr;
      cap_h_tally = 0;
      CU(cudaHostAlloc((void**)&h_tally, bs, cudaHostAllocDefault));
      cap_h_tally = bs;
    }
    return AMI_OK;
  }
  ~RunBuffers() {
    for (cudaStream_t st : {s_in, s_k, s_out})
      if (st) cudaStreamDestroy(st);
    for (int i = 0; i < 2; ++i) {
      for (cudaEvent_t ev : {ev_in[i], ev_k[i], ev_out[i]})
        if (ev) cudaEventDestroy(ev);
      cudaFree(k[i]); cudaFree(out[i]);
    }
    if (ev_start) cudaEventDestroy(ev_start);
    if (ev_stop) cudaEventDestroy(ev_stop);
    cudaFree(e); cudaFree(wp); cudaFree(partial); cudaFree(sum);
    if (h_tally) cudaFreeHost(h_tally);
  }
};

}  // namespace

static void free_run_workspace(ami_table* tab) {
  if (!tab->run_ws) return;
  if (tab->dev.device >= 0) cudaSetDevice(tab->dev.device);
  delete static_cast<RunBuffers*>(tab->run_ws);
  tab->run_ws = nullptr;
}

namespace {

RunBuffers* workspace_of(const ami_table* tab) {
  static std::mutex create_mu;
  std::lock_guard<std::mutex> lk(create_mu);
  ami_table* t = const_cast<ami_table*>(tab);
  if (!t->run_ws) t->run_ws = new RunBuffers;
  return static_cast<RunBuffers*>(t->run_ws);
}

}  // namespace

extern "C" int ami_run(const ami_table* tab, const ami_run_cfg* cfg, ami_run_stats* stats) {
  int rc = check_device(tab);
  if (rc) return rc;
  if (!cfg || cfg->n < 0 || cfg->n_f < 0 || cfg->n_b < 0 || cfg->chunk < 0 || cfg->first_sample < 0 ||
      (cfg->n_b > 0 && !cfg->beta) || (cfg->n_f > 0 && tab->flat.n_ext > 0 && !cfg->z_ext) ||
      (tab->flat.n_ext > 0 && !cfg->q) || (cfg->h_k && cfg->d_k) || (cfg->want_sum && !cfg->h_sum) ||
      (!cfg->want_sum && !cfg->h_out && !cfg->d_out) || cfg->dim < 0 || cfg->dim > 3 ||
      cfg->plan < AMI_PLAN_AUTO || cfg->plan > AMI_PLAN_TREE ||   /* the driver orders its own chunks: no AMI_PLAN_UNORDERED */
      (cfg->band != AMI_BAND_TIGHT_BINDING && cfg->band != AMI_BAND_FREE))
    return AMI_EINVAL;
  ami_run_stats local;
  memset(&local, 0, sizeof local);
  const int dim = cfg->dim ? cfg->dim : 2;
  const int64_t rows = (int64_t)cfg->n_b * cfg->n_f;
  const int n_comp = dim * tab->flat.n_int, n_eps = tab->flat.n_eps;
  if (cfg->n == 0 || rows == 0) {
    if (cfg->want_sum) {
      memset(cfg->h_sum, 0, (size_t)rows * 16);
      if (cfg->h_sumsq) memset(cfg->h_sumsq, 0, (size_t)rows * 16);
    }
    if (stats) *stats = local;
    return AMI_OK;
  }
  const bool host_io = cfg->h_k || cfg->h_out;
  const bool direct_out = cfg->d_out != nullptr;   // kernels write straight into the caller's buffer
  bool use_reg = false;   // the specialised kernels form the energies inline: no energy buffer
  ami::JitVariant var;
  var.dim = dim; var.band = cfg->band;
  rc = choose_plan(tab, cfg->plan, false, &use_reg, nullptr, var);
  if (rc) return rc;
  // Fused tally (register plan, a few rows): the evaluation kernel leaves one partial sum per (row, warp) and the
  // results are stored only if the caller wants them -- a seeded Monte-Carlo run then moves no sample data at all.
  const bool fused_tally = use_reg && cfg->want_sum && rows <= kFusedTallyMaxRows && ami::jit_fused_tally_ok(tab);
  const bool need_out = cfg->h_out || !use_reg || (cfg->want_sum && !fused_tally);
  const bool own_k = !cfg->d_k && (cfg->h_k || !use_reg);    // momenta pass through a buffer of the workspace
  const bool own_out = need_out && !direct_out;
  // default chunk: with host buffers small enough that the copies of one chunk overlap the kernels of the next
  // (measured: 2^17 samples); otherwise as large as the workspace allows (one chunk = no per-chunk overhead)
  int64_t chunk = cfg->chunk ? cfg->chunk : (host_io ? (int64_t)1 << 17 : (int64_t)1 << 26);
  while (chunk > 1024 && ((own_out && chunk * rows * 16 > ((int64_t)256 << 20)) ||
                          (fused_tally && chunk * rows > ((int64_t)1 << 30)) ||     // per-warp partials: rows x chunk bytes
                          (own_k && chunk * n_comp * 8 > ((int64_t)256 << 20)) ||
                          (!use_reg && chunk * n_eps * 8 > ((int64_t)256 << 20))))
    chunk /= 2;
  if (chunk > cfg->n) chunk = cfg->n;
  RunBuffers& rb = *workspace_of(tab);
  std::lock_guard<std::mutex> run_lock(rb.mu);
  cudaStream_t user = (cudaStream_t)cfg->stream;
  if ((rc = rb.init())) return rc;
  const int64_t wp_stride = (chunk + 31) / 32;
  if ((rc = rb.reserve(own_k ? (size_t)chunk * n_comp * 8 : 0, use_reg ? 0 : (size_t)chunk * n_eps * 8,
                       own_out ? (size_t)chunk * rows * 16 : 0, cfg->want_sum ? (size_t)rows * 32 : 0,
                       fused_tally ? (size_t)rows * wp_stride * 32 : 0)))
    return rc;
  const bool pipelined = host_io && cfg->n > chunk;
  cudaStream_t s_in = pipelined ? rb.s_in : user, s_k = pipelined ? rb.s_k : user, s_out = pipelined ? rb.s_out : user;
  CU(cudaEventRecord(rb.ev_start, user));
  if (pipelined)
    for (cudaStream_t st : {s_in, s_k, s_out}) CU(cudaStreamWaitEvent(st, rb.ev_start, 0));
  int launches = 0;
  // the chunk loop; any error leaves it through `rc` so that the internal streams are re-joined below
  auto run_chunks = [&]() -> int {
    for (int64_t c0 = 0, ci = 0; c0 < cfg->n; c0 += chunk, ++ci) {
      const int b = (int)(ci & 1);
      const int64_t nc = std::min(chunk, cfg->n - c0);
      const double* kbuf = nullptr;      // stays NULL when the specialised kernel draws the momenta itself
      if (cfg->d_k) {
        kbuf = cfg->d_k + c0 * n_comp;
      } else if (cfg->h_k) {
        if (pipelined && ci >= 2) CU(cudaStreamWaitEvent(s_in, rb.ev_k[b], 0));   // kernels of chunk c-2 have read k[b]
        CU(cudaMemcpyAsync(rb.k[b], cfg->h_k + c0 * n_comp, (size_t)nc * n_comp * 8, cudaMemcpyHostToDevice, s_in));
        if (pipelined) CU(cudaEventRecord(rb.ev_in[b], s_in));
        local.h2d_bytes += nc * n_comp * 8;
        kbuf = rb.k[b];
      }
      if (pipelined && cfg->h_k) CU(cudaStreamWaitEvent(s_k, rb.ev_in[b], 0));
      if (pipelined && cfg->h_out && ci >= 2) CU(cudaStreamWaitEvent(s_k, rb.ev_out[b], 0));   // out[b] has been copied out
      if (!cfg->d_k && !cfg->h_k && !use_reg) {
        CU(ami::launch_generate_momenta(cfg->seed, cfg->first_sample + c0, nc, n_comp, rb.k[b], s_k));
        ++launches;
        kbuf = rb.k[b];
      }
      MomentaSrc ms;
      ms.gen = !cfg->d_k && !cfg->h_k && use_reg; ms.seed = cfg->seed; ms.first_sample = cfg->first_sample + c0;
      ms.d_k = kbuf; ms.stride_sample = n_comp; ms.stride_comp = 1;
      ms.q = cfg->q; ms.t = cfg->t; ms.mu = cfg->mu; ms.dim = dim; ms.band = cfg->band;
      double* obuf = direct_out ? (double*)cfg->d_out + 2 * c0 : (need_out ? rb.out[b] : nullptr);
      int64_t tally_slots = 0;
      if (fused_tally) { ms.tally = rb.wp; ms.tally_stride = wp_stride; ms.tally_slots = &tally_slots; }
      const int64_t ostride = direct_out ? cfg->n : nc;
      int erc = evaluate_impl(tab, &ms, use_reg ? nullptr : rb.e, 0, nc, nc, cfg->z_ext, cfg->n_f, cfg->beta, cfg->n_b,
                              cfg->e_reg, cfg->plan, obuf, ostride, s_k, &launches);
      if (erc) return erc;
      if (cfg->want_sum) {   // on the kernel stream, in chunk order: the running sum is deterministic
        if (fused_tally)
          CU(ami::launch_warp_partial_sums(rb.wp, rows, tally_slots, wp_stride, rb.partial, rb.sum, ci == 0, s_k, &launches));
        else
          CU(ami::launch_block_sums(obuf, rows, nc, ostride, rb.partial, rb.sum, ci == 0, s_k, &launches));
      }
      if (pipelined) CU(cudaEventRecord(rb.ev_k[b], s_k));
      if (cfg->h_out) {
        if (pipelined) CU(cudaStreamWaitEvent(s_out, rb.ev_k[b], 0));
        if (rows == 1)
          CU(cudaMemcpyAsync((char*)cfg->h_out + (size_t)c0 * 16, obuf, (size_t)nc * 16, cudaMemcpyDeviceToHost, s_out));
        else
          CU(cudaMemcpy2DAsync((char*)cfg->h_out + (size_t)c0 * 16, (size_t)cfg->n * 16, obuf, (size_t)ostride * 16,
                               (size_t)nc * 16, (size_t)rows, cudaMemcpyDeviceToHost, s_out));
        if (pipelined) CU(cudaEventRecord(rb.ev_out[b], s_out));
        local.d2h_bytes += nc * rows * 16;
      }
      ++local.n_chunks;
    }
    return AMI_OK;
  };
  rc = run_chunks();
  if (pipelined) {   // the caller's stream continues after everything issued on the internal ones, error or not
    for (cudaStream_t st : {s_in, s_k, s_out}) {
      if (cudaEventRecord(rb.ev_stop, st) == cudaSuccess) cudaStreamWaitEvent(user, rb.ev_stop, 0);
    }
  }
  if (rc) return rc;
  const double* tally = rb.h_tally;
  if (cfg->want_sum) {
    CU(cudaMemcpyAsync(rb.h_tally, rb.sum, (size_t)rows * 32, cudaMemcpyDeviceToHost, user));
    local.d2h_bytes += rows * 32;
  }
  CU(cudaEventRecord(rb.ev_stop, user));
  CU(cudaEventSynchronize(rb.ev_stop));   // results in host buffers are complete on return
  for (int64_t r = 0; cfg->want_sum && r < rows; ++r) {
    ((double*)cfg->h_sum)[2 * r] = tally[4 * r];
    ((double*)cfg->h_sum)[2 * r + 1] = tally[4 * r + 1];
    if (cfg->h_sumsq) {
      ((double*)cfg->h_sumsq)[2 * r] = tally[4 * r + 2];
      ((double*)cfg->h_sumsq)[2 * r + 1] = tally[4 * r + 3];
    }
  }
  float ms = 0.f;
  CU(cudaEventElapsedTime(&ms, rb.ev_start, rb.ev_stop));
  local.gpu_ms = ms;
  local.kernel_launches = launches;
  if (stats) *stats = local;
  return AMI_OK;
}

// ---------------------------------------------------------------------------------------------
// ami_tally_static: the Monte-Carlo tally of PAPER.md:291 / :295 for callers that must not allocate (code
// under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  ami_run forms the same tally with
// per-block partial sums in a cudaMalloc'ed workspace and a second kernel; here the partial sums and the per-row
// arrival counters live in ONE file-scope device array that every GPU loading the library holds until exit, and
// one kernel does both stages: the CTA that arrives last for a row adds the row's partials in a fixed order.
// ---------------------------------------------------------------------------------------------
namespace {

constexpr int kStaticTallyMaxRows = AMI_TALLY_STATIC_MAX_ROWS;   // result rows (n_b * n_f) per call
constexpr int kStaticTallyMaxPartials = 16384;                   // double4 partial sums over all rows of a call
constexpr size_t kStaticCounterBytes = (size_t)kStaticTallyMaxRows * sizeof(unsigned int);            // 4 KiB
constexpr size_t kStaticTallyBytes = kStaticCounterBytes + (size_t)kStaticTallyMaxPartials * 32;      // 516 KiB
static_assert(kStaticCounterBytes % 256 == 0, "the partial sums start on a 256-byte boundary");
static_assert(kStaticTallyBytes == AMI_TALLY_STATIC_BYTES, "ami.h states the size of the array");

// [0, 4 KiB): arrival counter of each row; [4 KiB, 516 KiB): double4 partial sums [row][block].
// In host code this name is a stand-in, not a device address: static_tally_scratch() asks the runtime for it.
static __device__ __align__(256) unsigned char g_static_tally[kStaticTallyBytes];

// Device address of g_static_tally on the CURRENT device: looked up once per device, with that device current.
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_ptr[kStaticMaxDevices] = {};

cudaError_t static_tally_scratch(int device, void** ptr) {
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[device]) {
    void* p = nullptr;
    const cudaError_t rc = cudaGetSymbolAddress(&p, g_static_tally);
    if (rc != cudaSuccess) return rc;
    g_static_ptr[device] = p;
  }
  *ptr = g_static_ptr[device];
  return cudaSuccess;
}

// grid (blocks per row, rows) x 256 threads.  Stage 1 as row_partial_kernel (ami_kernels.cu): CTA x of row y adds
// its slice of the row, (re, im, re^2, im^2), and stores the partial.  Stage 2: the CTA whose ticket says that all
// others of its row have stored theirs adds the row's partials -- thread t takes partials t, t+256, ... in that
// order, then a tree of fixed shape -- so the result does not depend on WHICH CTA came last.
__global__ void __launch_bounds__(256) tally_static_kernel(const double2* __restrict__ v, long long n,
                                                           long long row_stride, unsigned int* done,
                                                           double4* partial, double4* __restrict__ tally) {
  __shared__ double4 sh[256];
  __shared__ bool last;
  const long long row = blockIdx.y;
  const double2* r = v + row * row_stride;
  const long long per = (n + gridDim.x - 1) / gridDim.x;
  const long long a = blockIdx.x * per, b = a + per < n ? a + per : n;
  double4 acc = make_double4(0.0, 0.0, 0.0, 0.0);
#pragma unroll 4
  for (long long i = a + threadIdx.x; i < b; i += blockDim.x) {
    const double2 x = r[i];
    acc.x += x.x;
    acc.y += x.y;
    acc.z = fma(x.x, x.x, acc.z);
    acc.w = fma(x.y, x.y, acc.w);
  }
  auto block_sum = [&]() {
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
      if (threadIdx.x < w) {
        sh[threadIdx.x].x += sh[threadIdx.x + w].x;
        sh[threadIdx.x].y += sh[threadIdx.x + w].y;
        sh[threadIdx.x].z += sh[threadIdx.x + w].z;
        sh[threadIdx.x].w += sh[threadIdx.x + w].w;
      }
      __syncthreads();
    }
  };
  block_sum();
  if (threadIdx.x == 0) {
    partial[row * gridDim.x + blockIdx.x] = sh[0];
    __threadfence();                                   // the partial is visible before the ticket is taken
    last = atomicAdd(&done[row], 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();                                     // the other CTAs' partials are visible to every thread here
  acc = make_double4(0.0, 0.0, 0.0, 0.0);
  for (int i = threadIdx.x; i < (int)gridDim.x; i += 256) {
    const double2* q = reinterpret_cast<const double2*>(&partial[row * gridDim.x + i]);   // L2 loads: not via a stale L1 line
    const double2 lo = __ldcg(q), hi = __ldcg(q + 1);
    acc.x += lo.x; acc.y += lo.y; acc.z += hi.x; acc.w += hi.y;
  }
  block_sum();
  if (threadIdx.x == 0) tally[row] = sh[0];
}

// blocks per row: a function of (rows, n) only, so the order of the sum is fixed
int static_tally_blocks(long long n_rows, long long n) {
  long long b = (8 * 148 + n_rows - 1) / n_rows;
  b = std::min<long long>(b, (n + 1023) / 1024);
  b = std::min<long long>(b, kStaticTallyMaxPartials / n_rows);
  return (int)std::max<long long>(1, b);
}

}  // namespace

extern "C" int ami_tally_static(int device, const void* d_vals, int64_t n_rows, int64_t n, int64_t row_stride,
                                double* d_tally, void* stream) {
  if (device < 0 || device >= kStaticMaxDevices || n_rows < 0 || n < 0 || (n_rows > 0 && !d_tally) ||
      (n_rows > 0 && n > 0 && !d_vals) || (n_rows > 1 && row_stride < n)) {
    g_cuda_err = "ami_tally_static: bad argument (device, null pointer, negative size, or row_stride < n)";
    return AMI_EINVAL;
  }
  if (n_rows > kStaticTallyMaxRows) {
    g_cuda_err = "ami_tally_static: " + std::to_string((long long)n_rows) + " rows exceed the static workspace's maximum of " +
                 std::to_string(kStaticTallyMaxRows) + " rows per call (split the rows over several calls)";
    return AMI_EUNSUPPORTED;
  }
  CU(cudaSetDevice(device));
  void* scratch = nullptr;
  CU(static_tally_scratch(device, &scratch));   // n_rows = 0: set-up only (do this once before a graph capture)
  if (n_rows == 0) return AMI_OK;
  const cudaStream_t st = (cudaStream_t)stream;
  unsigned int* done = (unsigned int*)scratch;
  double4* partial = (double4*)((unsigned char*)scratch + kStaticCounterBytes);
  // the array keeps what the last call left: the counters of the rows of THIS call start at zero
  CU(cudaMemsetAsync(done, 0, (size_t)n_rows * sizeof(unsigned int), st));
  dim3 grid((unsigned)static_tally_blocks(n_rows, n), (unsigned)n_rows);
  tally_static_kernel<<<grid, 256, 0, st>>>((const double2*)d_vals, n, row_stride, done, partial, (double4*)d_tally);
  ami::count_external_launch(nullptr);
  CU(cudaGetLastError());
  return AMI_OK;
}
