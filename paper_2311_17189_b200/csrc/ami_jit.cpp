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

struct Emitter {
  std::ostringstream o;
  int tmp = 0;
  std::string fresh(const char* p) { return std::string(p) + std::to_string(tmp++); }
};

// S_F(n) of group g as a named double (see ami_table.hpp); n has kids
std::string emit_f_sum(const std::vector<HNode>& f, int n, Emitter& E) {
  std::string acc;
  for (int c : f[n].kids) {
    if (f[c].kids.empty()) continue;
    const std::string sc = emit_f_sum(f, c, E);
    const std::string v = E.fresh("s");
    if (acc.empty()) E.o << "      const double " << v << " = F" << f[c].leaf << " * " << sc << ";\n";
    else E.o << "      const double " << v << " = fma(F" << f[c].leaf << ", " << sc << ", " << acc << ");\n";
    acc = v;
  }
  for (int c : f[n].kids) {
    if (!f[c].kids.empty()) continue;
    const bool plus = f[c].num == 1 && f[c].den == 1, minus = f[c].num == -1 && f[c].den == 1;
    const std::string leaf = "F" + std::to_string(f[c].leaf);
    if (acc.empty()) {
      if (plus) { acc = leaf; continue; }
      if (minus) { acc = "(-" + leaf + ")"; continue; }
      const std::string v = E.fresh("s");
      E.o << "      const double " << v << " = " << dlit((double)f[c].num / (double)f[c].den) << " * " << leaf << ";\n";
      acc = v;
      continue;
    }
    const std::string v = E.fresh("s");
    if (plus) E.o << "      const double " << v << " = " << acc << " + " << leaf << ";\n";
    else if (minus) E.o << "      const double " << v << " = " << acc << " - " << leaf << ";\n";
    else
      E.o << "      const double " << v << " = fma(" << dlit((double)f[c].num / (double)f[c].den) << ", " << leaf << ", "
          << acc << ");\n";
    acc = v;
  }
  return acc;
}

struct CV {            // a complex value held in named doubles; im empty = purely real
  std::string re, im;
  bool real() const { return im.empty(); }
};

// S_D(n): group FT at this node plus sum over kids of Dinv[kid.leaf] * S_D(kid)
CV emit_d_sum(const HornerPlan& hp, int n, Emitter& E) {
  CV acc;
  bool have = false;
  if (hp.dn[n].group >= 0) {
    acc.re = "FT" + std::to_string(hp.dn[n].group);
    have = true;
  }
  for (int c : hp.dn[n].kids) {
    const CV s = emit_d_sum(hp, c, E);
    const int u = hp.dn[c].leaf;
    const bool dreal = hp.d_is_real[u] != 0;
    const std::string dr = "Dr" + std::to_string(u), di = "Di" + std::to_string(u);
    CV r;
    r.re = E.fresh("r");
    // real part: dr*s.re - di*s.im (+ acc.re)
    {
      std::string inner = have ? acc.re : "";
      if (!dreal && !s.real()) {
        const std::string t = E.fresh("r");
        if (inner.empty()) E.o << "        const double " << t << " = -" << di << " * " << s.im << ";\n";
        else E.o << "        const double " << t << " = fma(-" << di << ", " << s.im << ", " << inner << ");\n";
        inner = t;
      }
      if (inner.empty()) E.o << "        const double " << r.re << " = " << dr << " * " << s.re << ";\n";
      else E.o << "        const double " << r.re << " = fma(" << dr << ", " << s.re << ", " << inner << ");\n";
    }
    // imaginary part: dr*s.im + di*s.re (+ acc.im)
    {
      std::string inner = (have && !acc.real()) ? acc.im : "";
      if (!s.real()) {
        const std::string t = E.fresh("r");
        if (inner.empty()) E.o << "        const double " << t << " = " << dr << " * " << s.im << ";\n";
        else E.o << "        const double " << t << " = fma(" << dr << ", " << s.im << ", " << inner << ");\n";
        inner = t;
      }
      if (!dreal) {
        const std::string t = E.fresh("r");
        if (inner.empty()) E.o << "        const double " << t << " = " << di << " * " << s.re << ";\n";
        else E.o << "        const double " << t << " = fma(" << di << ", " << s.re << ", " << inner << ");\n";
        inner = t;
      }
      r.im = inner;   // stays empty when the product and the running sum are both real
    }
    acc = r;
    have = true;
  }
  if (!have) acc.re = "0.0";
  return acc;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// The translation unit handed to NVRTC.
// ---------------------------------------------------------------------------------------------
std::string jit_generate_source(const FlatTable& ft, const HornerPlan& hp, int block_threads) {
  const int L = ft.n_int + ft.n_ext;
  Emitter E;
  std::ostringstream& o = E.o;
  o << kAmiParamsSrc << "\n" << kAmiDeviceSrc << "\n";
  o << "using namespace amidev;\n#define AMI_NT " << block_threads << "\n";
  // ---- body: one sample, energies e0..e{n_eps-1} in registers ------------------------------
  o << "__device__ __forceinline__ void ami_body(const AmiBatch& p, const long long s";
  for (int i = 0; i < ft.n_eps; ++i) o << ", const double e" << i;
  o << ") {\n";
  o << "#pragma unroll 1\n  for (int b = 0; b < p.n_b; ++b) {\n    const double beta = p.beta[b];\n";
  // Fermi/Bose leaves (independent of the external frequency)
  for (size_t u = 0; u < ft.leafF.size(); ++u) {
    const LeafF& l = ft.leafF[u];
    std::string arg = combo(l.c, "e");
    if (l.sigma < 0) arg = "(" + arg + ") + p.e_reg";          // P10(a)
    o << "    double F" << u << ";\n    {\n      double f, g;\n      fermi_fg<" << (l.sigma > 0 ? 1 : -1)
      << ", " << (l.k > 0 ? "true" : "false") << ">(beta * (" << arg << "), f, g);\n";
    if (l.k == 0) {
      o << "      F" << u << " = f;\n";
    } else {
      const std::vector<double> q = deriv_poly(l.k);
      o << "      double q = " << dlit(q.back()) << ";\n";
      for (int i = (int)q.size() - 2; i >= 0; --i) o << "      q = fma(q, f, " << dlit(q[i]) << ");\n";
      o << "      double bk = beta;\n";
      for (int i = 1; i < l.k; ++i) o << "      bk *= beta;\n";
      o << "      F" << u << " = bk * f * g * q;\n";
    }
    o << "    }\n";
  }
  // FT sums of every group (per beta)
  for (size_t g = 0; g < hp.groups.size(); ++g) {
    const std::vector<HNode>& f = hp.groups[g].f;
    o << "    double FT" << g << ";\n    {\n";
    if (f[0].kids.empty()) {
      o << "      FT" << g << " = " << dlit(f[0].terminal ? (double)f[0].num / (double)f[0].den : 0.0) << ";\n";
    } else {
      const std::string v = emit_f_sum(f, 0, E);
      o << "      FT" << g << " = " << v << ";\n";
    }
    o << "    }\n";
  }
  // frequencies
  o << "#pragma unroll 1\n    for (int f = 0; f < p.n_f; ++f) {\n";
  for (int x = 0; x < ft.n_ext; ++x) {
    o << "      const double zr" << x << " = p.z[2 * (f * " << ft.n_ext << " + " << x << ")], zi" << x
      << " = p.z[2 * (f * " << ft.n_ext << " + " << x << ") + 1];\n";
    o << "      const bool zz" << x << " = (zr" << x << " == 0.0 && zi" << x << " == 0.0);\n";
  }
  for (size_t u = 0; u < ft.leafD.size(); ++u) {
    const LeafD& l = ft.leafD[u];
    std::string re = combo(l.a, "zr"), im = combo(l.a, "zi"), en = combo(l.c, "e");
    std::string cond;
    for (int x = 0; x < ft.n_ext; ++x)
      if (l.a[x]) cond += (cond.empty() ? "" : " && ") + std::string("zz") + std::to_string(x);
    if (hp.d_is_real[u]) {
      // no frequency part: purely real, regulator always applies (P10(b))
      o << "      const double Dr" << u << " = fast_rcp((" << en << ") + p.e_reg);\n";
    } else {
      o << "      double Dr" << u << ", Di" << u << ";\n      {\n";
      o << "        const cplx d = crcp(cplx{((" << re << ") + (" << en << ")) + ((" << cond << ") ? p.e_reg : 0.0), "
        << im << "});\n";
      o << "        Dr" << u << " = d.re; Di" << u << " = d.im;\n      }\n";
    }
  }
  o << "      {\n";
  const CV res = emit_d_sum(hp, 0, E);
  o << "        double2* out = reinterpret_cast<double2*>(p.out) + ((long long)(p.b0 + b) * p.n_f_total + (p.f0 + f)) * "
       "p.out_row_stride + s;\n";
  o << "        *out = make_double2(p.prefactor * (" << res.re << "), "
    << (res.real() ? std::string("0.0") : "p.prefactor * (" + res.im + ")") << ");\n";
  o << "      }\n    }\n  }\n}\n\n";
  // ---- kernel 1: energies from memory ---------------------------------------------------------
  o << "extern \"C\" __global__ void __launch_bounds__(AMI_NT) ami_jit_eval(const __grid_constant__ AmiBatch p) {\n"
       "  const long long s = blockIdx.x * (long long)AMI_NT + threadIdx.x;\n  if (s >= p.n) return;\n";
  for (int i = 0; i < ft.n_eps; ++i) o << "  const double e" << i << " = p.e[" << i << " * p.e_stride + s];\n";
  o << "  ami_body(p, s";
  for (int i = 0; i < ft.n_eps; ++i) o << ", e" << i;
  o << ");\n}\n\n";
  // ---- kernel 2: momenta from memory, dispersion inline (Eqs. 8-18) ----------
  o << "extern \"C\" __global__ void __launch_bounds__(AMI_NT) ami_jit_fused(const __grid_constant__ AmiBatch p) {\n"
       "  const long long s = blockIdx.x * (long long)AMI_NT + threadIdx.x;\n  if (s >= p.n) return;\n"
       "  const double* ks = p.k + s * p.k_stride_sample;\n";
  for (int l = 0; l < ft.n_int; ++l)
    o << "  const double kx" << l << " = ks[" << 2 * l << " * p.k_stride_comp], ky" << l << " = ks[" << 2 * l + 1
      << " * p.k_stride_comp];\n";
  for (int x = 0; x < ft.n_ext; ++x)
    o << "  const double kx" << ft.n_int + x << " = p.q[" << 2 * x << "], ky" << ft.n_int + x << " = p.q[" << 2 * x + 1
      << "];\n";
  for (int i = 0; i < ft.n_eps; ++i) {
    std::vector<int> a(ft.sym_alpha.begin() + (size_t)i * L, ft.sym_alpha.begin() + (size_t)(i + 1) * L);
    o << "  const double e" << i << " = fma(2.0 * p.t, cos_bounded(" << combo(a, "kx") << ") + cos_bounded(" << combo(a, "ky")
      << "), p.mu);\n";
  }
  o << "  if (p.e_out) {\n";
  for (int i = 0; i < ft.n_eps; ++i) o << "    p.e_out[" << i << " * p.e_stride + s] = e" << i << ";\n";
  o << "  }\n  ami_body(p, s";
  for (int i = 0; i < ft.n_eps; ++i) o << ", e" << i;
  o << ");\n}\n";
  return o.str();
}

bool jit_eligible(const FlatTable& ft, const HornerPlan& hp) {
  if (const char* off = getenv("AMI_DISABLE_JIT"))
    if (off[0] == '1') return false;
  long long leaf_doubles = (long long)ft.leafF.size();
  for (size_t u = 0; u < ft.leafD.size(); ++u) leaf_doubles += hp.d_is_real[u] ? 1 : 2;
  return leaf_doubles <= 160 && hp.n_fnodes + 4 * hp.n_dnodes <= 24000;
}

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
  const char* opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo", "--ptxas-options=-v",
                        "-default-device"};
  const int rc = n.CompileProgram(prog, (int)(sizeof opts / sizeof opts[0]), opts);
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
  CUfunction fn_eval = nullptr, fn_fused = nullptr;
};

namespace {

struct Driver {
  CUresult (*ModuleLoadData)(CUmodule*, const void*) = nullptr;
  CUresult (*ModuleGetFunction)(CUfunction*, CUmodule, const char*) = nullptr;
  CUresult (*ModuleUnload)(CUmodule) = nullptr;
  CUresult (*LaunchKernel)(CUfunction, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, CUstream,
                           void**, void**) = nullptr;
  CUresult (*GetErrorString)(CUresult, const char**) = nullptr;
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
  const std::string src = jit_generate_source(tab->flat, tab->horner, kJitBlockThreads);
  js.status = jit_compile(src, cubin, js.log);
  if (js.status != AMI_OK) { err = js.log; return js.status; }
  Driver& d = driver();
  if (!d.ok) { js.log = "CUDA driver entry points unavailable"; js.status = AMI_ECUDA; err = js.log; return js.status; }
  cudaSetDevice(tab->dev.device);
  cudaFree(nullptr);   // makes the primary context current
  CUresult rc = d.ModuleLoadData(&js.mod, cubin.data());
  if (rc == CUDA_SUCCESS) rc = d.ModuleGetFunction(&js.fn_eval, js.mod, "ami_jit_eval");
  if (rc == CUDA_SUCCESS) rc = d.ModuleGetFunction(&js.fn_fused, js.mod, "ami_jit_fused");
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

cudaError_t jit_launch(const ami_table* tab, bool fused, const AmiBatch& b, cudaStream_t st) {
  const JitState* js = tab->jit;
  if (!js || js->status != AMI_OK) return cudaErrorInvalidDeviceFunction;
  if (b.n == 0) return cudaSuccess;
  AmiBatch copy = b;
  void* args[] = {&copy};
  const unsigned grid = (unsigned)((b.n + kJitBlockThreads - 1) / kJitBlockThreads);
  const CUresult rc = driver().LaunchKernel(fused ? js->fn_fused : js->fn_eval, grid, 1, 1, kJitBlockThreads, 1, 1, 0,
                                            (CUstream)st, args, nullptr);
  return rc == CUDA_SUCCESS ? cudaSuccess : cudaErrorLaunchFailure;
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
