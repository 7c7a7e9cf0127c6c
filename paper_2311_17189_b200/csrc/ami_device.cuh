// Device-side arithmetic shared by the evaluation kernels: complex helpers, fast reciprocals,
// overflow-safe Fermi/Bose functions and their derivatives (readings P11, P12).
#ifndef AMI_DEVICE_CUH
#define AMI_DEVICE_CUH
#ifndef __CUDACC_RTC__
#include <cuda_runtime.h>
#endif

namespace amidev {

struct cplx {
  double re, im;
};
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return cplx{fma(a.re, b.re, -a.im * b.im), fma(a.re, b.im, a.im * b.re)};
}
__device__ __forceinline__ cplx cscale(double s, cplx a) { return cplx{s * a.re, s * a.im}; }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return cplx{a.re + b.re, a.im + b.im}; }

// 1/x to 1 ulp for normal x: hardware seed (MUFU.RCP64H, measured max relative error 2^-19.9 on
// B200) + ONE third-order step r(1 + e + e^2), e = 1 - x r (error e^3 = 2^-60; measured max error
// 1.00 ulp over 4M arguments across 600 binades), no branch.  x = 0, inf or nan give a non-finite
// result (0 * inf in the correction), as the division would for the singular samples it stands
// for; arguments below 1e-290 in magnitude are outside the method's range (reading P10).
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  const double t = fma(e, e, e);
  return fma(r, t, r);
}
// The same for N independent arguments, step by step across the batch: the correction is three
// dependent DFMAs, so a batch gives the FP64 pipe N independent instructions per step.
template <int N>
__device__ __forceinline__ void fast_rcp_n(double (&x)[N]) {
  double r[N], e[N];
#pragma unroll
  for (int j = 0; j < N; ++j) asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r[j]) : "d"(x[j]));
#pragma unroll
  for (int j = 0; j < N; ++j) e[j] = fma(-x[j], r[j], 1.0);
#pragma unroll
  for (int j = 0; j < N; ++j) e[j] = fma(e[j], e[j], e[j]);
#pragma unroll
  for (int j = 0; j < N; ++j) x[j] = fma(r[j], e[j], r[j]);
}
__device__ __forceinline__ cplx crcp(cplx a) {
  const double n = fma(a.re, a.re, a.im * a.im);
  const double r = fast_rcp(n);
  return cplx{a.re * r, -a.im * r};
}

// ---- exponential core ---------------------------------------------------------------------------
// e^x = 2^n (1 + r q(r)),  n = rint(x log2 e),  r = x - n ln 2 in [-0.347, 0.347],
// q(r) ~ (e^r - 1)/r as a degree-10 Chebyshev-node fit on that interval (max error of e^r 7e-18).  The coefficients sit in constant memory so
// that every DFMA takes its constant straight from the bank (no register moves).  n is clamped to
// [-1021, 1010] in the integer domain: beyond it the Fermi/Bose value is 0 or 1 to double precision.
// Returns s = 2^n and rq = r q(r):  e^x = fma(s, rq, s),  e^x - 1 = fma(s, rq, s - 1).
__constant__ double kAmiExpQ[11] = {
    1.0, 0.5000000000000006, 0.1666666666666667, 0.04166666666657314, 0.008333333333326141, 0.0013888888932488599,
    0.00019841269874800493, 2.4801504346997686e-05, 2.7557255425746435e-06, 2.7626357241447223e-07,
    2.510520637395701e-08};

template <int N>
__device__ __forceinline__ void exp_core_n(const double (&x)[N], double (&s)[N], double (&rq)[N]) {
  double t[N], r[N], q[N];
#pragma unroll
  for (int j = 0; j < N; ++j) t[j] = fma(x[j], 1.4426950408889634, 6755399441055744.0);
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const double nd = t[j] - 6755399441055744.0;
    r[j] = fma(nd, -0.6931471805599453, x[j]);
    r[j] = fma(nd, -2.3190468138462996e-17, r[j]);
    q[j] = kAmiExpQ[10];
  }
#pragma unroll
  for (int i = 9; i >= 0; --i) {
#pragma unroll
    for (int j = 0; j < N; ++j) q[j] = fma(q[j], r[j], kAmiExpQ[i]);
  }
#pragma unroll
  for (int j = 0; j < N; ++j) {
    rq[j] = r[j] * q[j];
    int n = __double2loint(t[j]);
    n = max(-1021, min(1010, n));
    s[j] = __hiloint2double((n + 1023) << 20, 0);
  }
}
// e^x = 2^n m with integer n (not clamped) and m = 1 + r q(r) in [0.70, 1.42]: the form in which
// exponentials of SUMS are built from exponentials of the summands without ever overflowing
// (exponents add as integers, mantissas multiply).
template <int N>
__device__ __forceinline__ void exp_split_n(const double (&x)[N], int (&n)[N], double (&m)[N]) {
  double t[N], r[N], q[N];
#pragma unroll
  for (int j = 0; j < N; ++j) t[j] = fma(x[j], 1.4426950408889634, 6755399441055744.0);
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const double nd = t[j] - 6755399441055744.0;
    r[j] = fma(nd, -0.6931471805599453, x[j]);
    r[j] = fma(nd, -2.3190468138462996e-17, r[j]);
    q[j] = kAmiExpQ[10];
  }
#pragma unroll
  for (int i = 9; i >= 0; --i) {
#pragma unroll
    for (int j = 0; j < N; ++j) q[j] = fma(q[j], r[j], kAmiExpQ[i]);
  }
#pragma unroll
  for (int j = 0; j < N; ++j) {
    m[j] = fma(r[j], q[j], 1.0);
    n[j] = __double2loint(t[j]);
  }
}
// 2^n with n clamped to [-1021, 1010] (beyond it a Fermi/Bose value is 0 or 1 to double precision)
__device__ __forceinline__ double pow2_clamped(int n) {
  n = max(-1021, min(1010, n));
  return __hiloint2double((n + 1023) << 20, 0);
}

__device__ __forceinline__ void exp_core(double x, double& s, double& rq) {
  double xa[1] = {x}, sa[1], ra[1];
  exp_core_n<1>(xa, sa, ra);
  s = sa[0];
  rq = ra[0];
}

// ---- cosine of a bounded argument -----------------------------------------------------------------
// cos K = (-1)^n cos r,  n = rint(K/pi),  r = K - n pi in [-pi/2, pi/2] (two-part pi, exact for
// |K| < 5e5), even Taylor polynomial of degree 20 (next term 1.9e-17).  A degree-16 fit (5e-17) is two FMAs
// cheaper but differs from the correctly rounded cosine in the last bit often enough that results
// which are ill-conditioned in the ENERGIES (double pole at zero frequency) moved by 4e-11 against a
// quad-precision check fed with libm energies; this one stays at 5e-13.  Momentum sums of a diagram
// are a few pi; anything beyond 5e5 takes the library routine.
__constant__ double kAmiCosC[11] = {
    1.0, -0.5, 0.041666666666666664, -0.001388888888888889, 2.48015873015873e-05, -2.755731922398589e-07,
    2.08767569878681e-09, -1.1470745597729725e-11, 4.779477332387385e-14, -1.5619206968586225e-16,
    4.110317623312165e-19};

__device__ __noinline__ double cos_unbounded(double K) { return cos(K); }

template <int N>
__device__ __forceinline__ void cos_bounded_n(double (&K)[N]) {
  double t[N], r[N], r2[N], c[N];
#pragma unroll
  for (int j = 0; j < N; ++j) t[j] = fma(K[j], 0.3183098861837907, 6755399441055744.0);
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const double nd = t[j] - 6755399441055744.0;
    r[j] = fma(nd, -3.1415926534682512, K[j]);
    r[j] = fma(nd, -1.2154201013012384e-10, r[j]);
    r2[j] = r[j] * r[j];
    c[j] = kAmiCosC[10];
  }
#pragma unroll
  for (int i = 9; i >= 0; --i) {
#pragma unroll
    for (int j = 0; j < N; ++j) c[j] = fma(c[j], r2[j], kAmiCosC[i]);
  }
  double v[N];
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const int flip = (__double2loint(t[j]) & 1) << 31;
    v[j] = __hiloint2double(__double2hiint(c[j]) ^ flip, __double2loint(c[j]));
    asm volatile("" : "+d"(v[j]));   // keeps the batch together: the rare path below must not pull it apart
  }
  // |K| >= 5e5, inf, nan anywhere in the batch: the library routine for those elements (never taken
  // for momentum sums of a diagram).  One test per batch: the largest high word decides.
  int big = 0;
#pragma unroll
  for (int j = 0; j < N; ++j) big = max(big, __double2hiint(K[j]) & 0x7fffffff);
  if (big >= 0x411e8480) {
#pragma unroll
    for (int j = 0; j < N; ++j)
      if ((__double2hiint(K[j]) & 0x7fffffff) >= 0x411e8480) v[j] = cos_unbounded(K[j]);
  }
#pragma unroll
  for (int j = 0; j < N; ++j) K[j] = v[j];
}
__device__ __forceinline__ double cos_bounded(double K) {
  double a[1] = {K};
  cos_bounded_n<1>(a);
  return a[0];
}

// Counter-based momenta (reading P22; specification in ami_inputs/rng.py): splitmix64 finaliser of
// seed + GOLDEN (ctr + 1), top 53 bits, k = (u - 1/2) 2 pi with one correctly rounded multiply.
// momentum_from_state takes z = seed + GOLDEN (ctr + 1) so that consecutive counters cost an addition.
__device__ __forceinline__ double momentum_from_state(unsigned long long z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  z = z ^ (z >> 31);
  return __dmul_rn((double)(z >> 11) * 0x1.0p-53 - 0.5, 6.283185307179586);
}
__device__ __forceinline__ double momentum_of(unsigned long long seed, unsigned long long ctr) {
  return momentum_from_state(seed + 0x9E3779B97F4A7C15ull * (ctr + 1ull));
}

// f_sigma(E) = 1/(sigma e^x + 1) and g = 1 - f = sigma e^x f for x = beta E, any real x, without
// overflow, cancellation, branch or select (reading P12): sigma = +1 uses 1 + e^x = fma(s, rq, s + 1),
// sigma = -1 uses 1 - e^x = -fma(s, rq, s - 1), which is exact where e^x is close to 1 (n = 0: -rq).
template <int SIG, bool WANT_G>
__device__ __forceinline__ void fermi_fg(double x, double& f, double& g) {
  double s, rq;
  exp_core(x, s, rq);
  if (SIG > 0) {
    f = fast_rcp(fma(s, rq, s + 1.0));
    if (WANT_G) g = fma(s, rq, s) * f;
  } else {
    f = -fast_rcp(fma(s, rq, s - 1.0));
    if (WANT_G) g = -fma(s, rq, s) * f;
  }
}

// f^{(k)} = beta^k f g Q_k(f), Q_1 = -1, Q_{k+1} = (2f-1) Q_k - (f - f^2) Q_k'   (from f' = -beta f g,
// g' = beta f g, g = 1 - f).  Q holds the integer coefficients, row k, ascending powers of f.
#define AMI_QSTRIDE 8

// real argument, run-time statistics and derivative order (table-driven kernels)
__device__ __forceinline__ double fermi_real(double E, double beta, int sigma, int k,
                                             const double* __restrict__ Q) {
  double f, g;
  if (sigma > 0) fermi_fg<1, true>(beta * E, f, g);
  else fermi_fg<-1, true>(beta * E, f, g);
  if (k == 0) return f;
  double q = Q[k * AMI_QSTRIDE + (k - 1)];
  for (int i = k - 2; i >= 0; --i) q = fma(q, f, Q[k * AMI_QSTRIDE + i]);
  double bk = beta;
  for (int i = 1; i < k; ++i) bk *= beta;
  return bk * f * g * q;
}

// complex argument (complex energies, reading P19 variant 5b)
__device__ __forceinline__ cplx fermi_cplx(cplx E, double beta, int sigma, int k,
                                           const double* __restrict__ Q) {
  const double xr = beta * E.re, xi = beta * E.im;
  const bool pos = xr > 0.0;
  // y = x if Re x <= 0 else -x, so that |e^y| <= 1
  const double yr = pos ? -xr : xr, yi = pos ? -xi : xi;
  double s, c;
  sincos(yi, &s, &c);
  const double m = exp(yr);
  const cplx u{m * c, m * s};
  cplx den;   // 1 + sigma e^y, formed without cancellation for sigma = -1
  if (sigma > 0) {
    den = cplx{1.0 + u.re, u.im};
  } else {
    double sh, ch;
    sincos(0.5 * yi, &sh, &ch);
    // -(e^y - 1) = -(expm1(yr) cos yi - 2 sin^2(yi/2)) - i e^{yr} sin yi
    den = cplx{-(expm1(yr) * c - 2.0 * sh * sh), -u.im};
  }
  const cplx inv = crcp(den);
  const cplx su = sigma > 0 ? u : cplx{-u.re, -u.im};
  const cplx small = cmul(su, inv);
  const cplx f = pos ? small : inv;
  const cplx g = pos ? inv : small;
  if (k == 0) return f;
  cplx q{Q[k * AMI_QSTRIDE + (k - 1)], 0.0};
  for (int i = k - 2; i >= 0; --i) {
    q = cmul(q, f);
    q.re += Q[k * AMI_QSTRIDE + i];
  }
  double bk = beta;
  for (int i = 1; i < k; ++i) bk *= beta;
  return cscale(bk, cmul(cmul(f, g), q));
}

}  // namespace amidev
#endif  // AMI_DEVICE_CUH
