// Device-side arithmetic shared by the evaluation kernels: complex helpers, fast reciprocals,
// overflow-safe Fermi/Bose functions and their derivatives (readings P11, P12).
#pragma once
#include <cuda_runtime.h>

namespace amidev {

struct cplx {
  double re, im;
};
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return cplx{fma(a.re, b.re, -a.im * b.im), fma(a.re, b.im, a.im * b.re)};
}
__device__ __forceinline__ cplx cscale(double s, cplx a) { return cplx{s * a.re, s * a.im}; }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return cplx{a.re + b.re, a.im + b.im}; }

// 1/x to ~1 ulp: hardware seed (MUFU.RCP64H) + two Newton steps.  Falls back to the IEEE
// division when the seed is not a normal number (0, inf, nan, denormal range), so that
// singular samples produce the same non-finite results as the division would.
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  const double ax = fabs(x);
  if (!(ax > 1e-290 && ax < 1e290)) r = 1.0 / x;
  return r;
}
__device__ __forceinline__ cplx crcp(cplx a) {
  const double n = fma(a.re, a.re, a.im * a.im);
  const double r = fast_rcp(n);
  return cplx{a.re * r, -a.im * r};
}

// f^{(k)} = beta^k f g Q_k(f), Q_1 = -1, Q_{k+1} = (2f-1) Q_k - (f - f^2) Q_k'   (from f' = -beta f g,
// g' = beta f g, g = 1 - f).  Q holds the integer coefficients, row k, ascending powers of f.
#define AMI_QSTRIDE 8

// real argument.  f_sigma(E) = 1/(sigma e^{beta E} + 1); the exponential is only ever taken of
// -|x| (no overflow) and 1 - e^{-|x|} comes from expm1 for sigma = -1 (no cancellation).
__device__ __forceinline__ double fermi_real(double E, double beta, int sigma, int k,
                                             const double* __restrict__ Q) {
  const double x = beta * E;
  const double ax = -fabs(x);
  const double u = exp(ax);
  double f, g;
  if (sigma > 0) {
    const double inv = fast_rcp(1.0 + u);
    const double small = u * inv;
    f = x > 0.0 ? small : inv;
    g = x > 0.0 ? inv : small;
  } else {
    const double inv = fast_rcp(-expm1(ax));
    const double small = -u * inv;
    f = x > 0.0 ? small : inv;
    g = x > 0.0 ? inv : small;
  }
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
