// dex_voigt.cuh -- Voigt function H(a,x) = Re w(x + i a), "HUM1WEI24" (Schreier 2018):
// Humlicek (1982) region I rational for |x| + a >= 15, Weideman (1994) N = 24 expansion otherwise.
// fp64: in fp32 the real part of w is a small difference of O(1/x) terms.
// The Weideman coefficients are not printed in the paper; dex_weideman_coefficients() computes them
// on the host from their definition (cosine sums of f(t) = exp(-t^2)(L^2 + t^2), t = L tan(theta/2)).
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#define DEX_WEI_N 24

// c[n-1] = c_n, n = 1..24;  p(Z) = sum_n c_n Z^{n-1}
inline void dex_weideman_coefficients(double* c, double* L_out) {
  const int N = DEX_WEI_N, M = 2 * N;
  const double pi = 3.14159265358979323846;
  const double L = sqrt((double)N / sqrt(2.0));
  for (int n = 1; n <= N; ++n) {
    double acc = 0.0;
    for (int k = 1 - M; k <= M - 1; ++k) {
      const double theta = pi * (double)k / (double)M;
      const double t = L * tan(0.5 * theta);
      acc += exp(-t * t) * (L * L + t * t) * cos((double)n * theta);
    }
    c[n - 1] = acc / (double)(2 * M);
  }
  *L_out = L;
}

__device__ __forceinline__ double dex_voigt_H(const double* __restrict__ wc, double L, double a, double x) {
  const double inv_sqrt_pi = 0.56418958354775628695;
  if (fabs(x) + a >= 15.0) {
    // w = (i/sqrt(pi)) z / (z^2 - 1/2),  z = x + i a   =>   Re w = (x Im(den) - a Re(den)) / (|den|^2 sqrt(pi))
    const double dr = x * x - a * a - 0.5;
    const double di = 2.0 * a * x;
    return (x * di - a * dr) / (dr * dr + di * di) * inv_sqrt_pi;
  }
  // lmiz = L - i z = (L + a) - i x ;  lpiz = L + i z = (L - a) + i x
  const double lr = L + a, li = -x;
  const double n2 = lr * lr + li * li;
  const double ir = lr / n2, ii = -li / n2;              // 1 / lmiz
  const double pr_ = L - a, pi_ = x;
  const double Zr = pr_ * ir - pi_ * ii, Zi = pr_ * ii + pi_ * ir;   // Z = lpiz / lmiz
  double pr = wc[DEX_WEI_N - 1], pi = 0.0;
#pragma unroll
  for (int n = DEX_WEI_N - 2; n >= 0; --n) {
    const double tr = pr * Zr - pi * Zi + wc[n];
    pi = pr * Zi + pi * Zr;
    pr = tr;
  }
  const double i2r = ir * ir - ii * ii, i2i = 2.0 * ir * ii;          // 1 / lmiz^2
  return 2.0 * (pr * i2r - pi * i2i) + ir * inv_sqrt_pi;
}

// eqs. 14-20: contribution of one line at wavelength lam for projected velocity vproj
__device__ __forceinline__ void dex_line_terms(const double* __restrict__ wc, double L, double lam, double lam0,
                                               double eta_star0, double chi_star0, double a0, double inv_dlamD,
                                               double vproj, double c_light, double& eta_l, double& chi_l) {
  const double x = ((lam - lam0) + (vproj / c_light) * lam0) * inv_dlamD;
  const double r = lam / lam0;
  const double a = r * r * a0;
  const double phi = dex_voigt_H(wc, L, a, x) * inv_dlamD * 0.56418958354775628695;
  const double s = lam0 / lam;
  eta_l = s * eta_star0 * phi;
  chi_l = s * chi_star0 * phi;
}
