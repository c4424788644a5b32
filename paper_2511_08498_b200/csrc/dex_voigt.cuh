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

// ---- march-side evaluation ---------------------------------------------------------------------------
// The same HUM1WEI24 formula, arranged for the march's inner loop (one evaluation per segment, wavelength and
// active line: the Core-and-Voigt path is bound by this arithmetic, profiles/).  Still fp64 where the formula
// cancels, but
//   * p(Z) has REAL coefficients, so Horner at the complex point Z is done on the quadratic Z^2 - rZ + s
//     (r = 2 Re Z, s = |Z|^2; Goertzel / Knuth 4.6.4): b_k = c_k + r b_{k+1} - s b_{k+2}, p = c_0 + Z b_1 - s b_2:
//     2 DFMA per coefficient instead of 4, and the -s b_{k+2} term is off the critical path;
//   * the one reciprocal is an fp32 MUFU.RCP seed refined by two fp64 Newton steps (no division subroutine);
//   * region I is written as a (x^2 + a^2 + 1/2) / |z^2 - 1/2|^2, which has no cancellation.
// Agreement with dex_voigt_H: <= 5e-11 relative for |x| + a < 15 (checked in tests through the intensities).
__device__ __forceinline__ double dex_rcp64(double v) {
  float s;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"((float)v));
  double r = (double)s;
  r = fma(r, fma(-v, r, 1.0), r);
  r = fma(r, fma(-v, r, 1.0), r);
  return r;
}

__device__ __forceinline__ double dex_voigt_H_march(const double* __restrict__ wc, double L, double a, double x) {
  const double inv_sqrt_pi = 0.56418958354775628695;
  const double x2 = x * x;
  if (fabs(x) + a >= 15.0) {
    const double a2 = a * a;
    const double dr = x2 - a2 - 0.5;
    const double di = 2.0 * a * x;
    return (a * inv_sqrt_pi) * (x2 + a2 + 0.5) * dex_rcp64(fma(dr, dr, di * di));
  }
  // 1/(L - i z) = ((L + a) + i x) / ((L + a)^2 + x^2);  Z = (L + i z)/(L - i z),  L + i z = (L - a) + i x
  const double lr = L + a, pr_ = L - a;
  const double inv = dex_rcp64(fma(lr, lr, x2));
  const double ir = lr * inv, ii = x * inv;
  const double Zr = fma(pr_, ir, -(x * ii)), Zi = fma(pr_, ii, x * ir);
  const double r = Zr + Zr, ns = -fma(Zr, Zr, Zi * Zi);
  double b1 = wc[DEX_WEI_N - 1], b2 = 0.0;
#pragma unroll
  for (int n = DEX_WEI_N - 2; n >= 1; --n) {
    const double b0 = fma(r, b1, fma(ns, b2, wc[n]));
    b2 = b1;
    b1 = b0;
  }
  const double pr = fma(Zr, b1, fma(ns, b2, wc[0]));
  const double pi = Zi * b1;
  const double i2r = fma(ir, ir, -(ii * ii)), i2i = 2.0 * ir * ii;   // 1/(L - i z)^2
  return fma(2.0, fma(pr, i2r, -(pi * i2i)), ir * inv_sqrt_pi);
}
