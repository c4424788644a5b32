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

// ---- fp32 evaluation for small damping ---------------------------------------------------------------
// The fp64 Goertzel form above keeps the Core-and-Voigt march on the fp64 pipe (profiles/r01g: 50 % of its
// peak, everything else idle).  For the damping range of solar lines the same number is reached in fp32 from
//     w(z) = e^{-z^2} + (2i / sqrt(pi)) F(z),   F = Dawson's function,   z = x + i a
//     H(a, x) = Re w = e^{a^2 - x^2} cos(2 a x) - (2 / sqrt(pi)) Im F(x + i a),
// which has no cancellation: the Gaussian core and the algebraic wing are separate, positive terms.  F is entire,
// so Im F(x + i a) is summed from its Taylor series about the nearest node x_k = k / 32 of a table,
//     Im F(x_k + zeta) = Im sum_{m=1..4} c_m(k) zeta^m,   zeta = (x - x_k) + i a,   c_m = F^(m)(x_k) / m!,
// and the core is e^{-x_k^2} (tabulated) times short series in the small quantities (x - x_k), a.
// With |x - x_k| <= 1/64 and a <= 0.03 the truncated terms are below 2e-7 of H; measured against the exact
// Voigt function the fp32 evaluation is within 4e-7 relative for |x| + a < 15.  HUM1WEI24 itself deviates from
// the exact function by 2.6e-9 / a relative in the wings (its Weideman part has ~1e-11 ABSOLUTE error), so the
// two agree to <= 8e-7 only for a >= DEX_VF_A_LO; below that, and above DEX_VF_A_HI, the march evaluates the
// literal formula in fp64.  x must be supplied as an unevaluated fp32 pair (hi + lo): the Gaussian core turns an
// error dx into a relative error 2 x dx.
#define DEX_VF_INVDX 32
#define DEX_VF_NODES (15 * DEX_VF_INVDX + 1)
#define DEX_VF_A_LO 0.005f
#define DEX_VF_A_HI 0.03f

// Dawson's function in extended precision: Rybicki's exponentially convergent sampling sum
// F(x) = (1/sqrt(pi)) sum_{n odd} e^{-(x - n h)^2} / n  (error ~ e^{-(pi/h)^2}), h = 1/4.
inline long double dex_dawson_ld(long double x) {
  const long double h = 0.25L, inv_sqrt_pi = 0.564189583547756286948079451560772586L;
  const int n0 = 2 * (int)floorl(x / (2.0L * h)) + 1;   // odd n nearest to x / h
  long double acc = 0.0L;
  for (int j = -40; j <= 40; ++j) {
    const int n = n0 + 2 * j;
    const long double t = x - (long double)n * h;
    acc += expl(-t * t) / (long double)n;
  }
  return acc * inv_sqrt_pi;
}

// wing[k][m-1] = c_m(k) = F^(m)(x_k)/m!, m = 1..4;  core[k] = e^{-x_k^2};  x_k = k / DEX_VF_INVDX
inline void dex_voigt_fast_table(float* wing, float* core) {
  for (int k = 0; k < DEX_VF_NODES; ++k) {
    const long double x = (long double)k / (long double)DEX_VF_INVDX;
    long double c[5];
    if (x < 6.0L) {
      // F' = 1 - 2 x F,  F^(n+1) = -2 x F^(n) - 2 n F^(n-1)
      long double d[5];
      d[0] = dex_dawson_ld(x);
      d[1] = 1.0L - 2.0L * x * d[0];
      for (int n = 1; n < 4; ++n) d[n + 1] = -2.0L * x * d[n] - 2.0L * (long double)n * d[n - 1];
      long double fact = 1.0L;
      for (int m = 1; m <= 4; ++m) { fact *= (long double)m; c[m] = d[m] / fact; }
    } else {
      // the recurrence cancels like x^m at large x; differentiate the asymptotic series term by term instead:
      // F(x) ~ sum_j (2j-1)!! / (2^(j+1) x^(2j+1)),  d^m/dx^m x^-p / m! = (-1)^m C(p+m-1, m) x^-(p+m)
      for (int m = 1; m <= 4; ++m) {
        long double sum = 0.0L, coef = 0.5L, prev = 1e300L;   // coef = (2j-1)!!/2^(j+1)
        for (int j = 0; j < 60; ++j) {
          const int p = 2 * j + 1;
          long double binom = 1.0L;
          for (int i = 1; i <= m; ++i) binom *= (long double)(p + m - i) / (long double)i;
          const long double term = coef * binom * powl(x, -(long double)(p + m));
          if (term >= prev) break;          // asymptotic: stop at the smallest term (< 1e-17 relative for x >= 6)
          sum += term;
          prev = term;
          coef *= (long double)(2 * j + 1) / 2.0L;
        }
        c[m] = (m & 1) ? -sum : sum;
      }
    }
    for (int m = 1; m <= 4; ++m) wing[4 * k + (m - 1)] = (float)c[m];
    core[k] = (float)expl(-x * x);
  }
}

// H(a, x) for DEX_VF_A_LO <= a <= DEX_VF_A_HI and |x| + a < 15, x = xh + xl (|xl| <= ulp(xh)/2).  wing / core: the
// tables above (shared memory in the march).  Branch free, so that the march can interleave the evaluations of a
// batch's wavelengths; for |x| + a >= 15 the value is finite but meaningless and the caller replaces it with
// dex_voigt_H_region1.
__device__ __forceinline__ float dex_voigt_H_table(const float4* __restrict__ wing, const float* __restrict__ core,
                                                   float a, float xh, float xl) {
  const float ax = fminf(fabsf(xh), 15.0f);
  const float el = (fabsf(xh) < 15.0f) ? ((xh < 0.0f) ? -xl : xl) : 0.0f;
  const float t = fmaf(ax, (float)DEX_VF_INVDX, 12582912.0f);      // 2^23 + 2^22: the sum rounds |x| * 32 to an integer
  const int k = __float_as_int(t) - 0x4B400000;
  const float xk = (t - 12582912.0f) * (1.0f / (float)DEX_VF_INVDX);
  const float d = (ax - xk) + el;                                   // ax - xk is exact
  // core: e^{-x_k^2} * e^{a^2 - d (2 x_k + d)} * cos(2 a x)
  const float s = fmaf(a, a, -d * fmaf(2.0f, xk, d));
  float ex = fmaf(s, 1.0f / 120.0f, 1.0f / 24.0f);
  ex = fmaf(ex, s, 1.0f / 6.0f);
  ex = fmaf(ex, s, 0.5f);
  ex = fmaf(ex, s, 1.0f);
  ex = fmaf(ex, s, 1.0f);
  const float ph = 2.0f * a * ax, u = ph * ph;
  float cs = fmaf(u, 1.0f / 40320.0f, -1.0f / 720.0f);
  cs = fmaf(cs, u, 1.0f / 24.0f);
  cs = fmaf(cs, u, -0.5f);
  cs = fmaf(cs, u, 1.0f);
  const float g = core[k];
  const float4 c = wing[k];
  // Im[((c4 zeta + c3) zeta + c2) zeta + c1) zeta],  zeta = d + i a
  float sr = fmaf(c.w, d, c.z), si = c.w * a;
  float tr = fmaf(sr, d, fmaf(-si, a, c.y));
  si = fmaf(sr, a, si * d);
  sr = tr;
  tr = fmaf(sr, d, fmaf(-si, a, c.x));
  si = fmaf(sr, a, si * d);
  sr = tr;
  const float im = fmaf(sr, a, si * d);
  return fmaf(-1.1283791670955126f, im, g * ex * cs);
}

// The same for two wavelengths at once on Blackwell's packed fp32 pipe (FFMA2 / FMUL2 / FADD2): the Core-and-Voigt
// march is bound by instruction issue (profiles/r01h), and a packed instruction does two evaluations per slot.
__device__ __forceinline__ float2 dex_f2(float v) { return make_float2(v, v); }
__device__ __forceinline__ float2 dex_neg2(float2 v) { return make_float2(-v.x, -v.y); }
__device__ __forceinline__ float dex_xorsign(float v, float s) {
  return __int_as_float(__float_as_int(v) ^ (__float_as_int(s) & 0x80000000));
}
__device__ __forceinline__ float2 dex_voigt_H_table2(const float4* __restrict__ wing, const float* __restrict__ core,
                                                     float2 a, float2 xh, float2 xl) {
  const float2 ax = make_float2(fminf(fabsf(xh.x), 15.0f), fminf(fabsf(xh.y), 15.0f));
  const float2 el = make_float2(dex_xorsign(xl.x, xh.x), dex_xorsign(xl.y, xh.y));   // only read where |x| < 15
  const float2 t = __ffma2_rn(ax, dex_f2((float)DEX_VF_INVDX), dex_f2(12582912.0f));
  const int k0 = __float_as_int(t.x) - 0x4B400000, k1 = __float_as_int(t.y) - 0x4B400000;
  const float2 xk = __fmul2_rn(__fadd2_rn(t, dex_f2(-12582912.0f)), dex_f2(1.0f / (float)DEX_VF_INVDX));
  const float2 d = __fadd2_rn(__fadd2_rn(ax, dex_neg2(xk)), el);
  const float2 s = __ffma2_rn(dex_neg2(d), __ffma2_rn(dex_f2(2.0f), xk, d), __fmul2_rn(a, a));
  float2 ex = __ffma2_rn(s, dex_f2(1.0f / 120.0f), dex_f2(1.0f / 24.0f));
  ex = __ffma2_rn(ex, s, dex_f2(1.0f / 6.0f));
  ex = __ffma2_rn(ex, s, dex_f2(0.5f));
  ex = __ffma2_rn(ex, s, dex_f2(1.0f));
  ex = __ffma2_rn(ex, s, dex_f2(1.0f));
  const float2 ph = __fmul2_rn(__fadd2_rn(a, a), ax), u = __fmul2_rn(ph, ph);
  float2 cs = __ffma2_rn(u, dex_f2(1.0f / 40320.0f), dex_f2(-1.0f / 720.0f));
  cs = __ffma2_rn(cs, u, dex_f2(1.0f / 24.0f));
  cs = __ffma2_rn(cs, u, dex_f2(-0.5f));
  cs = __ffma2_rn(cs, u, dex_f2(1.0f));
  const float2 g = make_float2(core[k0], core[k1]);
  const float4 c0 = wing[k0], c1 = wing[k1];
  const float2 na = dex_neg2(a);
  float2 sr = __ffma2_rn(make_float2(c0.w, c1.w), d, make_float2(c0.z, c1.z));
  float2 si = __fmul2_rn(make_float2(c0.w, c1.w), a);
  float2 tr = __ffma2_rn(sr, d, __ffma2_rn(si, na, make_float2(c0.y, c1.y)));
  si = __ffma2_rn(sr, a, __fmul2_rn(si, d));
  sr = tr;
  tr = __ffma2_rn(sr, d, __ffma2_rn(si, na, make_float2(c0.x, c1.x)));
  si = __ffma2_rn(sr, a, __fmul2_rn(si, d));
  sr = tr;
  const float2 im = __ffma2_rn(sr, a, __fmul2_rn(si, d));
  return __ffma2_rn(dex_f2(-1.1283791670955126f), im, __fmul2_rn(__fmul2_rn(g, ex), cs));
}

// |x| + a >= 15: region I of Humlicek (1982) in the cancellation-free form of dex_voigt_H_march, fine in fp32
__device__ __forceinline__ float dex_voigt_H_region1(float a, float xh) {
  const float ax = fminf(fabsf(xh), 1.0e9f);
  const float x2 = ax * ax, a2 = a * a;
  const float dr = x2 - a2 - 0.5f, di = 2.0f * a * ax;
  return __fdividef((a * 0.5641895835477563f) * (x2 + a2 + 0.5f), fmaf(dr, dr, di * di));
}

__device__ __forceinline__ float dex_voigt_H_fast(const float4* __restrict__ wing, const float* __restrict__ core,
                                                  float a, float xh, float xl) {
  return (fabsf(xh) + a >= 15.0f) ? dex_voigt_H_region1(a, xh) : dex_voigt_H_table(wing, core, a, xh, xl);
}
