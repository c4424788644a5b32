// march.cu -- a5-a10: ray set-up, HDDA traversal, emissivity/opacity providers, segment integral,
// fused angular reduction to J, and the visit-list capture kernel.
//
// Mapping: LPR lanes share one probe and hold W/LPR wavelengths each, so one
// cell fetch of a ray is a single contiguous [cell][lambda][eta,chi] read split across its lanes;
// consecutive lane groups of a warp are consecutive probes (neighbouring voxels) tracing the same
// direction at the same time, so brick / level lookups and cell fetches of a warp hit the same lines.
// Each lane group loops over all quadrature directions and accumulates J in registers: the angular
// reduction needs no atomics and is deterministic.
#include <mutex>

#include "dex_internal.h"
#include "dex_voigt.cuh"

namespace {

__device__ __forceinline__ float dex_ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float dex_rcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// I_out = I_in e^{-tau} + eta h ds E(tau), E(tau) = (1 - e^{-tau})/tau, accumulated front to back from
// the probe outward:  I += T * eta h ds E(tau);  T *= e^{-tau}   (eq. 3 with constant eta, chi;
// PAPER.md:31-34, :347).  E needs expm1 quality in the thin regime: Taylor series
// to degree 6 below tau = 0.25 (truncation < 1.6e-9), (1 - e)/tau above.  hl = -hds * log2(e).
__device__ __forceinline__ void dex_accumulate(float eta, float chi, float hds, float hl, float& I, float& T) {
  const float tau = chi * hds;
  const float e = dex_ex2(chi * hl);
  float p = -1.0f / 5040.0f;
  p = fmaf(p, tau, 1.0f / 720.0f);
  p = fmaf(p, tau, -1.0f / 120.0f);
  p = fmaf(p, tau, 1.0f / 24.0f);
  p = fmaf(p, tau, -1.0f / 6.0f);
  p = fmaf(p, tau, 0.5f);
  p = fmaf(-p, tau, 1.0f);
  const float ome = 1.0f - e;
  const float q = ome * dex_rcp(fmaxf(tau, 0.25f));
  const bool thin = tau < 0.25f;
  const float E = thin ? p : q;
  I = fmaf(T, (eta * hds) * E, I);
  // T <- T e^-tau as T - T (1 - e^-tau) with the expm1-quality (1 - e^-tau): in the thin regime the product of a
  // thousand ex2.approx results (2^-22 each) is what limited long rays to ~1e-5; one rounding per segment now
  T = fmaf(-T, thin ? tau * p : ome, T);
}

// The same for two wavelengths at once with Blackwell's packed fp32 pipe (FFMA2 / FMUL2): the kernel is
// instruction-issue bound (profiles/), and a packed instruction does two wavelengths per issue slot.
__device__ __forceinline__ void dex_accumulate2(float2 eta, float2 chi, float2 hds2, float2 hl2, float2& I, float2& T) {
  const float2 tau = __fmul2_rn(chi, hds2);
  const float2 y = __fmul2_rn(chi, hl2);
  float2 e;
  e.x = dex_ex2(y.x);
  e.y = dex_ex2(y.y);
  float2 p = make_float2(-1.0f / 5040.0f, -1.0f / 5040.0f);
  p = __ffma2_rn(p, tau, make_float2(1.0f / 720.0f, 1.0f / 720.0f));
  p = __ffma2_rn(p, tau, make_float2(-1.0f / 120.0f, -1.0f / 120.0f));
  p = __ffma2_rn(p, tau, make_float2(1.0f / 24.0f, 1.0f / 24.0f));
  p = __ffma2_rn(p, tau, make_float2(-1.0f / 6.0f, -1.0f / 6.0f));
  p = __ffma2_rn(p, tau, make_float2(0.5f, 0.5f));
  p = __ffma2_rn(p, make_float2(-tau.x, -tau.y), make_float2(1.0f, 1.0f));
  float2 r;
  r.x = dex_rcp(fmaxf(tau.x, 0.25f));
  r.y = dex_rcp(fmaxf(tau.y, 0.25f));
  const float2 ome = __ffma2_rn(e, make_float2(-1.0f, -1.0f), make_float2(1.0f, 1.0f));
  const float2 q = __fmul2_rn(ome, r);
  const float2 tp = __fmul2_rn(tau, p);
  float2 E, w;
  E.x = (tau.x < 0.25f) ? p.x : q.x;
  E.y = (tau.y < 0.25f) ? p.y : q.y;
  w.x = (tau.x < 0.25f) ? tp.x : ome.x;
  w.y = (tau.y < 0.25f) ? tp.y : ome.y;
  I = __ffma2_rn(T, __fmul2_rn(__fmul2_rn(eta, hds2), E), I);
  T = __ffma2_rn(make_float2(-T.x, -T.y), w, T);      // T - T (1 - e^-tau), see dex_accumulate
}

// ISO march records (make_march_records_kernel): plane 0 holds chi2 = chi log2(e), plane 1 holds S = eta/chi.
//   y = -chi2 h ds  (= -tau log2 e),  e = 2^y = e^-tau,  I += T S (1 - e),  T *= e.
// 1 - e needs expm1 quality in the thin regime: below tau = 1/8 it is the degree-5 Taylor
// polynomial of -expm1(y ln 2) in y (truncation < 4.2e-8 relative), above it 1 - ex2(y) (error of ex2.approx
// relative to 1 - e^-1/8: < 1e-6).  Everything but the two MUFUs and the two selects of a wavelength pair is a
// packed FFMA2 / FMUL2: the kernel is issue-bound (profiles/), a packed instruction does two wavelengths per slot.
#define DEX_OME_A1 -0.6931471805599453f      // -ln2
#define DEX_OME_A2 -0.2402265069591007f      // -ln2^2 / 2
#define DEX_OME_A3 -0.05550410866482158f     // -ln2^3 / 6
#define DEX_OME_A4 -0.009618129107628477f    // -ln2^4 / 24
#define DEX_OME_A5 -0.0013333558146428443f   // -ln2^5 / 120
#define DEX_OME_YTHR -0.18033688011112042f   // -(1/8) log2(e)

__device__ __forceinline__ void dex_accumulate_S2(float2 S, float2 chi2, float2 nhds2, float2& I, float2& T) {
  const float2 y = __fmul2_rn(chi2, nhds2);
  float2 e;
  e.x = dex_ex2(y.x);
  e.y = dex_ex2(y.y);
  float2 p = __ffma2_rn(make_float2(DEX_OME_A5, DEX_OME_A5), y, make_float2(DEX_OME_A4, DEX_OME_A4));
  p = __ffma2_rn(p, y, make_float2(DEX_OME_A3, DEX_OME_A3));
  p = __ffma2_rn(p, y, make_float2(DEX_OME_A2, DEX_OME_A2));
  p = __ffma2_rn(p, y, make_float2(DEX_OME_A1, DEX_OME_A1));
  p = __fmul2_rn(p, y);
  if (y.x < DEX_OME_YTHR) p.x = 1.0f - e.x;
  if (y.y < DEX_OME_YTHR) p.y = 1.0f - e.y;
  I = __ffma2_rn(T, __fmul2_rn(S, p), I);
  T = __ffma2_rn(make_float2(-T.x, -T.y), p, T);      // T - T (1 - e^-tau), see dex_accumulate
}

__device__ __forceinline__ void dex_accumulate_S1(float S, float chi2, float nhds, float& I, float& T) {
  const float y = chi2 * nhds;
  const float e = dex_ex2(y);
  float p = fmaf(DEX_OME_A5, y, DEX_OME_A4);
  p = fmaf(p, y, DEX_OME_A3);
  p = fmaf(p, y, DEX_OME_A2);
  p = fmaf(p, y, DEX_OME_A1);
  p *= y;
  if (y < DEX_OME_YTHR) p = 1.0f - e;
  I = fmaf(T, S * p, I);
  T = fmaf(-T, p, T);
}

template <int LPT>
__device__ __forceinline__ void dex_accumulate_all_S(const float (&S)[LPT], const float (&chi2)[LPT], float hds,
                                                     float (&I)[LPT], float (&T)[LPT]) {
  const float nhds = -hds;
  if (LPT == 1) {
    dex_accumulate_S1(S[0], chi2[0], nhds, I[0], T[0]);
  } else {
    const float2 nhds2 = make_float2(nhds, nhds);
#pragma unroll
    for (int i = 0; i < LPT / 2; ++i) {
      float2 Ii = make_float2(I[2 * i], I[2 * i + 1]), Ti = make_float2(T[2 * i], T[2 * i + 1]);
      dex_accumulate_S2(make_float2(S[2 * i], S[2 * i + 1]), make_float2(chi2[2 * i], chi2[2 * i + 1]), nhds2, Ii, Ti);
      I[2 * i] = Ii.x; I[2 * i + 1] = Ii.y;
      T[2 * i] = Ti.x; T[2 * i + 1] = Ti.y;
    }
  }
}

// Providers that deliver (eta, chi) instead of march records (velocity interpolation, Core-and-Voigt, Classic): the
// record form is made on the fly, chi' = max(chi, 2^-60), S = eta rcp(chi'), and the S integrator above does the rest
// -- one MUFU.RCP per wavelength buys ~10 fewer issue slots per wavelength pair than the E(tau) form below (the kernel
// is issue-bound, profiles/).  chi < 2^-60 (a pure emitter) gives S (1 - e^-tau) = eta h ds to 1e-18 h ds.
#define DEX_CHI_TINY 8.673617379884035e-19f      // 2^-60
template <int LPT>
__device__ __forceinline__ void dex_accumulate_all_EC(const float (&eta)[LPT], const float (&chi)[LPT], float hds,
                                                      float (&I)[LPT], float (&T)[LPT]) {
  const float nhl = hds * -1.4426950408889634f;      // y = chi' (-h ds log2 e)
  if (LPT == 1) {
    const float c = fmaxf(chi[0], DEX_CHI_TINY);
    dex_accumulate_S1(eta[0] * dex_rcp(c), c, nhl, I[0], T[0]);
  } else {
    const float2 nhl2 = make_float2(nhl, nhl);
#pragma unroll
    for (int i = 0; i < LPT / 2; ++i) {
      const float2 c = make_float2(fmaxf(chi[2 * i], DEX_CHI_TINY), fmaxf(chi[2 * i + 1], DEX_CHI_TINY));
      const float2 S = __fmul2_rn(make_float2(eta[2 * i], eta[2 * i + 1]), make_float2(dex_rcp(c.x), dex_rcp(c.y)));
      float2 Ii = make_float2(I[2 * i], I[2 * i + 1]), Ti = make_float2(T[2 * i], T[2 * i + 1]);
      dex_accumulate_S2(S, c, nhl2, Ii, Ti);
      I[2 * i] = Ii.x; I[2 * i + 1] = Ii.y;
      T[2 * i] = Ti.x; T[2 * i + 1] = Ti.y;
    }
  }
}

template <int LPT>
__device__ __forceinline__ void dex_accumulate_all(const float (&eta)[LPT], const float (&chi)[LPT], float hds,
                                                   float (&I)[LPT], float (&T)[LPT]) {
  const float hl = hds * -1.4426950408889634f;
  if (LPT == 1) {
    dex_accumulate(eta[0], chi[0], hds, hl, I[0], T[0]);
  } else {
    const float2 hds2 = make_float2(hds, hds), hl2 = make_float2(hl, hl);
#pragma unroll
    for (int i = 0; i < LPT / 2; ++i) {
      float2 Ii = make_float2(I[2 * i], I[2 * i + 1]), Ti = make_float2(T[2 * i], T[2 * i + 1]);
      dex_accumulate2(make_float2(eta[2 * i], eta[2 * i + 1]), make_float2(chi[2 * i], chi[2 * i + 1]), hds2, hl2, Ii, Ti);
      I[2 * i] = Ii.x; I[2 * i + 1] = Ii.y;
      T[2 * i] = Ti.x; T[2 * i + 1] = Ti.y;
    }
  }
}

// LPT consecutive floats of a 32-byte plane record: one LDG.E.256 / .128 / .64 / .32
template <int LPT>
__device__ __forceinline__ void dex_load_plane(const float* __restrict__ p, float (&v)[LPT]) {
  if (LPT == 8) {
    asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[LPT - 4]), "=f"(v[LPT - 3]), "=f"(v[LPT - 2]), "=f"(v[LPT - 1])
        : "l"(p));
  } else if (LPT == 4) {
    const float4 q = __ldg(reinterpret_cast<const float4*>(p));
    v[0] = q.x; v[1] = q.y; v[LPT - 2] = q.z; v[LPT - 1] = q.w;
  } else if (LPT == 2) {
    const float2 q = __ldg(reinterpret_cast<const float2*>(p));
    v[0] = q.x; v[LPT - 1] = q.y;
  } else {
    v[0] = __ldg(p);
  }
}

// record layout: chi[0..7] then eta[0..7]; this lane owns wavelengths sub*LPT .. sub*LPT+LPT-1
template <int LPT>
__device__ __forceinline__ void dex_load_rec(const float* __restrict__ rec, int sub, float (&eta)[LPT], float (&chi)[LPT]) {
  const float* pc = rec + sub * LPT;
  const float* pe = rec + DEX_W + sub * LPT;
  if (LPT == 8) {          // one thread per ray: each 32-byte plane of the 64-byte record is one LDG.E.256
    dex_load_plane<LPT>(pc, chi);
    dex_load_plane<LPT>(pe, eta);
  } else if (LPT == 1) {
    chi[0] = __ldg(pc);
    eta[0] = __ldg(pe);
  } else if (LPT == 2) {
    const float2 c = __ldg(reinterpret_cast<const float2*>(pc));
    const float2 e = __ldg(reinterpret_cast<const float2*>(pe));
    chi[0] = c.x; chi[1] = c.y; eta[0] = e.x; eta[1] = e.y;
  } else {
#pragma unroll
    for (int i = 0; i < LPT / 4; ++i) {
      const float4 c = __ldg(reinterpret_cast<const float4*>(pc) + i);
      chi[4 * i] = c.x; chi[4 * i + 1] = c.y; chi[4 * i + 2] = c.z; chi[4 * i + 3] = c.w;
    }
#pragma unroll
    for (int i = 0; i < LPT / 4; ++i) {
      const float4 e = __ldg(reinterpret_cast<const float4*>(pe) + i);
      eta[4 * i] = e.x; eta[4 * i + 1] = e.y; eta[4 * i + 2] = e.z; eta[4 * i + 3] = e.w;
    }
  }
}

// Core-and-Voigt: what depends on (wavelength of the batch, active line) only -- eqs. 14, 18-20
struct DexCavTab {
  double dlam[DEX_NLINES][DEX_W];    // lambda - lambda0
  double r2[DEX_NLINES][DEX_W];      // (lambda / lambda0)^2:  a(lambda) = r2 a(lambda0)                 (eq. 20)
  float dlam_h[DEX_NLINES][DEX_W];   // the same two as fp32 (dlam as an unevaluated pair hi + lo) for the fp32 Voigt
  float dlam_l[DEX_NLINES][DEX_W];
  float r2f[DEX_NLINES][DEX_W];
  float dlam_min[DEX_NLINES], dlam_max[DEX_NLINES];   // extremes of lambda - lambda0 over the batch (region-I pre-test)
  float r2lo[DEX_NLINES], r2hi[DEX_NLINES];   // min / max of r2f over the batch (slightly widened): damping window test
  float scale[DEX_NLINES][DEX_W];    // (lambda0 / lambda) / sqrt(pi): eta*(lambda) phi = eta*0 invD scale H (eqs. 18-19)
  double lam0_over_c[DEX_NLINES];    // Doppler shift of the line centre per unit projected velocity     (eq. 14)
  int line[DEX_NLINES];              // the batch's active lines, compacted: slots 0 .. nq-1
  int nq;                            // number of active lines of the batch
};

// the literal fp64 formula for damping outside the fp32 window: rare, so kept out of line (it would otherwise be
// inlined 8 x DEX_NLINES times and set the register count of the whole kernel)
// The Weideman coefficients come from __constant__ memory, not from the kernel's DexMipsDev parameter: passing
// &M.wei_c[0] to an out-of-line function needs a generic address, for which the compiler copied the whole 464-byte
// parameter struct to local memory at the start of EVERY thread (58 STL.64: invisible in the march, whose threads live
// for millions of segments, but 3x the DRAM writes of the records themselves in dex_dir_records_kernel).
__constant__ double dex_c_wei[DEX_WEI_N];
__constant__ double dex_c_wei_L;
__device__ __noinline__ float dex_voigt_H_outside_window(double a, double x) {
  return (float)dex_voigt_H_march(dex_c_wei, dex_c_wei_L, a, x);
}

// eta, chi of one cell for this lane's wavelengths, seen along propagation direction om (a7)
template <int D, int VAR, int LPT>
__device__ __forceinline__ void dex_provider(const DexMipsDev& M, size_t batch_base, int cell, int sub,
                                             const float (&om)[D], float sin_incl, const DexCavTab& CT,
                                             const float4* __restrict__ vfw, const float* __restrict__ vfc,
                                             const float* __restrict__ iso0, const float* __restrict__ iso1,
                                             float (&eta)[LPT], float (&chi)[LPT]) {
  if (VAR == DEX_ISO) {   // march records, two planes of 32-byte rows: chi[] receives chi log2(e), eta[] S = eta/chi
    dex_load_plane<LPT>(iso0 + (unsigned)cell * DexRecStride<D>::value, chi);
    dex_load_plane<LPT>(iso1 + (unsigned)cell * DexRecStride<D>::value, eta);
    return;
  }
  // projected velocity of the cell's box-filtered bulk velocity, fp64 (DESIGN.md R-vel)
  // velocity-interpolation marches keep the velocities dense (stride 1, compile time); Core-and-Voigt / Classic read
  // the cell's contiguous [velocity, lines] record (dex_device.cuh)
  const float4* __restrict__ arec = M.aux + ((VAR == DEX_VELINTERP) ? (size_t)(unsigned)cell : dex_aux_vel(M, (size_t)(unsigned)cell));
  const float4 v4 = __ldg(arec);
  double vproj = __dmul_rn((double)v4.x, (double)om[0]);
  vproj = __dadd_rn(vproj, __dmul_rn((double)v4.y, (double)om[1]));
  if (D == 3) vproj = __dadd_rn(vproj, __dmul_rn((double)v4.z, (double)om[D - 1]));
  if (D == 2) vproj = __dmul_rn(vproj, (double)sin_incl);   // 2.5D: in-plane part of the 3D direction (1 for in-plane rays)
  if (VAR == DEX_VELINTERP) {
    // linear interpolation on the cell's uniform velocity grid [-V, V]:
    // f = (vproj + V) / (2V) (n - 1) clamped to [0, n-1], i0 = min(floor f, n-2), w = f - i0.  f needs fp64 (adjacent
    // bins of a Gaussian core differ by factors of 1e2, so an fp32 f would cost 1e-4 in eta), the division does not:
    // 1/(2V) is the fp32 MUFU.RCP refined by one fp64 Newton step (2^-44).  The bin is taken from f rounded to fp32;
    // where that rounding crosses an integer the pair (i0, w) describes the same point of the same piecewise-linear
    // function from the neighbouring interval (w within 3e-7 of 0 or 1), so only the two ends need the clamp.
    const int nvb = M.n_vbins;
    int i0 = 0;
    float w = 0.0f;
    if (v4.w > 0.0f) {
      const double V = (double)v4.w, d2 = V + V;
      double r = (double)dex_rcp(v4.w + v4.w);
      r = fma(r, fma(-d2, r, 1.0), r);
      const double f = (vproj + V) * (r * (double)(nvb - 1));
      const float top = (float)(nvb - 2);
      const float fi = fminf(fmaxf(floorf((float)f), 0.0f), top);
      i0 = (int)fi;
      w = (float)(f - (double)fi);
      w = fminf(fmaxf(w, (fi <= 0.0f) ? 0.0f : -1.0f), (fi >= top) ? 1.0f : 2.0f);
    }
    // this batch's tables start at vt0 (kept in a register pair by the caller through iso0); 32-bit record index
    const float* r0 = iso0 + (size_t)((unsigned)cell * (unsigned)nvb + (unsigned)i0) * DEX_REC;
    float e1[LPT], c1[LPT];
    dex_load_rec<LPT>(r0, sub, eta, chi);
    dex_load_rec<LPT>(r0 + DEX_REC, sub, e1, c1);
    const float omw = 1.0f - w;
    if (LPT == 1) {
      eta[0] = fmaf(w, e1[0], omw * eta[0]);
      chi[0] = fmaf(w, c1[0], omw * chi[0]);
    } else {
      const float2 w2 = dex_f2(w), omw2 = dex_f2(omw);
#pragma unroll
      for (int i = 0; i < LPT / 2; ++i) {
        const float2 e = __ffma2_rn(w2, make_float2(e1[2 * i], e1[2 * i + 1]), __fmul2_rn(omw2, make_float2(eta[2 * i], eta[2 * i + 1])));
        const float2 c = __ffma2_rn(w2, make_float2(c1[2 * i], c1[2 * i + 1]), __fmul2_rn(omw2, make_float2(chi[2 * i], chi[2 * i + 1])));
        eta[2 * i] = e.x; eta[2 * i + 1] = e.y;
        chi[2 * i] = c.x; chi[2 * i + 1] = c.y;
      }
    }
    return;
  }
  // Core-and-Voigt / Classic: background + sum over the active lines (eqs. 10-11).  Only H(a, x) needs fp64 (the
  // Weideman form cancels in the wings); the line sum itself is fp32.  Everything that depends
  // on (wavelength, line) alone comes from the block's shared table CT (one batch per block).
  dex_load_rec<LPT>(iso0 + (size_t)(unsigned)cell * DEX_REC, sub, eta, chi);   // iso0 = this batch's background records
  const int nq = CT.nq;                    // block-uniform
#pragma unroll 1
  for (int q = 0; q < nq; ++q) {           // not unrolled: the body is ~350 instructions and would be copied 4 times
    const int l = CT.line[q];
    const float4 ln = __ldg(arec + 1 + l);
    const double shift = vproj * CT.lam0_over_c[q];
    const float sh_h = (float)shift, sh_l = (float)(shift - (double)sh_h);
    const float es = ln.x * ln.w, cs = ln.y * ln.w;
    float H[LPT];
    if (M.voigt_fp32 && ln.z * CT.r2lo[q] >= DEX_VF_A_LO && ln.z * CT.r2hi[q] <= DEX_VF_A_HI) {
      // fp32 table form for every wavelength of the batch, branch free so that the LPT evaluations interleave
      bool far = false;
      float xh[LPT], af[LPT];
      if (LPT == 1) {
        const int j = sub;
        af[0] = CT.r2f[q][j] * ln.z;
        const float dh = CT.dlam_h[q][j];
        const float sm = dh + sh_h, bb = sm - dh;
        const float se = ((dh - (sm - bb)) + (sh_h - bb)) + (CT.dlam_l[q][j] + sh_l);
        xh[0] = sm * ln.w;
        const float xl = fmaf(se, ln.w, fmaf(sm, ln.w, -xh[0]));
        H[0] = dex_voigt_H_table(vfw, vfc, af[0], xh[0], xl);
        far = fabsf(xh[0]) + af[0] >= 15.0f;
      } else {
        // x = (dlam + shift) / dlamD as an fp32 pair: two-sum of the leading parts, two-product with 1/dlamD;
        // two wavelengths per packed instruction
        const float2 shh = dex_f2(sh_h), nshh = dex_f2(-sh_h), shl = dex_f2(sh_l), inv2 = dex_f2(ln.w), a02 = dex_f2(ln.z);
#pragma unroll
        for (int i = 0; i < LPT / 2; ++i) {
          const int j = sub * LPT + 2 * i;
          const float2 a2 = __fmul2_rn(*reinterpret_cast<const float2*>(&CT.r2f[q][j]), a02);
          const float2 dh = *reinterpret_cast<const float2*>(&CT.dlam_h[q][j]);
          const float2 dl = *reinterpret_cast<const float2*>(&CT.dlam_l[q][j]);
          const float2 sm = __fadd2_rn(dh, shh);
          const float2 bb = __fadd2_rn(sm, dex_neg2(dh));
          const float2 e1 = __fadd2_rn(dh, dex_neg2(__fadd2_rn(sm, dex_neg2(bb))));
          const float2 e2 = __fadd2_rn(shh, dex_neg2(bb));
          const float2 se = __fadd2_rn(__fadd2_rn(e1, e2), __fadd2_rn(dl, shl));
          const float2 x2 = __fmul2_rn(sm, inv2);
          const float2 xl = __ffma2_rn(se, inv2, __ffma2_rn(sm, inv2, dex_neg2(x2)));
          const float2 h2 = dex_voigt_H_table2(vfw, vfc, a2, x2, xl);
          af[2 * i] = a2.x; af[2 * i + 1] = a2.y;
          xh[2 * i] = x2.x; xh[2 * i + 1] = x2.y;
          H[2 * i] = h2.x; H[2 * i + 1] = h2.y;
        }
        (void)nshh;
        // can any wavelength of the batch be in region I?  One bound per (segment, line) instead of a test per
        // evaluation: |x_j| <= max(|dlam_min + shift|, |dlam_max + shift|) / dlamD, a_j <= a0 r2hi (slightly widened)
        const float xb = fmaxf(fabsf(CT.dlam_min[q] + sh_h), fabsf(CT.dlam_max[q] + sh_h)) * ln.w;
        far = fmaf(xb, 1.0001f, ln.z * CT.r2hi[q]) >= 14.99f;
      }
      if (far) {
#pragma unroll
        for (int i = 0; i < LPT; ++i)
          if (fabsf(xh[i]) + af[i] >= 15.0f) H[i] = dex_voigt_H_region1(af[i], xh[i]);
      }
    } else {
      // unrolled on purpose: a run-time index into H[] would put H -- and with it the fast path's results -- into local
      // memory (two STL.128 per segment in the march; in the records kernel, whose threads each own fresh local lines,
      // 5x the DRAM writes of the records themselves).  The callee is out of line, so this is 8 call sites, not 8 bodies.
#pragma unroll
      for (int i = 0; i < LPT; ++i) {
        const int j = sub * LPT + i;
        const double x = (CT.dlam[q][j] + shift) * (double)ln.w;
        H[i] = dex_voigt_H_outside_window(CT.r2[q][j] * (double)ln.z, x);
      }
    }
    if (LPT == 1) {
      const float phi = H[0] * CT.scale[q][sub];
      eta[0] = fmaf(es, phi, eta[0]);
      chi[0] = fmaf(cs, phi, chi[0]);
    } else {
      const float2 es2 = dex_f2(es), cs2 = dex_f2(cs);
#pragma unroll
      for (int i = 0; i < LPT / 2; ++i) {
        const float2 sc = *reinterpret_cast<const float2*>(&CT.scale[q][sub * LPT + 2 * i]);
        const float2 phi = __fmul2_rn(make_float2(H[2 * i], H[2 * i + 1]), sc);
        const float2 e2 = __ffma2_rn(es2, phi, make_float2(eta[2 * i], eta[2 * i + 1]));
        const float2 c2 = __ffma2_rn(cs2, phi, make_float2(chi[2 * i], chi[2 * i + 1]));
        eta[2 * i] = e2.x; eta[2 * i + 1] = e2.y;
        chi[2 * i] = c2.x; chi[2 * i + 1] = c2.y;
      }
    }
  }
}

// Block prologue of the Core-and-Voigt evaluation: the fp32 Voigt tables and everything that depends on (wavelength of
// the batch, active line) only go to shared memory (eqs. 14, 18-20).  Ends with a barrier.
__device__ __forceinline__ void dex_cav_block_setup(const DexMipsDev& M, int batch, DexCavTab& CT, float4* vfw, float* vfc) {
  {
    for (int i = threadIdx.x; i < DEX_VF_NODES; i += blockDim.x) {
      vfw[i] = __ldg(M.vf_wing + i);
      vfc[i] = __ldg(M.vf_core + i);
    }
    if (threadIdx.x < DEX_NLINES * DEX_W) {
      // the caller's active set may have gaps (-1 anywhere): slot q of the table = the q-th ACTIVE line
      const int q0 = threadIdx.x / DEX_W, j = threadIdx.x % DEX_W;
      const int l = M.active_lines[batch * DEX_NLINES + q0];
      int q = 0, total = 0;
      for (int qq = 0; qq < DEX_NLINES; ++qq) {
        const int on = (M.active_lines[batch * DEX_NLINES + qq] >= 0) ? 1 : 0;
        q += (qq < q0) ? on : 0;
        total += on;
      }
      if (threadIdx.x == 0) CT.nq = total;
      if (j == 0 && l >= 0) CT.line[q] = l;
      if (l >= 0) {
        const double lm = (double)__ldg(M.lam + batch * DEX_W + j), l0 = (double)M.lambda0[l];
        const double r = lm / l0;
        CT.dlam[q][j] = lm - l0;
        CT.r2[q][j] = r * r;
        CT.dlam_h[q][j] = (float)(lm - l0);
        CT.dlam_l[q][j] = (float)((lm - l0) - (double)CT.dlam_h[q][j]);
        CT.r2f[q][j] = (float)(r * r);
        CT.scale[q][j] = (float)((l0 / lm) * 0.56418958354775628695);
        if (j == 0) {
          CT.lam0_over_c[q] = l0 / M.c_light;
          double lo = 1e300, hi = 0.0, dmin = 1e300, dmax = -1e300;
          for (int jj = 0; jj < DEX_W; ++jj) {
            const double lj = (double)__ldg(M.lam + batch * DEX_W + jj);
            const double rr = lj / l0;
            lo = fmin(lo, rr * rr);
            hi = fmax(hi, rr * rr);
            dmin = fmin(dmin, lj - l0);
            dmax = fmax(dmax, lj - l0);
          }
          CT.dlam_min[q] = (float)dmin;
          CT.dlam_max[q] = (float)dmax;
          CT.r2lo[q] = (float)(lo * (1.0 - 1e-6));
          CT.r2hi[q] = (float)(hi * (1.0 + 1e-6));
        }
      }
    }
    __syncthreads();
  }
}

// Each lane group owns one probe and loops over the quadrature directions.
//
// Control structure (profiles/r01c-r01e): the loop over HDDA events is warp-synchronous.  Every iteration each live
// lane leaves one cell (dex_ray_advance: segment, in-brick move) and the emitting lanes integrate together.  A lane
// whose ray reaches a brick face does NOT take the general crossing at once: it waits (`blocked`) until a quorum of
// the warp's lanes wait too, or nobody else can move, and then they cross together.  With 29 rays per warp each
// meeting a face every ~17 steps, crossing at once would run the ~100-instruction general path on 4 lanes in 82 % of
// the iterations (measured); batched, it runs on >= DEX_CROSS_QUORUM lanes a quarter as often.
#ifndef DEX_MARCH_THREADS
#define DEX_MARCH_THREADS 128
#endif
#ifndef DEX_MARCH_MINB
#define DEX_MARCH_MINB 8
#endif
// resident blocks per SM asked of the compiler per variant: the ISO march fits 64 registers; the velocity tables
// want two records in flight, and Core-and-Voigt runs 8 independent fp64 Goertzel chains per line
#ifndef DEX_MINB_VEL
#define DEX_MINB_VEL 7   // swept 4..8 on C3: 774 / 675 / 665 / 631 / 678 ms (profiles/r01k)
#endif
#ifndef DEX_MINB_CAV
#define DEX_MINB_CAV 4
#endif
// which marches cross a whole box of empty bricks in one step (dex_device.cuh): the 2D ones.  In 3D the two extra
// coordinate searches per box exit cost what the skipped bricks save (C5 in the ray loop 139.7 -> 142.0 ms, C5 memoised
// with the 3D ISO march 94.2 -> 95.1 ms), so 3D rays take empty bricks one at a time
#define DEX_BOX(D, VAR) ((D) == 2)
#ifndef DEX_REC_THREADS
#define DEX_REC_THREADS 128   // block of dex_dir_records_kernel
#endif
#ifndef DEX_REC_GROUP
#define DEX_REC_GROUP 8       // runs of DEX_REC_THREADS cells per block of dex_dir_records_kernel
#endif
#ifndef DEX_MINB_ISO3D
#define DEX_MINB_ISO3D 7   // swept on C5 memoised: 6 / 7 / 8 / 10 blocks per SM give 97.2 / 94.0 / 99.2 / 126.8 ms (8 spills 40 B at 64 registers)
#endif
constexpr int dex_march_minb(int var, int ndim) {
  return var == DEX_ISO ? (ndim == 3 ? DEX_MINB_ISO3D : DEX_MARCH_MINB) : (var == DEX_VELINTERP ? DEX_MINB_VEL : DEX_MINB_CAV);
}
#ifndef DEX_FOLD_EVERY
#define DEX_FOLD_EVERY 32   // power of two
#endif
#ifndef DEX_CROSS_QUORUM
#define DEX_CROSS_QUORUM 8
#endif
#ifndef DEX_MEMO_MIN_REUSE
#define DEX_MEMO_MIN_REUSE 3.0   // estimated rays per (cell, direction) from which the memoised march is taken: C5 (estimate
                                 // 5.3; 3.4 segments per evaluated record) is 1.35x faster memoised, C3 / C4 (590) 1.8x / 5.9x
#endif



template <int D, int VAR, int LPR, bool FUSE_J, bool CLIP>
__global__ void __launch_bounds__(DEX_MARCH_THREADS, dex_march_minb(VAR, D))
dex_march_kernel(const DexGridDev G, const DexMipsDev M, const DexRaysDev R, const int* __restrict__ perm,
                 float* __restrict__ out, unsigned long long* __restrict__ seg_count,
                 unsigned long long* __restrict__ line_seg_count) {
  constexpr int LPT = DEX_W / LPR;
  constexpr unsigned FULL = 0xffffffffu;
  __shared__ float Jsm[FUSE_J ? LPT * DEX_MARCH_THREADS : 1];
  const int batch = blockIdx.y;
  const long long slot_id = ((long long)blockIdx.x * blockDim.x + threadIdx.x) / LPR;
  const bool valid = slot_id < R.n_probes;          // lanes past the end stay in the warp-synchronous loops, idle
  // probes are handed to lanes in tile order (dex_tile_probes): a warp's probes are spatial neighbours
  const long long gid = !valid ? 0 : (perm != nullptr ? (long long)perm[slot_id] : slot_id);
  const int sub = threadIdx.x % LPR;
  const int lam_off = batch * DEX_W + sub * LPT;
  unsigned nseg = 0;
  const int* binfo = M.binfo + (size_t)batch * G.n_bricks;
  asm volatile("" : "+l"(binfo));   // opaque for the same reason as iso0 / iso1 below
  const size_t batch_base = ((size_t)batch * G.n_active) * M.cps;
  // this lane's rows of the two ISO record planes (cell 0 of the batch); kept opaque so that the pointers stay in
  // registers instead of being rebuilt from the kernel parameters at every segment
  // (velocity interpolation: iso0 = this batch's velocity tables; Core-and-Voigt / Classic: its background records)
  const float* iso0 = (VAR == DEX_ISO) ? M.mrec + batch_base * DexRecStride<D>::value + sub * LPT
                      : (VAR == DEX_VELINTERP) ? M.vtab + batch_base * (size_t)M.n_vbins * DEX_REC
                                               : M.store + batch_base * DEX_REC;
  const float* iso1 = iso0 + M.mplane;
  asm volatile("" : "+l"(iso0), "+l"(iso1));
  const float* __restrict__ probe = R.probe_pos + gid * D;
  __shared__ DexCavTab CT;
  __shared__ float4 vfw[VAR == DEX_CAV ? DEX_VF_NODES : 1];
  __shared__ float vfc[VAR == DEX_CAV ? DEX_VF_NODES : 1];
  if (VAR == DEX_CAV) dex_cav_block_setup(M, batch, CT, vfw, vfc);
  // J is touched once per direction, I and T once per segment: J lives in shared memory ([i][thread], conflict-free)
  // I is accumulated on two levels: I[] (registers) holds the sum over the last <= DEX_FOLD_EVERY iterations of the
  // warp's loop, Ih[] (shared memory, [i][thread], conflict free) everything before.  With one level, a ray of ~1000
  // thin segments whose optical depth builds up slowly loses every far contribution below ulp(I)/2: -1.07e-5 relative
  // on C3's longest rays (measured; the rounding of I alone, everything else held in fp64); with two levels the same
  // rays are within 1.6e-6.  The fold points depend on the warp's iteration count, i.e. on which rays share a warp;
  // dex_tile_probes makes that a pure function of the probe array, so results are reproducible bit for bit.
#ifndef DEX_IH_REGISTERS
  __shared__ float Ihs[LPT * DEX_MARCH_THREADS];
#define DEX_IH(i) Ihs[(i) * DEX_MARCH_THREADS + threadIdx.x]
#else
  float Ih[LPT];
#define DEX_IH(i) Ih[i]
#endif
  float I[LPT], T[LPT];
  if (FUSE_J) {
#pragma unroll
    for (int i = 0; i < LPT; ++i) Jsm[i * DEX_MARCH_THREADS + threadIdx.x] = 0.0f;
  }
  DexRay3<D> ray;
  const bool caps = M.n_caps > 0;     // block-uniform: which of the two crossing routines (dex_device.cuh) this launch runs
  // one direction at a time: the lanes of a warp trace the same direction together (coherent fetches)
  const int k_begin = (!FUSE_J && R.k_per_block > 0) ? (int)blockIdx.z * R.k_per_block : 0;
  if (VAR == DEX_ISO && M.mdir != 0) {   // per-direction records (memoised Core-and-Voigt, below): direction k's start at k mdir
    iso0 += (size_t)k_begin * M.mdir;
    iso1 += (size_t)k_begin * M.mdir;
  }
  const int k_end = (!FUSE_J && R.k_per_block > 0) ? min(R.n_dirs, k_begin + R.k_per_block) : R.n_dirs;
  for (int k = k_begin; k < k_end; ++k) {
    const float* __restrict__ om = R.dirs + k * D;
    float omf[D];
#pragma unroll
    for (int a = 0; a < D; ++a) omf[a] = __ldg(om + a);
    // 2.5D rays: path lengths are divided by the sine of the inclination to the homogeneous axis (dex.h d_sin_incl)
    const float sin_incl = (D == 2 && R.sin_incl != nullptr) ? __ldg(R.sin_incl + k) : 1.0f;
    const float hk = (D == 2 && R.sin_incl != nullptr) ? __fdiv_rn(G.h, sin_incl) : G.h;
#pragma unroll
    for (int i = 0; i < LPT; ++i) { I[i] = 0.0f; DEX_IH(i) = 0.0f; T[i] = 1.0f; }
    bool alive = valid && dex_ray_init3<D>(ray, G, M, binfo, probe, om);
    bool blocked = false;   // waiting at a brick face for dex_ray_cross (implies alive)
    for (unsigned it = 1;; ++it) {
      const unsigned am = __ballot_sync(FULL, alive);
      if (am == 0u) break;
      if ((it & (DEX_FOLD_EVERY - 1)) == 0) {   // warp-uniform, so the fold costs < 1 % (a per-ray trigger diverges: +8 %)
#pragma unroll
        for (int i = 0; i < LPT; ++i) { DEX_IH(i) += I[i]; I[i] = 0.0f; }
      }
      const unsigned bm = __ballot_sync(FULL, blocked);
      if (bm == am || __popc(bm) >= DEX_CROSS_QUORUM) {
        if (blocked) {
          alive = caps ? dex_ray_cross<D>(ray, G, M, binfo, probe, om) : dex_ray_cross_nocap<D, DEX_BOX(D, VAR)>(ray, G, binfo, probe, om);
          blocked = false;
        }
      }
      if (alive && !blocked) {
        bool emit;
        int cell;
        float ds;
        const float t0 = ray.t;
        blocked = !dex_ray_advance<D>(ray, emit, cell, ds);
        if (CLIP) {   // T10 (compile time: the full-ray kernels do not pay for it): visit [t0, ray.t] clipped to the interval
          ds = __fsub_rn(fminf(ray.t, R.t_end), fmaxf(t0, R.t_begin));
          emit = emit && ds > 0.0f;
          if (ray.t >= R.t_end) { alive = false; blocked = false; }
        }
        // 3D ISO march over records that miss the L2 (C5 memoised: long_scoreboard 9 warps per issue, DRAM at 45 %): after an
        // in-brick step the next cell's 64-byte record is known one iteration early and is requested into the L2 now
        // (C5 102.5 -> 99.2 ms; into the L1, or one request per 32-byte half, is slower: profiles/r02_experiments.md)
        if (D == 3 && VAR == DEX_ISO && !blocked && ray.cell >= 0) {
          const float* pn = iso0 + (size_t)(unsigned)ray.cell * DexRecStride<D>::value;
          asm volatile("prefetch.global.L2 [%0];" ::"l"(pn));
        }
        if (emit) {
          ++nseg;
          const float hds = hk * ds;
          float eta[LPT], chi[LPT];
          dex_provider<D, VAR, LPT>(M, batch_base, cell, sub, omf, sin_incl, CT, vfw, vfc, iso0, iso1, eta, chi);
          if (VAR == DEX_ISO) dex_accumulate_all_S<LPT>(eta, chi, hds, I, T);
          // velocity interpolation keeps the E(tau) integrator: the record form costs it registers it does not have at
          // 7 blocks per SM (measured on C3: 583 ms against 616; Core-and-Voigt gains 3 % from the record form)
          else if (VAR == DEX_VELINTERP) dex_accumulate_all<LPT>(eta, chi, hds, I, T);
          else dex_accumulate_all_EC<LPT>(eta, chi, hds, I, T);
        }
      }
    }
    if (VAR == DEX_ISO && M.mdir != 0) { iso0 += M.mdir; iso1 += M.mdir; }
    if (valid) {
#pragma unroll
      for (int i = 0; i < LPT; ++i) I[i] += DEX_IH(i);
      if (R.i0 != nullptr) {
#pragma unroll
        for (int i = 0; i < LPT; ++i) I[i] = fmaf(T[i], __ldg(R.i0 + (size_t)k * M.io_stride + M.io_base + lam_off + i), I[i]);
      }
      if (FUSE_J) {
        const float wk = __ldg(R.weights + k);
#pragma unroll
        for (int i = 0; i < LPT; ++i) Jsm[i * DEX_MARCH_THREADS + threadIdx.x] = fmaf(wk, I[i], Jsm[i * DEX_MARCH_THREADS + threadIdx.x]);
      } else {
        float* dst = out + ((size_t)gid * R.n_dirs + k) * M.io_stride + M.io_base + lam_off;
#pragma unroll
        for (int i = 0; i < LPT; ++i) dst[i] = I[i];
      }
    }
  }
  if (FUSE_J && valid) {
    float* dst = out + (size_t)gid * M.io_stride + M.io_base + lam_off;
#pragma unroll
    for (int i = 0; i < LPT; ++i) {
      const float j = Jsm[i * DEX_MARCH_THREADS + threadIdx.x];
      dst[i] = R.accumulate ? __fadd_rn(dst[i], j) : j;
    }
  }
  if (seg_count != nullptr) {
    unsigned v = (sub == 0) ? nseg : 0u;
    v = __reduce_add_sync(FULL, v);
    if ((threadIdx.x & 31) == 0 && v) atomicAdd(seg_count, (unsigned long long)v);
  }
  if (VAR != DEX_ISO && line_seg_count != nullptr) {   // bench.py's roofline: provider evaluations (x active lines of the batch)
    const int nact = (VAR == DEX_CAV) ? CT.nq : 1;
    unsigned v = (sub == 0) ? nseg : 0u;
    v = __reduce_add_sync(FULL, v);
    if ((threadIdx.x & 31) == 0 && v && nact) atomicAdd(line_seg_count, (unsigned long long)v * (unsigned long long)nact);
  }
}

// ---- anisotropic providers, memoised per direction ----------------------------------------------------------------
// eta, chi of a cell along direction k (eqs. 10-20; the velocity-bin interpolation of PAPER.md:196-198) depend on
// (cell, k, wavelength) only, and with a probe in every voxel each (cell, direction) is crossed by hundreds of rays
// (C3, C4: ~600), every one of which would evaluate the same Voigt profiles / interpolate the same two bins.
// This kernel evaluates the provider ONCE per (cell of the brick's selected level, direction, batch)
// -- the very routine the march calls, so the numbers are the march's own -- and stores them as march records
// (chi' log2 e | S, the ISO layout); the rays are then marched by the ISO kernel with M.mdir stepping the record
// pointers from direction to direction.
template <int D, int VAR>
__global__ void __launch_bounds__(DEX_REC_THREADS)
dex_dir_records_kernel(const DexGridDev G, const DexMipsDev M, const DexRaysDev R, const int* __restrict__ active_bricks,
                       int b0, float* __restrict__ rec, size_t plane, unsigned long long* __restrict__ line_eval_count) {
  __shared__ DexCavTab CT;
  __shared__ float4 vfw[VAR == DEX_CAV ? DEX_VF_NODES : 1];
  __shared__ float vfc[VAR == DEX_CAV ? DEX_VF_NODES : 1];
  // blockIdx.x = cell block * n_dirs + direction: the blocks that evaluate the same cells for different directions are
  // neighbours in launch order and share the cells' background / line / velocity records in the L2 (direction-major
  // order re-read them from DRAM for every direction: 63 GB per C5 step)
  const int bl = blockIdx.y, batch = b0 + bl, k = (int)(blockIdx.x % (unsigned)R.n_dirs);
  const unsigned cell_group = blockIdx.x / (unsigned)R.n_dirs;
  if (VAR == DEX_CAV) dex_cav_block_setup(M, batch, CT, vfw, vfc);
  unsigned done = 0;
  // a block evaluates DEX_REC_GROUP consecutive runs of blockDim.x cells, so that the table set-up above (9.6 KB of Voigt
  // tables into shared memory, the per-line constants in fp64, a barrier) is paid once per ~1000 evaluations
#pragma unroll 1
  for (int run = 0; run < DEX_REC_GROUP; ++run) {
  // one thread per pyramid cell of an active brick: the brick's selected level for this batch is the one the rays visit;
  // under a near-field cap (T8) they also visit the finer levels of the same brick
  const long long t = ((long long)cell_group * DEX_REC_GROUP + run) * blockDim.x + threadIdx.x;
  bool work = t < (long long)G.n_active * M.cps;
  const int cell = (int)t;                         // record index: slot * cps + position in the slot's pyramid
  if (work) {
    const int slot = (int)(t / M.cps), c = (int)(t - (long long)slot * M.cps);
    const int info = __ldg(M.binfo + (size_t)batch * G.n_bricks + active_bricks[slot]);
    const int m = (info & 15) - 1;
    int l = 0;
    for (int i = 1; i <= M.max_level; ++i) l += (c >= M.lvloff[i]) ? 1 : 0;
    work = m >= 0 && (l == m || (M.n_caps > 0 && l < m));
  }
  if (work) {
    float omf[D];
#pragma unroll
    for (int a = 0; a < D; ++a) omf[a] = __ldg(R.dirs + (size_t)k * D + a);
    const float sin_incl = (D == 2 && R.sin_incl != nullptr) ? __ldg(R.sin_incl + k) : 1.0f;
    const size_t batch_base = ((size_t)batch * G.n_active) * M.cps;
    // what the march keeps in iso0: this batch's background records (Core-and-Voigt) / velocity tables
    const float* bg = (VAR == DEX_VELINTERP) ? M.vtab + batch_base * (size_t)M.n_vbins * DEX_REC : M.store + batch_base * DEX_REC;
    float eta[DEX_W], chi[DEX_W];
    dex_provider<D, VAR, DEX_W>(M, batch_base, cell, 0, omf, sin_incl, CT, vfw, vfc, bg, bg, eta, chi);
    float* o0 = rec + (size_t)k * M.mdir + (((size_t)bl * G.n_active) * M.cps + (size_t)(unsigned)cell) * DexRecStride<D>::value;
    float* o1 = o0 + ((D == 3) ? (size_t)DEX_W : plane);
    float c2[DEX_W], S[DEX_W];
#pragma unroll
    for (int j = 0; j < DEX_W; ++j) {
      const float cj = fmaxf(chi[j], DEX_CHI_TINY);
      c2[j] = cj * 1.4426950408889634f;
      S[j] = eta[j] * dex_rcp(cj);
    }
    // whole 32-byte rows: scalar stores left every sector half written, and the L2 read each one back from DRAM to merge
    // (C5: 103 GB written + 46 GB read for 53 GB of records)
#pragma unroll
    for (int j = 0; j < DEX_W; j += 4) {
      *reinterpret_cast<float4*>(o0 + j) = make_float4(c2[j], c2[j + 1], c2[j + 2], c2[j + 3]);
      *reinterpret_cast<float4*>(o1 + j) = make_float4(S[j], S[j + 1], S[j + 2], S[j + 3]);
    }
    done += 1;
  }
  }
  if (line_eval_count != nullptr && k == 0) {
    // bench.py's roofline counts provider evaluations: records (x active lines) here.  Every direction evaluates the same
    // cells, so direction 0 counts for all of them: one atomic per block instead of 1e8 on one address (C4)
    __shared__ unsigned n_done;
    if (threadIdx.x == 0) n_done = 0;
    __syncthreads();
    const unsigned w = __reduce_add_sync(0xffffffffu, done);
    if ((threadIdx.x & 31) == 0 && w) atomicAdd(&n_done, w);
    __syncthreads();
    const int nact = (VAR == DEX_CAV) ? CT.nq : 1;
    if (threadIdx.x == 0 && n_done && nact)
      atomicAdd(line_eval_count, (unsigned long long)n_done * (unsigned long long)nact * (unsigned long long)R.n_dirs);
  }
}

// a10: traversal only, one thread per ray, for one batch's level table -- the same stepping code as
// the march kernel, crossing routine included (the capped dex_ray_cross under a near-field cap, else the cap-free
// dex_ray_cross_nocap with the march's empty-space boxes), so the recorded list is the one the production path
// integrates over.
template <int D>
__global__ void __launch_bounds__(128)
dex_capture_kernel(const DexGridDev G, const DexMipsDev M, const DexRaysDev R, long long* __restrict__ counts,
                   unsigned long long* __restrict__ records, float* __restrict__ ds_out,
                   const long long* __restrict__ offsets, long long capacity, int batch, int* __restrict__ overflow) {
  const long long ray_id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long n_rays = R.n_probes * R.n_dirs;
  if (ray_id >= n_rays) return;
  const long long p = ray_id / R.n_dirs;
  const int k = (int)(ray_id - p * R.n_dirs);
  const float* __restrict__ probe = R.probe_pos + p * D;
  const float* __restrict__ om = R.dirs + k * D;
  const int* __restrict__ binfo = M.binfo + (size_t)batch * G.n_bricks;
  const long long begin = offsets[ray_id];
  const long long room = ((ray_id + 1 < n_rays) ? offsets[ray_id + 1] : capacity) - begin;
  long long n = 0;
  DexRay3<D> ray;
  const bool caps = M.n_caps > 0;     // as in dex_march_kernel
  bool alive = dex_ray_init3<D>(ray, G, M, binfo, probe, om);
  while (alive) {
    int c[D];
    dex_ray_cell_coords<D>(ray, c);
    const int m = ray.sh;
    bool emit;
    int cell;
    float ds;
    const float t0 = ray.t;
    const bool inside = dex_ray_advance<D>(ray, emit, cell, ds);
    if (R.t_end > 0.0f) {
      ds = __fsub_rn(fminf(ray.t, R.t_end), fmaxf(t0, R.t_begin));
      emit = emit && ds > 0.0f;
    }
    if (R.t_end > 0.0f && ray.t >= R.t_end) alive = false;
    else if (!inside)
      alive = caps ? dex_ray_cross<D>(ray, G, M, binfo, probe, om)
                   : dex_ray_cross_nocap<D, DEX_BOX(D, DEX_ISO)>(ray, G, binfo, probe, om);
    if (emit) {
      if (n < room) {
        unsigned long long rec = ((unsigned long long)(unsigned)m << 56) | (unsigned long long)(unsigned)(c[0] >> m);
        rec |= (unsigned long long)(unsigned)(c[1] >> m) << 18;
        if (D == 3) rec |= (unsigned long long)(unsigned)(c[D - 1] >> m) << 36;
        records[begin + n] = rec;
        if (ds_out) ds_out[begin + n] = ds;
      }
      ++n;
    }
  }
  counts[ray_id] = n;
  if (n > room) *overflow = 1;
}

// ---- probe tiling: counting sort of the probes into compact spatial tiles ------------------------------
// Lane coherence is what the march lives on (profiles/): 32 probes of a 4x8 (2D) or 4x4x2 (3D) block of
// the probe lattice trace almost the same cells, 32 probes of one row do not.  The tile edge is scaled by
// the mean probe spacing, so a regular lattice fills every tile with exactly one warp.
struct DexTiling {
  float inv_tile[3];
  int nt[3];
  int n_tiles;
};

template <int D>
__device__ __forceinline__ int dex_tile_of(const DexTiling& TL, const float* __restrict__ pos) {
  int t[3] = {0, 0, 0};
#pragma unroll
  for (int a = 0; a < D; ++a) t[a] = max(0, min(TL.nt[a] - 1, (int)floorf(pos[a] * TL.inv_tile[a])));
  return (t[2] * TL.nt[1] + t[1]) * TL.nt[0] + t[0];
}

template <int D>
__global__ void dex_tile_count_kernel(const DexTiling TL, long long n, const float* __restrict__ pos, int* __restrict__ count) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) atomicAdd(count + dex_tile_of<D>(TL, pos + i * D), 1);
}

__global__ void __launch_bounds__(1024) dex_tile_scan_kernel(int* __restrict__ count, int n) {
  __shared__ int part[1024];
  const int t = threadIdx.x;
  const int chunk = (n + 1023) / 1024;
  const int lo = min(n, t * chunk), hi = min(n, lo + chunk);
  int sum = 0;
  for (int i = lo; i < hi; ++i) sum += count[i];
  part[t] = sum;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {
    int v = (t >= off) ? part[t - off] : 0;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  int base = part[t] - sum;
  for (int i = lo; i < hi; ++i) { const int c = count[i]; count[i] = base; base += c; }
}

template <int D>
__global__ void dex_tile_scatter_kernel(const DexTiling TL, long long n, const float* __restrict__ pos,
                                        int* __restrict__ cursor, int* __restrict__ perm) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) perm[atomicAdd(cursor + dex_tile_of<D>(TL, pos + i * D), 1)] = (int)i;
}

// The atomic scatter leaves the members of a tile in arrival order; ranking them by probe index makes perm -- and with
// it the composition of every warp -- a pure function of the probe array.  One thread per probe counts the members of
// its tile with a smaller index (tiles hold ~32 probes on a regular lattice; any size is handled, in O(size) reads).
template <int D>
__global__ void dex_tile_rank_kernel(const DexTiling TL, long long n, const float* __restrict__ pos,
                                     const int* __restrict__ cursor, const int* __restrict__ perm_in,
                                     int* __restrict__ perm_out) {
  const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  const int p = perm_in[s];
  const int t = dex_tile_of<D>(TL, pos + (long long)p * D);
  const int begin = (t == 0) ? 0 : cursor[t - 1];      // after the scatter cursor[t] is the END of tile t
  const int end = cursor[t];
  int rank = 0;
  for (int q = begin; q < end; ++q) rank += (perm_in[q] < p) ? 1 : 0;
  perm_out[begin + rank] = p;
}

// J(p, lambda) = sum_k w_k I(p, k, lambda) from a materialised I: one thread per (probe, lambda);
// consecutive threads read consecutive lambda (coalesced).
// The sum runs in direction order with one fma per term, exactly as the fused march accumulates it: both give the same bits.
__global__ void dex_reduce_j_kernel(long long n_probes, int n_dirs, int n_lambda, const float* __restrict__ w,
                                    const float* __restrict__ I, float* __restrict__ J, int accumulate) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_probes * n_lambda) return;
  const long long p = i / n_lambda;
  const int j = (int)(i - p * n_lambda);
  float acc = 0.0f;
  for (int k = 0; k < n_dirs; ++k) acc = fmaf(__ldg(w + k), __ldg(I + (p * n_dirs + k) * n_lambda + j), acc);
  J[i] = accumulate ? __fadd_rn(J[i], acc) : acc;
}

// validation (dex_voigt_profile): the march's own Voigt routines on caller-supplied (a, x)
struct DexWeideman { double c[DEX_WEI_N]; double L; };
__global__ void dex_voigt_profile_kernel(const float* __restrict__ a, const double* __restrict__ x, long long n,
                                         double* __restrict__ H, int mode, const DexWeideman Wc,
                                         const float4* __restrict__ wing, const float* __restrict__ core) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float af = a[i];
  const double xd = x[i];
  if (mode == 0 && af >= DEX_VF_A_LO && af <= DEX_VF_A_HI) {
    const float xh = (float)xd, xl = (float)(xd - (double)xh);
    H[i] = (double)dex_voigt_H_fast(wing, core, af, xh, xl);
  } else {
    H[i] = dex_voigt_H_march(Wc.c, Wc.L, (double)af, xd);
  }
}

template <int D, int VAR, int LPR, bool CLIP = false>
dex_status launch_march_t(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays, float* d_out, bool fuse_j,
                          unsigned long long* d_seg, const int* perm, cudaStream_t st) {
  const int threads = DEX_MARCH_THREADS;
  const long long probes_per_block = threads / LPR;
  const long long gx = (rays.n_probes + probes_per_block - 1) / probes_per_block;
  if (gx <= 0) return DEX_OK;
  if (gx > 2147483647LL || m->n_batch > 65535) {
    dex_set_error("march: problem too large for one launch");
    return DEX_ERR_UNSUPPORTED;
  }
  unsigned gz = 1;
  if (!fuse_j && rays.k_per_block > 0) gz = (unsigned)((rays.n_dirs + rays.k_per_block - 1) / rays.k_per_block);
  if (gz > 65535u) { dex_set_error("march: too many direction groups for one launch"); return DEX_ERR_UNSUPPORTED; }
  dim3 grid((unsigned)gx, (unsigned)m->n_batch, gz);
  DexMipsDev md = m->dev;
  md.voigt_fp32 = dex_tuning_voigt_fp32();
  unsigned long long* d_work = dex_line_segment_counter();   // NULL unless march timing is enabled
  if (fuse_j)
    dex_march_kernel<D, VAR, LPR, true, CLIP><<<grid, threads, 0, st>>>(g->dev, md, rays, perm, d_out, d_seg, d_work);
  else
    dex_march_kernel<D, VAR, LPR, false, CLIP><<<grid, threads, 0, st>>>(g->dev, md, rays, perm, d_out, d_seg, d_work);
  dex_count_launch();
  DEX_CUDA_CHECK(cudaGetLastError());
  return DEX_OK;
}

template <int D, int VAR>
dex_status launch_march_v(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays, float* d_out, bool fuse_j,
                          unsigned long long* d_seg, int lpr, const int* perm, cudaStream_t st) {
  // finite radiance intervals (T10) are compiled for the production mapping only (lanes per ray is a performance knob:
  // results do not depend on it)
  if (rays.t_end > 0.0f) return launch_march_t<D, VAR, 1, true>(g, m, rays, d_out, fuse_j, d_seg, perm, st);
  switch (lpr) {
    case 8: return launch_march_t<D, VAR, 8>(g, m, rays, d_out, fuse_j, d_seg, perm, st);
    case 4: return launch_march_t<D, VAR, 4>(g, m, rays, d_out, fuse_j, d_seg, perm, st);
    case 2: return launch_march_t<D, VAR, 2>(g, m, rays, d_out, fuse_j, d_seg, perm, st);
    case 1: return launch_march_t<D, VAR, 1>(g, m, rays, d_out, fuse_j, d_seg, perm, st);
  }
  dex_set_error("lanes per ray must be 1, 2, 4 or 8");
  return DEX_ERR_INVALID_ARG;
}

template <int D>
dex_status launch_march_d(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays, float* d_out, bool fuse_j,
                          unsigned long long* d_seg, int lpr, const int* perm, cudaStream_t st) {
  switch (m->variant) {
    case DEX_ISO: return launch_march_v<D, DEX_ISO>(g, m, rays, d_out, fuse_j, d_seg, lpr, perm, st);
    case DEX_VELINTERP: return launch_march_v<D, DEX_VELINTERP>(g, m, rays, d_out, fuse_j, d_seg, lpr, perm, st);
    case DEX_CAV:
    case DEX_CLASSIC: return launch_march_v<D, DEX_CAV>(g, m, rays, d_out, fuse_j, d_seg, lpr, perm, st);
  }
  dex_set_error("unknown variant");
  return DEX_ERR_INVALID_ARG;
}

}  // namespace

// perm[i] = probe handled by lane group i.  *d_perm is allocated on the stream (stream-ordered) and must be
// released with cudaFreeAsync by the caller after the march has been enqueued.
template <int D>
static dex_status tile_probes_t(const dex_grid* g, const DexRaysDev& rays, int** d_perm, cudaStream_t st) {
  *d_perm = nullptr;
  const long long n = rays.n_probes;
  if (n < 64 || n > 2147483647LL) return DEX_OK;        // nothing to gain / index range
  DexTiling TL;
  double vol = 1.0;
  for (int a = 0; a < D; ++a) vol *= (double)g->dev.dims[a];
  const double spacing = fmax(1.0, pow(vol / (double)n, 1.0 / D));   // mean probe spacing in voxels
  const int shape2[3] = {4, 8, 1}, shape3[3] = {4, 4, 2};
  long long nt_total = 1;
  for (int a = 0; a < 3; ++a) {
    const double edge = spacing * (double)((D == 2) ? shape2[a] : shape3[a]);
    TL.inv_tile[a] = (float)(1.0 / edge);
    TL.nt[a] = (a < D) ? (int)ceil((double)g->dev.dims[a] / edge) : 1;
    nt_total *= TL.nt[a];
  }
  if (nt_total > (1LL << 28)) return DEX_OK;
  TL.n_tiles = (int)nt_total;
  int* d_count = nullptr;
  DEX_CUDA_CHECK(dex_alloc((void**)&d_count, sizeof(int) * (size_t)(TL.n_tiles + 1), st));
  cudaError_t e = dex_alloc((void**)d_perm, sizeof(int) * (size_t)n, st);
  if (e != cudaSuccess) { cudaFreeAsync(d_count, st); *d_perm = nullptr; DEX_CUDA_CHECK(e); }
  cudaMemsetAsync(d_count, 0, sizeof(int) * (size_t)(TL.n_tiles + 1), st);
  const unsigned blocks = (unsigned)((n + 255) / 256);
  dex_tile_count_kernel<D><<<blocks, 256, 0, st>>>(TL, n, rays.probe_pos, d_count);
  dex_tile_scan_kernel<<<1, 1024, 0, st>>>(d_count, TL.n_tiles);
  int* d_arrival = nullptr;
  e = dex_alloc((void**)&d_arrival, sizeof(int) * (size_t)n, st);
  if (e != cudaSuccess) { cudaFreeAsync(d_count, st); cudaFreeAsync(*d_perm, st); *d_perm = nullptr; DEX_CUDA_CHECK(e); }
  dex_tile_scatter_kernel<D><<<blocks, 256, 0, st>>>(TL, n, rays.probe_pos, d_count, d_arrival);
  dex_tile_rank_kernel<D><<<blocks, 256, 0, st>>>(TL, n, rays.probe_pos, d_count, d_arrival, *d_perm);
  dex_count_launch(4);
  cudaFreeAsync(d_arrival, st);
  cudaFreeAsync(d_count, st);
  DEX_CUDA_CHECK(cudaGetLastError());
  return DEX_OK;
}

dex_status dex_make_probe_tiling(const dex_grid* g, const DexRaysDev& rays, int** d_perm, cudaStream_t st) {
  return (g->desc.ndim == 2) ? tile_probes_t<2>(g, rays, d_perm, st) : tile_probes_t<3>(g, rays, d_perm, st);
}

// Anisotropic marches with many rays per (cell, direction): evaluate the provider once per (cell, direction, batch) into
// per-direction march records (dex_dir_records_kernel) and march them with the ISO kernel, a group of
// wavelength batches at a time so that the records fit the memory set aside for them.  J columns of different batches
// are disjoint, so the groups need no accumulation.
// Returns through *fell_back = true (and DEX_OK, nothing marched) when not even one batch's records could be allocated
// before the first group: the caller then evaluates eta, chi in the ray loop instead (launch_march_d).
template <int D>
static dex_status launch_march_memo(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays, float* d_out,
                                        bool fuse_j, unsigned long long* d_seg, int lpr, const int* perm, cudaStream_t st,
                                        int& batches_per_group, bool* fell_back) {
  const size_t A = (size_t)g->n_active, cps = (size_t)m->dev.cps;
  *fell_back = false;
  for (int b0 = 0; b0 < m->n_batch;) {
    // The budget of memo_group is an estimate: the pool's idle bytes may be fragmented or still owned by another stream,
    // and the rebuild pipeline's build stream allocates at the same time.  A failed allocation is retried with half
    // the batches; if one batch does not fit, the first group falls back, a later one reports the failure (the
    // batches already marched have been added to J and to the segment counter: they cannot be redone).
    int nb = (b0 + batches_per_group <= m->n_batch) ? batches_per_group : m->n_batch - b0;
    float* d_rec = nullptr;
    size_t plane = 0;
    for (;;) {
      plane = (size_t)nb * A * cps * DEX_W;
      cudaError_t e = dex_tuning_memo_fail_alloc() ? cudaErrorMemoryAllocation
                                                   : dex_alloc((void**)&d_rec, sizeof(float) * 2 * plane * (size_t)rays.n_dirs, st);
      if (e == cudaSuccess) break;
      cudaGetLastError();
      d_rec = nullptr;
      if (e != cudaErrorMemoryAllocation) { dex_set_error(std::string("march records: ") + cudaGetErrorString(e)); return DEX_ERR_CUDA; }
      if (nb > 1) { nb = (nb + 1) / 2; batches_per_group = nb; continue; }
      if (b0 == 0) { *fell_back = true; return DEX_OK; }
      dex_set_error("march records: out of device memory for one wavelength batch of per-direction records");
      return DEX_ERR_OOM;
    }
    dex_mips mm = *m;                       // a view of the group's batches as an ISO handle over the records
    mm.variant = DEX_ISO;
    mm.n_batch = nb;
    DexMipsDev& d = mm.dev;
    d.variant = DEX_ISO;
    d.n_batch = nb;
    d.mdir = 2 * plane;
    const long long tasks = (long long)A * (long long)cps;
    const long long per_block = (long long)DEX_REC_THREADS * DEX_REC_GROUP;
    const long long gx = ((tasks + per_block - 1) / per_block) * (long long)rays.n_dirs;
    if (gx > 2147483647LL) { dex_free(d_rec, st); dex_set_error("march: too many (cell, direction) blocks for one records launch"); return DEX_ERR_UNSUPPORTED; }
    dim3 grid((unsigned)gx, (unsigned)nb, 1);
    DexMipsDev full = m->dev;
    full.mdir = 2 * plane;
    full.voigt_fp32 = dex_tuning_voigt_fp32();
    dex_status s = DEX_OK;
    if (tasks > 0) {
      if (m->variant == DEX_VELINTERP)
        dex_dir_records_kernel<D, DEX_VELINTERP><<<grid, DEX_REC_THREADS, 0, st>>>(g->dev, full, rays, g->d_active_bricks, b0,
                                                                                    d_rec, plane, dex_line_segment_counter());
      else
        dex_dir_records_kernel<D, DEX_CAV><<<grid, DEX_REC_THREADS, 0, st>>>(g->dev, full, rays, g->d_active_bricks, b0, d_rec,
                                                                              plane, dex_line_segment_counter());
      dex_count_launch();
      if (cudaGetLastError() != cudaSuccess) { dex_set_error("record kernel launch failed"); s = DEX_ERR_CUDA; }
    }
    if (s == DEX_OK) {
      d.mrec = d_rec;
      d.mplane = (D == 3) ? (size_t)DEX_W : plane;
      d.binfo = m->dev.binfo + (size_t)b0 * g->n_bricks;
      d.io_base = m->dev.io_base + b0 * DEX_W;
      s = launch_march_v<D, DEX_ISO>(g, &mm, rays, d_out, fuse_j, d_seg, lpr, perm, st);
    }
    dex_free(d_rec, st);
    if (s != DEX_OK) return s;
    b0 += nb;
  }
  return DEX_OK;
}

// How many wavelength batches' per-direction records the memoised march may hold at once; 0 = do not memoise (a static
// medium, too few rays per cell and direction for the evaluation to be shared, or no room for one batch).
static int memo_group(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays) {
  if (m->variant == DEX_ISO) return 0;
  const int knob = dex_tuning_memo();
  if (knob == 0 || rays.n_dirs <= 0 || g->n_active <= 0) return 0;
  const int D = g->desc.ndim;
  double cells0 = 1.0, mean_dim = 0.0;
  for (int a = 0; a < D; ++a) { cells0 *= (double)g->dev.B; mean_dim += (double)g->dev.dims[a] / D; }
  // rays through a level-0 cell per direction: probes x a typical path length (0.4 of the box) / active cells
  const double reuse = (double)rays.n_probes * 0.4 * mean_dim / ((double)g->n_active * cells0);
  if (knob < 0 && reuse < DEX_MEMO_MIN_REUSE) return 0;
  const double per_batch = (double)rays.n_dirs * 2.0 * (double)g->n_active * (double)m->dev.cps * DEX_W * sizeof(float);
  size_t free_b = 0, total_b = 0;
  if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { cudaGetLastError(); return 0; }
  // half of what is available (the driver's free memory plus what the library's own pool holds idle from earlier calls),
  // at most 32 GB in 2D and 40 GB in 3D.  Measured in round 3 (profiles/r03_memo_budget.md): C3 36 -> 16 GB of records
  // costs 0.8 % of a step, C4 65 -> 34 GB 1.6 %, C5 72 -> 37 GB 2.2 % (19 GB: 8.4 %); the round-2 caps (64 / 96 GB) left
  // a second tenant of the GPU nothing.  "memo_budget_mb" moves the cap either way.
  double budget = fmin(0.5 * ((double)free_b + (double)dex_pool_idle_bytes()), D == 3 ? 40.0e9 : 32.0e9);
  const int cap_mb = dex_tuning_memo_budget_mb();       // "memo_budget_mb": the caller's own bound on these temporaries;
  if (cap_mb > 0) {                                      // one batch is the smallest group, so it is taken even above the bound
    budget = fmin(budget, fmax((double)cap_mb * 1.0e6, fmin(per_batch, budget)));
  }
  const int nb = (int)fmin((double)m->n_batch, floor(budget / per_batch));
  return nb < 1 ? 0 : nb;
}

// one upload of the Weideman coefficients per device (they are constants of the method)
static dex_status ensure_march_constants() {
  static std::mutex mu;
  static bool done[64] = {false};
  int dev = 0;
  DEX_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return DEX_OK;
  std::lock_guard<std::mutex> lk(mu);
  if (!done[dev]) {
    double c[DEX_WEI_N], L = 0.0;
    dex_weideman_coefficients(c, &L);
    DEX_CUDA_CHECK(cudaMemcpyToSymbol(dex_c_wei, c, sizeof(c)));
    DEX_CUDA_CHECK(cudaMemcpyToSymbol(dex_c_wei_L, &L, sizeof(L)));
    done[dev] = true;
  }
  return DEX_OK;
}

// what the last dex_launch_march of this thread actually ran with (dex_last_march_mapping)
static thread_local int t_map_lanes = 0, t_map_dirs_per_block = 0, t_map_memo_group = 0;
void dex_last_mapping(int* lanes_per_ray, int* dirs_per_block, int* memo_batches_per_group) {
  if (lanes_per_ray) *lanes_per_ray = t_map_lanes;
  if (dirs_per_block) *dirs_per_block = t_map_dirs_per_block;
  if (memo_batches_per_group) *memo_batches_per_group = t_map_memo_group;
}

bool dex_auto_dir_split(long long n_probes, int n_dirs, int n_lambda) {
  const int split = dex_tuning_dir_split();
  const size_t i_floats = (size_t)n_probes * (size_t)n_dirs * (size_t)n_lambda;
  const bool small = n_probes < 148LL * 128 && n_dirs > 1 && i_floats <= (64u << 20);
  return split > 0 || (split < 0 && small);
}

int dex_auto_lanes(int set, long long n_probes, bool dir_split) {
  if (set != 0) return set;
  if (n_probes >= 148LL * 128) return 1;
  return dir_split ? 2 : 8;      // swept on C1 with the split: 1 / 2 / 4 / 8 lanes give 0.254 / 0.236 / 0.251 / 0.265 ms per step
}

dex_status dex_launch_march(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays, float* d_out, bool fuse_j,
                            unsigned long long* d_seg, int lanes_per_ray, bool tile, cudaStream_t st,
                            const int* perm_in) {
  int* d_perm = nullptr;
  dex_status s = (m->variant == DEX_ISO) ? DEX_OK : ensure_march_constants();
  if (s != DEX_OK) return s;
  if (tile && !perm_in) s = dex_make_probe_tiling(g, rays, &d_perm, st);
  const int* perm = perm_in ? perm_in : d_perm;
  // Small problems (fewer probes than one wave of blocks) leave most SMs idle while every thread walks its directions
  // one after the other (C1: 4096 probes x 16 directions).  There the fused J is taken apart: one block per (probe tile,
  // batch, direction) writes I (a few MB), and dex_reduce_j_kernel sums it in the fused kernel's own order, so J is
  // bit-identical to the fused path.  Whole-spectrum handles only (a pipeline stage writes a window of J's columns).
  DexRaysDev r = rays;
  r.k_per_block = 0;
  float* d_I = nullptr;
  const size_t i_floats = (size_t)rays.n_probes * (size_t)rays.n_dirs * (size_t)m->n_lambda;
  const int split = dex_tuning_dir_split();
  if (s == DEX_OK && fuse_j && dex_auto_dir_split(rays.n_probes, rays.n_dirs, m->n_lambda) && m->dev.io_base == 0 &&
      m->dev.io_stride == m->n_lambda && rays.t_end <= 0.0f) {
    cudaError_t e = dex_alloc((void**)&d_I, sizeof(float) * i_floats, st);
    if (e != cudaSuccess) { cudaGetLastError(); d_I = nullptr; }     // no room: the fused path needs none
    else r.k_per_block = (split > 0) ? split : 1;
  }
  lanes_per_ray = dex_auto_lanes(lanes_per_ray, rays.n_probes, d_I != nullptr);
  if (s == DEX_OK) {
    float* out = d_I ? d_I : d_out;
    const bool fj = d_I ? false : fuse_j;
    int memo = memo_group(g, m, r);
    if (memo > 0) {
      bool fell_back = false;
      if (g->desc.ndim == 2) s = launch_march_memo<2>(g, m, r, out, fj, d_seg, lanes_per_ray, perm, st, memo, &fell_back);
      else s = launch_march_memo<3>(g, m, r, out, fj, d_seg, lanes_per_ray, perm, st, memo, &fell_back);
      if (fell_back) memo = 0;         // no room for one batch of records: evaluate in the ray loop
    }
    t_map_lanes = lanes_per_ray;
    t_map_dirs_per_block = r.k_per_block;
    t_map_memo_group = memo;
    if (memo == 0) {
      if (g->desc.ndim == 2) s = launch_march_d<2>(g, m, r, out, fj, d_seg, lanes_per_ray, perm, st);
      else s = launch_march_d<3>(g, m, r, out, fj, d_seg, lanes_per_ray, perm, st);
    }
    if (s == DEX_OK && d_I) s = dex_launch_reduce_j(r, m->n_lambda, d_I, d_out, st);
  }
  if (d_I) dex_free(d_I, st);
  if (d_perm) cudaFreeAsync(d_perm, st);
  return s;
}

dex_status dex_launch_capture(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays,
                              const dex_visit_capture* cap, int* d_overflow, cudaStream_t st) {
  const long long n_rays = rays.n_probes * rays.n_dirs;
  if (n_rays <= 0) return DEX_OK;
  const int threads = 128;
  const long long gx = (n_rays + threads - 1) / threads;
  if (gx > 2147483647LL) {
    dex_set_error("capture: too many rays");
    return DEX_ERR_UNSUPPORTED;
  }
  if (g->desc.ndim == 2)
    dex_capture_kernel<2><<<(unsigned)gx, threads, 0, st>>>(g->dev, m->dev, rays, (long long*)cap->d_counts,
                                                            (unsigned long long*)cap->d_records, cap->d_ds,
                                                            (const long long*)cap->d_offsets, cap->capacity,
                                                            cap->batch, d_overflow);
  else
    dex_capture_kernel<3><<<(unsigned)gx, threads, 0, st>>>(g->dev, m->dev, rays, (long long*)cap->d_counts,
                                                            (unsigned long long*)cap->d_records, cap->d_ds,
                                                            (const long long*)cap->d_offsets, cap->capacity,
                                                            cap->batch, d_overflow);
  dex_count_launch();
  DEX_CUDA_CHECK(cudaGetLastError());
  return DEX_OK;
}

dex_status dex_launch_voigt_profile(const float* d_a, const double* d_x, long long n, double* d_H, int mode, cudaStream_t st) {
  if (n <= 0) return DEX_OK;
  DexWeideman Wc;
  dex_weideman_coefficients(Wc.c, &Wc.L);
  float* d_tab = nullptr;
  DEX_CUDA_CHECK(dex_alloc((void**)&d_tab, sizeof(float) * DEX_VF_NODES * 5, st));
  cudaError_t e = cudaMemcpyAsync(d_tab, dex_voigt_fast_table_host(), sizeof(float) * DEX_VF_NODES * 5, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) {
    const long long gx = (n + 255) / 256;
    dex_voigt_profile_kernel<<<(unsigned)gx, 256, 0, st>>>(d_a, d_x, n, d_H, mode, Wc, (const float4*)d_tab,
                                                           d_tab + (size_t)DEX_VF_NODES * 4);
    dex_count_launch();
    e = cudaGetLastError();
  }
  cudaFreeAsync(d_tab, st);
  DEX_CUDA_CHECK(e);
  return DEX_OK;
}

dex_status dex_launch_reduce_j(const DexRaysDev& rays, int n_lambda, const float* d_I, float* d_J, cudaStream_t st) {
  const long long n = rays.n_probes * n_lambda;
  if (n <= 0) return DEX_OK;
  const int threads = 256;
  const long long gx = (n + threads - 1) / threads;
  dex_reduce_j_kernel<<<(unsigned)gx, threads, 0, st>>>(rays.n_probes, rays.n_dirs, n_lambda, rays.weights, d_I, d_J,
                                                        rays.accumulate);
  dex_count_launch();
  DEX_CUDA_CHECK(cudaGetLastError());
  return DEX_OK;
}

