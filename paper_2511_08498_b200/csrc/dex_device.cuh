// dex_device.cuh -- device-side structures and the HDDA stepping shared by the march kernels.
//
// Traversal follows Algorithm 1 of the paper under the T-rules of DESIGN.md
// (SURVEY.md 8(c)): plane times are a pure function tplane(a,k) = fma(k, inv[a], off[a]) of the ray,
// never accumulated, so the visit list is well defined bit for bit.  All traversal arithmetic uses
// explicit round-to-nearest intrinsics so that nvcc's FMA contraction cannot change it.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define DEX_W 8            // wavelengths per batch
#define DEX_REC (2 * DEX_W) // floats per cell record: chi[0..W-1] then eta[0..W-1] (pairs of wavelengths feed FFMA2)
#define DEX_MAXLEV 6
#define DEX_NLINES 4

// cell record accessors: record r (in units of DEX_REC floats) of a store, wavelength j of the batch
__host__ __device__ __forceinline__ size_t dex_rec_chi(size_t r, int j) { return r * DEX_REC + j; }
__host__ __device__ __forceinline__ size_t dex_rec_eta(size_t r, int j) { return r * DEX_REC + DEX_W + j; }

struct DexGridDev {
  int ndim;
  int dims[3];
  int nb[3];     // bricks per axis
  int B, logB;
  float h;
  int n_bricks;
  int n_active;
  const int* slot;  // [n_bricks] -> storage slot or -1
};

struct DexMipsDev {
  int variant;
  int n_lambda, n_batch;
  int max_level;
  int bits, per_word, words_per_batch;
  const unsigned long long* packed;  // [n_batch][words_per_batch]  PAPER.md:162 packed block states (exported)
  const int* binfo;                  // [n_batch][n_bricks]  (slot << 4) | (level + 1): what the march reads
  int cps;                           // cells per slot (all levels)
  int lvloff[DEX_MAXLEV];            // first cell of level m inside a slot
  const float* store;                // [n_batch][n_active][cps][DEX_REC]  chi|eta (ISO) or background
  const float* mrec;                 // ISO march records, same shape as store: chi'|S with S = eta/chi (see
                                     // make_march_records_kernel); what the ISO march reads
  const float4* line;                // [n_active][cps][n_lines]  (eta*, chi*, a0, 1/dlamD)
  const float4* vel;                 // [n_active][cps]           (vx, vy, vz, max|v|)
  const float* vtab;                 // [n_batch][n_active][cps][n_vbins][DEX_REC]
  const float* lam;                  // [n_lambda] device
  const signed char* active_lines;   // [n_batch][DEX_NLINES] device
  int n_lines, n_vbins;
  float lambda0[DEX_NLINES];
  double c_light;
  double wei_c[24];                  // Weideman N=24 coefficients c_1..c_24
  double wei_L;
};

struct DexRaysDev {
  long long n_probes;
  const float* probe_pos;
  int n_dirs;
  const float* dirs;
  const float* weights;
  const float* i0;
};

// ---- exact (uncontracted) fp32 helpers -------------------------------------------------
__device__ __forceinline__ float dex_tplane(int k, float inv, float off) {
  return __fmaf_rn((float)k, inv, off);  // T2
}

template <int D>
struct DexRay {
  float o[D], d[D], inv[D], off[D];
  float tn[D];
  int c[D];
  int m, size, slot;
  float t;
};

__device__ __forceinline__ int dex_brick_level(const DexMipsDev& M, int batch, int bi) {
  int q, r;
  if (M.bits == 3) { q = bi / 21; r = bi - q * 21; }
  else if (M.bits == 2) { q = bi >> 5; r = bi & 31; }
  else if (M.bits == 1) { q = bi >> 6; r = bi & 63; }
  else { q = bi / M.per_word; r = bi - q * M.per_word; }
  unsigned long long w = __ldg(M.packed + (size_t)batch * M.words_per_batch + q);
  return (int)((w >> (r * M.bits)) & ((1ull << M.bits) - 1ull)) - 1;
}

// plane (a,k) counts as crossed at the event (s, th) iff tplane < th, or == th and a < s  (T5)
__device__ __forceinline__ bool dex_crossed(int k, float inv, float off, float th, bool lower_axis) {
  float tp = dex_tplane(k, inv, off);
  return (tp < th) || (tp == th && lower_axis);
}

// level-0 coordinate on axis a (inside the cell [lo, lo+size)) that the plain DDA would hold when
// the ray crosses the exit plane of axis s at time th.  Guess from the position, then correct with
// the monotone `crossed` predicate -- the result is the unique one defined by T5.
__device__ __forceinline__ int dex_fine_coord(float o, float d, float inv, float off, int lo, int size,
                                              float th, bool lower_axis) {
  if (d == 0.0f) return (int)floorf(o);
  const int hi = lo + size - 1;
  int g = (int)floorf(__fmaf_rn(th, d, o));
  g = max(lo, min(hi, g));
  if (d > 0.0f) {
    while (g < hi && dex_crossed(g + 1, inv, off, th, lower_axis)) ++g;
    while (g > lo && !dex_crossed(g, inv, off, th, lower_axis)) --g;
  } else {
    while (g > lo && dex_crossed(g, inv, off, th, lower_axis)) --g;
    while (g < hi && !dex_crossed(g + 1, inv, off, th, lower_axis)) ++g;
  }
  return g;
}

template <int D>
__device__ __forceinline__ int dex_brick_of(const DexGridDev& G, const int* c) {
  int bi = (c[1] >> G.logB) * G.nb[0] + (c[0] >> G.logB);
  if (D == 3) bi += (c[2] >> G.logB) * G.nb[0] * G.nb[1];
  return bi;
}

template <int D>
__device__ __forceinline__ void dex_set_planes(DexRay<D>& r) {
#pragma unroll
  for (int a = 0; a < D; ++a) {
    int kp = (r.d[a] > 0.0f) ? r.c[a] + r.size : r.c[a];
    r.tn[a] = (r.d[a] != 0.0f) ? dex_tplane(kp, r.inv[a], r.off[a]) : __int_as_float(0x7f800000);
  }
}

// T1/T2/T6: trace from the probe outward, o = probe, d = -omega.  Returns false for a probe outside
// the grid or a null direction (such a ray has no segments).
template <int D>
__device__ __forceinline__ bool dex_ray_init(DexRay<D>& r, const DexGridDev& G, const DexMipsDev& M, int batch,
                                             const float* probe, const float* omega) {
  bool ok = true, any = false;
  int x[D];
#pragma unroll
  for (int a = 0; a < D; ++a) {
    r.o[a] = probe[a];
    r.d[a] = -omega[a];
    r.inv[a] = 0.0f;
    r.off[a] = 0.0f;
    if (r.d[a] != 0.0f) {
      any = true;
      r.inv[a] = __fdiv_rn(1.0f, r.d[a]);
      r.off[a] = __fmul_rn(-r.o[a], r.inv[a]);
    }
    x[a] = (int)floorf(r.o[a]);
    ok = ok && (x[a] >= 0) && (x[a] < G.dims[a]);
  }
  r.t = 0.0f;
  r.m = -1;
  r.size = 1;
  r.slot = -1;
  if (!(ok && any)) return false;
  int bi = dex_brick_of<D>(G, x);
  r.m = dex_brick_level(M, batch, bi);
  r.slot = __ldg(G.slot + bi);
  r.size = (r.m < 0) ? G.B : (1 << r.m);
#pragma unroll
  for (int a = 0; a < D; ++a) r.c[a] = x[a] & ~(r.size - 1);
  dex_set_planes<D>(r);
  return true;
}

// One HDDA event.  On return: `emit` says whether the cell that was just left contributes a segment
// (non-empty and th > t, T4); em_m / em_c / em_slot / ds describe it.  Returns false when the ray has
// left the grid (the segment, if any, is still valid).
template <int D>
struct DexSeg {
  bool emit;
  int m, slot;
  int c[D];
  float ds;
};

template <int D>
__device__ __forceinline__ bool dex_ray_step(DexRay<D>& r, const DexGridDev& G, const DexMipsDev& M, int batch,
                                             DexSeg<D>& seg) {
  // T4: lowest-index axis attaining the minimum
  int s = 0;
  float th = r.tn[0];
  if (r.tn[1] < th) { s = 1; th = r.tn[1]; }
  if (D == 3) { if (r.tn[D - 1] < th) { s = D - 1; th = r.tn[D - 1]; } }
  seg.emit = (r.m >= 0) && (th > r.t);
  seg.m = r.m;
  seg.slot = r.slot;
#pragma unroll
  for (int a = 0; a < D; ++a) seg.c[a] = r.c[a];
  seg.ds = __fsub_rn(th, r.t);
  r.t = fmaxf(r.t, th);
  // T5: cross the plane
  float ds_ = 0.f; int cs = 0, Ns = 0;
#pragma unroll
  for (int a = 0; a < D; ++a) if (a == s) { ds_ = r.d[a]; cs = r.c[a]; Ns = G.dims[a]; }
  const bool pos = ds_ > 0.0f;
  const int xs = pos ? cs + r.size : cs - 1;
  if (xs < 0 || xs >= Ns) return false;
  if ((xs >> G.logB) == (cs >> G.logB)) {
    // same brick: same level; only axis s moves
    const int ncs = pos ? cs + r.size : cs - r.size;
#pragma unroll
    for (int a = 0; a < D; ++a)
      if (a == s) {
        r.c[a] = ncs;
        r.tn[a] = dex_tplane(pos ? ncs + r.size : ncs, r.inv[a], r.off[a]);
      }
    return true;
  }
  // new brick: look up its level (MipLevel, Alg. 1 l.6-8) and re-initialise (l.32-39)
  int xb[D];
#pragma unroll
  for (int a = 0; a < D; ++a) xb[a] = (a == s) ? xs : r.c[a];
  const int bi = dex_brick_of<D>(G, xb);
  const int m2 = dex_brick_level(M, batch, bi);
  const int size2 = (m2 < 0) ? G.B : (1 << m2);
  if (size2 < r.size) {
#pragma unroll
    for (int a = 0; a < D; ++a)
      if (a != s) xb[a] = dex_fine_coord(r.o[a], r.d[a], r.inv[a], r.off[a], r.c[a], r.size, th, a < s);
  }
#pragma unroll
  for (int a = 0; a < D; ++a) r.c[a] = xb[a] & ~(size2 - 1);
  r.m = m2;
  r.size = size2;
  r.slot = __ldg(G.slot + bi);
  dex_set_planes<D>(r);
  return true;
}

// index of the cell inside its slot: level offset + row-major position at that level
template <int D>
__device__ __forceinline__ int dex_cell_in_slot(const DexGridDev& G, const DexMipsDev& M, int m, const int* c) {
  const int mask = G.B - 1;
  const int nb = G.B >> m;
  int idx = ((c[1] & mask) >> m) * nb + ((c[0] & mask) >> m);
  if (D == 3) idx += ((c[2] & mask) >> m) * nb * nb;
  return M.lvloff[m] + idx;
}


// ---------------------------------------------------------------------------------------------------
// v2 stepping used by the march kernel: same T-rules, fewer instructions.
//   * size = 1 << sh for cells and for empty bricks alike (sh = level, or log2 B for an empty brick)
//   * zero-direction axes carry inv = 0, off = +INF, so tplane = fma(k, 0, INF) = +INF without a select
//   * pm[a] = -1 if d[a] > 0 else 0: exit plane = c[a] + (size & pm[a])
//   * one 4-byte (slot, level) word per brick instead of the packed word + slot table
// ---------------------------------------------------------------------------------------------------
template <int D>
struct DexRay2 {
  float o[D], d[D], inv[D], off[D];
  float tn[D];
  int c[D], pm[D];
  int sh;        // log2 of the current cell (or empty-brick) size
  int cellbase;  // slot * cps + lvloff[level]; < 0 for an empty brick
  float t;
};

template <int D>
__device__ __forceinline__ void dex_planes2(DexRay2<D>& r) {
  const int size = 1 << r.sh;
#pragma unroll
  for (int a = 0; a < D; ++a) r.tn[a] = __fmaf_rn((float)(r.c[a] + (size & r.pm[a])), r.inv[a], r.off[a]);
}

__device__ __forceinline__ void dex_decode_brick(const DexGridDev& G, const DexMipsDev& M, int info, int& sh, int& cellbase) {
  const int m = (info & 15) - 1;
  sh = (m < 0) ? G.logB : m;
  cellbase = (m < 0) ? -1 : (info >> 4) * M.cps + M.lvloff[m];
}

template <int D>
__device__ __forceinline__ bool dex_ray_init2(DexRay2<D>& r, const DexGridDev& G, const DexMipsDev& M,
                                              const int* __restrict__ binfo, const float* probe, const float* omega) {
  bool ok = true, any = false;
  int x[D];
#pragma unroll
  for (int a = 0; a < D; ++a) {
    r.o[a] = probe[a];
    r.d[a] = -omega[a];
    r.pm[a] = (r.d[a] > 0.0f) ? -1 : 0;
    if (r.d[a] != 0.0f) {
      any = true;
      r.inv[a] = __fdiv_rn(1.0f, r.d[a]);
      r.off[a] = __fmul_rn(-r.o[a], r.inv[a]);
    } else {
      r.inv[a] = 0.0f;
      r.off[a] = __int_as_float(0x7f800000);
    }
    x[a] = (int)floorf(r.o[a]);
    ok = ok && (x[a] >= 0) && (x[a] < G.dims[a]);
  }
  r.t = 0.0f;
  r.sh = 0;
  r.cellbase = -1;
  if (!(ok && any)) return false;
  dex_decode_brick(G, M, __ldg(binfo + dex_brick_of<D>(G, x)), r.sh, r.cellbase);
  const int amask = ~((1 << r.sh) - 1);
#pragma unroll
  for (int a = 0; a < D; ++a) r.c[a] = x[a] & amask;
  dex_planes2<D>(r);
  return true;
}

// One HDDA event.  emit / cell / ds describe the cell that was just left (T4).  Returns false when the
// ray has left the grid.
template <int D>
__device__ __forceinline__ bool dex_ray_step2(DexRay2<D>& r, const DexGridDev& G, const DexMipsDev& M,
                                              const int* __restrict__ binfo, bool& emit, int& cell, float& ds) {
  int s = 0;
  float th = r.tn[0];
  if (r.tn[1] < th) { s = 1; th = r.tn[1]; }
  if (D == 3) { if (r.tn[D - 1] < th) { s = D - 1; th = r.tn[D - 1]; } }
  emit = (r.cellbase >= 0) && (th > r.t);
  ds = __fsub_rn(th, r.t);
  {
    const int mask = G.B - 1, lsh = G.logB - r.sh;
    int idx = (((r.c[1] & mask) >> r.sh) << lsh) + ((r.c[0] & mask) >> r.sh);
    if (D == 3) idx += ((r.c[D - 1] & mask) >> r.sh) << (2 * lsh);
    cell = r.cellbase + idx;
  }
  r.t = fmaxf(r.t, th);
  const int size = 1 << r.sh;
  int cs = r.c[0], pms = r.pm[0], Ns = G.dims[0];
  if (s == 1) { cs = r.c[1]; pms = r.pm[1]; Ns = G.dims[1]; }
  if (D == 3) { if (s == D - 1) { cs = r.c[D - 1]; pms = r.pm[D - 1]; Ns = G.dims[D - 1]; } }
  const int xs = pms ? cs + size : cs - 1;                      // T5
  if ((unsigned)xs >= (unsigned)Ns) return false;
  int x[D];
#pragma unroll
  for (int a = 0; a < D; ++a) x[a] = (a == s) ? xs : r.c[a];
  if (((xs ^ cs) >> G.logB) != 0) {
    // new brick: MipLevel (Alg. 1 l.6-8) and re-initialisation (l.32-39)
    int sh2, cb2;
    dex_decode_brick(G, M, __ldg(binfo + dex_brick_of<D>(G, x)), sh2, cb2);
    if (sh2 < r.sh) {
#pragma unroll
      for (int a = 0; a < D; ++a)
        if (a != s) x[a] = dex_fine_coord(r.o[a], r.d[a], r.inv[a], r.off[a], r.c[a], size, th, a < s);
    }
    r.sh = sh2;
    r.cellbase = cb2;
  }
  const int amask = ~((1 << r.sh) - 1);
#pragma unroll
  for (int a = 0; a < D; ++a) r.c[a] = x[a] & amask;
  dex_planes2<D>(r);
  return true;
}
