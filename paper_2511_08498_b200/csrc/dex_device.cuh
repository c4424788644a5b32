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
// floats between the march records of consecutive cells: 8 in 2D (two planes), 16 in 3D (interleaved), see DexMipsDev::mrec
template <int D> struct DexRecStride { static constexpr int value = (D == 3) ? 2 * DEX_W : DEX_W; };
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
  const int* binfo;                  // [n_batch][n_bricks]  ((slot * cps + lvloff[level]) << 4) | (level + 1), 0 = empty:
                                     // the one word the march reads per brick crossing
  int cps;                           // cells per slot (all levels)
  int lvloff[DEX_MAXLEV];            // first cell of level m inside a slot
  const float* store;                // [n_batch][n_active][cps][DEX_REC]  chi|eta (ISO) or background
  const float* mrec;                 // ISO march records (make_march_records_kernel), what the ISO march reads.  2D: two planes
  size_t mplane;                     // [2][n_batch][n_active][cps][DEX_W], plane 0 chi log2(e), plane 1 S = eta/chi, mplane =
                                     // floats per plane (lanes in x-adjacent cells share L1 lines).  3D: one 64-byte record per
                                     // cell, [n_batch][n_active][cps][chi log2(e) x 8 | S x 8], mplane = DEX_W: rays are sparse
                                     // there, and a record that misses the L2 costs one 64-byte DRAM burst instead of two
  size_t mdir;                       // 0, or floats between the records of consecutive DIRECTIONS (Core-and-Voigt memoised
                                     // per direction, march.cu: mrec then holds [n_dirs][2][n_batch][n_active][cps][DEX_W])
  const float4* aux;                 // [n_active][cps][1 + n_lines]: (vx, vy, vz, max|v|) then per line (eta*, chi*, a0,
                                     // 1/dlamD), see dex_aux_vel / dex_aux_line
  int aux_vs, aux_ls;                // float4 strides of the velocity and of a cell's line records
  size_t aux_lo;                     // float4 index of the first line record
  const float* vtab;                 // [n_batch][n_active][cps][n_vbins][DEX_REC]
  const float* lam;                  // [n_lambda] device
  const signed char* active_lines;   // [n_batch][DEX_NLINES] device
  int n_lines, n_vbins;
  float lambda0[DEX_NLINES];
  double c_light;
  double wei_c[24];                  // Weideman N=24 coefficients c_1..c_24
  double wei_L;
  const float4* vf_wing;             // [DEX_VF_NODES] Taylor coefficients of Im F about the nodes (dex_voigt.cuh)
  const float* vf_core;              // [DEX_VF_NODES] e^{-x_k^2}
  int n_caps;                        // near-field MIP cap (T8, dex_mips_set_level_caps): a cell entered at distance t is
  float cap_t[8];                    // formed at level min(brick level, #{i : t >= cap_t[i]}); n_caps = 0: no cap
  int voigt_fp32;                    // 0: fp64 HUM1WEI24 everywhere (tuning knob "voigt_fp32")
  int in_stride;                     // floats between consecutive voxels of the caller's [nvox][lambda] inputs (build)
  int io_stride, io_base;            // row length and first column of this handle's wavelengths in I / J / i0: n_lambda and
                                     // 0 unless the handle is one stage of dex_mean_intensity_pipelined
};

// Auxiliary chains of the anisotropic variants in one array `aux` of float4: velocity (vx, vy, vz, max|v|) and per line
// (eta*, chi*, a0, 1/dlamD).  Core-and-Voigt / Classic marches read both at every segment, so there a cell's record is
// contiguous, [velocity, line_0 .. line_{n-1}]: ONE 32-byte sector for one line (two for three lines) instead of a
// sector each from two arrays (C5 is bound by DRAM sectors: 184.7 -> 171.8 ms, profiles/r01k).  The velocity-
// interpolation march reads the velocity only, so there the velocities stay dense (16 B per cell) and the line records,
// which only the build uses, follow them.  vel(cell) = aux[cell * aux_vs], line(cell, l) = aux[aux_lo + cell * aux_ls + l].
__device__ __forceinline__ size_t dex_aux_vel(const DexMipsDev& M, size_t cell) { return cell * (size_t)M.aux_vs; }
__device__ __forceinline__ size_t dex_aux_line(const DexMipsDev& M, size_t cell, int l) {
  return M.aux_lo + cell * (size_t)M.aux_ls + (size_t)l;
}

struct DexRaysDev {
  long long n_probes;
  const float* probe_pos;
  int n_dirs;
  const float* dirs;
  const float* weights;
  const float* i0;
  const float* sin_incl;   // [n_dirs] or NULL: 2.5D rays
  float t_begin, t_end;    // finite radiance interval (T10); t_end <= 0: to the boundary
  int accumulate;          // fused J: d_J += sum_k w_k I_k instead of = (single-direction VLM sums its per-direction solves)
  int k_per_block;         // > 0: blockIdx.z selects a run of this many directions (materialised I only: small problems
                           // are spread over the machine direction by direction, dex_launch_march); 0: all directions
};

// ---- exact (uncontracted) fp32 helpers -------------------------------------------------
__device__ __forceinline__ float dex_tplane(int k, float inv, float off) {
  return __fmaf_rn((float)k, inv, off);  // T2
}

// plane (a,k) counts as crossed at the event (s, th) iff tplane < th, or == th and a < s  (T5)
__device__ __forceinline__ bool dex_crossed(int k, float inv, float off, float th, bool lower_axis) {
  float tp = dex_tplane(k, inv, off);
  return (tp < th) || (tp == th && lower_axis);
}

// level-0 coordinate on axis a (inside the cell [lo, lo+size)) that the plain DDA would hold when
// the ray crosses the exit plane of axis s at time th: the unique G in [lo, hi] with every plane up to G
// crossed and none beyond (T5; `crossed` is monotone along the ray).  The position o + th d locates it to
// within one voxel (plane times and position are fp32 evaluations of the same line, ~1e-4 voxel apart at
// coordinates below 2^18), so the guess is corrected by one step from two evaluations of the predicate --
// straight-line code (the correction loops this replaces were 11 % of the instructions of C2's march).
__device__ __forceinline__ int dex_fine_coord(float o, float d, float inv, float off, int lo, int size,
                                              float th, bool lower_axis) {
  if (d == 0.0f) return (int)floorf(o);
  const int hi = lo + size - 1;
  int g = (int)floorf(__fmaf_rn(th, d, o));
  g = max(lo, min(hi, g));
  const bool c0 = dex_crossed(g, inv, off, th, lower_axis);        // plane g
  const bool c1 = dex_crossed(g + 1, inv, off, th, lower_axis);    // plane g + 1
  if (d > 0.0f) {
    // cell g holds the ray iff plane g is crossed (or g == lo) and plane g + 1 is not (or g == hi)
    if (c1 && g < hi) return g + 1;
    if (!c0 && g > lo) return g - 1;
  } else {
    // moving down: cell g holds the ray iff plane g + 1 is crossed (or g == hi) and plane g is not (or g == lo)
    if (c0 && g > lo) return g - 1;
    if (!c1 && g < hi) return g + 1;
  }
  return g;
}

template <int D>
__device__ __forceinline__ int dex_brick_of(const DexGridDev& G, const int* c) {
  int bi = (c[1] >> G.logB) * G.nb[0] + (c[0] >> G.logB);
  if (D == 3) bi += (c[2] >> G.logB) * G.nb[0] * G.nb[1];
  return bi;
}

// ---------------------------------------------------------------------------------------------------
// HDDA state (Algorithm 1 under the T-rules), arranged so that a crossing that stays inside a brick --
// the common event -- costs a handful of instructions:
//   * kf[a] is the coordinate of the exit plane of axis a, kept as a float (integers below 2^24 are exact),
//     so the plane time is one fma, tn[a] = fma(kf[a], inv[a], off[a]) (T2), and an in-brick crossing of
//     axis s is  kf[s] += dk[s];  tn[s] = fma(..);  cell += cstep[s].
//   * tb = min over axes of the time of the BRICK's exit plane.  th < tb (strictly) proves that the plane
//     being crossed is not a brick face, so the level cannot change and only axis s moves.  Everything
//     else (brick faces, ties with a brick face, empty bricks, whole-brick cells) takes the general path,
//     which rebuilds the state from integer coordinates exactly as T3-T5 prescribe.
//   * zero-direction axes carry inv = 0, off = +INF, so tn = fma(k, 0, INF) = +INF without a select.
// ---------------------------------------------------------------------------------------------------
//   * the origin and direction themselves are not kept in registers: only the T5 re-entry into a finer brick
//     needs them, and reloads them from the (L1-resident) ray arrays.
template <int D>
struct DexRay3 {
  float inv[D], off[D];
  float tn[D], kf[D], dk[D];  // dk[a] > 0 iff d[a] > 0
  int cstep[D];
  int cell;   // record index (slot * cps + lvloff[level] + position) of the current cell; < 0 in an empty brick
  int sh;     // log2 of the current cell (or empty-brick) size
  int info;   // brick word of the current brick: (first record of the brick's level << 4) | (level + 1); 0 = empty
  float t, tb;
};

// Form the cell of brick word `info` that contains level-0 coordinate x (T3) and everything derived from it.
template <int D>
__device__ __forceinline__ void dex_set_cell(DexRay3<D>& r, const DexGridDev& G, const DexMipsDev& M, int info,
                                             const int* x) {
  int m = (info & 15) - 1;
  int base = info >> 4;
  float tcap = __int_as_float(0x7f800000);
  if (m > 0 && M.n_caps > 0) {
    // T8: the level of this visit is capped by the distance r.t at which the cell is entered; the cell is formed
    // again when the ray reaches the next threshold (folded into tb, so the in-brick fast step pays nothing)
    int cap = 0;
    for (int i = 0; i < M.n_caps; ++i) cap += (r.t >= M.cap_t[i]) ? 1 : 0;
    if (cap < m) {
      base += M.lvloff[cap] - M.lvloff[m];
      m = cap;
      tcap = M.cap_t[cap];
    }
  }
  const int sh = (m < 0) ? G.logB : m;
  const int size = 1 << sh, lsh = G.logB - sh, bmask = G.B - 1;
  r.info = info;
  r.sh = sh;
  int idx = 0;
  float tb = __int_as_float(0x7f800000);
#pragma unroll
  for (int a = 0; a < D; ++a) {
    const bool pos = r.dk[a] > 0.0f;
    const int c = x[a] & ~(size - 1);
    r.kf[a] = (float)(c + (pos ? size : 0));
    r.tn[a] = __fmaf_rn(r.kf[a], r.inv[a], r.off[a]);
    r.dk[a] = pos ? (float)size : -(float)size;
    const int bexit = (x[a] & ~bmask) + (pos ? G.B : 0);
    tb = fminf(tb, __fmaf_rn((float)bexit, r.inv[a], r.off[a]));
    idx += ((c & bmask) >> sh) << (a * lsh);
    r.cstep[a] = pos ? (1 << (a * lsh)) : -(1 << (a * lsh));
  }
  r.tb = fminf(tb, tcap);
  r.cell = (m < 0) ? -1 : base + idx;
}

// T1/T2/T6: trace from the probe outward, o = probe, d = -omega.  Returns false for a probe outside
// the grid or a null direction (such a ray has no segments).
template <int D>
__device__ __forceinline__ bool dex_ray_init3(DexRay3<D>& r, const DexGridDev& G, const DexMipsDev& M,
                                              const int* __restrict__ binfo, const float* probe, const float* omega) {
  bool ok = true, any = false;
  int x[D];
#pragma unroll
  for (int a = 0; a < D; ++a) {
    const float o = probe[a], d = -omega[a];
    r.dk[a] = d;              // only its sign is read (dex_set_cell), which then stores +-size
    if (d != 0.0f) {
      any = true;
      r.inv[a] = __fdiv_rn(1.0f, d);
      r.off[a] = __fmul_rn(-o, r.inv[a]);
    } else {
      r.inv[a] = 0.0f;
      r.off[a] = __int_as_float(0x7f800000);
    }
    x[a] = (int)floorf(o);
    ok = ok && (x[a] >= 0) && (x[a] < G.dims[a]);
  }
  r.t = 0.0f;
  if (!(ok && any)) return false;
  dex_set_cell<D>(r, G, M, __ldg(binfo + dex_brick_of<D>(G, x)), x);
  return true;
}

// level and level-0 low corner of the current cell (visit records, T7)
template <int D>
__device__ __forceinline__ void dex_ray_cell_coords(const DexRay3<D>& r, int* c) {
#pragma unroll
  for (int a = 0; a < D; ++a) c[a] = (int)r.kf[a] - ((r.dk[a] > 0.0f) ? (1 << r.sh) : 0);
}

// T4: lowest-index axis attaining the minimum exit time
template <int D>
__device__ __forceinline__ void dex_ray_next_plane(const DexRay3<D>& r, int& s, float& th) {
  s = 0;
  th = r.tn[0];
  if (r.tn[1] < th) { s = 1; th = r.tn[1]; }
  if (D == 3) { if (r.tn[D - 1] < th) { s = D - 1; th = r.tn[D - 1]; } }
}

// First half of an HDDA event: emit / cell / ds describe the cell being left (T4); if the crossing stays inside
// the brick it is carried out and true is returned.  false: the ray now waits at a brick face (or the grid
// boundary, or a tie with one) and dex_ray_cross completes the event.
template <int D>
__device__ __forceinline__ bool dex_ray_advance(DexRay3<D>& r, bool& emit, int& cell, float& ds) {
  int s;
  float th;
  dex_ray_next_plane<D>(r, s, th);
  emit = (r.cell >= 0) && (th > r.t);
  cell = r.cell;
  ds = __fsub_rn(th, r.t);
  r.t = fmaxf(r.t, th);
  const bool inside = th < r.tb;
  if (inside) {
    if (s == 0) {
      r.kf[0] = __fadd_rn(r.kf[0], r.dk[0]);
      r.tn[0] = __fmaf_rn(r.kf[0], r.inv[0], r.off[0]);
      r.cell += r.cstep[0];
    } else if (D == 2 || s == 1) {
      r.kf[1] = __fadd_rn(r.kf[1], r.dk[1]);
      r.tn[1] = __fmaf_rn(r.kf[1], r.inv[1], r.off[1]);
      r.cell += r.cstep[1];
    } else {
      r.kf[D - 1] = __fadd_rn(r.kf[D - 1], r.dk[D - 1]);
      r.tn[D - 1] = __fmaf_rn(r.kf[D - 1], r.inv[D - 1], r.off[D - 1]);
      r.cell += r.cstep[D - 1];
    }
  }
  return inside;
}

// Second half, general crossing (T5) for a ray that dex_ray_advance left waiting: the plane is found again (the
// exit times have not changed), the level-0 coordinates are rebuilt, the brick looked up (MipLevel, Alg. 1 l.6-8)
// and the state re-initialised (l.32-39).  Returns false when the ray has left the grid.
template <int D>
__device__ __forceinline__ bool dex_ray_cross(DexRay3<D>& r, const DexGridDev& G, const DexMipsDev& M,
                                              const int* __restrict__ binfo, const float* __restrict__ probe,
                                              const float* __restrict__ omega) {
  int s;
  float th;
  dex_ray_next_plane<D>(r, s, th);
  const int size = 1 << r.sh;
  int c[D];
  dex_ray_cell_coords<D>(r, c);
  int cs = c[0], Ns = G.dims[0];
  bool pos = r.dk[0] > 0.0f;
  if (s == 1) { cs = c[1]; Ns = G.dims[1]; pos = r.dk[1] > 0.0f; }
  if (D == 3) { if (s == D - 1) { cs = c[D - 1]; Ns = G.dims[D - 1]; pos = r.dk[D - 1] > 0.0f; } }
  const int xs = pos ? cs + size : cs - 1;
  const bool alive = (unsigned)xs < (unsigned)Ns;
  if (alive) {
    int x[D];
#pragma unroll
    for (int a = 0; a < D; ++a) x[a] = (a == s) ? xs : c[a];
    int info = r.info;
    if (((xs ^ cs) >> G.logB) != 0) {
      info = __ldg(binfo + dex_brick_of<D>(G, x));
      int m2 = (info & 15) - 1;
      if (m2 > 0 && M.n_caps > 0) {
        int cap = 0;
        for (int i = 0; i < M.n_caps; ++i) cap += (r.t >= M.cap_t[i]) ? 1 : 0;
        m2 = min(m2, cap);
      }
      const int sh2 = (m2 < 0) ? G.logB : m2;
      if (sh2 < r.sh) {
#pragma unroll
        for (int a = 0; a < D; ++a)
          if (a != s) x[a] = dex_fine_coord(__ldg(probe + a), -__ldg(omega + a), r.inv[a], r.off[a], c[a], size, th, a < s);
      }
    }
    dex_set_cell<D>(r, G, M, info, x);
  }
  return alive;
}

// ---- the same two routines without the near-field cap (M.n_caps == 0, the default): the march kernel picks the pair
// once per block.  The cap's threshold loops sit in the middle of the general routines; without them a crossing is
// straight-line code apart from the rare re-entry into a finer brick (profiles/r02: the crossing was 25 % of the
// instructions of C3's march).
template <int D, bool BOX>
__device__ __forceinline__ void dex_set_cell_nocap(DexRay3<D>& r, const DexGridDev& G, int info, const int* x) {
  const int m = (info & 15) - 1;
  r.info = info;
  if (m < 0) {
    // empty brick: the word carries the empty-space distance d (grid_build.cu); the cell is the (2d-1)^D box of empty
    // bricks around this one, clipped to the grid.  Its exit times are plane times like any other (T2), and a ray
    // leaves it through the face of the brick it enters next, so the times of the emitted visits are unchanged.
    // (2D only: in 3D the two extra coordinate searches per box exit and their registers cost the Core-and-Voigt march
    //  more than the skipped bricks save -- C5 139.7 -> 142.0 ms with boxes, C2 45.7 -> 44.4, C3 317.0 -> 311.5)
    const int d = BOX ? max(1, info >> 4) : 1;
    r.sh = (d > 1) ? G.logB + 1 : G.logB;        // sh > logB marks a multi-brick box (dex_ray_cross_nocap)
    const float fB = (float)G.B;
    float tb = __int_as_float(0x7f800000);
#pragma unroll
    for (int a = 0; a < D; ++a) {
      const bool pos = r.dk[a] > 0.0f;
      const int bq = x[a] >> G.logB;
      const int face = pos ? min(G.nb[a], bq + d) : max(0, bq - d + 1);
      r.kf[a] = (float)(face << G.logB);
      r.tn[a] = __fmaf_rn(r.kf[a], r.inv[a], r.off[a]);
      r.dk[a] = pos ? fB : -fB;                    // only the sign is read while the cell is empty
      if (BOX) r.cstep[a] = x[a] & ~(G.B - 1);     // low corner of the brick the box is entered in (dex_ray_cross_nocap)
      tb = fminf(tb, r.tn[a]);
    }
    r.tb = tb;
    r.cell = -1;
    return;
  }
  const int sh = m;
  const int size = 1 << sh, lsh = G.logB - sh, bmask = G.B - 1;
  const float fsize = (float)size;
  r.sh = sh;
  int idx = 0;
  float tb = __int_as_float(0x7f800000);
#pragma unroll
  for (int a = 0; a < D; ++a) {
    const bool pos = r.dk[a] > 0.0f;
    const int c = x[a] & -size;
    r.kf[a] = (float)(pos ? c + size : c);
    r.tn[a] = __fmaf_rn(r.kf[a], r.inv[a], r.off[a]);
    r.dk[a] = pos ? fsize : -fsize;
    const int bexit = pos ? (x[a] | bmask) + 1 : (x[a] & ~bmask);
    tb = fminf(tb, __fmaf_rn((float)bexit, r.inv[a], r.off[a]));
    idx += ((c & bmask) >> sh) << (a * lsh);
    const int st = 1 << (a * lsh);
    r.cstep[a] = pos ? st : -st;
  }
  r.tb = tb;
  r.cell = (info >> 4) + idx;
}

template <int D, bool BOX>
__device__ __forceinline__ bool dex_ray_cross_nocap(DexRay3<D>& r, const DexGridDev& G, const int* __restrict__ binfo,
                                                    const float* __restrict__ probe, const float* __restrict__ omega) {
  int s;
  float th;
  dex_ray_next_plane<D>(r, s, th);
  const int size = 1 << r.sh;
  int x[D], c[D];
  // exit plane kp, low corner c of the current cell per axis (T3); scalars of the crossed axis by select, not by index
  int kps = (int)r.kf[0], dims_s = G.dims[0];
  bool poss = r.dk[0] > 0.0f;
  c[0] = poss ? kps - size : kps;
  if (D >= 2) {
    const int kp1 = (int)r.kf[1];
    const bool pos1 = r.dk[1] > 0.0f;
    c[1] = pos1 ? kp1 - size : kp1;
    if (s == 1) { kps = kp1; poss = pos1; dims_s = G.dims[1]; }
  }
  if (D == 3) {
    const int kp2 = (int)r.kf[D - 1];
    const bool pos2 = r.dk[D - 1] > 0.0f;
    c[D - 1] = pos2 ? kp2 - size : kp2;
    if (s == D - 1) { kps = kp2; poss = pos2; dims_s = G.dims[D - 1]; }
  }
  const int xe = poss ? kps : kps - 1;           // level-0 coordinate just beyond the exit plane (T5)
  const int cs = poss ? kps - size : kps;
  const bool alive = (unsigned)xe < (unsigned)dims_s;
  const bool box = BOX && r.sh > G.logB;        // leaving a multi-brick box of empty space (dex_set_cell_nocap)
  const bool newbrick = box || ((xe ^ cs) >> G.logB) != 0;
#pragma unroll
  for (int a = 0; a < D; ++a) x[a] = (a == s) ? xe : c[a];
  if (!alive) return false;
  if (box) {
    // the box spans several bricks on the other axes: the brick being entered is the one holding the HDDA's
    // coordinates at this event (T5), searched over the whole axis (the position locates them to within one voxel).
    // Taking the empty bricks one at a time clamps the T5 coordinate to the current brick at every step; over the
    // box that composes to a clamp against the brick the box was entered in, on the side the ray comes from (the
    // T5 coordinate is monotone along the ray).  It only acts when a probe sits exactly on a cell plane and the
    // direction component is so small (|d| ~ 1e-16, a cos(pi/2) that is not quite 0) that the fp32 plane time of that
    // very plane is rounding noise: the plane then does not count as crossed although the ray started beyond it.
#pragma unroll
    for (int a = 0; a < D; ++a)
      if (a != s) {
        const float da = -__ldg(omega + a);
        int xa = dex_fine_coord(__ldg(probe + a), da, r.inv[a], r.off[a], 0, G.dims[a], th, a < s);
        if (da > 0.0f) xa = max(xa, r.cstep[a]);
        else if (da < 0.0f) xa = min(xa, r.cstep[a] + G.B - 1);
        x[a] = xa;
      }
  }
  int info = r.info;
  if (newbrick) {
    info = __ldg(binfo + dex_brick_of<D>(G, x));
    const int m2 = (info & 15) - 1;
    const int sh2 = (m2 < 0) ? G.logB : m2;
    if (!box && sh2 < r.sh) {
#pragma unroll
      for (int a = 0; a < D; ++a)
        if (a != s) x[a] = dex_fine_coord(__ldg(probe + a), -__ldg(omega + a), r.inv[a], r.off[a], c[a], size, th, a < s);
    }
  }
  dex_set_cell_nocap<D, BOX>(r, G, info, x);
  return true;
}
