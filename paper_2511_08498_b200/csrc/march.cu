// march.cu -- a5-a10: ray set-up, HDDA traversal, emissivity/opacity providers, segment integral,
// fused angular reduction to J, and the visit-list capture kernel.
//
// Mapping: LPR lanes share one probe and hold W/LPR wavelengths each, so one
// cell fetch of a ray is a single contiguous [cell][lambda][eta,chi] read split across its lanes;
// consecutive lane groups of a warp are consecutive probes (neighbouring voxels) tracing the same
// direction at the same time, so brick / level lookups and cell fetches of a warp hit the same lines.
// Each lane group loops over all quadrature directions and accumulates J in registers: the angular
// reduction needs no atomics and is deterministic.
#include "dex_internal.h"
#include "dex_voigt.cuh"

namespace {

// E(tau) = (1 - exp(-tau)) / tau with expm1-quality for small tau (1 - expf(-tau)
// loses the 1e-5 budget in the thin regime).  Returns e = exp(-tau) as well.
__device__ __forceinline__ float dex_E(float tau, float& e) {
  e = __expf(-tau);
  // Taylor series of E to degree 6: truncation < 1.6e-9 for tau < 0.25
  float p = -1.0f / 5040.0f;
  p = fmaf(p, tau, 1.0f / 720.0f);
  p = fmaf(p, tau, -1.0f / 120.0f);
  p = fmaf(p, tau, 1.0f / 24.0f);
  p = fmaf(p, tau, -1.0f / 6.0f);
  p = fmaf(p, tau, 0.5f);
  p = fmaf(-p, tau, 1.0f);
  const float q = __fdividef(1.0f - e, fmaxf(tau, 0.25f));
  return (tau < 0.25f) ? p : q;
}

// I_out = I_in e^{-tau} + eta h ds E(tau), accumulated front to back from the probe outward:
// I += T * eta h ds E(tau);  T *= e^{-tau}     (eq. 3 with constant eta, chi)
__device__ __forceinline__ void dex_accumulate(float eta, float chi, float hds, float& I, float& T) {
  const float tau = chi * hds;
  float e;
  const float E = dex_E(tau, e);
  I = fmaf(T, eta * hds * E, I);
  T *= e;
}

template <int LPT>
__device__ __forceinline__ void dex_load_rec(const float* __restrict__ rec, float (&eta)[LPT], float (&chi)[LPT]) {
  if (LPT == 1) {
    const float2 v = __ldg(reinterpret_cast<const float2*>(rec));
    eta[0] = v.x; chi[0] = v.y;
  } else {
#pragma unroll
    for (int i = 0; i < LPT / 2; ++i) {
      const float4 v = __ldg(reinterpret_cast<const float4*>(rec) + i);
      eta[2 * i] = v.x; chi[2 * i] = v.y; eta[2 * i + 1] = v.z; chi[2 * i + 1] = v.w;
    }
  }
}

template <int D, int VAR, int LPR, bool FUSE_J>
__global__ void __launch_bounds__(128)
dex_march_kernel(const DexGridDev G, const DexMipsDev M, const DexRaysDev R, float* __restrict__ out,
                 unsigned long long* __restrict__ seg_count) {
  constexpr int LPT = DEX_W / LPR;
  const int batch = blockIdx.y;
  const long long gid = ((long long)blockIdx.x * blockDim.x + threadIdx.x) / LPR;
  const int sub = threadIdx.x % LPR;
  const int lam_off = batch * DEX_W + sub * LPT;
  unsigned nseg = 0;
  if (gid < R.n_probes) {
    float probe[D];
#pragma unroll
    for (int a = 0; a < D; ++a) probe[a] = __ldg(R.probe_pos + gid * D + a);
    float J[LPT];
#pragma unroll
    for (int i = 0; i < LPT; ++i) J[i] = 0.0f;
    const size_t batch_base = ((size_t)batch * G.n_active) * M.cps;
    // per-thread wavelength constants of the anisotropic variants
    double lam[LPT];
    int al[DEX_NLINES];
    if (VAR == DEX_CAV) {
#pragma unroll
      for (int i = 0; i < LPT; ++i) lam[i] = (double)__ldg(M.lam + lam_off + i);
#pragma unroll
      for (int q = 0; q < DEX_NLINES; ++q) al[q] = M.active_lines[batch * DEX_NLINES + q];
    }
    for (int k = 0; k < R.n_dirs; ++k) {
      float om[D];
#pragma unroll
      for (int a = 0; a < D; ++a) om[a] = __ldg(R.dirs + k * D + a);
      float I[LPT], T[LPT];
#pragma unroll
      for (int i = 0; i < LPT; ++i) { I[i] = 0.0f; T[i] = 1.0f; }
      DexRay<D> ray;
      bool alive = dex_ray_init<D>(ray, G, M, batch, probe, om);
      while (alive) {
        DexSeg<D> seg;
        alive = dex_ray_step<D>(ray, G, M, batch, seg);
        if (seg.emit) {
          ++nseg;
          const float hds = G.h * seg.ds;
          const size_t cell = (size_t)seg.slot * M.cps + dex_cell_in_slot<D>(G, M, seg.m, seg.c);
          float eta[LPT], chi[LPT];
          if (VAR == DEX_ISO) {
            dex_load_rec<LPT>(M.store + (batch_base + cell) * DEX_REC + sub * LPT * 2, eta, chi);
          } else {
            // projected velocity of the cell's box-filtered bulk velocity, fp64 (DESIGN.md R-vel)
            const float4 v4 = __ldg(M.vel + cell);
            double vproj = __dmul_rn((double)v4.x, (double)om[0]);
            vproj = __dadd_rn(vproj, __dmul_rn((double)v4.y, (double)om[1]));
            if (D == 3) vproj = __dadd_rn(vproj, __dmul_rn((double)v4.z, (double)om[D - 1]));
            if (VAR == DEX_VELINTERP) {
              // linear interpolation on the cell's uniform velocity grid [-V, V]
              const int nvb = M.n_vbins;
              const double V = (double)v4.w;
              int i0 = 0;
              float w = 0.0f;
              if (V > 0.0) {
                double f = __dmul_rn(__ddiv_rn(__dadd_rn(vproj, V), __dmul_rn(2.0, V)), (double)(nvb - 1));
                f = fmin(fmax(f, 0.0), (double)(nvb - 1));
                i0 = min((int)floor(f), nvb - 2);
                w = (float)(f - (double)i0);
              }
              const float* r0 = M.vtab + ((batch_base + cell) * nvb + i0) * DEX_REC + sub * LPT * 2;
              float e1[LPT], c1[LPT];
              dex_load_rec<LPT>(r0, eta, chi);
              dex_load_rec<LPT>(r0 + DEX_REC, e1, c1);
#pragma unroll
              for (int i = 0; i < LPT; ++i) {
                eta[i] = fmaf(w, e1[i], (1.0f - w) * eta[i]);
                chi[i] = fmaf(w, c1[i], (1.0f - w) * chi[i]);
              }
            } else {
              // Core-and-Voigt / Classic: background + sum over the active lines (eqs. 10-11)
              dex_load_rec<LPT>(M.store + (batch_base + cell) * DEX_REC + sub * LPT * 2, eta, chi);
              double de[LPT], dc[LPT];
#pragma unroll
              for (int i = 0; i < LPT; ++i) { de[i] = (double)eta[i]; dc[i] = (double)chi[i]; }
#pragma unroll
              for (int q = 0; q < DEX_NLINES; ++q) {
                const int l = al[q];
                if (l < 0) continue;
                const float4 ln = __ldg(M.line + cell * M.n_lines + l);
                const double lam0 = (double)M.lambda0[l];
#pragma unroll
                for (int i = 0; i < LPT; ++i) {
                  double el, cl;
                  dex_line_terms(M.wei_c, M.wei_L, lam[i], lam0, (double)ln.x, (double)ln.y, (double)ln.z,
                                 (double)ln.w, vproj, M.c_light, el, cl);
                  de[i] += el;
                  dc[i] += cl;
                }
              }
#pragma unroll
              for (int i = 0; i < LPT; ++i) { eta[i] = (float)de[i]; chi[i] = (float)dc[i]; }
            }
          }
#pragma unroll
          for (int i = 0; i < LPT; ++i) dex_accumulate(eta[i], chi[i], hds, I[i], T[i]);
        }
      }
      if (R.i0 != nullptr) {
#pragma unroll
        for (int i = 0; i < LPT; ++i) I[i] = fmaf(T[i], __ldg(R.i0 + (size_t)k * M.n_lambda + lam_off + i), I[i]);
      }
      if (FUSE_J) {
        const float wk = __ldg(R.weights + k);
#pragma unroll
        for (int i = 0; i < LPT; ++i) J[i] = fmaf(wk, I[i], J[i]);
      } else {
        float* dst = out + ((size_t)gid * R.n_dirs + k) * M.n_lambda + lam_off;
#pragma unroll
        for (int i = 0; i < LPT; ++i) dst[i] = I[i];
      }
    }
    if (FUSE_J) {
      float* dst = out + (size_t)gid * M.n_lambda + lam_off;
#pragma unroll
      for (int i = 0; i < LPT; ++i) dst[i] = J[i];
    }
  }
  if (seg_count != nullptr) {
    unsigned v = (sub == 0) ? nseg : 0u;
    v = __reduce_add_sync(0xffffffffu, v);
    if ((threadIdx.x & 31) == 0 && v) atomicAdd(seg_count, (unsigned long long)v);
  }
}

// a10: traversal only, one thread per ray, for one batch's level table.
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
  float probe[D], om[D];
#pragma unroll
  for (int a = 0; a < D; ++a) { probe[a] = R.probe_pos[p * D + a]; om[a] = R.dirs[k * D + a]; }
  const long long begin = offsets[ray_id];
  const long long room = ((ray_id + 1 < n_rays) ? offsets[ray_id + 1] : capacity) - begin;
  long long n = 0;
  DexRay<D> ray;
  bool alive = dex_ray_init<D>(ray, G, M, batch, probe, om);
  while (alive) {
    DexSeg<D> seg;
    alive = dex_ray_step<D>(ray, G, M, batch, seg);
    if (seg.emit) {
      if (n < room) {
        unsigned long long rec = ((unsigned long long)(unsigned)seg.m << 56) |
                                 (unsigned long long)(unsigned)(seg.c[0] >> seg.m);
        rec |= (unsigned long long)(unsigned)(seg.c[1] >> seg.m) << 18;
        if (D == 3) rec |= (unsigned long long)(unsigned)(seg.c[D - 1] >> seg.m) << 36;
        records[begin + n] = rec;
        if (ds_out) ds_out[begin + n] = seg.ds;
      }
      ++n;
    }
  }
  counts[ray_id] = n;
  if (n > room) *overflow = 1;
}

// J(p, lambda) = sum_k w_k I(p, k, lambda) from a materialised I: one thread per (probe, lambda);
// consecutive threads read consecutive lambda (coalesced).
__global__ void dex_reduce_j_kernel(long long n_probes, int n_dirs, int n_lambda, const float* __restrict__ w,
                                    const float* __restrict__ I, float* __restrict__ J) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_probes * n_lambda) return;
  const long long p = i / n_lambda;
  const int j = (int)(i - p * n_lambda);
  float acc = 0.0f;
  for (int k = 0; k < n_dirs; ++k) acc = fmaf(__ldg(w + k), __ldg(I + (p * n_dirs + k) * n_lambda + j), acc);
  J[i] = acc;
}

template <int D, int VAR, int LPR>
dex_status launch_march_t(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays, float* d_out, bool fuse_j,
                          unsigned long long* d_seg, cudaStream_t st) {
  const int threads = 128;
  const long long probes_per_block = threads / LPR;
  const long long gx = (rays.n_probes + probes_per_block - 1) / probes_per_block;
  if (gx <= 0) return DEX_OK;
  if (gx > 2147483647LL || m->n_batch > 65535) {
    dex_set_error("march: problem too large for one launch");
    return DEX_ERR_UNSUPPORTED;
  }
  dim3 grid((unsigned)gx, (unsigned)m->n_batch, 1);
  if (fuse_j)
    dex_march_kernel<D, VAR, LPR, true><<<grid, threads, 0, st>>>(g->dev, m->dev, rays, d_out, d_seg);
  else
    dex_march_kernel<D, VAR, LPR, false><<<grid, threads, 0, st>>>(g->dev, m->dev, rays, d_out, d_seg);
  dex_count_launch();
  DEX_CUDA_CHECK(cudaGetLastError());
  return DEX_OK;
}

template <int D, int VAR>
dex_status launch_march_v(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays, float* d_out, bool fuse_j,
                          unsigned long long* d_seg, int lpr, cudaStream_t st) {
  switch (lpr) {
    case 8: return launch_march_t<D, VAR, 8>(g, m, rays, d_out, fuse_j, d_seg, st);
    case 4: return launch_march_t<D, VAR, 4>(g, m, rays, d_out, fuse_j, d_seg, st);
    case 2: return launch_march_t<D, VAR, 2>(g, m, rays, d_out, fuse_j, d_seg, st);
    case 1: return launch_march_t<D, VAR, 1>(g, m, rays, d_out, fuse_j, d_seg, st);
  }
  dex_set_error("lanes per ray must be 1, 2, 4 or 8");
  return DEX_ERR_INVALID_ARG;
}

template <int D>
dex_status launch_march_d(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays, float* d_out, bool fuse_j,
                          unsigned long long* d_seg, int lpr, cudaStream_t st) {
  switch (m->variant) {
    case DEX_ISO: return launch_march_v<D, DEX_ISO>(g, m, rays, d_out, fuse_j, d_seg, lpr, st);
    case DEX_VELINTERP: return launch_march_v<D, DEX_VELINTERP>(g, m, rays, d_out, fuse_j, d_seg, lpr, st);
    case DEX_CAV:
    case DEX_CLASSIC: return launch_march_v<D, DEX_CAV>(g, m, rays, d_out, fuse_j, d_seg, lpr, st);
  }
  dex_set_error("unknown variant");
  return DEX_ERR_INVALID_ARG;
}

}  // namespace

dex_status dex_launch_march(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays, float* d_out, bool fuse_j,
                            unsigned long long* d_seg, int lanes_per_ray, cudaStream_t st) {
  if (g->desc.ndim == 2) return launch_march_d<2>(g, m, rays, d_out, fuse_j, d_seg, lanes_per_ray, st);
  return launch_march_d<3>(g, m, rays, d_out, fuse_j, d_seg, lanes_per_ray, st);
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

dex_status dex_launch_reduce_j(const DexRaysDev& rays, int n_lambda, const float* d_I, float* d_J, cudaStream_t st) {
  const long long n = rays.n_probes * n_lambda;
  if (n <= 0) return DEX_OK;
  const int threads = 256;
  const long long gx = (n + threads - 1) / threads;
  dex_reduce_j_kernel<<<(unsigned)gx, threads, 0, st>>>(rays.n_probes, rays.n_dirs, n_lambda, rays.weights, d_I, d_J);
  dex_count_launch();
  DEX_CUDA_CHECK(cudaGetLastError());
  return DEX_OK;
}
