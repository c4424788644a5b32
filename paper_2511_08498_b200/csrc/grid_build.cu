// grid_build.cu -- a1: brick occupancy + compaction.
// A brick is populated iff any of its voxels is active; populated bricks get storage slots 0..A-1 in
// brick-index order (the offset lookup table of).
#include "dex_internal.h"

namespace {

// one warp per brick: OR-reduce the brick's voxels
template <int D>
__global__ void dex_brick_flags_kernel(const DexGridDev G, const uint8_t* __restrict__ active, int* __restrict__ flag) {
  const int warp = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  const int lane = threadIdx.x & 31;
  if (warp >= G.n_bricks) return;
  int bx = warp % G.nb[0];
  int by = (warp / G.nb[0]) % G.nb[1];
  int bz = (D == 3) ? warp / (G.nb[0] * G.nb[1]) : 0;
  const int B = G.B;
  const int nvb = (D == 3) ? B * B * B : B * B;
  int any = 0;
  for (int i = lane; i < nvb; i += 32) {
    const int x = i & (B - 1);
    const int y = (i >> G.logB) & (B - 1);
    const int z = (D == 3) ? (i >> (2 * G.logB)) : 0;
    const size_t v = ((size_t)(bz * B + z) * G.dims[1] + (by * B + y)) * G.dims[0] + (bx * B + x);
    any |= (int)active[v];
  }
  any = __any_sync(0xffffffffu, any != 0);
  if (lane == 0) flag[warp] = any;
}

__global__ void dex_fill_int_kernel(int* p, int n, int v) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

// single-block exclusive scan of the flags -> slot table, slot -> brick list, active count
__global__ void __launch_bounds__(1024)
dex_scan_slots_kernel(const int* __restrict__ flag, int n, int* __restrict__ slot, int* __restrict__ active_bricks,
                      int* __restrict__ n_active) {
  __shared__ int part[1024];
  const int t = threadIdx.x;
  const int chunk = (n + 1023) / 1024;
  const int lo = min(n, t * chunk), hi = min(n, lo + chunk);
  int cnt = 0;
  for (int i = lo; i < hi; ++i) cnt += (flag[i] != 0);
  part[t] = cnt;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {      // Hillis-Steele inclusive scan
    int v = (t >= off) ? part[t - off] : 0;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  int base = part[t] - cnt;
  for (int i = lo; i < hi; ++i) {
    if (flag[i] != 0) { slot[i] = base; active_bricks[base] = i; ++base; }
    else slot[i] = -1;
  }
  if (t == 1023) *n_active = part[1023];
}

// Empty-space distance: for an empty brick, the Chebyshev distance (in bricks, capped at DEX_EDIST_MAX) to the nearest
// populated brick; 0 for a populated one.  The (2d-1)^D box of bricks centred on an empty brick at distance d holds no
// populated brick, so a ray inside it can be taken to the box's face in ONE HDDA step (dex_set_cell_nocap): empty visits
// are never emitted, and the face a ray leaves through is the face of the brick it enters, so emitted lists are unchanged.
#define DEX_EDIST_MAX 8
template <int D>
__global__ void dex_empty_distance_kernel(const DexGridDev G, const int* __restrict__ flag, int* __restrict__ edist) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= G.n_bricks) return;
  if (flag[b] != 0) { edist[b] = 0; return; }
  const int bx = b % G.nb[0], by = (b / G.nb[0]) % G.nb[1], bz = (D == 3) ? b / (G.nb[0] * G.nb[1]) : 0;
  int d = DEX_EDIST_MAX;
  for (int r = 1; r < DEX_EDIST_MAX && d == DEX_EDIST_MAX; ++r) {       // shells of growing radius, stop at the first hit
    const int z0 = (D == 3) ? max(0, bz - r) : 0, z1 = (D == 3) ? min(G.nb[2] - 1, bz + r) : 0;
    for (int z = z0; z <= z1 && d == DEX_EDIST_MAX; ++z)
      for (int y = max(0, by - r); y <= min(G.nb[1] - 1, by + r) && d == DEX_EDIST_MAX; ++y) {
        const bool edge_zy = (D == 3 && (z == bz - r || z == bz + r)) || y == by - r || y == by + r;
        const int x0 = max(0, bx - r), x1 = min(G.nb[0] - 1, bx + r);
        if (edge_zy) {
          for (int x = x0; x <= x1; ++x)
            if (flag[(z * G.nb[1] + y) * G.nb[0] + x] != 0) { d = r; break; }
        } else {      // interior row of the shell: only its two end points belong to it
          if (bx - r >= 0 && flag[(z * G.nb[1] + y) * G.nb[0] + bx - r] != 0) d = r;
          if (bx + r < G.nb[0] && flag[(z * G.nb[1] + y) * G.nb[0] + bx + r] != 0) d = r;
        }
      }
  }
  edist[b] = d;
}

}  // namespace

dex_status dex_launch_grid_build(dex_grid* g, const uint8_t* d_active, cudaStream_t st) {
  const int nb = (int)g->n_bricks;
  int* d_flag = nullptr;
  int* d_count = nullptr;
  DEX_CUDA_CHECK(dex_alloc((void**)&d_flag, sizeof(int) * (size_t)nb, st));
  DEX_CUDA_CHECK(dex_alloc((void**)&d_count, sizeof(int), st));
  if (d_active == nullptr) {
    dex_fill_int_kernel<<<(nb + 255) / 256, 256, 0, st>>>(d_flag, nb, 1);
  } else {
    const long long threads = (long long)nb * 32;
    const unsigned blocks = (unsigned)((threads + 255) / 256);
    if (g->desc.ndim == 2) dex_brick_flags_kernel<2><<<blocks, 256, 0, st>>>(g->dev, d_active, d_flag);
    else dex_brick_flags_kernel<3><<<blocks, 256, 0, st>>>(g->dev, d_active, d_flag);
  }
  dex_count_launch();
  dex_scan_slots_kernel<<<1, 1024, 0, st>>>(d_flag, nb, g->d_slot, g->d_active_bricks, d_count);
  if (g->desc.ndim == 2) dex_empty_distance_kernel<2><<<(nb + 127) / 128, 128, 0, st>>>(g->dev, d_flag, g->d_edist);
  else dex_fill_int_kernel<<<(nb + 255) / 256, 256, 0, st>>>(g->d_edist, nb, 1);   // 3D rays take empty bricks one at a time (march.cu DEX_BOX)
  dex_count_launch(2);
  int h_count = 0;
  cudaError_t e = cudaMemcpyAsync(&h_count, d_count, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  dex_free(d_flag, st);
  dex_free(d_count, st);
  DEX_CUDA_CHECK(e);
  DEX_CUDA_CHECK(cudaGetLastError());
  g->n_active = h_count;
  g->dev.n_active = h_count;
  return DEX_OK;
}
