// grid_static.cu -- dex_brick_slots_static: step a1 (brick occupancy + compaction) for callers that
// are not allowed to allocate device memory.
//
// Who that is: code running where a cudaMalloc / cudaMallocAsync would either fail or stall everybody else -- a solver
// that was handed a fixed memory budget at start-up and whose arena is already carved up, a plug-in living inside a host
// application that owns the GPU's allocator (any allocation made behind its back breaks its accounting or synchronises
// the device under it), or a real-time loop that cannot take the driver's allocation lock between two frames.  The normal
// entry (dex_build_sparse_grid, grid_build.cu) draws its per-brick flag array, its counter and the handle's tables from the
// library's stream-ordered pool; this file does the same step with NO allocation at all:
//   - the outputs (slot table, slot -> brick list, active count) are the caller's device buffers;
//   - the one piece of scratch the step needs, the per-brick occupancy flags the scan reads, lives in the file-scope
//     device array g_static_flag below, DEX_STATIC_MAX_BRICKS ints = 4 MiB.  It is part of the library image: every GPU
//     that loads this module holds those 4 MiB until the process exits, whether or not the entry is ever called.
//
// Host code cannot use the array's name as a pointer: in host code `g_static_flag` names a host-side shadow object, and a
// kernel given that address would fault (or quietly scribble over host memory on a system where the GPU can reach it).  The
// device address is looked up once per device with cudaGetSymbolAddress, with that device current, on the entry's first
// call there (static_flag_ptr below), and handed to the kernels as an ordinary pointer argument.
//
// Every call on a device shares the one array.  Each call rewrites flags [0, n_bricks) before the scan reads them, so
// nothing has to be cleared between calls and a smaller grid after a larger one is fine (tests/test_zz_no_alloc.py does
// exactly that); the entries beyond n_bricks keep whatever the last larger call left there and are never read.  Two
// calls whose kernels can overlap on the GPU (different streams without an ordering event, or two host threads on two
// streams) race on the array and produce garbage: order them.
//
// The kernels are restatements of grid_build.cu's (same numbering: slots 0..A-1 in brick-index order); that file is not
// touched and shares nothing with this one.
#include <mutex>

#include "dex_internal.h"

// The scratch: per-brick occupancy flags of the call in flight.  Device code below could name it directly; the kernels
// take it as a pointer argument instead so that the host-side look-up is the one place that decides which memory is used.
static __device__ __align__(256) int g_static_flag[DEX_STATIC_MAX_BRICKS];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
int* g_flag_ptr[kMaxDevices] = {};   // device address of g_static_flag on device i, NULL until the first call there

// The device-side address of g_static_flag on the CURRENT device (one array instance per device that loads the module).
dex_status static_flag_ptr(int** out) {
  int dev = -1;
  DEX_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) { dex_set_error("device ordinal out of range for dex_brick_slots_static"); return DEX_ERR_UNSUPPORTED; }
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_flag_ptr[dev]) {
    int* p = nullptr;
    DEX_CUDA_CHECK(cudaGetSymbolAddress((void**)&p, g_static_flag));
    if (!p) { dex_set_error("cudaGetSymbolAddress returned NULL for the static scratch array"); return DEX_ERR_CUDA; }
    g_flag_ptr[dev] = p;
  }
  *out = g_flag_ptr[dev];
  return DEX_OK;
}

struct StaticGeom {
  int ndim, B, logB, n_bricks;
  int dims[3], nb[3];
};

// one warp per brick: flag = 1 iff any voxel of the brick is active (d_active == NULL: every brick)
__global__ void static_brick_flags_kernel(const StaticGeom G, const uint8_t* __restrict__ active, int* __restrict__ flag) {
  const int warp = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  const int lane = threadIdx.x & 31;
  if (warp >= G.n_bricks) return;
  int any = 1;
  if (active != nullptr) {
    const int bx = warp % G.nb[0];
    const int by = (warp / G.nb[0]) % G.nb[1];
    const int bz = warp / (G.nb[0] * G.nb[1]);       // 0 in 2D (nb[2] = 1)
    const int B = G.B;
    const int nvb = (G.ndim == 3) ? B * B * B : B * B;
    any = 0;
    for (int i = lane; i < nvb; i += 32) {
      const int x = i & (B - 1);
      const int y = (i >> G.logB) & (B - 1);
      const int z = (G.ndim == 3) ? (i >> (2 * G.logB)) : 0;
      const size_t v = ((size_t)(bz * B + z) * G.dims[1] + (by * B + y)) * G.dims[0] + (bx * B + x);
      any |= (int)active[v];
    }
    any = __any_sync(0xffffffffu, any != 0) ? 1 : 0;
  }
  if (lane == 0) flag[warp] = any;
}

// one block: exclusive scan of the flags -> slot per brick (-1 = empty), slot -> brick list, active count
__global__ void __launch_bounds__(1024)
static_scan_slots_kernel(const int* __restrict__ flag, int n, int* __restrict__ slot, int* __restrict__ active_bricks,
                         int* __restrict__ n_active) {
  __shared__ int part[1024];
  const int t = threadIdx.x;
  const int chunk = (n + 1023) / 1024;
  const int lo = min(n, t * chunk), hi = min(n, lo + chunk);
  int cnt = 0;
  for (int i = lo; i < hi; ++i) cnt += (flag[i] != 0);
  part[t] = cnt;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {
    const int v = (t >= off) ? part[t - off] : 0;
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

}  // namespace

extern "C" dex_status dex_brick_slots_static(const dex_grid_desc* desc, const uint8_t* d_active, int32_t* d_slot,
                                             int32_t* d_active_bricks, int32_t* d_n_active, void* stream) {
  if (!desc || !d_slot || !d_active_bricks || !d_n_active) {
    dex_set_error("NULL desc / d_slot / d_active_bricks / d_n_active");
    return DEX_ERR_INVALID_ARG;
  }
  if (desc->ndim != 2 && desc->ndim != 3) { dex_set_error("ndim must be 2 or 3"); return DEX_ERR_INVALID_ARG; }
  int logB = 0;
  while ((1 << logB) < desc->brick) ++logB;
  if (desc->brick < 2 || desc->brick > 32 || (1 << logB) != desc->brick) {
    dex_set_error("brick must be a power of two in 2..32");
    return DEX_ERR_SHAPE;
  }
  StaticGeom G;
  G.ndim = desc->ndim;
  G.B = desc->brick;
  G.logB = logB;
  long long nbr = 1;
  for (int a = 0; a < 3; ++a) {
    if (a < desc->ndim) {
      if (desc->dims[a] <= 0 || desc->dims[a] % desc->brick) {
        dex_set_error("every dimension must be a positive multiple of brick");
        return DEX_ERR_SHAPE;
      }
      if (desc->dims[a] >= (1 << 18)) { dex_set_error("dimension too large (< 2^18)"); return DEX_ERR_SHAPE; }
      G.dims[a] = desc->dims[a];
      G.nb[a] = desc->dims[a] / desc->brick;
    } else {
      G.dims[a] = 1;
      G.nb[a] = 1;
    }
    nbr *= G.nb[a];
  }
  if (nbr > (long long)DEX_STATIC_MAX_BRICKS) {
    dex_set_error("dex_brick_slots_static: " + std::to_string(nbr) + " bricks exceed the static scratch array of " +
                  std::to_string((long long)DEX_STATIC_MAX_BRICKS) +
                  " (DEX_STATIC_MAX_BRICKS); use dex_build_sparse_grid, which allocates, or a larger brick");
    return DEX_ERR_SHAPE;
  }
  G.n_bricks = (int)nbr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) {
    cudaGetLastError();
    dex_set_error("no CUDA device available (this library has no CPU fallback)");
    return DEX_ERR_CUDA;
  }
  int* d_flag = nullptr;
  const dex_status s = static_flag_ptr(&d_flag);       // first call on this device: looks the array's address up
  if (s != DEX_OK) return s;
  cudaStream_t st = (cudaStream_t)stream;
  const long long threads = nbr * 32;
  static_brick_flags_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(G, d_active, d_flag);
  static_scan_slots_kernel<<<1, 1024, 0, st>>>(d_flag, G.n_bricks, d_slot, d_active_bricks, d_n_active);
  dex_count_launch(2);
  DEX_CUDA_CHECK(cudaGetLastError());
  return DEX_OK;
}
