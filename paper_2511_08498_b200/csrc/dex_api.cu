// dex_api.cu -- the extern "C" boundary declared in include/dex.h: argument validation, handle
// ownership, and dispatch to the kernels.  No compute happens on the host.
#include <math.h>
#include <string.h>

#include <atomic>
#include <mutex>
#include <new>
#include <vector>

#include "dex_internal.h"
#include "dex_voigt.cuh"

namespace {
thread_local std::string g_last_error;
std::atomic<long long> g_launches{0};
std::atomic<int> g_lanes_per_ray{0};  // 0 = automatic, see lanes_for()
std::atomic<int> g_timing{0};
std::atomic<int> g_tile_probes{1};
std::atomic<int> g_voigt_fp32{1};
std::atomic<int> g_dir_split{-1};
std::atomic<int> g_memo{-1};
std::atomic<int> g_memo_budget_mb{0};     // 0 = automatic (memo_group in march.cu)
std::atomic<int> g_memo_fail_allocs{0};   // fault injection: this many record allocations of the memoised march fail
std::mutex g_timing_mu;
struct EvPair { cudaEvent_t a, b; };
std::vector<EvPair> g_events;
unsigned long long* g_d_line_segs = nullptr;   // device counter of (segment, active line) pairs, timing mode only

// Lanes that share one ray.  One thread per ray (all W wavelengths in registers) is the fastest mapping whenever the
// probes fill the machine (profiles/r01_history.md: 1.6-2.2x over 8 lanes on C2).  0 = automatic: dex_launch_march
// (march.cu) decides from the probe count -- small problems take 8 lanes per ray, or 2 when they are also spread over
// the machine direction by direction (C1: 0.415 -> 0.236 ms per step).
int lanes_for(long long) { return g_lanes_per_ray.load(); }

int ilog2_exact(int v) {
  if (v <= 0 || (v & (v - 1))) return -1;
  int l = 0;
  while ((1 << l) < v) ++l;
  return l;
}

bool have_device() {
  int n = 0;
  cudaError_t e = cudaGetDeviceCount(&n);
  if (e != cudaSuccess || n <= 0) {
    cudaGetLastError();
    dex_set_error("no CUDA device available (this library has no CPU fallback)");
    return false;
  }
  return true;
}

template <typename T>
dex_status dmalloc(T** p, size_t count, cudaStream_t st) {
  *p = nullptr;
  if (count == 0) count = 1;
  DEX_CUDA_CHECK(dex_alloc((void**)p, sizeof(T) * count, st));
  return DEX_OK;
}

void free_mips_memory(dex_mips* m) {
  void* ptrs[] = {m->d_store, m->d_mrec, m->aux_borrowed ? nullptr : (void*)m->d_aux, m->d_vtab, m->d_lam, m->d_active_lines,
                  m->d_levels, m->d_packed, m->d_fail, m->d_binfo, m->aux_borrowed ? nullptr : (void*)m->d_vftab};
  for (void* q : ptrs) dex_free(q, m->stream);
}

dex_status check_rays(const dex_grid* grid, const dex_mips* mips, const dex_rays* rays, DexRaysDev* out) {
  if (!grid || !mips || !rays) { dex_set_error("NULL grid / mips / rays"); return DEX_ERR_INVALID_ARG; }
  if (mips->grid != grid) { dex_set_error("mips were built for a different grid"); return DEX_ERR_INVALID_ARG; }
  if (rays->n_probes < 0 || rays->n_dirs < 0) { dex_set_error("negative ray counts"); return DEX_ERR_SHAPE; }
  if (rays->n_probes > 0 && rays->n_dirs > 0 && (!rays->d_probe_pos || !rays->d_dirs)) {
    dex_set_error("d_probe_pos / d_dirs is NULL");
    return DEX_ERR_INVALID_ARG;
  }
  out->n_probes = rays->n_probes;
  out->probe_pos = rays->d_probe_pos;
  out->n_dirs = rays->n_dirs;
  out->dirs = rays->d_dirs;
  out->weights = rays->d_weights;
  out->i0 = rays->d_i0;
  out->sin_incl = rays->d_sin_incl;
  out->t_begin = rays->t_begin;
  out->t_end = rays->t_end;
  out->accumulate = rays->accumulate;
  out->k_per_block = 0;
  if (rays->t_end > 0.0f && !(rays->t_begin >= 0.0f && rays->t_begin < rays->t_end)) {
    dex_set_error("radiance interval needs 0 <= t_begin < t_end");
    return DEX_ERR_INVALID_ARG;
  }
  if (rays->d_sin_incl && grid->dev.ndim != 2) { dex_set_error("d_sin_incl (2.5D rays) needs a 2D grid"); return DEX_ERR_INVALID_ARG; }
  return DEX_OK;
}

struct MarchTimer {
  cudaStream_t st;
  bool on;
  EvPair ev{};
  explicit MarchTimer(cudaStream_t s) : st(s), on(g_timing.load() != 0) {
    if (on) {
      cudaEventCreate(&ev.a);
      cudaEventCreate(&ev.b);
      cudaEventRecord(ev.a, st);
    }
  }
  ~MarchTimer() {
    if (on) {
      cudaEventRecord(ev.b, st);
      std::lock_guard<std::mutex> lk(g_timing_mu);
      g_events.push_back(ev);
    }
  }
};
}  // namespace

namespace {
// device copies of host inputs, released when the call returns
struct Uploads {
  cudaStream_t st;
  std::vector<void*> ptrs;
  int64_t bytes = 0;
  dex_status status = DEX_OK;
  explicit Uploads(cudaStream_t s) : st(s) {}
  ~Uploads() { for (void* p : ptrs) dex_free(p, st); }
  template <typename T>
  const T* put(const T* h, size_t count) {
    if (!h || status != DEX_OK) return nullptr;
    void* d = nullptr;
    const size_t nbytes = sizeof(T) * (count ? count : 1);
    if (dex_alloc(&d, nbytes, st) != cudaSuccess) {
      cudaGetLastError();
      dex_set_error("device allocation failed while uploading host inputs");
      status = DEX_ERR_OOM;
      return nullptr;
    }
    ptrs.push_back(d);
    if (count && cudaMemcpyAsync(d, h, sizeof(T) * count, cudaMemcpyHostToDevice, st) != cudaSuccess) {
      dex_set_error(cudaGetErrorString(cudaGetLastError()));
      status = DEX_ERR_CUDA;
      return nullptr;
    }
    bytes += (int64_t)(sizeof(T) * count);
    return (const T*)d;
  }
  template <typename T>
  T* alloc(size_t count) {
    if (status != DEX_OK) return nullptr;
    void* d = nullptr;
    if (dex_alloc(&d, sizeof(T) * (count ? count : 1), st) != cudaSuccess) {
      cudaGetLastError();
      dex_set_error("device allocation failed");
      status = DEX_ERR_OOM;
      return nullptr;
    }
    ptrs.push_back(d);
    return (T*)d;
  }
};
}  // namespace

const float* dex_voigt_fast_table_host() {
  static std::vector<float> tab;
  static std::once_flag once;
  std::call_once(once, [] {
    tab.resize((size_t)DEX_VF_NODES * 5);
    dex_voigt_fast_table(tab.data(), tab.data() + (size_t)DEX_VF_NODES * 4);
  });
  return tab.data();
}

// The library's own stream-ordered pool, one per device, created at first use: nothing is returned to the driver
// until dex_trim(), so a rebuild per iteration pays no cudaMalloc / cudaFree.  A PRIVATE pool: the device's default
// pool (and with it every other cudaMallocAsync user of the process) keeps its own release threshold and statistics.
namespace {
std::mutex g_pool_mu;
cudaMemPool_t g_pool[64] = {nullptr};
cudaMemPool_t pool_of_current_device() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return nullptr; }
  std::lock_guard<std::mutex> lk(g_pool_mu);
  if (!g_pool[dev]) {
    cudaMemPoolProps props;
    memset(&props, 0, sizeof(props));
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t pool = nullptr;
    if (cudaMemPoolCreate(&pool, &props) == cudaSuccess) {
      unsigned long long keep = ~0ULL;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
      g_pool[dev] = pool;
    } else {
      cudaGetLastError();
    }
  }
  return g_pool[dev];
}
}  // namespace

cudaError_t dex_alloc(void** p, size_t bytes, cudaStream_t st) {
  cudaMemPool_t pool = pool_of_current_device();
  if (!pool) return cudaMallocAsync(p, bytes, st);     // pool creation failed: the default pool, untouched
  return cudaMallocFromPoolAsync(p, bytes, pool, st);
}
size_t dex_pool_idle_bytes() {
  cudaMemPool_t pool = pool_of_current_device();
  if (!pool) return 0;
  unsigned long long reserved = 0, used = 0;
  if (cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReservedMemCurrent, &reserved) != cudaSuccess ||
      cudaMemPoolGetAttribute(pool, cudaMemPoolAttrUsedMemCurrent, &used) != cudaSuccess) {
    cudaGetLastError();
    return 0;
  }
  return reserved > used ? (size_t)(reserved - used) : 0;
}
void dex_free(void* p, cudaStream_t st) {
  if (p) cudaFreeAsync(p, st);
}

void dex_set_error(const std::string& msg) { g_last_error = msg; }
void dex_count_launch(int n) { g_launches.fetch_add(n); }
int dex_tuning_voigt_fp32() { return g_voigt_fp32.load(); }
int dex_tuning_dir_split() { return g_dir_split.load(); }
int dex_tuning_memo() { return g_memo.load(); }
int dex_tuning_memo_budget_mb() { return g_memo_budget_mb.load(); }
bool dex_tuning_memo_fail_alloc() {
  int n = g_memo_fail_allocs.load();
  while (n > 0 && !g_memo_fail_allocs.compare_exchange_weak(n, n - 1)) {}
  return n > 0;
}
unsigned long long* dex_line_segment_counter() { return g_timing.load() ? g_d_line_segs : nullptr; }

extern "C" {

const char* dex_last_error(void) { return g_last_error.c_str(); }
const char* dex_version(void) { return "dex-b200 0.1 (sm_100a)"; }
int64_t dex_launch_count(void) { return (int64_t)g_launches.load(); }

dex_status dex_pool_high_water(int64_t* bytes_in_use_high, int reset) {
  if (!have_device()) return DEX_ERR_CUDA;
  cudaMemPool_t pool = pool_of_current_device();
  if (!pool) { dex_set_error("the library's memory pool could not be created"); return DEX_ERR_CUDA; }
  DEX_CUDA_CHECK(cudaDeviceSynchronize());
  unsigned long long v = 0;
  DEX_CUDA_CHECK(cudaMemPoolGetAttribute(pool, cudaMemPoolAttrUsedMemHigh, &v));
  if (bytes_in_use_high) *bytes_in_use_high = (int64_t)v;
  if (reset) {
    v = 0;
    DEX_CUDA_CHECK(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrUsedMemHigh, &v));
  }
  return DEX_OK;
}

dex_status dex_trim(int64_t* bytes_reserved_after) {
  if (!have_device()) return DEX_ERR_CUDA;
  cudaMemPool_t pool = pool_of_current_device();
  if (!pool) { dex_set_error("the library's memory pool could not be created"); return DEX_ERR_CUDA; }
  DEX_CUDA_CHECK(cudaDeviceSynchronize());
  DEX_CUDA_CHECK(cudaMemPoolTrimTo(pool, 0));
  unsigned long long v = 0;
  DEX_CUDA_CHECK(cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReservedMemCurrent, &v));
  if (bytes_reserved_after) *bytes_reserved_after = (int64_t)v;
  return DEX_OK;
}

dex_status dex_set_lanes_per_ray(int lanes) {
  if (lanes != 0 && lanes != 1 && lanes != 2 && lanes != 4 && lanes != 8) {
    dex_set_error("lanes per ray must be 0 (automatic), 1, 2, 4 or 8");
    return DEX_ERR_INVALID_ARG;
  }
  g_lanes_per_ray.store(lanes);
  return DEX_OK;
}

dex_status dex_get_lanes_per_ray(int64_t n_probes, int n_dirs, int n_lambda, int* lanes) {
  if (!lanes) { dex_set_error("NULL lanes"); return DEX_ERR_INVALID_ARG; }
  *lanes = dex_auto_lanes(lanes_for((long long)n_probes), (long long)n_probes,
                          dex_auto_dir_split((long long)n_probes, n_dirs, n_lambda < 1 ? 1 : n_lambda));
  return DEX_OK;
}

dex_status dex_last_march_mapping(int* lanes_per_ray, int* dirs_per_block, int* memo_batches_per_group) {
  dex_last_mapping(lanes_per_ray, dirs_per_block, memo_batches_per_group);
  return DEX_OK;
}

dex_status dex_set_tuning(const char* name, int value) {
  if (!name) { dex_set_error("NULL tuning name"); return DEX_ERR_INVALID_ARG; }
  if (!strcmp(name, "lanes_per_ray")) return dex_set_lanes_per_ray(value);
  if (!strcmp(name, "tile_probes")) { g_tile_probes.store(value ? 1 : 0); return DEX_OK; }
  if (!strcmp(name, "voigt_fp32")) { g_voigt_fp32.store(value ? 1 : 0); return DEX_OK; }
  if (!strcmp(name, "dir_split")) { g_dir_split.store(value < 0 ? -1 : value); return DEX_OK; }
  if (!strcmp(name, "memo")) { g_memo.store(value < 0 ? -1 : (value ? 1 : 0)); return DEX_OK; }
  if (!strcmp(name, "memo_budget_mb")) { g_memo_budget_mb.store(value < 0 ? 0 : value); return DEX_OK; }
  if (!strcmp(name, "memo_fail_allocs")) { g_memo_fail_allocs.store(value < 0 ? 0 : value); return DEX_OK; }
  dex_set_error("unknown tuning knob");
  return DEX_ERR_INVALID_ARG;
}

void dex_march_timing_enable(int on) {
  if (on) {
    std::lock_guard<std::mutex> lk(g_timing_mu);
    if (!g_d_line_segs && cudaMalloc((void**)&g_d_line_segs, sizeof(unsigned long long)) == cudaSuccess)
      cudaMemset(g_d_line_segs, 0, sizeof(unsigned long long));
    else
      cudaGetLastError();
  }
  g_timing.store(on ? 1 : 0);
}

dex_status dex_march_work_read(int64_t* line_segments, int reset) {
  std::lock_guard<std::mutex> lk(g_timing_mu);
  unsigned long long v = 0;
  if (g_d_line_segs) {
    DEX_CUDA_CHECK(cudaDeviceSynchronize());
    DEX_CUDA_CHECK(cudaMemcpy(&v, g_d_line_segs, sizeof(v), cudaMemcpyDeviceToHost));
    if (reset) DEX_CUDA_CHECK(cudaMemset(g_d_line_segs, 0, sizeof(v)));
  }
  if (line_segments) *line_segments = (int64_t)v;
  return DEX_OK;
}

dex_status dex_march_timing_read(double* ms_total, int64_t* n_launches, int reset) {
  std::lock_guard<std::mutex> lk(g_timing_mu);
  double total = 0.0;
  for (auto& ev : g_events) {
    DEX_CUDA_CHECK(cudaEventSynchronize(ev.b));
    float ms = 0.f;
    DEX_CUDA_CHECK(cudaEventElapsedTime(&ms, ev.a, ev.b));
    total += (double)ms;
  }
  if (ms_total) *ms_total = total;
  if (n_launches) *n_launches = (int64_t)g_events.size();
  if (reset) {
    for (auto& ev : g_events) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
    g_events.clear();
  }
  return DEX_OK;
}

// ------------------------------------------------------------------------------------------- grid
dex_status dex_build_sparse_grid(const dex_grid_desc* desc, const uint8_t* d_active, void* stream, dex_grid** out) {
  if (!desc || !out) { dex_set_error("NULL desc / out"); return DEX_ERR_INVALID_ARG; }
  *out = nullptr;
  if (desc->ndim != 2 && desc->ndim != 3) { dex_set_error("ndim must be 2 or 3"); return DEX_ERR_INVALID_ARG; }
  const int logB = ilog2_exact(desc->brick);
  if (logB < 1 || desc->brick > 32) { dex_set_error("brick must be a power of two in 2..32"); return DEX_ERR_SHAPE; }
  if (!(desc->voxel_size > 0.0f)) { dex_set_error("voxel_size must be > 0"); return DEX_ERR_INVALID_ARG; }
  int64_t nvox = 1, nbr = 1;
  for (int a = 0; a < desc->ndim; ++a) {
    if (desc->dims[a] <= 0 || desc->dims[a] % desc->brick) {
      dex_set_error("every dimension must be a positive multiple of brick");
      return DEX_ERR_SHAPE;
    }
    if (desc->dims[a] >= (1 << 18)) { dex_set_error("dimension too large (< 2^18)"); return DEX_ERR_SHAPE; }
    nvox *= desc->dims[a];
    nbr *= desc->dims[a] / desc->brick;
  }
  if (nbr > 2147483647LL / 64) { dex_set_error("too many bricks"); return DEX_ERR_SHAPE; }
  if (!have_device()) return DEX_ERR_CUDA;
  dex_grid* g = new (std::nothrow) dex_grid();
  if (!g) { dex_set_error("host allocation failed"); return DEX_ERR_OOM; }
  g->desc = *desc;
  if (desc->ndim == 2) g->desc.dims[2] = 1;
  g->n_bricks = nbr;
  g->nvox = nvox;
  DexGridDev& d = g->dev;
  d.ndim = desc->ndim;
  for (int a = 0; a < 3; ++a) {
    d.dims[a] = (a < desc->ndim) ? desc->dims[a] : 1;
    d.nb[a] = (a < desc->ndim) ? desc->dims[a] / desc->brick : 1;
  }
  d.B = desc->brick;
  d.logB = logB;
  d.h = desc->voxel_size;
  d.n_bricks = (int)nbr;
  d.n_active = 0;
  g->stream = (cudaStream_t)stream;
  dex_status s = dmalloc(&g->d_slot, (size_t)nbr, g->stream);
  if (s == DEX_OK) s = dmalloc(&g->d_active_bricks, (size_t)nbr, g->stream);
  if (s == DEX_OK) s = dmalloc(&g->d_edist, (size_t)nbr, g->stream);
  if (s == DEX_OK) { d.slot = g->d_slot; s = dex_launch_grid_build(g, d_active, (cudaStream_t)stream); }
  if (s != DEX_OK) { dex_destroy_grid(g); return s; }
  *out = g;
  return DEX_OK;
}

dex_status dex_grid_info(const dex_grid* grid, int64_t* n_bricks, int64_t* n_active) {
  if (!grid) { dex_set_error("NULL grid"); return DEX_ERR_INVALID_ARG; }
  if (n_bricks) *n_bricks = grid->n_bricks;
  if (n_active) *n_active = grid->n_active;
  return DEX_OK;
}

dex_status dex_grid_get_slots(const dex_grid* grid, int32_t* h_slot) {
  if (!grid || !h_slot) { dex_set_error("NULL grid / h_slot"); return DEX_ERR_INVALID_ARG; }
  DEX_CUDA_CHECK(cudaDeviceSynchronize());
  DEX_CUDA_CHECK(cudaMemcpy(h_slot, grid->d_slot, sizeof(int) * (size_t)grid->n_bricks, cudaMemcpyDeviceToHost));
  return DEX_OK;
}

void dex_destroy_grid(dex_grid* grid) {
  if (!grid) return;
  dex_free(grid->d_slot, grid->stream);
  dex_free(grid->d_active_bricks, grid->stream);
  dex_free(grid->d_edist, grid->stream);
  delete grid;
}

// ------------------------------------------------------------------------------------------- mips
}  // extern "C"

// dex_build_vlm_mips with the wavelength-independent chains (velocity, line parameters: "shared by all
// batches") and the fp32 Voigt tables optionally BORROWED from an earlier build of the same atmosphere: the rebuild
// pipeline builds them with its first stage only.
static dex_status build_vlm_mips_impl(const dex_grid* grid, const dex_mips_desc* desc, void* stream, float4* donor_aux,
                                      float* donor_vftab, dex_mips** out) {
  if (!grid || !desc || !out) { dex_set_error("NULL grid / desc / out"); return DEX_ERR_INVALID_ARG; }
  *out = nullptr;
  const int v = (int)desc->variant;
  if (v < DEX_ISO || v > DEX_CLASSIC) { dex_set_error("unknown variant"); return DEX_ERR_INVALID_ARG; }
  if (desc->metric != DEX_METRIC_IOD_LOG && desc->metric != DEX_METRIC_RELVAR) {
    dex_set_error("unknown metric");
    return DEX_ERR_INVALID_ARG;
  }
  if (desc->lambda_batch != DEX_W) { dex_set_error("lambda_batch must be 8 in this build"); return DEX_ERR_UNSUPPORTED; }
  if (desc->n_lambda <= 0 || desc->n_lambda % desc->lambda_batch) {
    dex_set_error("n_lambda must be a positive multiple of lambda_batch");
    return DEX_ERR_SHAPE;
  }
  if (desc->lambda_stride != 0 && desc->lambda_stride < desc->n_lambda) {
    dex_set_error("lambda_stride must be 0 (dense) or >= n_lambda");
    return DEX_ERR_SHAPE;
  }
  int max_level = desc->max_level;
  if (max_level < 0 || max_level > grid->dev.logB || max_level >= DEX_MAXLEV) {
    dex_set_error("max_level must be in 0..log2(brick)");
    return DEX_ERR_SHAPE;
  }
  if (v == DEX_CLASSIC) max_level = 0;   // brute force at full resolution
  const int n_batch = desc->n_lambda / desc->lambda_batch;
  if (v == DEX_ISO) {
    if (!desc->d_eta || !desc->d_chi) { dex_set_error("ISO needs d_eta and d_chi"); return DEX_ERR_INVALID_ARG; }
  } else {
    if (!desc->d_eta_bg || !desc->d_chi_bg || !desc->d_vel || !desc->d_lambda || !desc->h_active_lines) {
      dex_set_error("anisotropic variants need d_eta_bg, d_chi_bg, d_vel, d_lambda, h_active_lines");
      return DEX_ERR_INVALID_ARG;
    }
    if (desc->n_lines < 0 || desc->n_lines > DEX_MAX_LINES) { dex_set_error("n_lines must be 0..4"); return DEX_ERR_SHAPE; }
    if (desc->n_lines > 0 && (!desc->h_lambda0 || !desc->d_eta_star0 || !desc->d_chi_star0 || !desc->d_a0 ||
                              !desc->d_inv_dlamD)) {
      dex_set_error("line arrays are NULL");
      return DEX_ERR_INVALID_ARG;
    }
    for (int i = 0; i < n_batch * DEX_MAX_LINES; ++i) {
      const int l = desc->h_active_lines[i];
      if (l < -1 || l >= desc->n_lines) { dex_set_error("active line id out of range"); return DEX_ERR_SHAPE; }
    }
    if (!(desc->c_light > 0.0f)) { dex_set_error("c_light must be > 0"); return DEX_ERR_INVALID_ARG; }
    if (v == DEX_VELINTERP && (desc->n_vbins < 2 || desc->n_vbins > 32)) {
      dex_set_error("n_vbins must be in 2..32");
      return DEX_ERR_UNSUPPORTED;
    }
  }
  if (!have_device()) return DEX_ERR_CUDA;
  dex_mips* m = new (std::nothrow) dex_mips();
  if (!m) { dex_set_error("host allocation failed"); return DEX_ERR_OOM; }
  m->grid = grid;
  m->variant = v;
  m->n_lambda = desc->n_lambda;
  m->n_batch = n_batch;
  m->max_level = max_level;
  m->metric = (int)desc->metric;
  m->thr_eta = desc->thr_eta;
  m->thr_chi = desc->thr_chi;
  m->tau_gate = desc->tau_gate;
  DexMipsDev& d = m->dev;
  memset(&d, 0, sizeof(d));
  d.variant = v;
  d.n_lambda = desc->n_lambda;
  d.n_batch = n_batch;
  d.max_level = max_level;
  d.in_stride = desc->lambda_stride ? desc->lambda_stride : desc->n_lambda;
  d.io_stride = desc->n_lambda;
  d.io_base = 0;
  int bits = 1;
  while ((1 << bits) < max_level + 2) ++bits;      // ceil(log2(max_level + 2))
  d.bits = bits;
  d.per_word = 64 / bits;
  d.words_per_batch = (int)((grid->n_bricks + d.per_word - 1) / d.per_word);
  int cps = 0;
  for (int lv = 0; lv <= max_level; ++lv) {
    d.lvloff[lv] = cps;
    const int n = grid->dev.B >> lv;
    cps += (grid->dev.ndim == 3) ? n * n * n : n * n;
  }
  d.cps = cps;
  d.n_lines = (v == DEX_ISO) ? 0 : desc->n_lines;
  d.n_vbins = (v == DEX_VELINTERP) ? desc->n_vbins : 0;
  d.c_light = (double)desc->c_light;
  for (int l = 0; l < d.n_lines; ++l) d.lambda0[l] = desc->h_lambda0[l];
  dex_weideman_coefficients(d.wei_c, &d.wei_L);
  const size_t A = (size_t)grid->n_active;
  if ((long long)A * cps >= (1LL << 27)) { dex_set_error("too many pyramid cells per batch (brick word holds 27 bits)"); delete m; return DEX_ERR_SHAPE; }
  cudaStream_t st = (cudaStream_t)stream;
  m->stream = st;
  dex_status s = DEX_OK;
  m->store_floats = (size_t)n_batch * A * cps * DEX_REC;
  s = dmalloc(&m->d_store, m->store_floats, st);
  if (s == DEX_OK && v == DEX_ISO) s = dmalloc(&m->d_mrec, m->store_floats, st);
  if (s == DEX_OK) s = dmalloc(&m->d_levels, (size_t)n_batch * grid->n_bricks, st);
  if (s == DEX_OK) s = dmalloc(&m->d_packed, (size_t)n_batch * d.words_per_batch, st);
  if (s == DEX_OK) s = dmalloc(&m->d_binfo, (size_t)n_batch * grid->n_bricks, st);
  if (s == DEX_OK) s = dmalloc(&m->d_fail, (size_t)n_batch * A * (max_level + 1), st);
  if (s == DEX_OK && v != DEX_ISO) {
    m->aux_borrowed = donor_aux != nullptr && donor_vftab != nullptr;
    if (m->aux_borrowed) { m->d_aux = donor_aux; m->d_vftab = donor_vftab; }
    else s = dmalloc(&m->d_aux, A * cps * (size_t)(d.n_lines + 1), st);
    if (s == DEX_OK) s = dmalloc(&m->d_lam, (size_t)desc->n_lambda, st);
    if (s == DEX_OK) s = dmalloc(&m->d_active_lines, (size_t)n_batch * DEX_MAX_LINES, st);
    if (s == DEX_OK && !m->aux_borrowed) s = dmalloc(&m->d_vftab, (size_t)DEX_VF_NODES * 5, st);
    if (s == DEX_OK && v == DEX_VELINTERP) {
      m->vtab_floats = m->store_floats * (size_t)d.n_vbins;
      s = dmalloc(&m->d_vtab, m->vtab_floats, st);
    }
    if (s == DEX_OK) {
      cudaError_t e = cudaMemcpyAsync(m->d_lam, desc->d_lambda, sizeof(float) * desc->n_lambda,
                                      cudaMemcpyDeviceToDevice, st);
      if (e == cudaSuccess)
        e = cudaMemcpyAsync(m->d_active_lines, desc->h_active_lines, (size_t)n_batch * DEX_MAX_LINES,
                            cudaMemcpyHostToDevice, st);
      if (e == cudaSuccess && !m->aux_borrowed)
        e = cudaMemcpyAsync(m->d_vftab, dex_voigt_fast_table_host(), sizeof(float) * DEX_VF_NODES * 5,
                            cudaMemcpyHostToDevice, st);
      if (e != cudaSuccess) { dex_set_error(cudaGetErrorString(e)); s = DEX_ERR_CUDA; }
    }
  }
  if (s == DEX_OK) {
    d.vf_wing = (const float4*)m->d_vftab;
    d.vf_core = m->d_vftab ? m->d_vftab + (size_t)DEX_VF_NODES * 4 : nullptr;
    d.packed = m->d_packed;
    d.binfo = m->d_binfo;
    d.store = m->d_store;
    d.mrec = m->d_mrec;
    d.mplane = (grid->dev.ndim == 3) ? (size_t)DEX_W : m->store_floats / 2;   // 3D: interleaved records (dex_device.cuh)
    d.aux = m->d_aux;
    if (v == DEX_VELINTERP) { d.aux_vs = 1; d.aux_lo = A * cps; d.aux_ls = d.n_lines; }      // dense velocities, lines behind
    else { d.aux_vs = d.n_lines + 1; d.aux_lo = 1; d.aux_ls = d.n_lines + 1; }             // one record per cell
    d.vtab = m->d_vtab;
    d.lam = m->d_lam;
    d.active_lines = m->d_active_lines;
    s = dex_launch_mips_build(m, desc, st);
  }
  if (s != DEX_OK) { free_mips_memory(m); delete m; return s; }
  *out = m;
  return DEX_OK;
}

extern "C" {

dex_status dex_build_vlm_mips(const dex_grid* grid, const dex_mips_desc* desc, void* stream, dex_mips** out) {
  return build_vlm_mips_impl(grid, desc, stream, nullptr, nullptr, out);
}

dex_status dex_mips_get_levels(const dex_mips* mips, int8_t* h_level) {
  if (!mips || !h_level) { dex_set_error("NULL mips / h_level"); return DEX_ERR_INVALID_ARG; }
  DEX_CUDA_CHECK(cudaDeviceSynchronize());
  DEX_CUDA_CHECK(cudaMemcpy(h_level, mips->d_levels, (size_t)mips->n_batch * mips->grid->n_bricks, cudaMemcpyDeviceToHost));
  return DEX_OK;
}

dex_status dex_mips_set_levels(dex_mips* mips, const int8_t* h_level) {
  if (!mips || !h_level) { dex_set_error("NULL mips / h_level"); return DEX_ERR_INVALID_ARG; }
  const size_t n = (size_t)mips->n_batch * mips->grid->n_bricks;
  std::vector<int32_t> slots((size_t)mips->grid->n_bricks);
  dex_status s = dex_grid_get_slots(mips->grid, slots.data());
  if (s != DEX_OK) return s;
  for (size_t i = 0; i < n; ++i) {
    const int lv = h_level[i];
    const bool active = slots[i % (size_t)mips->grid->n_bricks] >= 0;
    if (lv < -1 || lv > mips->max_level || (active != (lv >= 0))) {
      dex_set_error("injected level out of range or inconsistent with brick occupancy");
      return DEX_ERR_SHAPE;
    }
  }
  DEX_CUDA_CHECK(cudaMemcpy(mips->d_levels, h_level, n, cudaMemcpyHostToDevice));
  s = dex_launch_pack_levels(mips, 0);
  if (s != DEX_OK) return s;
  DEX_CUDA_CHECK(cudaDeviceSynchronize());
  return DEX_OK;
}

dex_status dex_mips_velocity_bin_report(const dex_mips* mips, float factor, float* h_max_ratio, int64_t* h_cells_over) {
  if (!mips || !h_max_ratio || !h_cells_over) { dex_set_error("NULL mips / outputs"); return DEX_ERR_INVALID_ARG; }
  if (mips->variant != DEX_VELINTERP) { dex_set_error("the bin-spacing report applies to DEX_VELINTERP mips"); return DEX_ERR_INVALID_ARG; }
  const int nl = mips->dev.n_lines;
  for (int l = 0; l < nl; ++l) { h_max_ratio[l] = 0.0f; h_cells_over[l] = 0; }
  if (nl == 0) return DEX_OK;
  unsigned* d_max = nullptr;
  unsigned long long* d_cnt = nullptr;
  DEX_CUDA_CHECK(cudaDeviceSynchronize());
  dex_status s = dmalloc(&d_max, (size_t)DEX_MAX_LINES, (cudaStream_t)0);
  if (s == DEX_OK) s = dmalloc(&d_cnt, (size_t)DEX_MAX_LINES, (cudaStream_t)0);
  cudaError_t e = cudaSuccess;
  if (s == DEX_OK) e = cudaMemsetAsync(d_max, 0, sizeof(unsigned) * DEX_MAX_LINES, 0);
  if (s == DEX_OK && e == cudaSuccess) e = cudaMemsetAsync(d_cnt, 0, sizeof(unsigned long long) * DEX_MAX_LINES, 0);
  if (s == DEX_OK && e == cudaSuccess) s = dex_launch_vbin_report(mips, factor, d_max, d_cnt, 0);
  unsigned hmax[DEX_MAX_LINES] = {0};
  unsigned long long hcnt[DEX_MAX_LINES] = {0};
  if (s == DEX_OK && e == cudaSuccess) e = cudaMemcpy(hmax, d_max, sizeof(hmax), cudaMemcpyDeviceToHost);
  if (s == DEX_OK && e == cudaSuccess) e = cudaMemcpy(hcnt, d_cnt, sizeof(hcnt), cudaMemcpyDeviceToHost);
  cudaDeviceSynchronize();
  dex_free(d_max, 0);
  dex_free(d_cnt, 0);
  if (s != DEX_OK) return s;
  DEX_CUDA_CHECK(e);
  for (int l = 0; l < nl; ++l) {
    memcpy(&h_max_ratio[l], &hmax[l], sizeof(float));
    h_cells_over[l] = (int64_t)hcnt[l];
  }
  return DEX_OK;
}

dex_status dex_mips_set_level_caps(dex_mips* mips, int n_caps, const float* h_cap_t) {
  if (!mips || (n_caps > 0 && !h_cap_t)) { dex_set_error("NULL mips / h_cap_t"); return DEX_ERR_INVALID_ARG; }
  if (n_caps < 0 || n_caps > 8) { dex_set_error("n_caps must be 0..8"); return DEX_ERR_SHAPE; }
  for (int i = 0; i < n_caps; ++i) {
    if (!(h_cap_t[i] >= 0.0f) || (i > 0 && h_cap_t[i] < h_cap_t[i - 1])) {
      dex_set_error("cap thresholds must be >= 0 and ascending");
      return DEX_ERR_INVALID_ARG;
    }
  }
  mips->dev.n_caps = n_caps;
  for (int i = 0; i < 8; ++i) mips->dev.cap_t[i] = (i < n_caps) ? h_cap_t[i] : 0.0f;
  return DEX_OK;
}

dex_status dex_mips_get_packed_levels(const dex_mips* mips, int batch, uint64_t* h_words, int64_t* n_words) {
  if (!mips) { dex_set_error("NULL mips"); return DEX_ERR_INVALID_ARG; }
  if (batch < 0 || batch >= mips->n_batch) { dex_set_error("batch out of range"); return DEX_ERR_SHAPE; }
  if (n_words) *n_words = mips->dev.words_per_batch;
  if (h_words) {
    DEX_CUDA_CHECK(cudaDeviceSynchronize());
    DEX_CUDA_CHECK(cudaMemcpy(h_words, mips->d_packed + (size_t)batch * mips->dev.words_per_batch,
                              sizeof(uint64_t) * (size_t)mips->dev.words_per_batch, cudaMemcpyDeviceToHost));
  }
  return DEX_OK;
}

dex_status dex_mips_get_level_data(const dex_mips* mips, int chain, int level, float* h_dense) {
  if (!mips || !h_dense) { dex_set_error("NULL mips / h_dense"); return DEX_ERR_INVALID_ARG; }
  if (level < 0 || level > mips->max_level) { dex_set_error("level out of range"); return DEX_ERR_SHAPE; }
  size_t width = 0;
  switch (chain) {
    case DEX_CHAIN_ETA: case DEX_CHAIN_CHI: width = (size_t)mips->n_lambda; break;
    case DEX_CHAIN_VEL: width = 4; if (mips->variant == DEX_ISO) width = 0; break;
    case DEX_CHAIN_LINE: width = 4 * (size_t)mips->dev.n_lines; break;
    case DEX_CHAIN_VTAB: width = (mips->variant == DEX_VELINTERP) ? 2 * (size_t)mips->dev.n_vbins * mips->n_lambda : 0; break;
    default: dex_set_error("unknown chain"); return DEX_ERR_INVALID_ARG;
  }
  if (width == 0) { dex_set_error("chain not present in this variant"); return DEX_ERR_INVALID_ARG; }
  size_t cells = 1;
  for (int a = 0; a < mips->grid->dev.ndim; ++a) cells *= (size_t)(mips->grid->dev.dims[a] >> level);
  float* d_dense = nullptr;
  DEX_CUDA_CHECK(cudaDeviceSynchronize());
  dex_status s = dmalloc(&d_dense, cells * width, (cudaStream_t)0);
  if (s != DEX_OK) return s;
  cudaError_t e = cudaMemset(d_dense, 0, sizeof(float) * cells * width);
  if (e == cudaSuccess) {
    s = dex_launch_level_data(mips, chain, level, d_dense, 0);
    if (s == DEX_OK) e = cudaMemcpy(h_dense, d_dense, sizeof(float) * cells * width, cudaMemcpyDeviceToHost);
  }
  cudaDeviceSynchronize();
  dex_free(d_dense, (cudaStream_t)0);
  if (s != DEX_OK) return s;
  DEX_CUDA_CHECK(e);
  return DEX_OK;
}

void dex_destroy_mips(dex_mips* mips) {
  if (!mips) return;
  free_mips_memory(mips);
  delete mips;
}

// ------------------------------------------------------------------------------------------- solve
dex_status dex_formal_solution(const dex_grid* grid, const dex_mips* mips, const dex_rays* rays, float* d_I,
                               dex_visit_capture* capture, int64_t* d_segment_count, void* stream) {
  DexRaysDev R;
  dex_status s = check_rays(grid, mips, rays, &R);
  if (s != DEX_OK) return s;
  if (rays->n_probes == 0 || rays->n_dirs == 0) return DEX_OK;   // nothing to trace
  if (!d_I && !capture) { dex_set_error("d_I is NULL and no capture requested"); return DEX_ERR_INVALID_ARG; }
  if (capture) {
    if (!capture->d_counts || !capture->d_records || !capture->d_offsets || capture->capacity < 0) {
      dex_set_error("capture buffers are NULL");
      return DEX_ERR_INVALID_ARG;
    }
    if (capture->batch < 0 || capture->batch >= mips->n_batch) { dex_set_error("capture batch out of range"); return DEX_ERR_SHAPE; }
  }
  if (!have_device()) return DEX_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  if (d_I) {
    MarchTimer tm(st);
    s = dex_launch_march(grid, mips, R, d_I, false, (unsigned long long*)d_segment_count, lanes_for(R.n_probes), g_tile_probes.load() != 0, st);
    if (s != DEX_OK) return s;
  }
  if (capture) {
    int* d_over = nullptr;
    s = dmalloc(&d_over, 1, st);
    if (s != DEX_OK) return s;
    int h_over = 0;
    cudaError_t e = cudaMemsetAsync(d_over, 0, sizeof(int), st);
    if (e == cudaSuccess) {
      s = dex_launch_capture(grid, mips, R, capture, d_over, st);
      if (s == DEX_OK) e = cudaMemcpyAsync(&h_over, d_over, sizeof(int), cudaMemcpyDeviceToHost, st);
      if (s == DEX_OK && e == cudaSuccess) e = cudaStreamSynchronize(st);
    }
    dex_free(d_over, st);
    if (s != DEX_OK) return s;
    DEX_CUDA_CHECK(e);
    if (h_over) { dex_set_error("visit capture overflow: counts are complete, records truncated"); return DEX_ERR_CAPACITY; }
  }
  return DEX_OK;
}

dex_status dex_mean_intensity(const dex_grid* grid, const dex_mips* mips, const dex_rays* rays, const float* d_I,
                              float* d_J, int64_t* d_segment_count, void* stream) {
  DexRaysDev R;
  dex_status s = check_rays(grid, mips, rays, &R);
  if (s != DEX_OK) return s;
  if (rays->n_probes == 0) return DEX_OK;                          // J has no rows
  if (!d_J) { dex_set_error("d_J is NULL"); return DEX_ERR_INVALID_ARG; }
  if (rays->n_dirs > 0 && !rays->d_weights) { dex_set_error("d_weights is NULL"); return DEX_ERR_INVALID_ARG; }
  if (!have_device()) return DEX_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  if (d_I) return dex_launch_reduce_j(R, mips->n_lambda, d_I, d_J, st);
  MarchTimer tm(st);
  return dex_launch_march(grid, mips, R, d_J, true, (unsigned long long*)d_segment_count, lanes_for(R.n_probes), g_tile_probes.load() != 0, st);
}

// ------------------------------------------------------------------------------------------- rebuild pipeline
dex_status dex_mean_intensity_pipelined(const dex_grid* grid, const dex_mips_desc* desc, const dex_rays* rays,
                                        int batches_per_stage, int n_caps, const float* h_cap_t, float* d_J,
                                        int64_t* d_segment_count, int8_t* h_levels, void* stream) {
  if (!grid || !desc || !rays) { dex_set_error("NULL grid / desc / rays"); return DEX_ERR_INVALID_ARG; }
  if (batches_per_stage < 1) { dex_set_error("batches_per_stage must be >= 1"); return DEX_ERR_INVALID_ARG; }
  if (desc->lambda_batch != DEX_W) { dex_set_error("lambda_batch must be 8 in this build"); return DEX_ERR_UNSUPPORTED; }
  if (desc->n_lambda <= 0 || desc->n_lambda % DEX_W) {
    dex_set_error("n_lambda must be a positive multiple of lambda_batch");
    return DEX_ERR_SHAPE;
  }
  if (desc->lambda_stride != 0 && desc->lambda_stride < desc->n_lambda) {
    dex_set_error("lambda_stride must be 0 (dense) or >= n_lambda");
    return DEX_ERR_SHAPE;
  }
  if (rays->n_probes > 0 && !d_J) { dex_set_error("d_J is NULL"); return DEX_ERR_INVALID_ARG; }
  if (rays->n_probes > 0 && rays->n_dirs > 0 && !rays->d_weights) { dex_set_error("d_weights is NULL"); return DEX_ERR_INVALID_ARG; }
  if (!have_device()) return DEX_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  const int n_batch = desc->n_lambda / DEX_W;
  const int n_stage = (n_batch + batches_per_stage - 1) / batches_per_stage;
  const int stride = desc->lambda_stride ? desc->lambda_stride : desc->n_lambda;
  const bool aniso = desc->variant != DEX_ISO;

  // Streams: builds on `sb`, which outranks the marches so that its small kernels take the first SM slots that fall
  // free; marches alternate between two streams so that stage s+1's blocks fill the SMs that stage s's last wave
  // leaves idle (a stage of one batch is only ~1.7 waves of blocks on C2: serialised, the tails cost 20 %).
  int prio_lo = 0, prio_hi = 0;
  cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
  cudaStream_t sb = nullptr, sm[2] = {nullptr, nullptr};
  DEX_CUDA_CHECK(cudaStreamCreateWithPriority(&sb, cudaStreamNonBlocking, prio_hi));
  for (int i = 0; i < 2; ++i) {
    cudaError_t ce = cudaStreamCreateWithPriority(&sm[i], cudaStreamNonBlocking, prio_lo);
    if (ce != cudaSuccess) { cudaStreamDestroy(sb); if (i) cudaStreamDestroy(sm[0]); DEX_CUDA_CHECK(ce); }
  }
  cudaEvent_t ev_in = nullptr, ev_built[2] = {nullptr, nullptr}, ev_marched[2] = {nullptr, nullptr};
  cudaEventCreateWithFlags(&ev_in, cudaEventDisableTiming);
  for (int i = 0; i < 2; ++i) {
    cudaEventCreateWithFlags(&ev_built[i], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&ev_marched[i], cudaEventDisableTiming);
  }

  dex_status s = DEX_OK;
  cudaError_t e = cudaSuccess;
  int* d_perm = nullptr;
  if (rays->n_probes > 0 && g_tile_probes.load() != 0) {   // the probe tiling is the same for every stage
    DexRaysDev R;
    R.n_probes = rays->n_probes;
    R.probe_pos = rays->d_probe_pos;
    if (!rays->d_probe_pos) { dex_set_error("d_probe_pos is NULL"); s = DEX_ERR_INVALID_ARG; }
    else s = dex_make_probe_tiling(grid, R, &d_perm, st);
  }
  cudaEventRecord(ev_in, st);            // the caller's inputs (and the tiling) are ordered on `stream`
  cudaStreamWaitEvent(sb, ev_in, 0);
  cudaStreamWaitEvent(sm[0], ev_in, 0);
  cudaStreamWaitEvent(sm[1], ev_in, 0);

  float4* keep_aux = nullptr;            // built by the first stage on `sb`, read by every stage, freed after the join
  float* keep_vftab = nullptr;
  dex_mips* prev = nullptr;              // stage s-1, released on the build stream once its march has finished
  int prev_ev = 0;
  for (int sg = 0; sg < n_stage && s == DEX_OK && e == cudaSuccess; ++sg) {
    const int b0 = sg * batches_per_stage;
    const int nb = (b0 + batches_per_stage <= n_batch) ? batches_per_stage : n_batch - b0;
    const size_t off = (size_t)b0 * DEX_W;
    dex_mips_desc sub = *desc;
    sub.n_lambda = nb * DEX_W;
    sub.lambda_stride = stride;
    if (desc->d_lambda) sub.d_lambda = desc->d_lambda + off;
    if (desc->d_eta) sub.d_eta = desc->d_eta + off;
    if (desc->d_chi) sub.d_chi = desc->d_chi + off;
    if (desc->d_eta_bg) sub.d_eta_bg = desc->d_eta_bg + off;
    if (desc->d_chi_bg) sub.d_chi_bg = desc->d_chi_bg + off;
    if (aniso && desc->h_active_lines) sub.h_active_lines = desc->h_active_lines + (size_t)b0 * DEX_MAX_LINES;
    dex_mips* cur = nullptr;
    s = build_vlm_mips_impl(grid, &sub, (void*)sb, keep_aux, keep_vftab, &cur);
    if (s != DEX_OK) break;
    if (aniso && !keep_aux && cur->d_aux && cur->d_vftab) {
      // the first stage's wavelength-independent chains and Voigt tables serve every later stage: this call keeps them
      keep_aux = cur->d_aux;
      keep_vftab = cur->d_vftab;
      cur->aux_borrowed = true;
    }
    cur->dev.io_stride = desc->n_lambda;
    cur->dev.io_base = (int)off;
    s = dex_mips_set_level_caps(cur, n_caps, h_cap_t);
    if (s == DEX_OK && h_levels)
      e = cudaMemcpyAsync(h_levels + (size_t)b0 * grid->n_bricks, cur->d_levels, (size_t)nb * grid->n_bricks,
                          cudaMemcpyDeviceToHost, sb);
    cudaEventRecord(ev_built[sg & 1], sb);
    if (prev) {   // enqueued AFTER this stage's build: stage s-1 is released when its march is done, and the build of
                  // stage s+1 queues behind that, so at most two stages' pyramids are resident
      cudaStreamWaitEvent(sb, ev_marched[prev_ev], 0);
      dex_destroy_mips(prev);
      prev = nullptr;
    }
    cudaStream_t ms = sm[sg & 1];
    if (s == DEX_OK && e == cudaSuccess && rays->n_probes > 0) {
      DexRaysDev R;
      s = check_rays(grid, cur, rays, &R);
      if (s == DEX_OK) {
        cudaStreamWaitEvent(ms, ev_built[sg & 1], 0);
        MarchTimer tm(ms);
        s = dex_launch_march(grid, cur, R, d_J, true, (unsigned long long*)d_segment_count, lanes_for(R.n_probes),
                             false, ms, d_perm);
      }
    }
    cudaEventRecord(ev_marched[sg & 1], ms);
    prev = cur;
    prev_ev = sg & 1;
  }
  if (prev) {
    cudaStreamWaitEvent(sb, ev_marched[prev_ev], 0);
    dex_destroy_mips(prev);
  }
  // join: `stream` waits for both march streams and for the build stream's tail (level copies, releases), so draining
  // `stream` drains the call
  for (int i = 0; i < 2; ++i) {
    cudaEventRecord(ev_built[i], sm[i]);
    cudaStreamWaitEvent(st, ev_built[i], 0);
  }
  cudaEventRecord(ev_in, sb);
  cudaStreamWaitEvent(st, ev_in, 0);
  if (d_perm) cudaFreeAsync(d_perm, st);
  dex_free(keep_aux, st);                // `st` has just been made to wait for every march and for the build stream
  dex_free(keep_vftab, st);
  if (h_levels && e == cudaSuccess) e = cudaStreamSynchronize(sb);
  cudaEventDestroy(ev_in);
  for (int i = 0; i < 2; ++i) { cudaEventDestroy(ev_built[i]); cudaEventDestroy(ev_marched[i]); }
  cudaStreamDestroy(sb);                 // deferred by the runtime until the streams' work has completed
  cudaStreamDestroy(sm[0]);
  cudaStreamDestroy(sm[1]);
  if (s != DEX_OK) return s;
  DEX_CUDA_CHECK(e);
  DEX_CUDA_CHECK(cudaGetLastError());
  return DEX_OK;
}

// ------------------------------------------------------------------------------------------- single-direction VLM
namespace {
dex_status check_aniso_desc(const dex_mips_desc* desc) {
  if (desc->variant == DEX_ISO) { dex_set_error("a static (DEX_ISO) medium has no direction dependence"); return DEX_ERR_INVALID_ARG; }
  if (desc->lambda_batch != DEX_W) { dex_set_error("lambda_batch must be 8 in this build"); return DEX_ERR_UNSUPPORTED; }
  if (desc->n_lambda <= 0 || desc->n_lambda % DEX_W) { dex_set_error("n_lambda must be a positive multiple of lambda_batch"); return DEX_ERR_SHAPE; }
  if (desc->lambda_stride != 0 && desc->lambda_stride < desc->n_lambda) { dex_set_error("lambda_stride must be 0 (dense) or >= n_lambda"); return DEX_ERR_SHAPE; }
  if (!desc->d_eta_bg || !desc->d_chi_bg || !desc->d_vel || !desc->d_lambda || !desc->h_active_lines) {
    dex_set_error("anisotropic media need d_eta_bg, d_chi_bg, d_vel, d_lambda, h_active_lines");
    return DEX_ERR_INVALID_ARG;
  }
  if (desc->n_lines < 0 || desc->n_lines > DEX_MAX_LINES) { dex_set_error("n_lines must be 0..4"); return DEX_ERR_SHAPE; }
  if (desc->n_lines > 0 && (!desc->h_lambda0 || !desc->d_eta_star0 || !desc->d_chi_star0 || !desc->d_a0 || !desc->d_inv_dlamD)) {
    dex_set_error("line arrays are NULL");
    return DEX_ERR_INVALID_ARG;
  }
  const int n_batch = desc->n_lambda / DEX_W;
  for (int i = 0; i < n_batch * DEX_MAX_LINES; ++i) {
    const int l = desc->h_active_lines[i];
    if (l < -1 || l >= desc->n_lines) { dex_set_error("active line id out of range"); return DEX_ERR_SHAPE; }
  }
  if (!(desc->c_light > 0.0f)) { dex_set_error("c_light must be > 0"); return DEX_ERR_INVALID_ARG; }
  return DEX_OK;
}

dex_status upload_active_lines(const dex_mips_desc* desc, signed char** d_al, cudaStream_t st) {
  const size_t n = (size_t)(desc->n_lambda / DEX_W) * DEX_MAX_LINES;
  dex_status s = dmalloc(d_al, n, st);
  if (s != DEX_OK) return s;
  cudaError_t e = cudaMemcpyAsync(*d_al, desc->h_active_lines, n, cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) { dex_free(*d_al, st); *d_al = nullptr; DEX_CUDA_CHECK(e); }
  return DEX_OK;
}
}  // namespace

dex_status dex_direction_fields(const dex_grid* grid, const dex_mips_desc* desc, const float* d_omega,
                                const float* d_sin_incl, float* d_eta, float* d_chi, void* stream) {
  if (!grid || !desc || !d_omega || !d_eta || !d_chi) { dex_set_error("NULL grid / desc / d_omega / d_eta / d_chi"); return DEX_ERR_INVALID_ARG; }
  if (d_sin_incl && grid->dev.ndim != 2) { dex_set_error("d_sin_incl (2.5D rays) needs a 2D grid"); return DEX_ERR_INVALID_ARG; }
  dex_status s = check_aniso_desc(desc);
  if (s != DEX_OK) return s;
  if (!have_device()) return DEX_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  signed char* d_al = nullptr;
  s = upload_active_lines(desc, &d_al, st);
  if (s != DEX_OK) return s;
  s = dex_launch_direction_fields(grid, desc, d_al, d_omega, d_sin_incl, d_eta, d_chi, st);
  dex_free(d_al, st);
  return s;
}

dex_status dex_mean_intensity_single_direction(const dex_grid* grid, const dex_mips_desc* desc, const dex_rays* rays,
                                               int n_caps, const float* h_cap_t, float* d_J, int64_t* d_segment_count,
                                               int8_t* h_levels, void* stream) {
  if (!grid || !desc || !rays) { dex_set_error("NULL grid / desc / rays"); return DEX_ERR_INVALID_ARG; }
  dex_status s = check_aniso_desc(desc);
  if (s != DEX_OK) return s;
  if (rays->n_probes < 0 || rays->n_dirs < 0) { dex_set_error("negative n_probes / n_dirs"); return DEX_ERR_INVALID_ARG; }
  if (rays->n_probes == 0) return DEX_OK;
  if (!d_J) { dex_set_error("d_J is NULL"); return DEX_ERR_INVALID_ARG; }
  if (rays->n_dirs > 0 && (!rays->d_weights || !rays->d_dirs || !rays->d_probe_pos)) {
    dex_set_error("d_probe_pos / d_dirs / d_weights is NULL");
    return DEX_ERR_INVALID_ARG;
  }
  if (rays->d_sin_incl && grid->dev.ndim != 2) { dex_set_error("d_sin_incl (2.5D rays) needs a 2D grid"); return DEX_ERR_INVALID_ARG; }
  if (!have_device()) return DEX_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t nl = (size_t)desc->n_lambda, D = (size_t)grid->dev.ndim;
  const size_t n_batch = nl / DEX_W;
  DEX_CUDA_CHECK(cudaMemsetAsync(d_J, 0, sizeof(float) * (size_t)rays->n_probes * nl, st));   // n_dirs == 0: J = 0
  if (rays->n_dirs == 0) return DEX_OK;
  float *d_eta = nullptr, *d_chi = nullptr;
  signed char* d_al = nullptr;
  int* d_perm = nullptr;
  s = dmalloc(&d_eta, (size_t)grid->nvox * nl, st);
  if (s == DEX_OK) s = dmalloc(&d_chi, (size_t)grid->nvox * nl, st);
  if (s == DEX_OK) s = upload_active_lines(desc, &d_al, st);
  if (s == DEX_OK && g_tile_probes.load() != 0) {     // one probe tiling serves every direction
    DexRaysDev R;
    R.n_probes = rays->n_probes;
    R.probe_pos = rays->d_probe_pos;
    s = dex_make_probe_tiling(grid, R, &d_perm, st);
  }
  dex_mips_desc iso = *desc;
  iso.variant = DEX_ISO;
  iso.d_eta = d_eta;
  iso.d_chi = d_chi;
  iso.lambda_stride = 0;
  cudaError_t e = cudaSuccess;
  for (int k = 0; k < rays->n_dirs && s == DEX_OK && e == cudaSuccess; ++k) {
    s = dex_launch_direction_fields(grid, desc, d_al, rays->d_dirs + (size_t)k * D,
                                    rays->d_sin_incl ? rays->d_sin_incl + k : nullptr, d_eta, d_chi, st);
    if (s != DEX_OK) break;
    dex_mips* m = nullptr;
    s = dex_build_vlm_mips(grid, &iso, stream, &m);
    if (s != DEX_OK) break;
    s = dex_mips_set_level_caps(m, n_caps, h_cap_t);
    if (s == DEX_OK && h_levels)
      e = cudaMemcpyAsync(h_levels + (size_t)k * n_batch * grid->n_bricks, m->d_levels, n_batch * (size_t)grid->n_bricks,
                          cudaMemcpyDeviceToHost, st);
    dex_rays rk = *rays;
    rk.n_dirs = 1;
    rk.d_dirs = rays->d_dirs + (size_t)k * D;
    rk.d_weights = rays->d_weights + k;
    rk.d_i0 = rays->d_i0 ? rays->d_i0 + (size_t)k * nl : nullptr;
    rk.d_sin_incl = rays->d_sin_incl ? rays->d_sin_incl + k : nullptr;
    rk.accumulate = 1;
    DexRaysDev R;
    if (s == DEX_OK) s = check_rays(grid, m, &rk, &R);
    if (s == DEX_OK) {
      MarchTimer tm(st);
      s = dex_launch_march(grid, m, R, d_J, true, (unsigned long long*)d_segment_count, lanes_for(R.n_probes), false, st,
                           d_perm);
    }
    dex_destroy_mips(m);     // stream-ordered: released after the march above
  }
  if (d_perm) cudaFreeAsync(d_perm, st);
  dex_free(d_al, st);
  dex_free(d_eta, st);
  dex_free(d_chi, st);
  if (s == DEX_OK && e == cudaSuccess && h_levels) e = cudaStreamSynchronize(st);
  if (s != DEX_OK) return s;
  DEX_CUDA_CHECK(e);
  return DEX_OK;
}

dex_status dex_voigt_profile(const float* d_a, const double* d_x, int64_t n, double* d_H, int mode, void* stream) {
  if (n < 0 || (n > 0 && (!d_a || !d_x || !d_H))) { dex_set_error("NULL d_a / d_x / d_H"); return DEX_ERR_INVALID_ARG; }
  if (mode != 0 && mode != 1) { dex_set_error("mode must be 0 (as the march chooses) or 1 (fp64 form)"); return DEX_ERR_INVALID_ARG; }
  if (!have_device()) return DEX_ERR_CUDA;
  return dex_launch_voigt_profile(d_a, d_x, (long long)n, d_H, mode, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------- host entry
dex_status dex_mean_intensity_host(const dex_grid_desc* desc, const uint8_t* h_active, const dex_mips_desc* hm,
                                   const dex_rays* hr, float* h_J, int64_t* h_segment_count, int64_t* h2d_bytes,
                                   int64_t* d2h_bytes, void* stream) {
  if (!desc || !hm || !hr || !h_J) { dex_set_error("NULL desc / host_mips / host_rays / h_J"); return DEX_ERR_INVALID_ARG; }
  if (desc->ndim != 2 && desc->ndim != 3) { dex_set_error("ndim must be 2 or 3"); return DEX_ERR_INVALID_ARG; }
  if (hm->n_lambda <= 0 || hr->n_probes < 0 || hr->n_dirs < 0 || hm->n_lines < 0 || hm->n_lines > DEX_MAX_LINES) {
    dex_set_error("bad n_lambda / n_probes / n_dirs / n_lines");
    return DEX_ERR_SHAPE;
  }
  if (hm->lambda_stride != 0 && hm->lambda_stride != hm->n_lambda) {
    dex_set_error("the host entry uploads dense [nvox][n_lambda] spectra: lambda_stride must be 0 (or n_lambda)");
    return DEX_ERR_SHAPE;
  }
  if (!have_device()) return DEX_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  size_t nvox = 1;
  for (int a = 0; a < desc->ndim; ++a) {
    if (desc->dims[a] <= 0) { dex_set_error("dims must be positive"); return DEX_ERR_SHAPE; }
    nvox *= (size_t)desc->dims[a];
  }
  const size_t nl = (size_t)hm->n_lambda, D = (size_t)desc->ndim;
  Uploads up(st);
  dex_mips_desc dm = *hm;                 // host-side members (h_lambda0, h_active_lines) are used as they are
  dm.d_lambda = up.put(hm->d_lambda, nl);
  dm.d_eta = up.put(hm->d_eta, nvox * nl);
  dm.d_chi = up.put(hm->d_chi, nvox * nl);
  dm.d_eta_bg = up.put(hm->d_eta_bg, nvox * nl);
  dm.d_chi_bg = up.put(hm->d_chi_bg, nvox * nl);
  dm.d_vel = up.put(hm->d_vel, nvox * D);
  dm.d_eta_star0 = up.put(hm->d_eta_star0, nvox * (size_t)hm->n_lines);
  dm.d_chi_star0 = up.put(hm->d_chi_star0, nvox * (size_t)hm->n_lines);
  dm.d_a0 = up.put(hm->d_a0, nvox * (size_t)hm->n_lines);
  dm.d_inv_dlamD = up.put(hm->d_inv_dlamD, nvox * (size_t)hm->n_lines);
  const uint8_t* d_active = up.put(h_active, nvox);
  dex_rays dr = *hr;
  dr.d_probe_pos = up.put(hr->d_probe_pos, (size_t)hr->n_probes * D);
  dr.d_dirs = up.put(hr->d_dirs, (size_t)hr->n_dirs * D);
  dr.d_weights = up.put(hr->d_weights, (size_t)hr->n_dirs);
  dr.d_i0 = up.put(hr->d_i0, (size_t)hr->n_dirs * nl);
  dr.d_sin_incl = up.put(hr->d_sin_incl, (size_t)hr->n_dirs);
  float* d_J = up.alloc<float>((size_t)hr->n_probes * nl);
  int64_t* d_seg = up.alloc<int64_t>(1);
  if (up.status != DEX_OK) return up.status;
  dex_grid* grid = nullptr;
  dex_mips* mips = nullptr;
  dex_status s = dex_build_sparse_grid(desc, d_active, stream, &grid);
  if (s == DEX_OK) s = dex_build_vlm_mips(grid, &dm, stream, &mips);
  cudaError_t e = cudaSuccess;
  if (s == DEX_OK) e = cudaMemsetAsync(d_seg, 0, sizeof(int64_t), st);
  if (s == DEX_OK && e == cudaSuccess) s = dex_mean_intensity(grid, mips, &dr, nullptr, d_J, d_seg, stream);
  int64_t out_bytes = 0;
  if (s == DEX_OK && e == cudaSuccess && hr->n_probes > 0) {
    e = cudaMemcpyAsync(h_J, d_J, sizeof(float) * (size_t)hr->n_probes * nl, cudaMemcpyDeviceToHost, st);
    out_bytes += (int64_t)(sizeof(float) * (size_t)hr->n_probes * nl);
  }
  if (s == DEX_OK && e == cudaSuccess && h_segment_count) {
    e = cudaMemcpyAsync(h_segment_count, d_seg, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
    out_bytes += (int64_t)sizeof(int64_t);
  }
  const cudaError_t e2 = cudaStreamSynchronize(st);     // the temporaries below must not be freed under running work
  dex_destroy_mips(mips);
  dex_destroy_grid(grid);
  if (s != DEX_OK) return s;
  DEX_CUDA_CHECK(e);
  DEX_CUDA_CHECK(e2);
  if (h2d_bytes) *h2d_bytes = up.bytes;
  if (d2h_bytes) *d2h_bytes = out_bytes;
  return DEX_OK;
}

}  // extern "C"
