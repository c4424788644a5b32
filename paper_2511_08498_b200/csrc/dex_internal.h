// dex_internal.h -- host-side declarations shared by the translation units of libdex.so.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>

#include "../../include/dex.h"
#include "dex_device.cuh"

struct dex_grid {
  dex_grid_desc desc;
  DexGridDev dev;          // device view (pointers into memory owned by this handle)
  int* d_slot = nullptr;   // [n_bricks]
  int* d_active_bricks = nullptr;  // [n_active] slot -> brick
  int* d_edist = nullptr;          // [n_bricks] 0 populated, else Chebyshev distance in bricks to the nearest populated brick
  int64_t n_bricks = 0, n_active = 0;
  int64_t nvox = 0;
  cudaStream_t stream = nullptr;   // the stream the handle was built on; its memory is released on it
};

struct dex_mips {
  const dex_grid* grid = nullptr;
  DexMipsDev dev;
  int variant = 0, n_lambda = 0, n_batch = 0, max_level = 0;
  int metric = 0;
  float thr_eta = 0, thr_chi = 0, tau_gate = -1;
  // owned device memory
  float* d_store = nullptr;
  float* d_mrec = nullptr;
  float4* d_aux = nullptr;                   // [n_active][cps][1 + n_lines] velocity + line records (dex_aux_vel / dex_aux_line)
  float* d_vtab = nullptr;
  float* d_lam = nullptr;
  signed char* d_active_lines = nullptr;
  signed char* d_levels = nullptr;           // [n_batch][n_bricks]
  unsigned long long* d_packed = nullptr;    // [n_batch][words_per_batch]
  int* d_binfo = nullptr;                    // [n_batch][n_bricks] (slot << 4) | (level + 1)
  float* d_vftab = nullptr;                  // fp32 Voigt tables: [NODES][4] wing then [NODES] core (anisotropic variants)
  int* d_fail = nullptr;                     // [n_batch][n_active][max_level+1]
  size_t store_floats = 0, vtab_floats = 0;
  bool aux_borrowed = false;       // d_aux / d_vftab belong to the caller (the rebuild pipeline shares the wavelength-
                                   // independent chains between its stages): not built, not freed by this handle
  cudaStream_t stream = nullptr;   // the stream the handle was built on; its memory is released on it
};

void dex_set_error(const std::string& msg);
// Stream-ordered device memory from the device's default pool (kept warm: release threshold = unlimited), so that a
// rebuild per iteration does not pay cudaMalloc / cudaFree (page mapping, device-wide synchronisation) every time.
cudaError_t dex_alloc(void** p, size_t bytes, cudaStream_t st);
void dex_free(void* p, cudaStream_t st);
size_t dex_pool_idle_bytes();      // memory the library's pool holds but no live allocation uses (reusable at once)
void dex_count_launch(int n = 1);
int dex_tuning_voigt_fp32();
int dex_tuning_memo();    // -1 automatic, 0 never, 1 always: anisotropic provider memoised per direction (march.cu)
int dex_tuning_memo_budget_mb();   // > 0: cap (MB) on the per-direction records the memoised march holds at once; 0 = automatic
bool dex_tuning_memo_fail_alloc(); // fault injection ("memo_fail_allocs"): true = treat the next records allocation as failed
int dex_tuning_dir_split();   // -1 automatic, 0 never, n > 0: n directions per block whenever J is fused
// automatic mapping of small problems (march.cu): does a fused-J march over n_probes x n_dirs spread its directions over
// blocks (n_lambda only bounds the temporary I), and how many lanes share a ray (`set` = the caller's knob, 0 = automatic)
bool dex_auto_dir_split(long long n_probes, int n_dirs, int n_lambda);
int dex_auto_lanes(int set, long long n_probes, bool dir_split);   // set: the caller's knob (0 = automatic, else 1/2/4/8 lanes per ray)
// the mapping the last dex_launch_march of the calling thread ran with (march.cu)
void dex_last_mapping(int* lanes_per_ray, int* dirs_per_block, int* memo_batches_per_group);
unsigned long long* dex_line_segment_counter();   // device counter, NULL unless march timing is enabled

// grid_build.cu
dex_status dex_launch_grid_build(dex_grid* g, const uint8_t* d_active, cudaStream_t st);
// mips_build.cu
dex_status dex_launch_mips_build(dex_mips* m, const dex_mips_desc* desc, cudaStream_t st);
dex_status dex_launch_pack_levels(dex_mips* m, cudaStream_t st);
dex_status dex_launch_vbin_report(const dex_mips* m, float factor, unsigned* d_max, unsigned long long* d_cnt, cudaStream_t st);
// single-direction VLM input: Classic fields along the direction d_omega[D] (device), dense [nvox][n_lambda]
dex_status dex_launch_direction_fields(const dex_grid* g, const dex_mips_desc* desc, const signed char* d_active_lines,
                                       const float* d_omega, const float* d_sin_incl, float* d_eta, float* d_chi,
                                       cudaStream_t st);
dex_status dex_launch_level_data(const dex_mips* m, int chain, int level, float* d_dense, cudaStream_t st);
// march.cu
dex_status dex_launch_march(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays, float* d_out, bool fuse_j,
                            unsigned long long* d_seg, int lanes_per_ray, bool tile, cudaStream_t st,
                            const int* perm_in = nullptr);
// perm[i] = probe handled by lane group i (compact spatial tiles); *d_perm stays NULL when tiling does not apply.
// Stream-ordered allocation: release with cudaFreeAsync on `st`.
dex_status dex_make_probe_tiling(const dex_grid* g, const DexRaysDev& rays, int** d_perm, cudaStream_t st);
dex_status dex_launch_capture(const dex_grid* g, const dex_mips* m, const DexRaysDev& rays,
                              const dex_visit_capture* cap, int* d_overflow, cudaStream_t st);
dex_status dex_launch_voigt_profile(const float* d_a, const double* d_x, long long n, double* d_H, int mode, cudaStream_t st);
const float* dex_voigt_fast_table_host();   // [NODES * 4 + NODES] floats, computed once
dex_status dex_launch_reduce_j(const DexRaysDev& rays, int n_lambda, const float* d_I, float* d_J, cudaStream_t st);

#define DEX_CUDA_CHECK(expr)                                                                   \
  do {                                                                                         \
    cudaError_t _e = (expr);                                                                   \
    if (_e != cudaSuccess) {                                                                   \
      dex_set_error(std::string(#expr) + ": " + cudaGetErrorString(_e));                       \
      return (_e == cudaErrorMemoryAllocation) ? DEX_ERR_OOM : DEX_ERR_CUDA;                   \
    }                                                                                          \
  } while (0)
