/*
 * dex.h -- C-ABI boundary of the B200-native long-characteristics formal solver
 * (hot path of arxiv/paper_2511_08498, "A Simple Ray Acceleration Structure for Non-LTE
 * Radiative Transfer").  PAPER.md below is /root/reference/PAPER.md; T-/V-rules are the
 * traversal / level contracts of SURVEY.md section 8(c), restated in DESIGN.md.
 *
 * Conventions
 *   - `d_*` pointers are CALLER-OWNED DEVICE memory (e.g. a torch tensor's data_ptr()),
 *     `h_*` pointers are caller-owned HOST memory.  The library never frees or retains them
 *     after the call returns; it copies what it needs into the opaque handles it owns until
 *     dex_destroy_*.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Work is enqueued
 *     asynchronously; only dex_build_sparse_grid (reads back the active-brick count),
 *     dex_*_info / dex_*_get_* and a formal solution with visit capture synchronise.
 *   - Index space: a level-0 voxel has side 1; its physical side is
 *     `voxel_size` (the "Delta s" of PAPER.md:130).  Voxel v = (z*Ny + y)*Nx + x.
 *   - Per-voxel spectra are [nvox][n_lambda] fp32 with lambda fastest; per-line fields are
 *     [n_lines][nvox]; velocities [nvox][ndim].
 *   - Every call returns a dex_status; nothing throws or aborts across the ABI.  Argument
 *     errors are detected before any launch.  dex_last_error() gives a thread-local message.
 *   - NaN / negative eta, chi are the caller's responsibility.
 *   - There is no CPU fallback: without a CUDA device every compute call returns DEX_ERR_CUDA.
 */
#ifndef DEX_H_
#define DEX_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DEX_MAX_LINES 4 /* maximum overlapping lines in a wavelength batch */

typedef enum {
  DEX_OK = 0,
  DEX_ERR_INVALID_ARG = 1,
  DEX_ERR_SHAPE = 2,
  DEX_ERR_UNSUPPORTED = 3,
  DEX_ERR_OOM = 4,
  DEX_ERR_CUDA = 5,
  DEX_ERR_CAPACITY = 6
} dex_status;

/* Thread-local description of the last failure on this thread; valid until the next call. */
const char* dex_last_error(void);
/* Library version string (static storage). */
const char* dex_version(void);

typedef struct dex_grid dex_grid; /* opaque, library-owned */
typedef struct dex_mips dex_mips; /* opaque, library-owned */

/* ------------------------------------------------------------------------------------------
 * Sparse brick grid: the model is split into cubic blocks of side
 * `brick` (16 in 2D / 8 in 3D typically) which are populated or empty.
 * ---------------------------------------------------------------------------------------- */
typedef struct {
  int ndim;         /* 2 or 3 */
  int dims[3];      /* Nx, Ny, Nz voxels (Nz ignored in 2D); each a multiple of brick */
  int brick;        /* power of two, 2..32 */
  float voxel_size; /* h > 0, physical side of a level-0 voxel */
} dex_grid_desc;

/* a1. Brick occupancy + compaction.  A brick is active iff any of its voxels has
 * d_active != 0 (the sparsity map is shared by all wavelengths);
 * d_active == NULL means all active.  Active bricks get storage slots 0..A-1 in brick-index
 * order.  Synchronises once to read A back.
 * Errors: DEX_ERR_INVALID_ARG (NULL desc/out, ndim), DEX_ERR_SHAPE (dims not multiple of
 * brick, brick not a power of two), DEX_ERR_OOM, DEX_ERR_CUDA. */
dex_status dex_build_sparse_grid(const dex_grid_desc* desc, const uint8_t* d_active /*[nvox] or NULL*/,
                                 void* stream, dex_grid** out);
dex_status dex_grid_info(const dex_grid* grid, int64_t* n_bricks, int64_t* n_active);
/* Validation: slot per brick, -1 = empty.  Brick b = (bz*NBy + by)*NBx + bx. */
dex_status dex_grid_get_slots(const dex_grid* grid, int32_t* h_slot /*[n_bricks]*/);
void dex_destroy_grid(dex_grid* grid);

/* a1 for callers that must not allocate device memory (same numbering as
 * dex_build_sparse_grid: active bricks get slots 0..A-1 in brick-index order).
 * Meant for code that runs where an allocation is not an option: a solver confined to a memory budget fixed at
 * start-up, a plug-in inside a host application that owns the device allocator, a latency-bound loop that cannot
 * wait on the driver's allocation lock.  dex_build_sparse_grid takes its flag array, its counter and the handle's
 * tables from the library's pool; this entry calls no cudaMalloc / cudaFree / pool routine and never synchronises:
 *   outputs   d_slot [n_bricks] (slot, -1 = empty brick), d_active_bricks [n_bricks] (entry s = brick of slot s for
 *             s < A; entries from A on are left as they were), d_n_active [1] (A) -- CALLER-OWNED DEVICE memory,
 *             written asynchronously on `stream`; no handle is created (the other calls of this header do not take
 *             these tables -- this entry serves callers that run the brick bookkeeping themselves);
 *   scratch   the per-brick occupancy flags sit in a fixed array inside the library image: DEX_STATIC_MAX_BRICKS
 *             ints (4 MiB), held by every GPU that loads libdex.so until the process exits.  More bricks than that
 *             -> DEX_ERR_SHAPE with a message naming the limit, nothing launched.
 * The first call on each device looks up the array's device address (cudaGetSymbolAddress, with the caller's
 * current device) and keeps it; make that first call outside any stream capture.  All calls on a device share the
 * array and it keeps the last call's contents; each call rewrites the part it reads, so nothing needs clearing, but
 * two calls that can overlap on the GPU (two streams with no ordering between them) race on it -- order them.
 * d_active: [nvox] device bytes or NULL (all active).
 * Errors: DEX_ERR_INVALID_ARG (NULL desc / outputs, ndim), DEX_ERR_SHAPE (brick, dims, too many bricks),
 * DEX_ERR_UNSUPPORTED (device ordinal >= 64), DEX_ERR_CUDA. */
#define DEX_STATIC_MAX_BRICKS (1 << 20)
dex_status dex_brick_slots_static(const dex_grid_desc* desc, const uint8_t* d_active /*[nvox] or NULL*/,
                                  int32_t* d_slot, int32_t* d_active_bricks, int32_t* d_n_active, void* stream);

/* ------------------------------------------------------------------------------------------
 * MIP pyramid + variance-limited mipmapping
 * ---------------------------------------------------------------------------------------- */
typedef enum {
  DEX_ISO = 0,       /* static medium: fetch eta, chi */
  DEX_VELINTERP = 1, /* velocity-grid AVLM */
  DEX_CAV = 2,       /* "Core and Voigt" AVLM */
  DEX_CLASSIC = 3    /* brute force at every level-0 cell for every direction; no mips */
} dex_variant;

typedef enum {
  DEX_METRIC_IOD_LOG = 0, /* eq. 8 on ln(eta h), ln(chi h) + chi h gate */
  DEX_METRIC_RELVAR = 1   /* Var[x]/Mean[x]^2 of eta, chi (BASELINE.json wording) */
} dex_metric;

typedef struct {
  dex_variant variant;
  int n_lambda;     /* total wavelengths; multiple of lambda_batch */
  int lambda_batch; /* W: wavelengths per batch sharing one level table (8). Must be 8. */
  int max_level;    /* 0 <= max_level <= log2(brick) */
  dex_metric metric;
  float thr_eta, thr_chi; /* a cell passes iff metric < thr for both (strict) */
  float tau_gate;         /* always average where mean(chi) h <= tau_gate; < 0 disables */
  const float* d_lambda;  /* [n_lambda] wavelengths (anisotropic variants; same unit as h_lambda0) */
  /* ISO */
  const float* d_eta; /* [nvox][n_lambda] */
  const float* d_chi;
  /* anisotropic variants (eqs. 10-20) */
  const float* d_eta_bg; /* [nvox][n_lambda] isotropic background */
  const float* d_chi_bg;
  const float* d_vel; /* [nvox][ndim] bulk velocity, unit of c_light */
  int n_lines;
  const float* h_lambda0;   /* [n_lines] rest wavelengths (HOST) */
  const float* d_eta_star0; /* [n_lines][nvox] eta*_l(lambda0)  (eq. 18) */
  const float* d_chi_star0; /* [n_lines][nvox] chi*_l(lambda0)  (eq. 19) */
  const float* d_a0;        /* [n_lines][nvox] damping a(lambda0) (eq. 20) */
  const float* d_inv_dlamD; /* [n_lines][nvox] 1 / Doppler width */
  const int8_t* h_active_lines; /* [n_batch][DEX_MAX_LINES] line ids, -1 padded (HOST) */
  int n_vbins;   /* DEX_VELINTERP: velocity bins per cell, 2..32 */
  float c_light; /* speed of light in the unit of d_vel */
  int lambda_stride; /* floats between consecutive voxels in d_eta, d_chi, d_eta_bg, d_chi_bg; 0 = n_lambda (dense).
                      * A larger stride lets a handle be built for a window of a wider spectrum (the stages of
                      * dex_mean_intensity_pipelined): pass the arrays offset to the window's first wavelength.
                      * Must be 0 or >= n_lambda (DEX_ERR_SHAPE). */
} dex_mips_desc;

/* a2-a4. Gather active bricks into brick-major storage, build the box-filter mips of every
 * chain of the variant (V1: fp64 sum of the 2^D children, one rounding), evaluate the VLM cell
 * test in fp64 (V2-V6) and select one level per (batch, brick) (V5), packed into 64-bit words
 * (PAPER.md:162).  Asynchronous on `stream`.
 * Errors: DEX_ERR_INVALID_ARG (NULL pointers required by the variant), DEX_ERR_SHAPE
 * (max_level > log2(brick), n_lambda % lambda_batch, n_lines > DEX_MAX_LINES, bad line ids),
 * DEX_ERR_UNSUPPORTED (lambda_batch != 8, n_vbins out of range), DEX_ERR_OOM, DEX_ERR_CUDA. */
dex_status dex_build_vlm_mips(const dex_grid* grid, const dex_mips_desc* desc, void* stream, dex_mips** out);
/* Validation accessors (synchronise). */
dex_status dex_mips_get_levels(const dex_mips* mips, int8_t* h_level /*[n_batch][n_bricks], -1 empty*/);
dex_status dex_mips_set_levels(dex_mips* mips, const int8_t* h_level /*same shape; injects a table*/);
/* Velocity-bin spacing diagnostic of DEX_VELINTERP mips (the code "warns if the spacing between bins
 * is greater than two times (configurable) the thermal width of the spectral line").  For every line l:
 * h_max_ratio[l] = max over the level-0 cells of the active bricks of (2 V / (n_vbins - 1)) / (c dlamD_l / lambda0_l),
 * V = |v| of the voxel; h_cells_over[l] = number of those cells whose ratio exceeds `factor` (the paper's default: 2).
 * Both arrays hold n_lines entries.  Synchronises.  Errors: DEX_ERR_INVALID_ARG (NULL, not a VELINTERP handle). */
dex_status dex_mips_velocity_bin_report(const dex_mips* mips, float factor, float* h_max_ratio, int64_t* h_cells_over);
/* Near-field MIP cap (the long-characteristics analogue of DexRT's per-cascade maximum MIP level
 * [0,0,1,2,3,4] over intervals ending at 1.5 * 4^i voxels; T8).  A cell entered at
 * distance t (index units) from the probe is formed at level min(brick level, #{i : t >= h_cap_t[i]}); thresholds
 * ascending, n_caps <= 8; n_caps = 0 (the default) removes the cap.  Host-side state of the handle: takes effect for
 * the marches launched afterwards.  Errors: DEX_ERR_INVALID_ARG, DEX_ERR_SHAPE. */
dex_status dex_mips_set_level_caps(dex_mips* mips, int n_caps, const float* h_cap_t);
/* Packed block states of one batch: state = level + 1 (0 = empty) in ceil(log2(max_level+2)) bits,
 * floor(64/bits) bricks per word, no straddling.  *n_words receives the word count; h_words may be
 * NULL to query it. */
dex_status dex_mips_get_packed_levels(const dex_mips* mips, int batch, uint64_t* h_words, int64_t* n_words);
typedef enum {
  DEX_CHAIN_ETA = 0,      /* ISO eta / background eta:  [cells_m][n_lambda] */
  DEX_CHAIN_CHI = 1,
  DEX_CHAIN_VEL = 2,      /* [cells_m][4]: box-filtered vx, vy, vz(0 in 2D), max |v| over the cell */
  DEX_CHAIN_LINE = 3,     /* [cells_m][n_lines][4]: eta*, chi*, a0, 1/dlamD */
  DEX_CHAIN_VTAB = 4      /* [cells_m][n_vbins][n_lambda][2] (eta, chi), DEX_VELINTERP */
} dex_chain;
/* Canonical dense level-m array of a chain (cells of empty bricks are 0). */
dex_status dex_mips_get_level_data(const dex_mips* mips, int chain, int level, float* h_dense);
/* Releases the handle's device memory with a stream-ordered free on the stream the handle was BUILT on.  Work that
 * uses the handle on another stream must be ordered before the destroy by the caller (event / synchronise): the pool
 * may hand the memory to the next allocation on the build stream at once.  The same holds for dex_destroy_grid. */
void dex_destroy_mips(dex_mips* mips);

/* ------------------------------------------------------------------------------------------
 * Rays: long characteristics from each probe along each quadrature direction to the grid
 * boundary.  I(p, w) is the intensity arriving at p propagating along w; the
 * library traces the upwind characteristic x(s) = p - s w (T1).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
  int64_t n_probes;
  const float* d_probe_pos; /* [n_probes][ndim], index space, inside [0, N) on every axis */
  int n_dirs;
  const float* d_dirs;    /* [n_dirs][ndim] unit propagation directions */
  const float* d_weights; /* [n_dirs] quadrature weights (dex_mean_intensity) */
  const float* d_i0;      /* [n_dirs][n_lambda] incoming boundary intensity, NULL = 0 */
  const float* d_sin_incl; /* [n_dirs] or NULL.  2.5D rays (in-plane samples "augmented with a 4 sample
                            * Gauss-Radau quadrature for different inclinations in y", y homogeneous and free of
                            * velocity): sin of the angle between direction k and the homogeneous
                            * out-of-plane axis, in (0, 1].  d_dirs stays the in-plane unit direction and the traversal
                            * is unchanged; every path length is divided by sin_incl[k] and the projected velocity is
                            * multiplied by it.  2D grids only (else DEX_ERR_INVALID_ARG); NULL = rays in the plane. */
  float t_begin, t_end;    /* Finite radiance interval (DexRT traces HDDA(t1, t2) per cascade: Algorithm 1 l.9, l.22,
                            * PAPER.md:347; T10): only the part of every ray with
                            * t_begin <= t <= t_end (index units from the probe) contributes; d_i0 enters at t_end.  The
                            * traversal still starts at the probe, so cells and plane times are those of the full ray
                            * and each visit is clipped to the interval.  t_end <= 0 (a zero-initialised struct): to the
                            * grid boundary.  Requires 0 <= t_begin < t_end otherwise (DEX_ERR_INVALID_ARG). */
  int accumulate;          /* fused dex_mean_intensity only: d_J += sum_k w_k I_k instead of d_J = ... (0: overwrite).  Lets a
                            * caller sum solves that use different level structures per direction (single-direction VLM). */
} dex_rays;

/* a10. Visit-list capture (validation mode).  Ray r = probe * n_dirs + dir.  Records of ray r
 * are written at d_records[d_offsets[r] + i] in trace order (probe outward) for the traversal of
 * batch `batch`; a record is level << 56 | z << 36 | y << 18 | x with (x,y,z) the cell coordinate
 * at that level (T7).  d_ds (optional) receives the fp32 path lengths.  d_counts[r] always gets the
 * full count; records beyond the ray's room (d_offsets[r+1] - d_offsets[r], last ray: capacity)
 * are dropped and the call returns DEX_ERR_CAPACITY after finishing. */
typedef struct {
  int64_t* d_counts;        /* [n_rays] */
  uint64_t* d_records;      /* [capacity] */
  float* d_ds;              /* [capacity] or NULL */
  int64_t capacity;
  const int64_t* d_offsets; /* [n_rays] */
  int batch;
} dex_visit_capture;

/* a5-a8. HDDA traversal (Algorithm 1, under the T-rules) + per-segment
 * I_out = I_in e^{-chi h ds} + eta h ds E(chi h ds), E(t) = (1 - e^{-t})/t, for every wavelength
 * (eq. 3 with piecewise-constant eta, chi).
 * d_I: [n_probes][n_dirs][n_lambda] fp32.  d_segment_count: NULL or one int64 counter that is
 * INCREMENTED by the number of emitted (non-empty, ds > 0) segments over all rays and batches. */
dex_status dex_formal_solution(const dex_grid* grid, const dex_mips* mips, const dex_rays* rays, float* d_I,
                               dex_visit_capture* capture /*NULL = off*/, int64_t* d_segment_count,
                               void* stream);

/* a9. J(p, lambda) = sum_k w_k I(p, k, lambda).  d_I == NULL: trace internally and
 * reduce in the same kernel (fused; I is never materialised).  d_J: [n_probes][n_lambda] fp32. */
dex_status dex_mean_intensity(const dex_grid* grid, const dex_mips* mips, const dex_rays* rays,
                              const float* d_I /*NULL = fused*/, float* d_J, int64_t* d_segment_count,
                              void* stream);

/* Per-iteration rebuild pipeline.  In the paper every iteration recomputes the MIP chains "from
 * scratch from MIP 0" and configures the refinement "at each wavelength batch": the pyramid of a
 * batch lives only as long as that batch's formal solution.  This entry does the same for a whole spectrum: the
 * n_lambda / lambda_batch batches of `desc` are taken in stages of `batches_per_stage` consecutive batches; stage s+1's
 * pyramid and level table (a2-a4) are built on an internal high-priority stream while stage s's fused march (a5-a9)
 * runs on `stream`, and a stage's pyramid is released as soon as its march has finished, so at most two stages' mips
 * are resident (instead of the whole spectrum's).  The probe tiling is computed once.  Results are those of
 * dex_build_vlm_mips + dex_mean_intensity on the whole spectrum, bit for bit (batches are independent: each has its
 * own level table).  d_J: [n_probes][n_lambda]; *d_segment_count (may be NULL) is incremented by the
 * emitted segments of all stages; n_caps / h_cap_t: near-field cap as in dex_mips_set_level_caps (0 / NULL: none);
 * h_levels (may be NULL): receives the level table [n_batch][n_bricks] (the call then synchronises).  The caller's
 * input arrays must stay valid until `stream` has drained.  Errors: as the calls it chains; DEX_ERR_INVALID_ARG for
 * batches_per_stage < 1. */
dex_status dex_mean_intensity_pipelined(const dex_grid* grid, const dex_mips_desc* desc, const dex_rays* rays,
                                        int batches_per_stage, int n_caps, const float* h_cap_t, float* d_J,
                                        int64_t* d_segment_count, int8_t* h_levels, void* stream);

/* Single-direction VLM ("the VLM method can be employed to generate the error-limited MIP
 * structure for a grid of emissivity and opacity given a single direction ... combined with the adaptive grid and ray
 * acceleration technique"; T11).
 * dex_direction_fields: eta, chi of the anisotropic medium `desc` describes (the inputs of DEX_CAV / DEX_CLASSIC: backgrounds,
 * velocity, line arrays, h_active_lines; thresholds and variant ignored) as seen along ONE direction d_omega[ndim] (device):
 * eqs. 10-20 at full resolution with v_proj = v . omega (times *d_sin_incl if not NULL, a device scalar: 2.5D ray), evaluated
 * in fp64 (HUM1WEI24) and rounded once.  d_eta, d_chi: dense [nvox][n_lambda] fp32, voxels of empty bricks written as 0;
 * they are inputs of a DEX_ISO dex_build_vlm_mips.  Asynchronous on `stream` (h_active_lines is copied at the call).
 * dex_mean_intensity_single_direction: for every quadrature direction k: direction fields, DEX_ISO mips with desc's metric,
 * thresholds, gate and max_level, fused march of direction k's rays (weight w_k, boundary row i0[k], sin_incl[k], interval),
 * accumulated into d_J [n_probes][n_lambda] (overwritten, not added to).  *d_segment_count (may be NULL) is incremented by
 * the emitted segments; h_levels (may be NULL) receives [n_dirs][n_batch][n_bricks] (the call then synchronises).  Holds
 * two dense [nvox][n_lambda] arrays and one direction's pyramid at a time.
 * Errors: DEX_ERR_INVALID_ARG (NULL pointers, desc->variant == DEX_ISO: a static medium has no direction dependence),
 * DEX_ERR_SHAPE, DEX_ERR_OOM, DEX_ERR_CUDA. */
dex_status dex_direction_fields(const dex_grid* grid, const dex_mips_desc* desc, const float* d_omega,
                                const float* d_sin_incl, float* d_eta, float* d_chi, void* stream);
dex_status dex_mean_intensity_single_direction(const dex_grid* grid, const dex_mips_desc* desc, const dex_rays* rays,
                                               int n_caps, const float* h_cap_t, float* d_J, int64_t* d_segment_count,
                                               int8_t* h_levels, void* stream);

/* Validation: the Voigt function H(a_i, x_i) = Re w(x_i + i a_i) of PAPER.md:329 ("HUM1WEI24") exactly as the
 * Core-and-Voigt march evaluates it, for n (damping, frequency offset) pairs in device memory.  mode 0: as the
 * march chooses (fp32 table form inside its damping window, the fp64 Weideman / Humlicek form outside it, see
 * csrc/dex_voigt.cuh); mode 1: the fp64 form everywhere.  Asynchronous on `stream`. */
dex_status dex_voigt_profile(const float* d_a, const double* d_x, int64_t n, double* d_H, int mode, void* stream);

/* The whole hot path (a1-a9) from HOST buffers in one call: the end-to-end entry a caller without
 * device memory of their own uses (bench.py's `e2e` leg).  `h_active` is [nvox] or NULL.  In `host_mips`
 * and `host_rays` EVERY pointer, including the ones named d_*, is HOST memory here (pinned memory makes the
 * copies asynchronous; pageable memory works, staged by the driver).  The call uploads the inputs, runs
 * dex_build_sparse_grid, dex_build_vlm_mips and the fused dex_mean_intensity on `stream`, copies J
 * ([n_probes][n_lambda]) and the emitted-segment count into h_J / h_segment_count (may be NULL), destroys
 * its temporaries and returns after the stream has drained.  *h2d_bytes / *d2h_bytes (may be NULL) receive
 * the bytes copied in each direction.  Errors: as the three calls it chains, plus DEX_ERR_OOM. */
dex_status dex_mean_intensity_host(const dex_grid_desc* desc, const uint8_t* h_active, const dex_mips_desc* host_mips,
                                   const dex_rays* host_rays, float* h_J, int64_t* h_segment_count,
                                   int64_t* h2d_bytes, int64_t* d2h_bytes, void* stream);

/* Number of kernel launches this library has enqueued since load (bench.py's gpu_launches). */
int64_t dex_launch_count(void);
/* High-water mark (bytes) of the device memory this library's handles and temporaries have held at once since the last
 * reset.  All of it comes from a stream-ordered pool of the library's own (one per device, created at first use), which
 * keeps freed memory for the next build instead of returning it to the driver; the device's default pool and other
 * allocators are not touched.  Synchronises.  bench.py reports it to show what the rebuild pipeline keeps resident. */
dex_status dex_pool_high_water(int64_t* bytes_in_use_high, int reset);
/* Return the pool's unused memory to the driver (e.g. before another allocator in the process needs the GBs that C3's
 * velocity tables held); *bytes_reserved_after (may be NULL) = what the pool still holds for live handles.  Synchronises. */
dex_status dex_trim(int64_t* bytes_reserved_after);
/* Device time (ms) and launch count of the march kernels since the last reset, measured with CUDA
 * events on the launching stream when timing is enabled (bench.py roofline leg).  Synchronises. */
void dex_march_timing_enable(int on);
dex_status dex_march_timing_read(double* ms_total, int64_t* n_launches, int reset);
/* Work counter of the anisotropic marches while timing is enabled: provider evaluations / W -- one per emitted segment
 * when eta, chi are evaluated inside the march, one per (cell, direction, batch) record when they are memoised per
 * direction ("memo" below) -- times the number of active lines of the batch for Core-and-Voigt / Classic (bench.py's
 * roofline leg multiplies by W and by the flops per evaluation stated in DESIGN.md).  Synchronises. */
dex_status dex_march_work_read(int64_t* line_segments, int reset);
/* Kernel configuration knob: lanes that share one ray, 1/2/4/8, or 0 (default) = automatic: one thread per ray unless
 * there are fewer probes than one wave of blocks (148 SMs x 128 threads), where 8 lanes per ray fill the machine better
 * (2 when the march is also spread over the machine direction by direction, see "dir_split"). */
dex_status dex_set_lanes_per_ray(int lanes);
/* PREDICTION of the lanes-per-ray mapping a whole-spectrum fused-J march over `n_probes` probes x `n_dirs` directions x
 * `n_lambda` wavelengths takes under the current settings.  It cannot see what only the launch knows (a wavelength window
 * of the rebuild pipeline, a finite radiance interval, a temporary I that fails to allocate -- each keeps the march
 * unsplit); dex_last_march_mapping reports what a march actually ran with. */
dex_status dex_get_lanes_per_ray(int64_t n_probes, int n_dirs, int n_lambda, int* lanes);
/* The mapping the LAST dex_formal_solution / dex_mean_intensity* march launched from the calling thread ran with:
 * lanes sharing a ray (1/2/4/8), directions per block of the direction-split launch (0 = not split: every thread walks
 * all directions), wavelength batches per group of the memoised march (0 = eta, chi evaluated in the ray loop; smaller
 * than the spectrum when the records budget or a failed allocation split it).  Any pointer may be NULL.  bench.py
 * records these instead of restating the rules. */
dex_status dex_last_march_mapping(int* lanes_per_ray, int* dirs_per_block, int* memo_batches_per_group);
/* MEASURED fp32 arithmetic peak of the current device in TFLOP/s (an FMA counts 2 flops): register-resident chains of
 * scalar FFMA (*tflops_ffma) and of the packed two-wide FFMA2 the march's integrators use (*tflops_ffma2), ~15 ms in all,
 * timed with CUDA events on `stream`.  The denominator of the "alu" roofline of the Core-and-Voigt / Classic march
 * (SURVEY.md 8(d) caveat 2).  Either pointer may be NULL.  Synchronises. */
dex_status dex_measure_fp32_peak(double* tflops_ffma, double* tflops_ffma2, void* stream);
/* Kernel-structure knobs for performance experiments (results do not change): "lanes_per_ray" 0/1/2/4/8;
 * "tile_probes" 0/1 (1, default: probes are handed to warps in compact spatial tiles by an internal counting
 * sort instead of in the caller's order); "voigt_fp32" 0/1 (1, default: the Core-and-Voigt march evaluates H(a, x) in
 * its fp32 table form inside the damping window of csrc/dex_voigt.cuh; 0: the fp64 form everywhere -- results agree
 * to ~1e-6); "dir_split" -1 (default: automatic), 0, n: a fused-J march over fewer probes than one wave of blocks is
 * launched as one block per (probe tile, batch, n directions) into a temporary I and summed by the reduction kernel in
 * the fused kernel's order (bit-identical J); 0 never, n > 0 always; "memo" -1 (default: automatic), 0, 1: the
 * anisotropic marches (velocity interpolation, Core-and-Voigt, Classic) evaluate eta, chi once per (cell, direction,
 * batch) into per-direction march records and march those with the ISO kernel, instead of once per ray segment, when a
 * cell is crossed by many rays per direction (a probe in every voxel: hundreds); same routine, same numbers up to the last bits of the record rounding;
 * "memo_budget_mb" 0 (default: automatic -- half of the free device memory, at most 32 GB in 2D / 40 GB in 3D), n > 0:
 * the memoised march holds at most n MB of per-direction records at once and takes the spectrum in more groups of
 * wavelength batches (one batch is the smallest group and is taken even when it exceeds n; J is bit-identical for every
 * grouping).  A records allocation that fails is retried with half the batches; if one batch does not fit, the solve
 * evaluates eta, chi in the ray loop as with "memo" 0 (DEX_ERR_OOM only when that happens after the first group);
 * "memo_fail_allocs" n: fault injection for the tests -- the next n records allocations are treated as failed. */
dex_status dex_set_tuning(const char* name, int value);

#ifdef __cplusplus
}
#endif
#endif /* DEX_H_ */
