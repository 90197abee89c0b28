/*
 * cpm.h -- C ABI of the B200-native checkerboard Cellular Potts sweep (arXiv 2312.09317).
 *
 * The library implements ONE thing: the data-parallel hot path of the paper's parallel CPM --
 * the checkerboard-partitioned Metropolis copy-attempt sweep over a 2D/3D lattice of cell ids
 * ("Designing a parallel execution scheme", Methods L218-264 Eq 1-9, and
 * "GPU implementation details" L270-284), with the optional motility terms of the Methods: Act (Eq 8-9),
 * chemotaxis along a vector field (Eq 4) and persistence along one vector per cell (Eq 5-7).  All compute runs in hand-written CUDA kernels for
 * sm_100a; there is no CPU fallback: every entry point that needs the device fails with
 * CPM_ERR_CUDA when no usable GPU is present.
 *
 * Conventions
 *   - every call returns CPM_OK (0) or a negative CPM_ERR_* code; nothing throws or aborts;
 *     cpm_last_error() returns a message for the last failing call on that context.
 *   - the CALLER owns every buffer it passes.  "set" calls copy from it, "get" calls fill it.
 *     `on_device` says whether the pointer is a device pointer (1; must be on the context's
 *     device) or a host pointer (0).  NULL output pointers are skipped.
 *   - lattice arrays are dense, x fastest: index = x + dims[0]*(y + dims[1]*z); N = prod(dims).
 *     per-cell arrays have max_cells+1 entries (entry 0 = medium, always reported as 0).
 *   - the context owns all device state until cpm_destroy.  One context is not thread-safe.
 *   - cpm_step is asynchronous on the context's stream; getters synchronise that stream.
 */
#ifndef CPM_H
#define CPM_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct cpm_ctx cpm_ctx; /* opaque; owned by the library */

enum { CPM_OK = 0, CPM_ERR_ARG = -1, CPM_ERR_DIMS = -2, CPM_ERR_UNSUPPORTED = -3,
       CPM_ERR_CUDA = -4, CPM_ERR_OOM = -5, CPM_ERR_STATE = -6 };
enum { CPM_MOORE = 0 }; /* the only neighbourhood the paper uses (L225): 8 / 26 neighbours */
enum {
  CPM_FLAG_WARP_KERNEL = 1, /* use the warp-per-subsection kernel even where the pooled kernel applies */
  CPM_FLAG_NO_TMA = 2,      /* warp-per-subsection kernel: stage tiles with plain loads instead of TMA */
  CPM_FLAG_NO_GRAPH = 4     /* launch the kernels of an MCS one by one instead of as one CUDA graph per MCS */
};
enum {
  CPM_MODE_DETERMINISTIC = 0, /* per-cell state read from a phase-start snapshot + the worker's own
                                 deltas; integer atomic deltas applied after (bit-exact, schedule-free) */
  CPM_MODE_LIVE_ATOMICS = 1   /* paper-faithful: live reads (possibly stale, L53), immediate atomics (L51) */
};

/* Problem statement (L220-234, Tables 1-3): lattice geometry, J between cell TYPES,
 * lambda / target per type, temperature, RNG seed, and the checkerboard schedule knobs (L77). */
typedef struct {
  int32_t  ndim;                  /* 2 or 3 */
  int32_t  dims[3];               /* x fastest; dims[2] ignored (1) when ndim == 2 */
  int32_t  neighbourhood;         /* CPM_MOORE */
  int32_t  periodic[3];           /* 0 = closed: the lattice is embedded in immutable medium */
  int32_t  n_types;               /* 1..127; type 0 = medium */
  const int32_t *J;               /* host, n_types*n_types, symmetric, |J| <= 2^24 (Eq 1) */
  const int32_t *lambda_V, *target_V;   /* host [n_types] or NULL (= 0): volume constraint, Eq 1 */
  const int32_t *lambda_P, *target_P;   /* perimeter constraint, Eq 3 */
  const int32_t *lambda_act, *max_act;  /* Act model, Eq 8-9; max_act in [0,255] */
  double   T;                     /* >= 0; 0 = no uphill move, +inf = accept every evaluated move (Eq 2) */
  uint64_t seed;                  /* Philox4x32-10 key */
  int32_t  subsection;            /* S, checkerboard subsection edge; 0 = scheduler's choice */
  int32_t  attempts_per_activation; /* k; 0 = S^d (one activation per subsection per MCS) */
  int32_t  mode;                  /* CPM_MODE_* */
  uint32_t max_cells;             /* cell ids are 0..max_cells; < 2^24 */
  int32_t  device;                /* CUDA device ordinal */
  void    *stream;                /* cudaStream_t (e.g. torch's current stream); NULL = default stream */
  uint32_t flags;                 /* CPM_FLAG_*; 0 = the library chooses (debug / A-B switches for tests) */
  /* Vector terms (Methods L236-253; readings S21, S22); NULL / 0 = off.  With x^ the unit vector of the
   * copy direction (source site -> target site), a copy's dH is lowered by
   *   round( lambda_pers(tau_A) x^.p^_A + lambda_pers(tau_B) x^.p^_B + (lambda_chem(tau_A) + lambda_chem(tau_B)) x^.C_source )
   * (A = source cell, B = target cell, a side only for a real cell), in Q14 fixed point. */
  const int32_t *lambda_pers;     /* host [n_types], |.| <= 2^24: persistence strength, Eq 5 */
  const double  *mu_pers;         /* host [n_types], in [0,1]: directional memory mu of Eq 6 */
  int32_t  dt_pers;               /* look-back Delta t of Eq 6 in MCS; >= 1 when any lambda_pers != 0 */
  const int32_t *lambda_chem;     /* host [n_types], |.| <= 2^24: chemotaxis strength, Eq 4 */
  /* Periodic centroid tracking (L297 "Composite variable tracking"; reading S23).  != 0: on periodic axes a
   * site's coordinate enters its cell's sum as the periodic image nearest to the cell (its anchor = floor of the
   * centroid at the last MCS boundary), and after every MCS the sum is shifted by dim x volume so that the centroid
   * sum/volume (Eq 10) stays inside [0, dim): cells smaller than half the lattice keep a meaningful centroid when
   * they straddle or cross a periodic border; Eq 6 then uses the shortest displacement through the border.
   * 0: sums are the plain coordinate sums of the cell's sites. */
  int32_t  unwrap_centroids;
} cpm_params;

/* Validate parameters, build the type tables, the Metropolis threshold table (Eq 2) and the
 * Act log/exp tables on the host, allocate device state, choose S, k and the phase list
 * (checkerboard scheduler, L49/L77).  Errors: CPM_ERR_ARG (bad value, non-symmetric J, T < 0),
 * CPM_ERR_DIMS (dims not a multiple of S, odd subsection count on a periodic axis),
 * CPM_ERR_UNSUPPORTED (max_cells >= 2^24, S too large for shared memory), CPM_ERR_CUDA,
 * CPM_ERR_OOM. */
int  cpm_create(const cpm_params *params, cpm_ctx **out);
int  cpm_destroy(cpm_ctx *ctx);

/* Load the state of the model: ids[N] cell id per site (0 = medium), frozen[N] (NULL = none;
 * non-zero = obstacle voxel that is never copied from or into, L139 stroma), cell_type
 * [max_cells+1] (type of each cell id; cell_type[0] must be 0).  Resets the Act field to 0 and
 * recounts volume, perimeter (Eq 3's A) and coordinate sums (L288) on the device.
 * Errors: CPM_ERR_ARG (NULL ids/cell_type, an id > max_cells or a type >= n_types).
 * Host buffers (on_device = 0; pinned or pageable) are read before the call returns.  A lattice of >= 2^24 sites on the
 * tiled layout crosses PCIe in 8 slabs on a stream of the context's own while the slabs that have arrived are packed and
 * recounted (cpm_get_lattice likewise, the other way); the result does not depend on it.  The environment variable
 * CPM_PIPE_MIN_SITES, read by cpm_create, moves that threshold (tests). */
int  cpm_set_lattice(cpm_ctx *ctx, const uint32_t *ids, const uint8_t *frozen,
                     const uint8_t *cell_type, int on_device);
/* Optional: set the per-site Act field (integers 0..255 stored as float, L255). */
int  cpm_set_act(cpm_ctx *ctx, const float *act, int on_device);
/* Chemotaxis (Eq 4): the vector field C, field[N][ndim] (component fastest), float32 components in
 * [-1,1] (the paper's fields are unit vectors); stored in Q14.  Default: all zero.  Needs a type with
 * lambda_chem != 0 (else CPM_ERR_UNSUPPORTED); a component outside [-1,1] or NaN -> CPM_ERR_ARG. */
int  cpm_set_chemotaxis_field(cpm_ctx *ctx, const float *field, int on_device);
/* Persistence (Eq 5-7): p[(max_cells+1)][3] doubles, the direction p^ of every cell (unit or zero
 * vectors, components in [-1,1]; entry 0 ignored).  cpm_set_lattice resets every p^ to 0 (no bias) and starts the
 * look-back window at the present centroids; after every MCS of cpm_step each cell's p^ is updated by Eq 6-7 from its
 * centroid (Eq 10) now and dt_pers MCS ago, on the device, in IEEE double without fused multiply-adds.
 * Needs a type with lambda_pers != 0 (else CPM_ERR_UNSUPPORTED). */
int  cpm_set_persistence(cpm_ctx *ctx, const double *p, int on_device);
int  cpm_get_persistence(cpm_ctx *ctx, double *p, int on_device);
/* Set the MCS counter (checkpoint/resume: the RNG is keyed by (seed, MCS, phase, subsection, attempt)). */
int  cpm_set_mcs(cpm_ctx *ctx, uint32_t mcs);

/* Run n_mcs Monte Carlo steps (one MCS = N copy attempts, L65): for each repetition and each
 * of the 2^d checkerboard colours, all subsections of that colour run k sequential copy
 * attempts concurrently (L49); then the Act field decays by 1 (L255).  Asynchronous: the launches of one
 * MCS are captured once into a CUDA graph and replayed on the context's stream. */
int  cpm_step(cpm_ctx *ctx, uint32_t n_mcs);

int  cpm_get_lattice(cpm_ctx *ctx, uint32_t *ids, int on_device);
int  cpm_get_act(cpm_ctx *ctx, float *act, int on_device);
/* Per-cell globals kept by integer atomics (L51, L57, L288): volume, perimeter, coordinate sums.  Volume and perimeter
 * share one 64-bit word {V:hi32, P:lo32} (the paper's interleaved pair, L297): a cell whose perimeter reaches 2^32
 * (only an obstacle id owning > 1.6e8 surface-like voxels could) would carry into its volume -- outside this build. */
int  cpm_get_cell_stats(cpm_ctx *ctx, uint32_t *volume, uint32_t *perimeter,
                        uint64_t *sum_x, uint64_t *sum_y, uint64_t *sum_z, int on_device);
/* Centroid of every cell (Eq 10): xyz[(max_cells+1)][3] doubles = coordinate sums / volume, one IEEE division each,
 * computed on the device from the integer tallies (never accumulated in floating point, L288); (0,0,0) for ids without
 * sites and for medium.  With unwrap_centroids the centroid of a cell that straddles a periodic border lies inside
 * [0, dim) at the cell's true position on the torus. */
int  cpm_get_centroids(cpm_ctx *ctx, double *xyz, int on_device);
/* out (host) = {attempts, evaluated, accepted, mcs}. */
int  cpm_get_counters(cpm_ctx *ctx, uint64_t out[4]);
int  cpm_get_schedule(cpm_ctx *ctx, int32_t *S, int32_t *k, int32_t *phase_steps_per_mcs);
/* ---- instrumentation (Fig 3, Fig 4; not on the sweep's hot path) ----
 * Sorting observable (L69, Fig 4): out (host) [n_types*n_types], out[a*n_types+b] == out[b*n_types+a] = number of unordered
 * Moore pairs of lattice positions held by DIFFERENT cells whose types are a and b -- the interfaces Eq 1 sums J over
 * (diagonal: homotypic, off-diagonal: heterotypic).  A position outside a closed lattice counts as medium. */
int  cpm_get_interface_counts(cpm_ctx *ctx, uint64_t *out);
/* Update statistics of the schedule (L65-79, Fig 3): which positions the copy attempts of the NEXT n_mcs MCS pick as
 * targets; the lattice and the MCS counter are not touched.  Active subsections advance in lock-step (L75), so attempt a of
 * the e-th non-empty phase-step of the m-th MCS happens at tick (m E + e) k + a, E = non-empty phase-steps per MCS.
 *   freq (host) [n_freq]: (position, MCS) pairs in which the position was picked exactly j times (last bin: >= n_freq-1);
 *   wait (host) [n_wait]: consecutive picks of one position whose ticks differ by dt, binned (dt-1)/wait_bin (last bin: beyond).
 * Needs n_mcs * 2^d * S^d < 2^32 and n_freq + n_wait <= 4096 (CPM_ERR_ARG); allocates 8 bytes per site while it runs. */
int  cpm_update_statistics(cpm_ctx *ctx, uint32_t n_mcs, uint64_t *freq, int32_t n_freq, uint64_t *wait, int32_t n_wait,
                           uint32_t wait_bin);
/* The same statistics for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it): this call allocates NOTHING, on the device or the host -- no cudaMalloc, cudaFree or allocating
 * library routine.  The kernel's per-site scratch (8 bytes per site) and its histograms live in ONE file-scope
 * `static __device__` array of CPM_NOALLOC_MAX_SITES * 8 + CPM_NOALLOC_MAX_BINS * 8 bytes (8 MiB + 32 KiB) that every GPU
 * which loads the library holds until exit.  Limits: dims[0]*dims[1]*dims[2] <= CPM_NOALLOC_MAX_SITES and n_freq + n_wait
 * <= CPM_NOALLOC_MAX_BINS, else CPM_ERR_ARG with a message that names the limit (plus the limits of cpm_update_statistics).
 * freq / wait: caller-owned, host pointers (on_device = 0; the call returns after the stream has drained) or device
 * pointers on the context's device (on_device != 0; results are ready in stream order, no synchronisation).  Results are
 * bit-identical to cpm_update_statistics.  All contexts on one device share the array, which keeps the last call's
 * contents (cleared by this call where it must start at zero): calls that overlap on the GPU -- two contexts on different
 * streams -- RACE; serialise them.  cpm_noalloc_setup(device) resolves the array's device address (cudaGetSymbolAddress,
 * once per device, with that device current); the first cpm_update_statistics_noalloc on a device does it itself, so
 * call cpm_noalloc_setup before a graph capture begins.  Returns CPM_ERR_CUDA when the address cannot be had. */
#define CPM_NOALLOC_MAX_SITES (1u << 20)
#define CPM_NOALLOC_MAX_BINS  4096
int  cpm_noalloc_setup(int device);
int  cpm_update_statistics_noalloc(cpm_ctx *ctx, uint32_t n_mcs, uint64_t *freq, int32_t n_freq, uint64_t *wait, int32_t n_wait,
                                   uint32_t wait_bin, int on_device);
/* Introspection for tests: host copy of the Metropolis table, thr[h] = floor(exp(-h/T) 2^32),
 * h = 1..Hmax; returns Hmax (>= 0) or a negative error; fills at most cap entries (thr[0] unused). */
int64_t cpm_get_threshold_table(cpm_ctx *ctx, uint32_t *thr, uint64_t cap);
/* Introspection: kernels launched by this context so far, and the launch geometry of the sweep
 * kernel: out = {launches, sweep_launches, warps_per_cta, smem_bytes_per_cta, uses_tma,
 * pooled (1: pooled kernel on the tiled lattice layout -- one warp per group of 8 subsections,
 * small power-of-two S; 0: one warp per subsection on the row-major layout)}. */
int  cpm_get_launch_info(cpm_ctx *ctx, uint64_t out[6]);
/* Average device time (ms) of the sweep kernel launches since the last call with reset != 0,
 * measured with CUDA events on the context's stream when timing is enabled. */
int  cpm_set_kernel_timing(cpm_ctx *ctx, int enabled);
int  cpm_get_kernel_timing(cpm_ctx *ctx, double *sweep_ms_total, uint64_t *sweep_launches, int reset);
const char *cpm_last_error(const cpm_ctx *ctx);
/* Device-side Philox4x32-10 of n (ctr[4], key[2]) pairs (host arrays) -> out[4n]; test hook that
 * runs the same device function the sweep uses. */
int  cpm_debug_philox(int device, const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n);

#ifdef __cplusplus
}
#endif
#endif
