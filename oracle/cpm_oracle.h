/*
 * cpm_oracle.h -- C interface of the CPU ORACLE of the checkerboard Cellular Potts sweep.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may load it.  It shares no source, header,
 * table generator or helper with the CUDA path under paper_2312_09317_b200/.
 *
 * What it computes and which passage each part follows is documented in cpm_oracle.cpp.
 * All pointers are HOST pointers.  Every function returns 0 on success, a negative code on
 * error (ORACLE_ERR_*); oracle_last_error() gives a message.
 */
#ifndef CPM_ORACLE_H
#define CPM_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_ctx oracle_ctx;

enum { ORACLE_OK = 0, ORACLE_ERR_ARG = -1, ORACLE_ERR_DIMS = -2, ORACLE_ERR_UNSUPPORTED = -3,
       ORACLE_ERR_STATE = -6 };
enum { ORACLE_MODE_DETERMINISTIC = 0, ORACLE_MODE_LIVE = 1 };

/* Same field order as the product's parameter block so the tests can fill both from one dict;
 * declared here independently (no shared header). */
typedef struct {
  int32_t ndim;            /* 2 or 3 */
  int32_t dims[3];         /* x fastest; dims[2] = 1 when ndim == 2 */
  int32_t neighbourhood;   /* 0 = Moore, the only one the paper uses */
  int32_t periodic[3];     /* 0 = closed: outside is immutable medium */
  int32_t n_types;         /* type 0 = medium */
  const int32_t *J;        /* n_types*n_types, symmetric */
  const int32_t *lambda_V, *target_V, *lambda_P, *target_P, *lambda_act, *max_act; /* [n_types] or NULL */
  double   T;              /* 0 = no uphill move; +inf = accept every evaluated move */
  uint64_t seed;
  int32_t  subsection;     /* S; 0 = default (8 in 2D, 4 in 3D, halved while it does not divide dims; R4) */
  int32_t  attempts_per_activation; /* k; 0 = S^d */
  int32_t  mode;
  uint32_t max_cells;      /* cell IDs are 0..max_cells */
  int32_t  device;         /* ignored */
  void    *stream;         /* ignored */
  /* vector terms (Eq 4-7; readings S21, S22); NULL / 0 = off */
  const int32_t *lambda_pers; /* [n_types] persistence strength, Eq 5 */
  const double  *mu_pers;     /* [n_types] directional memory mu in [0,1], Eq 6 */
  int32_t  dt_pers;           /* look-back in MCS, Eq 6; >= 1 when any lambda_pers != 0 */
  const int32_t *lambda_chem; /* [n_types] chemotaxis strength, Eq 4 */
  int32_t  unwrap_centroids;  /* != 0: coordinate sums follow the cell through periodic borders (L297; reading S23) */
} oracle_params;

int  oracle_create(const oracle_params *p, oracle_ctx **out);
int  oracle_destroy(oracle_ctx *c);
int  oracle_set_lattice(oracle_ctx *c, const uint32_t *ids, const uint8_t *frozen, const uint8_t *cell_type);
int  oracle_set_act(oracle_ctx *c, const float *act);
int  oracle_set_mcs(oracle_ctx *c, uint32_t mcs);
int  oracle_step(oracle_ctx *c, uint32_t n_mcs);
int  oracle_get_lattice(oracle_ctx *c, uint32_t *ids);
int  oracle_get_act(oracle_ctx *c, float *act);
int  oracle_get_cell_stats(oracle_ctx *c, uint32_t *volume, uint32_t *perimeter,
                           uint64_t *sum_x, uint64_t *sum_y, uint64_t *sum_z);
int  oracle_get_counters(oracle_ctx *c, uint64_t out[4]); /* attempts, evaluated, accepted, mcs */
int  oracle_get_schedule(oracle_ctx *c, int32_t *S, int32_t *k, int32_t *phase_steps_per_mcs);
const char *oracle_last_error(const oracle_ctx *c);

/* ---- hooks used only by the pins in tests/ ---- */
/* order in which the subsections of one phase-step are visited: 0 forward, 1 reversed,
 * 2 pseudo-random (from order_seed).  The result must not depend on it. */
int  oracle_set_visit_order(oracle_ctx *c, int32_t order, uint64_t order_seed);
/* Incremental dH of "copy the state of neighbour nb of site t into t", against the current
 * lattice and LIVE tallies.  status: 0 = early-out (same cell / frozen), 1 = evaluated,
 * 2 = refused by the extinction rule.  dH_hamiltonian excludes the Act bias, dH_act is the
 * integer Act bias that is SUBTRACTED from it. */
int  oracle_probe(oracle_ctx *c, uint64_t t_index, int32_t nb, int32_t *status,
                  int64_t *dH_hamiltonian, int64_t *dH_act);
/* Apply that copy unconditionally (same commit code as the sweep). */
int  oracle_force_copy(oracle_ctx *c, uint64_t t_index, int32_t nb);
/* Per-attempt trace of the next oracle_step calls: rec[6] = {t_index, nb, status, dH, accepted, u32}
 * appended to buf (up to cap records); pass NULL to stop. */
int  oracle_set_trace(oracle_ctx *c, int64_t *buf, uint64_t cap, uint64_t *count);
/* ---- vector terms (Eq 4-7) ---- */
/* field[N][ndim] (component fastest), components in [-1,1] (the paper's fields are unit vectors, L240) */
int  oracle_set_chemotaxis_field(oracle_ctx *c, const float *field);
/* p[(max_cells+1)][3]: persistence direction per cell (unit or zero vectors); default 0 after set_lattice */
int  oracle_set_persistence(oracle_ctx *c, const double *p);
int  oracle_get_persistence(oracle_ctx *c, double *p);
/* xyz[(max_cells+1)][3]: centroid of every cell, Eq 10 (coordinate sums / volume) */
int  oracle_get_centroids(oracle_ctx *c, double *xyz);
/* the integer chemotaxis + persistence bias that is SUBTRACTED from dH for this copy (0 for early-outs) */
int  oracle_probe_dir(oracle_ctx *c, uint64_t t_index, int32_t nb, int64_t *dH_dir);
/* Q14 unit vectors of the copy direction (source -> target) per neighbour index: out[nb*3 + {0,1,2}] */
int  oracle_direction_table(int32_t ndim, int64_t *out);
/* ---- instrumentation ---- */
/* out[n_types*n_types]: unordered Moore pairs of positions held by different cells, by the two cells' types (symmetric) */
int  oracle_get_interface_counts(oracle_ctx *c, uint64_t *out);
/* target-pick statistics of the next n_mcs MCS of the schedule (lattice untouched): see cpm_oracle.cpp */
int  oracle_update_statistics(oracle_ctx *c, uint32_t n_mcs, uint64_t *freq, int32_t n_freq, uint64_t *wait, int32_t n_wait,
                              uint32_t bin);
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* proposal decode of one 32-bit word: local site index l in [0,S^d) and neighbour index nb */
void oracle_decode_proposal(uint32_t w, uint32_t sites, uint32_t n_nb, uint32_t *l, uint32_t *nb);
/* acceptance table: returns Hmax; fills thr[1..min(Hmax,cap-1)] (thr[0] unused = 0xffffffff) */
int64_t oracle_threshold_table(double T, uint32_t *thr, uint64_t cap);
/* fixed-point geometric mean in Q16 of n activity values (0..255) */
int64_t oracle_gm_q16(const int32_t *act, int32_t n);
/* neighbour offset table in the order the proposal index nb uses: out[nb*3 + {0,1,2}] = dx,dy,dz */
int  oracle_neighbour_offsets(int32_t ndim, int32_t *out);

#ifdef __cplusplus
}
#endif
#endif
