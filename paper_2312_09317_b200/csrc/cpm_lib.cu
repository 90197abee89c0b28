// cpm_lib.cu -- host side of the C ABI declared in include/cpm.h: parameter validation, the
// checkerboard phase scheduler (a1), host-built tables (Metropolis thresholds, Act log/exp),
// device state, TMA descriptors, kernel launches.  No compute happens on the host; without a
// usable CUDA device every entry point that needs one returns CPM_ERR_CUDA.
#include "../../include/cpm.h"
#include "cpm_device.cuh"
#include "cpm_pool_kernel.cuh"
#include "cpm_stats_kernels.cuh"

#include <nvtx3/nvToolsExt.h>   // header-only: ranges around the API calls for nsys / ncu timelines

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

using namespace cpm;

namespace {
struct NvtxRange {   // RAII range on the calling thread
  explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};
}  // namespace

typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

typedef void (*SweepFn)(const CUtensorMap, const SweepParams);
typedef void (*ThreadFn)(const SweepParams);

constexpr int PIPE_SLABS = 8;                   // slabs of a pipelined host transfer
constexpr long long PIPE_MIN_SITES = 1ll << 24; // lattices below this go in one piece

struct cpm_ctx {
  int d = 0, device = 0;
  cudaStream_t stream = nullptr;
  int dim[3] = {1, 1, 1};
  int per[3] = {0, 0, 0};
  int nT = 0;
  double T = 0;
  uint64_t seed = 0;
  int mode = 0;
  uint32_t max_cells = 0;
  long long N = 0;
  int S = 0, sites = 0, k = 0, R = 0, nNb = 0;
  int nsub[3] = {1, 1, 1};
  bool act_enabled = false;
  bool have_lattice = false;
  int nsets = 1;
  int wpc = 4;           // warps per CTA
  size_t cta_smem = 0;
  bool use_tma = true;
  SweepFn fn = nullptr;
  bool pooled = false;          // pooled kernel on the tiled layout (small power-of-two S), else one warp per subsection
  ThreadFn tfn = nullptr;
  unsigned long long n_act_col[8] = {0}, grp_col[8] = {0};   // active subsections / groups of 8 per colour
  size_t tile_words = 0;
  SweepParams sp;        // template of the launch parameters
  CUtensorMap tm_lat;
  uint32_t *tl_tiles() const { return sp.tl.tiles; }

  // device state
  uint32_t *lat = nullptr;
  uint8_t *act = nullptr;
  unsigned long long *liveVP = nullptr, *snapVP = nullptr, *sumx = nullptr, *sumy = nullptr, *sumz = nullptr;
  unsigned long long *counters = nullptr;
  int *error_flag = nullptr;
  uint32_t *mcs_dev = nullptr;
  int32_t *J_dev = nullptr, *D_dev = nullptr, *log_dev = nullptr, *exp_dev = nullptr;
  TypeParams *types_dev = nullptr;
  int4 *lane_tab_dev = nullptr;
  unsigned char *img_dev = nullptr;   // pooled kernel: types + adhesion table as one shared-memory image
  size_t img_bytes = 0;
  std::vector<int32_t> Dtab;
  uint32_t *thr_dev = nullptr;
  uint32_t *ovf_keys = nullptr;
  unsigned long long *ovf_dvp = nullptr;
  int *ovf_count = nullptr;
  // vector terms (Eq 4-7)
  bool pers_on = false, chem_on = false;
  int dt_pers = 0;
  int2 *vec_types_dev = nullptr;
  double *mu_dev = nullptr, *phat = nullptr, *ring = nullptr;
  short4 *pq = nullptr, *chem = nullptr;
  uint8_t *ctype_dev = nullptr;
  uint32_t *pers_n = nullptr;
  bool unwrap = false;                       // periodic centroid tracking (reading S23)
  int *anc = nullptr;
  unsigned long long *first_site = nullptr;
  // staging buffers for host-pointer I/O, kept between calls
  void *stage_a = nullptr, *stage_b = nullptr, *stage_c = nullptr;
  size_t stage_a_cap = 0, stage_b_cap = 0, stage_c_cap = 0;
  // host <-> device transfers of a large lattice run slab by slab on a stream of their own, overlapped with the pack /
  // recount / unpack kernels of the slabs that have arrived (pipe_plan)
  cudaStream_t io_stream = nullptr;
  cudaEvent_t io_ev[PIPE_SLABS + 2] = {};
  long long pipe_min_sites = PIPE_MIN_SITES;   // the environment variable CPM_PIPE_MIN_SITES overrides it (tests)

  std::vector<uint32_t> thr;
  std::vector<TypeParams> types;   // host copy of the per-type records
  int act_cap = 0;                 // largest Act value the field can hold right now
  long long Hmax = 0;
  uint32_t mcs_host = 0;      // mirror of the device counter
  uint64_t mcs_run = 0;       // MCS executed by this context (for the attempts counter)
  uint64_t launches = 0, sweep_launches = 0;

  // one CUDA graph = one MCS (every launch parameter but the MCS counter, which the kernels read from device
  // memory, repeats from MCS to MCS); captured on a stream of the context's own, launched on the caller's
  bool use_graph = true;
  cudaStream_t cap_stream = nullptr;
  cudaGraphExec_t mcs_graph = nullptr;
  uint64_t graph_launches = 0, graph_sweeps = 0;   // kernels / sweep kernels in one MCS

  bool timing = false;
  std::vector<cudaEvent_t> ev_pool;
  size_t ev_used = 0;

  std::string err;
};

namespace {

int fail(cpm_ctx *c, int code, const std::string &msg) {
  if (c) c->err = msg;
  return code;
}
#define CK(call)                                                                                      \
  do {                                                                                                \
    cudaError_t e_ = (call);                                                                          \
    if (e_ != cudaSuccess)                                                                            \
      return fail(c, e_ == cudaErrorMemoryAllocation ? CPM_ERR_OOM : CPM_ERR_CUDA,                    \
                  std::string(#call) + ": " + cudaGetErrorString(e_));                                \
  } while (0)

template <int DIM, bool ACT, bool LIVE>
SweepFn pick_sets(int nsets) {
  return nsets == 1 ? (SweepFn)sweep_kernel<DIM, ACT, LIVE, 1> : (SweepFn)sweep_kernel<DIM, ACT, LIVE, 4>;
}
template <int DIM>
SweepFn pick_flags(bool act, bool live, int nsets) {
  if (act) return live ? pick_sets<DIM, true, true>(nsets) : pick_sets<DIM, true, false>(nsets);
  return live ? pick_sets<DIM, false, true>(nsets) : pick_sets<DIM, false, false>(nsets);
}
// pre-generated specialised kernels per extension set
SweepFn pick_kernel(int d, bool act, bool live, int nsets) {
  return d == 2 ? pick_flags<2>(act, live, nsets) : pick_flags<3>(act, live, nsets);
}

template <int DIM, int S, bool VEC>
ThreadFn pick_pool_flags(bool act, bool live, int nT, size_t *smem) {
  *smem = PSmem<DIM, S>::bytes(nT);
  if (act) return live ? (ThreadFn)sweep_pool_kernel<DIM, S, true, true, VEC> : (ThreadFn)sweep_pool_kernel<DIM, S, true, false, VEC>;
  return live ? (ThreadFn)sweep_pool_kernel<DIM, S, false, true, VEC> : (ThreadFn)sweep_pool_kernel<DIM, S, false, false, VEC>;
}
template <int DIM, int S>
ThreadFn pick_pool_vec(bool act, bool live, bool vec, int nT, size_t *smem) {
  return vec ? pick_pool_flags<DIM, S, true>(act, live, nT, smem) : pick_pool_flags<DIM, S, false>(act, live, nT, smem);
}
// pooled kernel: 3D S = 2, 4, 8; 2D S = 2, 4, 8, 16; one specialisation per extension set (L282)
ThreadFn pick_pool_kernel(int d, int S, bool act, bool live, bool vec, int nT, size_t *smem) {
  if (d == 3) {
    if (S == 2) return pick_pool_vec<3, 2>(act, live, vec, nT, smem);
    if (S == 4) return pick_pool_vec<3, 4>(act, live, vec, nT, smem);
    if (S == 8) return pick_pool_vec<3, 8>(act, live, vec, nT, smem);
    return nullptr;
  }
  if (S == 2) return pick_pool_vec<2, 2>(act, live, vec, nT, smem);
  if (S == 4) return pick_pool_vec<2, 4>(act, live, vec, nT, smem);
  if (S == 8) return pick_pool_vec<2, 8>(act, live, vec, nT, smem);
  if (S == 16) return pick_pool_vec<2, 16>(act, live, vec, nT, smem);
  return nullptr;
}

int grid_for(long long n, int block = 256) {
  long long g = (n + block - 1) / block;
  const long long cap = 148LL * 32;  // grid-stride loops: a few waves over the 148 SMs
  if (g > cap) g = cap;
  if (g < 1) g = 1;
  return (int)g;
}

int roundup(int v, int m) { return (v + m - 1) / m * m; }

// a device pointer to n elements of T holding the caller's data: the caller's own pointer when it is
// already on the device, otherwise one of the context's staging buffers (kept between calls)
cudaError_t stage_reserve(void **buf, size_t *cap, size_t bytes) {
  if (*cap >= bytes) return cudaSuccess;
  if (*buf) { cudaFree(*buf); *buf = nullptr; *cap = 0; }
  cudaError_t e = cudaMalloc(buf, bytes);
  if (e == cudaSuccess) *cap = bytes;
  return e;
}
template <class T>
cudaError_t stage_in(T **out, void **buf, size_t *cap, const T *src, size_t n, int on_device, cudaStream_t st) {
  *out = nullptr;
  if (!src) return cudaSuccess;
  if (on_device) { *out = const_cast<T *>(src); return cudaSuccess; }
  cudaError_t e = stage_reserve(buf, cap, n * sizeof(T));
  if (e != cudaSuccess) return e;
  *out = reinterpret_cast<T *>(*buf);
  return cudaMemcpyAsync(*buf, src, n * sizeof(T), cudaMemcpyHostToDevice, st);
}
template <class T>
cudaError_t stage_out_begin(T **out, void **buf, size_t *cap, T *dst, size_t n, int on_device) {
  *out = nullptr;
  if (!dst) return cudaSuccess;
  if (on_device) { *out = dst; return cudaSuccess; }
  cudaError_t e = stage_reserve(buf, cap, n * sizeof(T));
  if (e == cudaSuccess) *out = reinterpret_cast<T *>(*buf);
  return e;
}
template <class T>
cudaError_t stage_out_end(T *staged, T *dst, size_t n, int on_device, cudaStream_t st) {
  if (!dst || on_device) return cudaSuccess;
  return cudaMemcpyAsync(dst, staged, n * sizeof(T), cudaMemcpyDeviceToHost, st);
}

int make_tensor_map(cpm_ctx *c, CUtensorMap *tm, CUtensorMapDataType dt, int elem, void *base, long long pitch_elems,
                    int bx) {
  void *fnp = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fnp, cudaEnableDefault, &qres);
  if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fnp)
    return fail(c, CPM_ERR_CUDA, "cuTensorMapEncodeTiled entry point not available");
  PFN_encodeTiled enc = (PFN_encodeTiled)fnp;
  const cuuint32_t rank = (cuuint32_t)c->d;
  cuuint64_t gdim[3] = {(cuuint64_t)c->dim[0], (cuuint64_t)c->dim[1], (cuuint64_t)c->dim[2]};
  cuuint64_t gstr[2] = {(cuuint64_t)pitch_elems * elem, (cuuint64_t)pitch_elems * elem * c->dim[1]};
  cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)c->sp.TY, (cuuint32_t)c->sp.TZ};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(tm, dt, rank, base, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(c, CPM_ERR_CUDA, "cuTensorMapEncodeTiled failed with code " + std::to_string((int)r));
  return CPM_OK;
}

int check_device_flag(cpm_ctx *c) {
  int flag = 0;
  CK(cudaMemcpyAsync(&flag, c->error_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  if (flag & 1) return fail(c, CPM_ERR_UNSUPPORTED, "a subsection changed more distinct cells in one activation than its own-delta table holds");
  if (flag & 2) return fail(c, CPM_ERR_ARG, "cell id above max_cells in the lattice");
  if (flag & 4) return fail(c, CPM_ERR_ARG, "Act values must be integers in [0,255]");
  if (flag & 8) return fail(c, CPM_ERR_ARG, "vector components must lie in [-1,1]");
  return CPM_OK;
}

// (Re)build the bound of one side of the Act bias and upload the per-type records.  The pooled kernel works a
// geometric mean out only when the bias can change the outcome: a side lies in [0, lamA * GM / maxA] and GM <= the
// largest Act value in the field: the largest Max_act after cpm_set_lattice (the field starts at 0 and only ever
// receives Max_act values, L255), 255 once cpm_set_act has loaded caller-chosen values.  The slack covers the
// rounding of the fixed-point mean (relative 2^-10 at most) and of the final shift.
int upload_types(cpm_ctx *c, int user_values) {
  int cap_val = 0;
  for (int i = 0; i < c->nT; ++i) cap_val = std::max(cap_val, (int)c->types[i].maxA);
  if (user_values) cap_val = 255;
  c->act_cap = cap_val;
  for (int i = 0; i < c->nT; ++i) {
    TypeParams &t = c->types[i];
    long long cap = 0;
    if (t.lamA != 0) { const long long v = ((long long)t.lamA * cap_val) / t.maxA; cap = v + v / 1024 + 2; }
    t.cap = (int32_t)std::min<long long>(cap, 0x3fffffffLL);
  }
  cudaError_t e = cudaMemcpyAsync(c->types_dev, c->types.data(), c->types.size() * sizeof(TypeParams), cudaMemcpyHostToDevice, c->stream);
  std::vector<unsigned char> img;
  if (e == cudaSuccess && c->img_dev) {   // the same records, followed by the adhesion table, as the pooled kernel's shared memory holds them
    img.assign(c->img_bytes, 0);
    memcpy(img.data(), c->types.data(), c->types.size() * sizeof(TypeParams));
    memcpy(img.data() + c->types.size() * sizeof(TypeParams), c->Dtab.data(), c->Dtab.size() * 4);
    e = cudaMemcpyAsync(c->img_dev, img.data(), c->img_bytes, cudaMemcpyHostToDevice, c->stream);
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  return e == cudaSuccess ? CPM_OK : fail(c, CPM_ERR_CUDA, cudaGetErrorString(e));
}

void free_all(cpm_ctx *c) {
  cudaFree(c->lat); cudaFree(c->act); cudaFree(c->liveVP); cudaFree(c->snapVP); cudaFree(c->sumx); cudaFree(c->sumy);
  cudaFree(c->sumz); cudaFree(c->counters); cudaFree(c->error_flag); cudaFree(c->mcs_dev); cudaFree(c->J_dev); cudaFree(c->D_dev);
  cudaFree(c->log_dev); cudaFree(c->exp_dev); cudaFree(c->types_dev); cudaFree(c->thr_dev);
  cudaFree(c->tl_tiles()); cudaFree(c->ovf_keys); cudaFree(c->ovf_dvp); cudaFree(c->ovf_count);
  cudaFree(c->stage_a); cudaFree(c->stage_b); cudaFree(c->stage_c);
  cudaFree(c->vec_types_dev); cudaFree(c->mu_dev); cudaFree(c->phat); cudaFree(c->ring); cudaFree(c->pq); cudaFree(c->chem);
  cudaFree(c->lane_tab_dev); cudaFree(c->img_dev); cudaFree(c->ctype_dev); cudaFree(c->pers_n); cudaFree(c->anc); cudaFree(c->first_site);
  for (auto e : c->ev_pool) cudaEventDestroy(e);
  if (c->mcs_graph) cudaGraphExecDestroy(c->mcs_graph);
  if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
  for (auto e : c->io_ev) if (e) cudaEventDestroy(e);
  if (c->io_stream) cudaStreamDestroy(c->io_stream);
}

// the transfer stream and its events, made on first use
cudaError_t pipe_ready(cpm_ctx *c) {
  if (c->io_stream) return cudaSuccess;
  cudaError_t e = cudaStreamCreateWithFlags(&c->io_stream, cudaStreamNonBlocking);
  for (int i = 0; e == cudaSuccess && i < PIPE_SLABS + 2; ++i) e = cudaEventCreateWithFlags(&c->io_ev[i], cudaEventDisableTiming);
  return e;
}

// Slabs of the slowest axis for the pipelined cpm_set_lattice on the tiled layout: slab i = the planes of the pairs of
// subsection layers [a[i], a[i+1]).  A chain with slow index a of either colour bit reads the planes 2 S a - 1 ..
// 2 S (a + 1): its own slab plus one plane of each neighbour slab.  False: the lattice goes in one piece.
bool pipe_plan(const cpm_ctx *c, int a[PIPE_SLABS + 1]) {
  if (!c->pooled || c->unwrap || c->N < c->pipe_min_sites) return false;
  const int ax = c->d - 1;
  const int pairs = (c->nsub[ax] + 1) / 2;
  if (pairs < 2 * PIPE_SLABS) return false;
  // the slabs shrink towards the end: what is left to do when the last byte has arrived is the last two slabs' work
  static const double upto[PIPE_SLABS + 1] = {0.0, 0.2, 0.4, 0.6, 0.75, 0.87, 0.94, 0.98, 1.0};
  for (int i = 0; i <= PIPE_SLABS; ++i) a[i] = (int)(upto[i] * pairs + 0.5);
  for (int i = 1; i <= PIPE_SLABS; ++i) a[i] = std::max(a[i], a[i - 1] + 1);           // no empty slab (pairs >= 2 PIPE_SLABS)
  a[PIPE_SLABS] = pairs;
  for (int i = PIPE_SLABS - 1; i >= 0; --i) a[i] = std::min(a[i], a[i + 1] - 1);
  for (int col = 0; col < (1 << c->d); ++col) {
    if (c->n_act_col[col] == 0) continue;
    const unsigned long long slow = (unsigned long long)c->sp.tl.nact[col][ax];
    if (slow == 0 || c->n_act_col[col] / slow < (unsigned long long)PK_GC) return false;   // a group never reaches back beyond the previous slab
  }
  return true;
}

// a1: the work of ONE Monte Carlo step on stream st: R repetitions x 2^d colours of the sweep kernel, the
// snapshot refresh after each, then the Act decay (which also advances the device MCS counter)
int enqueue_mcs(cpm_ctx *c, cudaStream_t st, bool timed) {
  const int ncol = 1 << c->d;
  const size_t ncell = (size_t)c->max_cells + 1;
  for (int rep = 0; rep < c->R; ++rep)
    for (int col = 0; col < ncol; ++col) {
      SweepParams sp = c->sp;
      sp.p = (uint32_t)(rep * ncol + col);
      unsigned long long n_active = 1;
      for (int a = 0; a < 3; ++a) {
        sp.col[a] = (a < c->d) ? ((col >> a) & 1) : 0;
        sp.nact[a] = (a < c->d) ? (c->nsub[a] - sp.col[a] + 1) / 2 : 1;
        n_active *= (unsigned long long)sp.nact[a];
      }
      if (n_active == 0) continue;  // this colour does not occur (a single subsection along an axis)
      sp.n_active = n_active;
      for (int a = 0; a < 2; ++a) {   // exact reciprocal for dividends below 2^31 (Granlund-Montgomery): m = ceil(2^(31+l) / d), l = ceil(log2 d)
        const uint32_t dv = (uint32_t)sp.nact[a];
        int l = 0;
        while ((1u << l) < dv) ++l;
        if (dv <= 1) { sp.nact_mul[a] = 0; sp.nact_shr[a] = 0; }
        else {
          const unsigned long long num = 1ull << (31 + l);
          sp.nact_mul[a] = (uint32_t)((num + dv - 1) / dv);   // < 2^32 because d > 2^(l-1)
          sp.nact_shr[a] = (uint32_t)(l - 1);                  // umulhi takes 32 of the 31 + l bits
        }
      }
      sp.grp_base = sp.tl.base[col];
      const unsigned long long per_cta = c->pooled ? (unsigned long long)PK_GC : (unsigned long long)c->wpc;
      const unsigned long long grid = (n_active + per_cta - 1) / per_cta;
      if (grid > 0x7fffffffULL || (c->pooled && n_active > 0x7fffffffULL)) return fail(c, CPM_ERR_UNSUPPORTED, "too many subsections for one launch");
      cudaEvent_t e0 = nullptr, e1 = nullptr;
      if (timed) {
        while (c->ev_pool.size() < c->ev_used + 2) { cudaEvent_t e; CK(cudaEventCreate(&e)); c->ev_pool.push_back(e); }
        e0 = c->ev_pool[c->ev_used++]; e1 = c->ev_pool[c->ev_used++];
        CK(cudaEventRecord(e0, st));
      }
      if (c->pooled) c->tfn<<<(unsigned)grid, PK_THREADS, c->cta_smem, st>>>(sp);
      else c->fn<<<(unsigned)grid, 32 * c->wpc, c->cta_smem, st>>>(c->tm_lat, sp);
      if (timed) CK(cudaEventRecord(e1, st));
      c->launches++; c->sweep_launches++;
      // deterministic mode: the next phase-step reads the values as of its own start
      if (c->snapVP) {
        const long long n_pairs = (long long)((ncell + 1) / 2);   // the arrays are allocated in whole 16-byte pairs
        snapshot_kernel<<<grid_for(n_pairs), 256, 0, st>>>((const ulonglong2 *)c->liveVP, (ulonglong2 *)c->snapVP, n_pairs, c->ovf_count);
        c->launches++;
      }
    }
  if (c->unwrap) {   // L297: centroids back inside the lattice on periodic axes, anchors follow
    const long long ncl = (long long)ncell;
    centroid_normalise_kernel<<<(unsigned)((ncl + 255) / 256), 256, 0, st>>>(ncl, c->liveVP, c->sumx, c->sumy, c->sumz, c->anc, c->dim[0],
                                                                           c->dim[1], c->dim[2], c->per[0], c->per[1], c->per[2]);
    c->launches++;
  }
  if (c->pers_on) {   // Eq 6-7: every cell's persistence direction from its centroid now and dt MCS ago
    const long long ncl = (long long)ncell;
    persistence_update_kernel<<<(unsigned)((ncl + 255) / 256), 256, 0, st>>>(ncl, c->dt_pers + 1, c->liveVP, c->sumx, c->sumy, c->sumz,
                                                                           c->ctype_dev, c->mu_dev, c->phat, c->pq, c->ring, c->pers_n,
                                                                           (c->unwrap && c->per[0]) ? c->dim[0] : 0,
                                                                           (c->unwrap && c->per[1]) ? c->dim[1] : 0,
                                                                           (c->unwrap && c->per[2]) ? c->dim[2] : 0);
    c->launches++;
  }
  if (c->act_enabled) {
    const long long n_vec = c->sp.apitch * c->dim[1] * c->dim[2] / 16;
    act_decay_kernel<<<grid_for(n_vec), 256, 0, st>>>((uint4 *)c->act, n_vec, c->mcs_dev, c->pers_n);
  } else {
    mcs_increment_kernel<<<1, 1, 0, st>>>(c->mcs_dev, c->pers_n);
  }
  c->launches++;
  return CPM_OK;
}

// capture one MCS into a graph (once per context)
int build_mcs_graph(cpm_ctx *c) {
  if (!c->cap_stream) CK(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
  const uint64_t l0 = c->launches, s0 = c->sweep_launches;
  CK(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
  int rc = enqueue_mcs(c, c->cap_stream, false);
  cudaGraph_t g = nullptr;
  cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
  c->graph_launches = c->launches - l0; c->graph_sweeps = c->sweep_launches - s0;
  c->launches = l0; c->sweep_launches = s0;   // nothing ran yet
  if (rc != CPM_OK) { if (g) cudaGraphDestroy(g); return rc; }
  if (e != cudaSuccess) return fail(c, CPM_ERR_CUDA, std::string("stream capture: ") + cudaGetErrorString(e));
  e = cudaGraphInstantiate(&c->mcs_graph, g, 0);
  cudaGraphDestroy(g);
  if (e != cudaSuccess) { c->mcs_graph = nullptr; return fail(c, CPM_ERR_CUDA, std::string("graph instantiate: ") + cudaGetErrorString(e)); }
  return CPM_OK;
}

}  // namespace

extern "C" {

// every entry point catches allocation failures of the host containers: nothing throws through the C ABI
#define CPM_GUARD_BEGIN try {
#define CPM_GUARD_END(ctx)                                                     \
  } catch (const std::bad_alloc &) { return fail(ctx, CPM_ERR_OOM, "host allocation failed"); } \
  catch (...) { return fail(ctx, CPM_ERR_STATE, "unexpected host exception"); }

static int create_impl(const cpm_params *p, cpm_ctx **out) {
  if (!p || !out) return CPM_ERR_ARG;
  *out = nullptr;
  if (p->ndim != 2 && p->ndim != 3) return CPM_ERR_DIMS;
  if (p->neighbourhood != CPM_MOORE) return CPM_ERR_UNSUPPORTED;
  if (p->n_types < 1 || p->n_types > 127 || !p->J) return CPM_ERR_ARG;
  if (!(p->T >= 0)) return CPM_ERR_ARG;
  // the Metropolis table has floor(T 32 ln 2) + 1 entries: a finite T above 2^20 is outside this build
  if (!std::isinf(p->T) && p->T > 1048576.0) return CPM_ERR_UNSUPPORTED;
  if (p->mode != CPM_MODE_DETERMINISTIC && p->mode != CPM_MODE_LIVE_ATOMICS) return CPM_ERR_ARG;
  if (p->max_cells >= (1u << 24)) return CPM_ERR_UNSUPPORTED;
  const int d = p->ndim, nT = p->n_types;
  for (int a = 0; a < d; ++a) if (p->dims[a] < 1) return CPM_ERR_DIMS;
  for (int i = 0; i < nT; ++i)
    for (int j = 0; j < nT; ++j) {
      if (p->J[i * nT + j] != p->J[j * nT + i]) return CPM_ERR_ARG;
      if (p->J[i * nT + j] > (1 << 24) || p->J[i * nT + j] < -(1 << 24)) return CPM_ERR_ARG;
    }
  bool any_act = false;
  for (int i = 0; i < nT; ++i) {
    if (p->max_act && (p->max_act[i] < 0 || p->max_act[i] > 255)) return CPM_ERR_ARG;
    if (p->lambda_act && p->lambda_act[i] < 0) return CPM_ERR_ARG;
    // ranges that keep the 32x32->64 products and the int32 sums of the dH assembly exact
    if (p->lambda_P && (p->lambda_P[i] > (1 << 24) || p->lambda_P[i] < -(1 << 24))) return CPM_ERR_ARG;
    if (p->lambda_V && (p->lambda_V[i] > (1 << 30) || p->lambda_V[i] < -(1 << 30))) return CPM_ERR_ARG;
    if (p->max_act && p->max_act[i] != 0) any_act = true;
  }
  bool pers_on = false, chem_on = false;
  for (int i = 0; i < nT; ++i) {
    if (p->lambda_pers && (p->lambda_pers[i] > (1 << 24) || p->lambda_pers[i] < -(1 << 24))) return CPM_ERR_ARG;
    if (p->lambda_chem && (p->lambda_chem[i] > (1 << 24) || p->lambda_chem[i] < -(1 << 24))) return CPM_ERR_ARG;
    if (p->mu_pers && !(p->mu_pers[i] >= 0.0 && p->mu_pers[i] <= 1.0)) return CPM_ERR_ARG;
    if (p->lambda_pers && p->lambda_pers[i] != 0) pers_on = true;
    if (p->lambda_chem && p->lambda_chem[i] != 0) chem_on = true;
  }
  if (p->dt_pers < 0 || p->dt_pers > 4096 || (pers_on && p->dt_pers < 1)) return CPM_ERR_ARG;

  // ---- checkerboard scheduler (a1): subsection edge S, attempts per activation k ----
  int S = p->subsection;
  if (S == 0) {
    S = (d == 2) ? 8 : 4;   // small subsections: many independent chains per warp (R4)
    auto divides = [&](int s) { for (int a = 0; a < d; ++a) if (p->dims[a] % s) return false; return true; };
    while (S > 2 && !divides(S)) S /= 2;
  }
  if (S < 2) return CPM_ERR_DIMS;
  long long sites = 1;
  for (int a = 0; a < d; ++a) {
    if (p->dims[a] % S) return CPM_ERR_DIMS;
    if (p->periodic[a] && ((p->dims[a] / S) & 1)) return CPM_ERR_DIMS;
    sites *= S;
  }
  if (sites > (1 << 24)) return CPM_ERR_UNSUPPORTED;
  {   // the kernels index lattice rows (y + Y z) with 32 bits
    long long nrows = 1;
    for (int a = 1; a < d; ++a) nrows *= p->dims[a];
    if (nrows >= (1LL << 31)) return CPM_ERR_UNSUPPORTED;
  }
  long long k = p->attempts_per_activation ? p->attempts_per_activation : sites;
  if (k < 1 || sites % k) return CPM_ERR_ARG;

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1 || p->device < 0 || p->device >= ndev) return CPM_ERR_CUDA;
  if (cudaSetDevice(p->device) != cudaSuccess) return CPM_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, p->device) != cudaSuccess) return CPM_ERR_CUDA;
  if (prop.major < 10) return CPM_ERR_CUDA;  // kernels are built for sm_100a only

  cpm_ctx *c = new cpm_ctx();
  if (const char *e = std::getenv("CPM_PIPE_MIN_SITES")) c->pipe_min_sites = std::atoll(e);
  c->d = d; c->device = p->device; c->stream = (cudaStream_t)p->stream;
  c->nT = nT; c->T = p->T; c->seed = p->seed; c->mode = p->mode; c->max_cells = p->max_cells;
  c->N = 1;
  for (int a = 0; a < 3; ++a) {
    c->dim[a] = (a < d) ? p->dims[a] : 1;
    c->per[a] = (a < d) ? (p->periodic[a] != 0) : 0;
    c->nsub[a] = (a < d) ? c->dim[a] / S : 1;
    c->N *= c->dim[a];
  }
  c->S = S; c->sites = (int)sites; c->k = (int)k; c->R = (int)(sites / k);
  c->nNb = (d == 2) ? 8 : 26;
  c->act_enabled = any_act;
  c->pers_on = pers_on; c->chem_on = chem_on; c->dt_pers = p->dt_pers;
  c->unwrap = p->unwrap_centroids != 0 && (c->per[0] || c->per[1] || c->per[2]);
  c->use_graph = !(p->flags & CPM_FLAG_NO_GRAPH);
  c->nsets = (sites <= 512) ? 1 : 4;
  // TMA wants the tile's first word at a 16-byte boundary: x0-4 with x0 a multiple of S
  c->use_tma = !(p->flags & CPM_FLAG_NO_TMA) && (S % 4 == 0);
  size_t pool_smem = 0;
  c->tfn = (nT <= 8 && !(p->flags & CPM_FLAG_WARP_KERNEL))
               ? pick_pool_kernel(d, S, c->act_enabled, p->mode == CPM_MODE_LIVE_ATOMICS, pers_on || chem_on || c->unwrap, nT, &pool_smem) : nullptr;
  c->pooled = c->tfn != nullptr;
  if (c->pooled) c->use_tma = true;   // one bulk copy per group of 8 tiles

  // ---- tile geometry (a2) ----
  SweepParams &sp = c->sp;
  memset(&sp, 0, sizeof(sp));
  sp.h = c->act_enabled ? 2 : 1;
  sp.hx = 4;
  sp.TX = roundup(S + 2 * sp.hx, 4);
  sp.TY = S + 2 * sp.h;
  sp.TZ = (d == 3) ? S + 2 * sp.h : 1;
  sp.AX = sp.TX;
  sp.tile_bytes = sp.TX * sp.TY * sp.TZ * 4;
  sp.act_tile_bytes = c->act_enabled ? sp.AX * sp.TY * sp.TZ : 0;
  sp.warp_smem_bytes = roundup(sp.tile_bytes, 128) + roundup(sp.act_tile_bytes, 128);
  if (!c->pooled && ((long long)sp.TX * sp.TY * sp.TZ > 65535 || sp.TX > 256 || sp.TY > 256 || sp.AX > 256)) {
    delete c;
    return CPM_ERR_UNSUPPORTED;
  }
  const size_t smem_cap = 227 * 1024;
  c->wpc = 4;
  while (c->wpc > 1 && (size_t)c->wpc * sp.warp_smem_bytes + 64 > 100 * 1024) c->wpc /= 2;
  if (c->wpc > 8) c->wpc = 8;  // 64 B of mbarriers
  // per CTA: warp tiles, 64 B of mbarriers, neighbour-offset tables (256 B), type records, J
  const size_t table_bytes = 64 + 256 + (size_t)(nT + 1) * sizeof(TypeParams) + (size_t)nT * nT * 4;
  c->cta_smem = (size_t)c->wpc * sp.warp_smem_bytes + table_bytes;
  if (c->pooled) { c->wpc = PK_THREADS / 32; c->cta_smem = pool_smem; }
  if (c->cta_smem > smem_cap) { delete c; return CPM_ERR_UNSUPPORTED; }

  // ---- host-built tables ----
  // Metropolis thresholds (Eq 2): thr[h] = floor(exp(-h/T) 2^32), h = 1..Hmax = floor(T 32 ln 2)
  const bool accept_all = std::isinf(p->T);
  c->Hmax = (p->T > 0 && !accept_all) ? (long long)std::floor(p->T * 32.0 * std::log(2.0)) : 0;
  c->thr.assign((size_t)c->Hmax + 1, 0xffffffffu);
  for (long long h = 1; h <= c->Hmax; ++h) {
    double v = std::floor(std::exp(-(double)h / p->T) * 4294967296.0);
    c->thr[(size_t)h] = v >= 4294967295.0 ? 0xffffffffu : (v < 0 ? 0u : (uint32_t)v);
  }
  // Act fixed-point tables: log2 in Q16 for 1..255, 2^(f/1024) in Q16
  std::vector<int32_t> logq(256, 0), expq(1024, 0);
  for (int a = 1; a < 256; ++a) logq[a] = (int32_t)std::llround(65536.0 * std::log2((double)a));
  for (int f = 0; f < 1024; ++f) expq[f] = (int32_t)std::llround(65536.0 * std::exp2((double)f / 1024.0));
  // per-type records; row nT is all zero (what medium, id 0, reads: no constraints, reading S3);
  // lamA is stored as 0 when Max_act is 0 so that one test decides whether a side has an Act bias
  std::vector<TypeParams> types(nT + 1);
  for (int i = 0; i < nT; ++i) {
    TypeParams t{};
    t.lamV = p->lambda_V ? p->lambda_V[i] : 0; t.tgtV = p->target_V ? p->target_V[i] : 0;
    t.lamP = p->lambda_P ? p->lambda_P[i] : 0; t.tgtP = p->target_P ? p->target_P[i] : 0;
    t.maxA = p->max_act ? p->max_act[i] : 0;
    t.lamA = (p->lambda_act && t.maxA != 0) ? p->lambda_act[i] : 0;
    types[i] = t;
  }
  c->types = types;
  types[nT] = TypeParams{};
  // adhesion difference table of the pooled kernel: D[a][b][n][frozen] = J(a,n) - J(b,n) (the byte offset into a
  // row is the top byte of a lattice word: type * 8 + frozen * 4), then the diagonal J(t,t)
  std::vector<int32_t> Dtab((size_t)2 * nT * nT * nT + nT);
  for (int a = 0; a < nT; ++a)
    for (int b2 = 0; b2 < nT; ++b2)
      for (int n = 0; n < nT; ++n)
        for (int f = 0; f < 2; ++f) Dtab[(((size_t)a * nT + b2) * nT + n) * 2 + f] = p->J[a * nT + n] - p->J[b2 * nT + n];
  for (int t = 0; t < nT; ++t) Dtab[(size_t)2 * nT * nT * nT + t] = p->J[t * nT + t];

  // ---- tiled layout of the pooled kernel: per colour, groups of 8 tiles of (S+2)^d words ----
  TileLayout &tl = sp.tl;
  tl.S = S; tl.TW = 1;
  for (int a = 0; a < d; ++a) tl.TW *= S + 2;
  c->tile_words = 0;
  for (int col = 0; col < 8; ++col) {
    unsigned long long na = 1;
    for (int a = 0; a < 3; ++a) {
      const int bit = (col >> a) & 1;
      tl.nact[col][a] = (a < d) ? (c->nsub[a] - bit + 1) / 2 : (bit ? 0 : 1);
      na *= (unsigned long long)tl.nact[col][a];
    }
    c->n_act_col[col] = na;
    c->grp_col[col] = (na + (unsigned long long)(PK_GC - 1)) / (unsigned long long)PK_GC;
    tl.base[col] = c->tile_words;
    c->tile_words += (size_t)(c->grp_col[col] * (unsigned long long)tl.TW * (unsigned long long)PK_GC);
  }

  // ---- device state ----
  const long long pitch = roundup(c->dim[0], 4), apitch = roundup(c->dim[0], 16);
  const long long rows = (long long)c->dim[1] * c->dim[2];
  const size_t ncell = (size_t)c->max_cells + 1;
  int rc = CPM_OK;
  auto alloc = [&](void **ptr, size_t bytes) {
    if (rc != CPM_OK) return;
    cudaError_t e = cudaMalloc(ptr, bytes);
    if (e != cudaSuccess) rc = fail(c, e == cudaErrorMemoryAllocation ? CPM_ERR_OOM : CPM_ERR_CUDA, cudaGetErrorString(e));
    else if (cudaMemsetAsync(*ptr, 0, bytes, c->stream) != cudaSuccess) rc = CPM_ERR_CUDA;
  };
  sp.ovf_cap = 0;
  if (c->pooled) {
    alloc((void **)&tl.tiles, c->tile_words * 4);
    if (c->mode == CPM_MODE_DETERMINISTIC) {
      // spill slots for chains that change more than PK_DCAP distinct cells in one activation: one for every chain of
      // the largest colour (12 * PK_SPILL bytes each: 0.7 GB at 1024^3), so the pool itself can never run out; beyond
      // 8 Mi chains per colour one for every 8th chain
      unsigned long long most = 0;
      for (int col = 0; col < 8; ++col) most = std::max(most, c->n_act_col[col]);
      sp.ovf_cap = (int)(most <= (8ull << 20) ? std::max<unsigned long long>(most, 1ull) : std::max<unsigned long long>(most / 8, 8ull << 20));
      alloc((void **)&c->ovf_keys, (size_t)sp.ovf_cap * PK_SPILL * 4);
      alloc((void **)&c->ovf_dvp, (size_t)sp.ovf_cap * PK_SPILL * 8);
    }
    alloc((void **)&c->ovf_count, 4);
  } else {
    alloc((void **)&c->lat, (size_t)pitch * rows * 4);
  }
  if (c->act_enabled) alloc((void **)&c->act, (size_t)apitch * rows);
  alloc((void **)&c->liveVP, (ncell + 1) / 2 * 16);
  if (c->mode == CPM_MODE_DETERMINISTIC) alloc((void **)&c->snapVP, (ncell + 1) / 2 * 16);
  alloc((void **)&c->sumx, ncell * 8); alloc((void **)&c->sumy, ncell * 8); alloc((void **)&c->sumz, ncell * 8);
  alloc((void **)&c->counters, COUNTER_SLOTS * 2 * 8);
  alloc((void **)&c->error_flag, 4); alloc((void **)&c->mcs_dev, 4);
  alloc((void **)&c->J_dev, (size_t)nT * nT * 4); alloc((void **)&c->D_dev, Dtab.size() * 4); alloc((void **)&c->log_dev, 256 * 4); alloc((void **)&c->exp_dev, 1024 * 4);
  alloc((void **)&c->types_dev, (nT + 1) * sizeof(TypeParams)); alloc((void **)&c->thr_dev, c->thr.size() * 4);
  // vector terms: per-type strengths (row nT, what medium reads, stays zero), per-cell directions, the look-back ring
  std::vector<int2> vtypes(nT + 1, make_int2(0, 0));
  std::vector<double> mus(nT, 0.0);
  for (int i = 1; i < nT; ++i) {   // type 0 is medium: no terms (reading S3)
    vtypes[i] = make_int2(p->lambda_pers ? p->lambda_pers[i] : 0, p->lambda_chem ? p->lambda_chem[i] : 0);
  }
  for (int i = 0; i < nT; ++i) mus[i] = p->mu_pers ? p->mu_pers[i] : 0.0;
  if (pers_on || chem_on) alloc((void **)&c->vec_types_dev, (nT + 1) * sizeof(int2));
  if (pers_on) {
    alloc((void **)&c->mu_dev, nT * sizeof(double));
    alloc((void **)&c->phat, ncell * 3 * sizeof(double));
    alloc((void **)&c->ring, (size_t)(p->dt_pers + 1) * ncell * 3 * sizeof(double));
    alloc((void **)&c->pq, ncell * sizeof(short4));
    alloc((void **)&c->ctype_dev, ncell);
    alloc((void **)&c->pers_n, 4);
  }
  if (chem_on) alloc((void **)&c->chem, (size_t)c->N * sizeof(short4));
  if (c->unwrap) { alloc((void **)&c->anc, ncell * 3 * sizeof(int)); alloc((void **)&c->first_site, ncell * 8); }
  if (rc == CPM_OK && c->vec_types_dev) {
    cudaError_t e = cudaMemcpyAsync(c->vec_types_dev, vtypes.data(), vtypes.size() * sizeof(int2), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess && c->mu_dev) e = cudaMemcpyAsync(c->mu_dev, mus.data(), nT * sizeof(double), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) rc = fail(c, CPM_ERR_CUDA, cudaGetErrorString(e));
  }
  if (rc == CPM_OK) {
    cudaError_t e = cudaMemcpyAsync(c->J_dev, p->J, (size_t)nT * nT * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->D_dev, Dtab.data(), Dtab.size() * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->log_dev, logq.data(), 256 * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->exp_dev, expq.data(), 1024 * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->thr_dev, c->thr.data(), c->thr.size() * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) rc = fail(c, CPM_ERR_CUDA, cudaGetErrorString(e));
  }
  c->Dtab = Dtab;
  c->img_bytes = (((size_t)(nT + 1) * sizeof(TypeParams) + Dtab.size() * 4) + 15) / 16 * 16;
  if (c->pooled) alloc((void **)&c->img_dev, c->img_bytes);
  if (c->pooled) {   // neighbour n of the enumeration (dz, dy, dx) lexicographic, centre skipped (reading S16), in a tile of edge S + 2
    alloc((void **)&c->lane_tab_dev, 32 * sizeof(int4));
    int4 tab[32];
    const int Tt = S + 2, nNb = c->nNb;
    for (int n = 0; n < 32; ++n) {
      tab[n] = make_int4(0, 0, 0, 0);
      if (n >= nNb) continue;
      const int i = n + (n >= nNb / 2 ? 1 : 0);
      const int dx = i % 3 - 1, dy = (i / 3) % 3 - 1, dz = (d == 3) ? i / 9 - 1 : 0;
      tab[n] = make_int4((dz * Tt + dy) * Tt + dx, dx, dy, dz);
    }
    if (rc == CPM_OK && cudaMemcpyAsync(c->lane_tab_dev, tab, sizeof(tab), cudaMemcpyHostToDevice, c->stream) != cudaSuccess) rc = CPM_ERR_CUDA;
    if (rc == CPM_OK && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = CPM_ERR_CUDA;
  }
  if (rc == CPM_OK) rc = upload_types(c, 0);
  if (rc != CPM_OK) { free_all(c); delete c; return rc; }

  // ---- launch-parameter template ----
  sp.lat = c->lat; sp.act = c->act; sp.pitch = pitch; sp.apitch = apitch;
  sp.X = c->dim[0]; sp.Y = c->dim[1]; sp.Z = c->dim[2];
  for (int a = 0; a < 3; ++a) { sp.per[a] = c->per[a]; sp.nsub[a] = c->nsub[a]; }
  sp.S = S; sp.sites = c->sites; sp.k = c->k;
  sp.log2S = -1;
  for (int b = 1; b < 16; ++b) if ((1 << b) == S) sp.log2S = b;
  sp.mcs_ptr = c->mcs_dev;
  sp.key0 = (uint32_t)c->seed; sp.key1 = (uint32_t)(c->seed >> 32);
  sp.use_tma = c->use_tma ? 1 : 0;
  sp.J = c->J_dev; sp.D = c->D_dev; sp.nT = nT; sp.types = c->types_dev;
  sp.thr = c->thr_dev; sp.Hmax = c->Hmax; sp.accept_all = accept_all ? 1 : 0;
  sp.logq16 = c->log_dev; sp.expq16 = c->exp_dev;
  sp.snapVP = c->snapVP; sp.liveVP = c->liveVP; sp.sumx = c->sumx; sp.sumy = c->sumy; sp.sumz = c->sumz;
  sp.cell_arr[0] = c->liveVP; sp.cell_arr[1] = c->sumx; sp.cell_arr[2] = c->sumy; sp.cell_arr[3] = c->sumz;
  sp.counters = c->counters; sp.error_flag = c->error_flag;
  sp.ovf_keys = c->ovf_keys; sp.ovf_dvp = c->ovf_dvp; sp.ovf_count = c->ovf_count;
  sp.vec_on = (pers_on || chem_on) ? 1 : 0; sp.vec_types = c->vec_types_dev; sp.pq = c->pq; sp.chem = c->chem;
  sp.anc = c->anc; sp.img = c->img_dev; sp.img_bytes = (int)c->img_bytes; sp.lane_tab = c->lane_tab_dev;
  for (int n2 = 1; n2 <= 3; ++n2) sp.xq_len[n2 - 1] = (int)std::llround(16384.0 / std::sqrt((double)n2));

  memset(&c->tm_lat, 0, sizeof(CUtensorMap));
  if (c->use_tma && !c->pooled) {
    rc = make_tensor_map(c, &c->tm_lat, CU_TENSOR_MAP_DATA_TYPE_UINT32, 4, c->lat, pitch, sp.TX);
    if (rc != CPM_OK) { free_all(c); delete c; return rc; }
  }
  c->fn = pick_kernel(d, c->act_enabled, c->mode == CPM_MODE_LIVE_ATOMICS, c->nsets);
  cudaError_t e = cudaFuncSetAttribute(c->pooled ? (const void *)c->tfn : (const void *)c->fn,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->cta_smem);
  if (e != cudaSuccess) { free_all(c); delete c; return CPM_ERR_CUDA; }
  *out = c;
  return CPM_OK;
}

int cpm_create(const cpm_params *p, cpm_ctx **out) {
  CPM_GUARD_BEGIN
  return create_impl(p, out);
  CPM_GUARD_END(nullptr)
}

int cpm_destroy(cpm_ctx *c) {
  if (!c) return CPM_OK;
  cudaSetDevice(c->device);
  cudaStreamSynchronize(c->stream);
  free_all(c);
  delete c;
  return CPM_OK;
}

int cpm_set_lattice(cpm_ctx *c, const uint32_t *ids, const uint8_t *frozen, const uint8_t *cell_type, int on_device) {
  if (!c) return CPM_ERR_ARG;
  if (!ids || !cell_type) return fail(c, CPM_ERR_ARG, "ids and cell_type are required");
  NvtxRange nvtx("cpm_set_lattice");
  CPM_GUARD_BEGIN
  CK(cudaSetDevice(c->device));
  const size_t ncell = (size_t)c->max_cells + 1;
  // the type table is validated on the host
  std::vector<uint8_t> ct(ncell);
  if (on_device) { CK(cudaMemcpyAsync(ct.data(), cell_type, ncell, cudaMemcpyDeviceToHost, c->stream)); CK(cudaStreamSynchronize(c->stream)); }
  else memcpy(ct.data(), cell_type, ncell);
  if (ct[0] != 0) return fail(c, CPM_ERR_ARG, "cell 0 must have type 0 (medium)");
  for (size_t i = 0; i < ncell; ++i) if (ct[i] >= c->nT) return fail(c, CPM_ERR_ARG, "cell type out of range");
  const uint32_t *sid; const uint8_t *sfz, *sct;
  int slab[PIPE_SLABS + 1];
  const bool piped = !on_device && pipe_plan(c, slab);
  if (piped) {
    // the lattice comes over slab by slab on the transfer stream; the kernels below follow the slabs
    CK(pipe_ready(c));
    CK(stage_reserve(&c->stage_a, &c->stage_a_cap, (size_t)c->N * 4));
    if (frozen) CK(stage_reserve(&c->stage_b, &c->stage_b_cap, (size_t)c->N));
    sid = reinterpret_cast<const uint32_t *>(c->stage_a);
    sfz = frozen ? reinterpret_cast<const uint8_t *>(c->stage_b) : nullptr;
    CK(cudaEventRecord(c->io_ev[PIPE_SLABS], c->stream));            // earlier work on the staging buffers is done first
    CK(cudaStreamWaitEvent(c->io_stream, c->io_ev[PIPE_SLABS], 0));
    // (the slab copies themselves are issued further down, each just before the first kernels that need it, so that a
    // pageable source, whose copies hold up the host, still overlaps with the kernels of the slabs before it)
  } else {
    CK(stage_in(const_cast<uint32_t **>(&sid), &c->stage_a, &c->stage_a_cap, ids, (size_t)c->N, on_device, c->stream));
    CK(stage_in(const_cast<uint8_t **>(&sfz), &c->stage_b, &c->stage_b_cap, frozen, (size_t)c->N, on_device, c->stream));
  }
  CK(stage_in(const_cast<uint8_t **>(&sct), &c->stage_c, &c->stage_c_cap, cell_type, ncell, on_device, c->stream));

  CK(cudaMemsetAsync(c->error_flag, 0, 4, c->stream));
  if (c->act) CK(cudaMemsetAsync(c->act, 0, (size_t)c->sp.apitch * c->dim[1] * c->dim[2], c->stream));
  if (c->act && c->act_cap == 255) { int rc0 = upload_types(c, 0); if (rc0 != CPM_OK) return rc0; }
  CK(cudaMemsetAsync(c->liveVP, 0, ncell * 8, c->stream));
  CK(cudaMemsetAsync(c->sumx, 0, ncell * 8, c->stream));
  CK(cudaMemsetAsync(c->sumy, 0, ncell * 8, c->stream));
  CK(cudaMemsetAsync(c->sumz, 0, ncell * 8, c->stream));
  if (c->unwrap) {   // reading S23: the first site of a cell in scan order anchors the images of its other sites
    CK(cudaMemsetAsync(c->first_site, 0xff, ncell * 8, c->stream));
    anchor_first_site_kernel<<<grid_for(c->N), 256, 0, c->stream>>>(sid, c->N, c->max_cells, c->first_site);
    anchor_from_first_kernel<<<(unsigned)((ncell + 255) / 256), 256, 0, c->stream>>>((long long)ncell, c->first_site, c->dim[0], c->dim[1], c->anc);
    c->launches += 2;
  }
  if (c->pooled) {
    const TileLayout &tl = c->sp.tl;
    // pack then recount, for the chains [w0, w1) of every colour that the slab `piece` holds (one piece: all of them)
    auto pack_and_recount = [&](int piece) {
      const int ax = c->d - 1;
      unsigned long long gb[8], ge[8], wb[8], we[8];
      for (int col = 0; col < (1 << c->d); ++col) {
        const unsigned long long n = c->n_act_col[col];
        gb[col] = 0; ge[col] = c->grp_col[col]; wb[col] = 0; we[col] = n;
        if (piece < 0 || n == 0) continue;
        const unsigned long long slow = (unsigned long long)tl.nact[col][ax], fast = n / slow;
        const unsigned long long w0 = std::min<unsigned long long>((unsigned long long)slab[piece], slow) * fast;
        const unsigned long long w1 = std::min<unsigned long long>((unsigned long long)slab[piece + 1], slow) * fast;
        // a group that straddles two slabs goes with the later one, whose data arrives last
        gb[col] = w0 >> PK_GS; wb[col] = gb[col] << PK_GS;
        if (piece < PIPE_SLABS - 1) { ge[col] = w1 >> PK_GS; we[col] = ge[col] << PK_GS; }
      }
      for (int col = 0; col < (1 << c->d); ++col) {
        if (c->n_act_col[col] == 0 || ge[col] <= gb[col]) continue;
        const int grid = grid_for((long long)(ge[col] - gb[col]), 1);
        if (c->d == 2)
          tile_pack_kernel<2><<<grid, 256, 0, c->stream>>>(sid, sfz, sct, c->max_cells, tl, col, c->n_act_col[col], gb[col], ge[col], c->dim[0],
                                                          c->dim[1], c->dim[2], c->per[0], c->per[1], c->per[2], c->error_flag);
        else
          tile_pack_kernel<3><<<grid, 256, 0, c->stream>>>(sid, sfz, sct, c->max_cells, tl, col, c->n_act_col[col], gb[col], ge[col], c->dim[0],
                                                          c->dim[1], c->dim[2], c->per[0], c->per[1], c->per[2], c->error_flag);
        c->launches++;
      }
      RecountRanges rr{};
      unsigned long long most = 0;
      for (int col = 0; col < (1 << c->d); ++col) {
        if (c->n_act_col[col] == 0 || we[col] <= wb[col]) continue;
        rr.w_begin[col] = wb[col]; rr.w_end[col] = we[col];
        most = std::max(most, we[col] - wb[col]);
      }
      if (most > 0) {   // one launch for all colours (blockIdx.y)
        const dim3 grid((unsigned)grid_for((long long)most, 128), (unsigned)(1 << c->d));
        if (c->d == 2)
          tile_recount_kernel<2><<<grid, 128, 0, c->stream>>>(tl, rr, c->liveVP, c->sumx, c->sumy, c->sumz,
                                                             c->anc, c->dim[0], c->dim[1], c->dim[2], c->per[0], c->per[1], c->per[2]);
        else
          tile_recount_kernel<3><<<grid, 128, 0, c->stream>>>(tl, rr, c->liveVP, c->sumx, c->sumy, c->sumz,
                                                             c->anc, c->dim[0], c->dim[1], c->dim[2], c->per[0], c->per[1], c->per[2]);
        c->launches++;
      }
    };
    if (!piped) pack_and_recount(-1);
    else {
      // slab i needs one plane of slab i + 1 (its upper halo) and one of slab i - 1; slab 0 reaches the LAST slab through a
      // periodic border, so it goes last then
      const bool wrap = c->per[c->d - 1] != 0;
      const int ax = c->d - 1;
      const size_t plane = (size_t)(c->N / c->dim[ax]);
      int issued = 0;   // slabs whose copies are on the transfer stream
      for (int n = 0; n < PIPE_SLABS; ++n) {
        const int i = wrap ? (n + 1) % PIPE_SLABS : n;
        const int need = (wrap && i == 0) ? PIPE_SLABS - 1 : std::min(i + 1, PIPE_SLABS - 1);
        for (; issued <= need; ++issued) {
          const size_t p0 = std::min<size_t>((size_t)slab[issued] * 2 * c->S, (size_t)c->dim[ax]) * plane;
          const size_t p1 = (issued == PIPE_SLABS - 1) ? (size_t)c->N : std::min<size_t>((size_t)slab[issued + 1] * 2 * c->S, (size_t)c->dim[ax]) * plane;
          CK(cudaMemcpyAsync(const_cast<uint32_t *>(sid) + p0, ids + p0, (p1 - p0) * 4, cudaMemcpyHostToDevice, c->io_stream));
          if (frozen) CK(cudaMemcpyAsync(const_cast<uint8_t *>(sfz) + p0, frozen + p0, p1 - p0, cudaMemcpyHostToDevice, c->io_stream));
          CK(cudaEventRecord(c->io_ev[issued], c->io_stream));
        }
        CK(cudaStreamWaitEvent(c->stream, c->io_ev[need], 0));
        pack_and_recount(i);
      }
      CK(cudaStreamWaitEvent(c->stream, c->io_ev[PIPE_SLABS - 1], 0));
    }
  } else {
    pack_kernel<<<grid_for(c->N), 256, 0, c->stream>>>(sid, sfz, sct, c->max_cells, c->lat, c->sp.pitch, c->dim[0],
                                                        c->dim[1], c->dim[2], c->error_flag);
    c->launches++;
    if (c->d == 2)
      recount_kernel<2><<<grid_for(c->N), 256, 0, c->stream>>>(c->lat, c->sp.pitch, c->dim[0], c->dim[1], c->dim[2], c->per[0],
                                                                c->per[1], c->per[2], c->liveVP, c->sumx, c->sumy, c->sumz, c->anc);
    else
      recount_kernel<3><<<grid_for(c->N), 256, 0, c->stream>>>(c->lat, c->sp.pitch, c->dim[0], c->dim[1], c->dim[2], c->per[0],
                                                                c->per[1], c->per[2], c->liveVP, c->sumx, c->sumy, c->sumz, c->anc);
    c->launches++;
  }
  if (c->snapVP) CK(cudaMemcpyAsync(c->snapVP, c->liveVP, ncell * 8, cudaMemcpyDeviceToDevice, c->stream));
  if (c->unwrap) {
    centroid_normalise_kernel<<<(unsigned)((ncell + 255) / 256), 256, 0, c->stream>>>((long long)ncell, c->liveVP, c->sumx, c->sumy, c->sumz, c->anc,
                                                                                   c->dim[0], c->dim[1], c->dim[2], c->per[0], c->per[1], c->per[2]);
    c->launches++;
  }
  if (c->pers_on) {   // reading S22: p^ = 0, the look-back window starts at the present centroids
    CK(cudaMemcpyAsync(c->ctype_dev, sct, ncell, cudaMemcpyDeviceToDevice, c->stream));
    persistence_init_kernel<<<(unsigned)((ncell + 255) / 256), 256, 0, c->stream>>>((long long)ncell, c->dt_pers + 1, c->liveVP, c->sumx, c->sumy,
                                                                                   c->sumz, c->phat, c->pq, c->ring, c->pers_n);
    c->launches++;
  }
  CK(cudaGetLastError());
  int rc = check_device_flag(c);
  if (rc != CPM_OK) return rc;
  c->have_lattice = true;
  return CPM_OK;
  CPM_GUARD_END(c)
}

int cpm_set_act(cpm_ctx *c, const float *act, int on_device) {
  if (!c || !act) return fail(c, CPM_ERR_ARG, "null argument");
  if (!c->act_enabled) return fail(c, CPM_ERR_UNSUPPORTED, "the Act field needs at least one type with max_act > 0");
  CK(cudaSetDevice(c->device));
  int rc = check_device_flag(c);   // a pending error of an earlier cpm_step is reported, not discarded
  if (rc != CPM_OK) return rc;
  if (c->act_cap != 255) { rc = upload_types(c, 1); if (rc != CPM_OK) return rc; }
  const float *s;
  CK(stage_in(const_cast<float **>(&s), &c->stage_a, &c->stage_a_cap, act, (size_t)c->N, on_device, c->stream));
  act_set_kernel<<<grid_for(c->N), 256, 0, c->stream>>>(s, c->act, c->sp.apitch, c->dim[0], c->dim[1], c->dim[2], c->error_flag);
  c->launches++;
  CK(cudaGetLastError());
  rc = check_device_flag(c);
  if (rc != CPM_OK) CK(cudaMemsetAsync(c->error_flag, 0, 4, c->stream));   // bad input: reported once, state stays usable
  return rc;
}

int cpm_set_chemotaxis_field(cpm_ctx *c, const float *field, int on_device) {
  if (!c || !field) return fail(c, CPM_ERR_ARG, "null argument");
  if (!c->chem_on) return fail(c, CPM_ERR_UNSUPPORTED, "no cell type has lambda_chem != 0");
  CK(cudaSetDevice(c->device));
  int rc = check_device_flag(c);
  if (rc != CPM_OK) return rc;
  const float *s;
  CK(stage_in(const_cast<float **>(&s), &c->stage_a, &c->stage_a_cap, field, (size_t)c->N * c->d, on_device, c->stream));
  // validate first: a refused field leaves the loaded one untouched
  chem_set_kernel<<<grid_for(c->N), 256, 0, c->stream>>>(s, c->chem, c->N, c->d, c->error_flag, 0);
  c->launches++;
  CK(cudaGetLastError());
  rc = check_device_flag(c);
  if (rc != CPM_OK) { CK(cudaMemsetAsync(c->error_flag, 0, 4, c->stream)); return rc; }   // bad input: reported once
  chem_set_kernel<<<grid_for(c->N), 256, 0, c->stream>>>(s, c->chem, c->N, c->d, c->error_flag, 1);
  c->launches++;
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(c->stream));   // the staging buffer may be reused by the next call
  return CPM_OK;
}

int cpm_set_persistence(cpm_ctx *c, const double *p, int on_device) {
  if (!c || !p) return fail(c, CPM_ERR_ARG, "null argument");
  if (!c->pers_on) return fail(c, CPM_ERR_UNSUPPORTED, "no cell type has lambda_pers != 0");
  if (!c->have_lattice) return fail(c, CPM_ERR_STATE, "cpm_set_lattice first");
  CK(cudaSetDevice(c->device));
  int rc = check_device_flag(c);
  if (rc != CPM_OK) return rc;
  const size_t ncell = (size_t)c->max_cells + 1;
  const double *s;
  CK(stage_in(const_cast<double **>(&s), &c->stage_a, &c->stage_a_cap, p, ncell * 3, on_device, c->stream));
  persistence_set_kernel<<<(unsigned)((ncell + 255) / 256), 256, 0, c->stream>>>((long long)ncell, s, c->phat, c->pq, c->error_flag, 0);
  c->launches++;
  CK(cudaGetLastError());
  rc = check_device_flag(c);
  if (rc != CPM_OK) { CK(cudaMemsetAsync(c->error_flag, 0, 4, c->stream)); return rc; }
  persistence_set_kernel<<<(unsigned)((ncell + 255) / 256), 256, 0, c->stream>>>((long long)ncell, s, c->phat, c->pq, c->error_flag, 1);
  c->launches++;
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(c->stream));
  return CPM_OK;
}

int cpm_get_persistence(cpm_ctx *c, double *p, int on_device) {
  if (!c || !p) return fail(c, CPM_ERR_ARG, "null argument");
  if (!c->pers_on) return fail(c, CPM_ERR_UNSUPPORTED, "no cell type has lambda_pers != 0");
  if (!c->have_lattice) return fail(c, CPM_ERR_STATE, "cpm_set_lattice first");
  CK(cudaSetDevice(c->device));
  CK(cudaMemcpyAsync(p, c->phat, ((size_t)c->max_cells + 1) * 3 * sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
  return check_device_flag(c);
}

int cpm_set_mcs(cpm_ctx *c, uint32_t mcs) {
  if (!c) return CPM_ERR_ARG;
  CK(cudaSetDevice(c->device));
  CK(cudaMemcpyAsync(c->mcs_dev, &mcs, 4, cudaMemcpyHostToDevice, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  c->mcs_host = mcs;
  return CPM_OK;
}

int cpm_step(cpm_ctx *c, uint32_t n_mcs) {
  if (!c) return CPM_ERR_ARG;
  if (!c->have_lattice) return fail(c, CPM_ERR_STATE, "cpm_set_lattice first");
  NvtxRange nvtx("cpm_step");
  CPM_GUARD_BEGIN
  CK(cudaSetDevice(c->device));
  // per-launch events need the plain launch sequence; otherwise one graph launch per MCS
  const bool graph = c->use_graph && !c->timing;
  if (graph && !c->mcs_graph) { int rc = build_mcs_graph(c); if (rc != CPM_OK) return rc; }
  for (uint32_t m = 0; m < n_mcs; ++m) {
    if (graph) {
      CK(cudaGraphLaunch(c->mcs_graph, c->stream));
      c->launches += c->graph_launches; c->sweep_launches += c->graph_sweeps;
    } else {
      int rc = enqueue_mcs(c, c->stream, c->timing);
      if (rc != CPM_OK) return rc;
    }
    c->mcs_host++; c->mcs_run++;
  }
  CK(cudaGetLastError());
  return CPM_OK;
  CPM_GUARD_END(c)
}

int cpm_get_lattice(cpm_ctx *c, uint32_t *ids, int on_device) {
  if (!c || !ids) return fail(c, CPM_ERR_ARG, "null argument");
  NvtxRange nvtx("cpm_get_lattice");
  CK(cudaSetDevice(c->device));
  uint32_t *s;
  CK(stage_out_begin(&s, &c->stage_a, &c->stage_a_cap, ids, (size_t)c->N, on_device));
  if (c->pooled) {
    const bool piped = !on_device && c->N >= c->pipe_min_sites;
    if (piped) CK(pipe_ready(c));
    const int pieces = piped ? PIPE_SLABS : 1;
    // the pieces are unpacked on the context's stream; each goes to the host on the transfer stream while the next is unpacked
    for (int i = 0; i < pieces; ++i) {
      const long long i0 = c->N * i / pieces, i1 = c->N * (i + 1) / pieces;
      if (c->d == 2) tile_unpack_kernel<2><<<grid_for(i1 - i0), 256, 0, c->stream>>>(c->sp.tl, c->dim[0], c->dim[1], c->dim[2], s, i0, i1);
      else tile_unpack_kernel<3><<<grid_for(i1 - i0), 256, 0, c->stream>>>(c->sp.tl, c->dim[0], c->dim[1], c->dim[2], s, i0, i1);
      c->launches++;
      if (piped) CK(cudaEventRecord(c->io_ev[i], c->stream));
    }
    for (int i = 0; piped && i < pieces; ++i) {
      const long long i0 = c->N * i / pieces, i1 = c->N * (i + 1) / pieces;
      CK(cudaStreamWaitEvent(c->io_stream, c->io_ev[i], 0));
      CK(cudaMemcpyAsync(ids + i0, s + i0, (size_t)(i1 - i0) * 4, cudaMemcpyDeviceToHost, c->io_stream));
    }
    CK(cudaGetLastError());
    if (piped) {   // the context's stream ends behind the last transfer: the synchronisation below covers it
      CK(cudaEventRecord(c->io_ev[PIPE_SLABS + 1], c->io_stream));
      CK(cudaStreamWaitEvent(c->stream, c->io_ev[PIPE_SLABS + 1], 0));
      return check_device_flag(c);
    }
    c->launches--;   // counted once below
  } else {
    unpack_kernel<<<grid_for(c->N), 256, 0, c->stream>>>(c->lat, c->sp.pitch, c->dim[0], c->dim[1], c->dim[2], s);
  }
  c->launches++;
  CK(cudaGetLastError());
  CK(stage_out_end(s, ids, (size_t)c->N, on_device, c->stream));
  return check_device_flag(c);
}

int cpm_get_act(cpm_ctx *c, float *act, int on_device) {
  if (!c || !act) return fail(c, CPM_ERR_ARG, "null argument");
  CK(cudaSetDevice(c->device));
  float *s;
  CK(stage_out_begin(&s, &c->stage_a, &c->stage_a_cap, act, (size_t)c->N, on_device));
  act_get_kernel<<<grid_for(c->N), 256, 0, c->stream>>>(c->act, c->sp.apitch, c->dim[0], c->dim[1], c->dim[2], s);
  c->launches++;
  CK(cudaGetLastError());
  CK(stage_out_end(s, act, (size_t)c->N, on_device, c->stream));
  return check_device_flag(c);
}

int cpm_get_cell_stats(cpm_ctx *c, uint32_t *volume, uint32_t *perimeter, uint64_t *sx, uint64_t *sy, uint64_t *sz,
                       int on_device) {
  if (!c) return CPM_ERR_ARG;
  CK(cudaSetDevice(c->device));
  const size_t n = (size_t)c->max_cells + 1;
  uint32_t *sv, *spm;
  CK(stage_out_begin(&sv, &c->stage_b, &c->stage_b_cap, volume, n, on_device));
  CK(stage_out_begin(&spm, &c->stage_c, &c->stage_c_cap, perimeter, n, on_device));
  if (volume || perimeter) {
    stats_unpack_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->liveVP, (long long)n, sv, spm);
    c->launches++;
    CK(cudaGetLastError());
  }
  CK(stage_out_end(sv, volume, n, on_device, c->stream));
  CK(stage_out_end(spm, perimeter, n, on_device, c->stream));
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  if (sx) CK(cudaMemcpyAsync(sx, c->sumx, n * 8, kind, c->stream));
  if (sy) CK(cudaMemcpyAsync(sy, c->sumy, n * 8, kind, c->stream));
  if (sz) CK(cudaMemcpyAsync(sz, c->sumz, n * 8, kind, c->stream));
  return check_device_flag(c);
}

int cpm_get_centroids(cpm_ctx *c, double *xyz, int on_device) {
  if (!c || !xyz) return fail(c, CPM_ERR_ARG, "null argument");
  if (!c->have_lattice) return fail(c, CPM_ERR_STATE, "cpm_set_lattice first");
  CK(cudaSetDevice(c->device));
  const size_t n = (size_t)c->max_cells + 1;
  double *s;
  CK(stage_out_begin(&s, &c->stage_a, &c->stage_a_cap, xyz, n * 3, on_device));
  centroid_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>((long long)n, c->liveVP, c->sumx, c->sumy, c->sumz, s);
  c->launches++;
  CK(cudaGetLastError());
  CK(stage_out_end(s, xyz, n * 3, on_device, c->stream));
  return check_device_flag(c);
}

int cpm_get_counters(cpm_ctx *c, uint64_t out[4]) {
  if (!c || !out) return fail(c, CPM_ERR_ARG, "null argument");
  CK(cudaSetDevice(c->device));
  unsigned long long h[COUNTER_SLOTS * 2];
  CK(cudaMemcpyAsync(h, c->counters, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  uint64_t ev = 0, ac = 0;
  for (int i = 0; i < COUNTER_SLOTS; ++i) { ev += h[2 * i]; ac += h[2 * i + 1]; }
  out[0] = (uint64_t)c->N * c->mcs_run; out[1] = ev; out[2] = ac; out[3] = c->mcs_host;
  return CPM_OK;
}

int cpm_get_schedule(cpm_ctx *c, int32_t *S, int32_t *k, int32_t *steps) {
  if (!c) return CPM_ERR_ARG;
  if (S) *S = c->S;
  if (k) *k = c->k;
  if (steps) *steps = (1 << c->d) * c->R;
  return CPM_OK;
}

int cpm_get_interface_counts(cpm_ctx *c, uint64_t *out) {
  if (!c || !out) return fail(c, CPM_ERR_ARG, "null argument");
  if (!c->have_lattice) return fail(c, CPM_ERR_STATE, "cpm_set_lattice first");
  CK(cudaSetDevice(c->device));
  const size_t n = (size_t)c->nT * c->nT;
  unsigned long long *d = nullptr;
  CK(stage_reserve(&c->stage_c, &c->stage_c_cap, n * 8));
  d = reinterpret_cast<unsigned long long *>(c->stage_c);
  CK(cudaMemsetAsync(d, 0, n * 8, c->stream));
  LatView V{};
  V.lat = c->lat; V.pitch = c->sp.pitch; V.tl = c->sp.tl; V.pooled = c->pooled ? 1 : 0;
  V.X = c->dim[0]; V.Y = c->dim[1]; V.Z = c->dim[2];
  for (int a = 0; a < 3; ++a) V.per[a] = c->per[a];
  const int use_smem = n * 8 <= 32768 ? 1 : 0;   // block-local counts for up to 64 types, else global atomics only
  const size_t shm = use_smem ? n * 8 : 0;
  if (c->d == 2) interface_count_kernel<2><<<grid_for(c->N), 256, shm, c->stream>>>(V, c->nT, d, use_smem);
  else interface_count_kernel<3><<<grid_for(c->N), 256, shm, c->stream>>>(V, c->nT, d, use_smem);
  c->launches++;
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(out, d, n * 8, cudaMemcpyDeviceToHost, c->stream));
  return check_device_flag(c);
}

int cpm_update_statistics(cpm_ctx *c, uint32_t n_mcs, uint64_t *freq, int32_t n_freq, uint64_t *wait, int32_t n_wait, uint32_t wait_bin) {
  if (!c || !freq || !wait) return fail(c, CPM_ERR_ARG, "null argument");
  if (n_freq < 1 || n_wait < 1 || wait_bin < 1 || n_freq + n_wait > 4096) return fail(c, CPM_ERR_ARG, "histogram sizes");
  const unsigned long long ticks = (unsigned long long)n_mcs * (unsigned long long)(1 << c->d) * (unsigned long long)c->sites;
  if (ticks >= (1ull << 32)) return fail(c, CPM_ERR_ARG, "n_mcs * 2^d * S^d must stay below 2^32");
  CK(cudaSetDevice(c->device));
  StatParams P{};
  P.S = c->S; P.sites = c->sites; P.k = c->k; P.R = c->R; P.nNb = c->nNb;
  for (int a = 0; a < 3; ++a) P.nsub[a] = c->nsub[a];
  P.X = c->dim[0]; P.Y = c->dim[1];
  int rank = 0;
  for (int col = 0; col < 8; ++col) P.rank[col] = (col < (1 << c->d) && c->n_act_col[col] > 0) ? rank++ : -1;
  P.E_per_rep = rank;
  P.mcs0 = c->mcs_host; P.n_mcs = n_mcs; P.key0 = (uint32_t)c->seed; P.key1 = (uint32_t)(c->seed >> 32); P.bin = wait_bin;
  P.n_freq = n_freq; P.n_wait = n_wait;
  const long long nsub_total = (long long)c->nsub[0] * c->nsub[1] * c->nsub[2];
  const size_t nh = (size_t)n_freq + (size_t)n_wait;
  uint32_t *scratch = nullptr;
  unsigned long long *hist = nullptr;
  cudaError_t e = cudaMalloc(&scratch, (size_t)c->N * 8);
  if (e == cudaSuccess) e = cudaMalloc(&hist, nh * 8);
  if (e != cudaSuccess) { cudaFree(scratch); cudaFree(hist); return fail(c, CPM_ERR_OOM, cudaGetErrorString(e)); }
  std::vector<unsigned long long> h(nh);
  e = cudaMemsetAsync(scratch, 0, (size_t)c->N * 8, c->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(hist, 0, nh * 8, c->stream);
  if (e == cudaSuccess) {
    const unsigned blocks = (unsigned)((nsub_total + 127) / 128);
    if (c->d == 2) update_stats_kernel<2><<<blocks, 128, nh * 8, c->stream>>>(P, nsub_total, scratch, scratch + c->N, hist);
    else update_stats_kernel<3><<<blocks, 128, nh * 8, c->stream>>>(P, nsub_total, scratch, scratch + c->N, hist);
    c->launches++;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(h.data(), hist, nh * 8, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  cudaFree(scratch); cudaFree(hist);
  if (e != cudaSuccess) return fail(c, CPM_ERR_CUDA, cudaGetErrorString(e));
  for (int i = 0; i < n_freq; ++i) freq[i] = h[(size_t)i];
  for (int i = 0; i < n_wait; ++i) wait[i] = h[(size_t)n_freq + i];
  return CPM_OK;
}

}  // extern "C"

// ---- cpm_update_statistics_noalloc: the same kernel on a file-scope scratch array; no allocation of any kind ----
// Layout of the array: [hist: 4096 x u64 | last: MAX_SITES x u32 | cnt: MAX_SITES x u32].  Every GPU that loads the
// library holds it until exit.  In host code the NAME below is a host-side stand-in, never a device address: the
// address the kernel gets comes from cudaGetSymbolAddress, once per device, with that device current.
namespace {
constexpr size_t NOALLOC_HIST_BYTES = (size_t)CPM_NOALLOC_MAX_BINS * 8;
constexpr size_t NOALLOC_BYTES = NOALLOC_HIST_BYTES + (size_t)CPM_NOALLOC_MAX_SITES * 8;
}  // namespace
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];
namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
unsigned char *g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};

// device address of the scratch array on `device`, which must be the current device; nullptr + *e on failure
unsigned char *noalloc_scratch_on(int device, cudaError_t *e) {
  *e = cudaSuccess;
  if (device < 0 || device >= NOALLOC_MAX_DEVICES) { *e = cudaErrorInvalidDevice; return nullptr; }
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[device]) {
    void *p = nullptr;
    *e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (*e != cudaSuccess) return nullptr;
    g_noalloc_ptr[device] = static_cast<unsigned char *>(p);
  }
  return g_noalloc_ptr[device];
}
}  // namespace

extern "C" {

int cpm_noalloc_setup(int device) {
  if (cudaSetDevice(device) != cudaSuccess) return CPM_ERR_CUDA;
  cudaError_t e;
  return noalloc_scratch_on(device, &e) ? CPM_OK : CPM_ERR_CUDA;
}

int cpm_update_statistics_noalloc(cpm_ctx *c, uint32_t n_mcs, uint64_t *freq, int32_t n_freq, uint64_t *wait, int32_t n_wait,
                                  uint32_t wait_bin, int on_device) {
  if (!c || !freq || !wait) return fail(c, CPM_ERR_ARG, "null argument");
  if (n_freq < 1 || n_wait < 1 || wait_bin < 1 || n_freq + n_wait > CPM_NOALLOC_MAX_BINS)
    return fail(c, CPM_ERR_ARG, "histogram sizes: n_freq + n_wait must be in [2, 4096]");
  if (c->N > (long long)CPM_NOALLOC_MAX_SITES)
    return fail(c, CPM_ERR_ARG, "cpm_update_statistics_noalloc: the lattice has more than CPM_NOALLOC_MAX_SITES (1048576) sites; "
                                "use cpm_update_statistics");
  const unsigned long long ticks = (unsigned long long)n_mcs * (unsigned long long)(1 << c->d) * (unsigned long long)c->sites;
  if (ticks >= (1ull << 32)) return fail(c, CPM_ERR_ARG, "n_mcs * 2^d * S^d must stay below 2^32");
  CK(cudaSetDevice(c->device));
  cudaError_t e;
  unsigned char *base = noalloc_scratch_on(c->device, &e);
  if (!base) return fail(c, CPM_ERR_CUDA, std::string("cudaGetSymbolAddress(g_noalloc_scratch): ") + cudaGetErrorString(e));
  unsigned long long *hist = reinterpret_cast<unsigned long long *>(base);
  uint32_t *last = reinterpret_cast<uint32_t *>(base + NOALLOC_HIST_BYTES);
  uint32_t *cnt = last + c->N;
  StatParams P{};
  P.S = c->S; P.sites = c->sites; P.k = c->k; P.R = c->R; P.nNb = c->nNb;
  for (int a = 0; a < 3; ++a) P.nsub[a] = c->nsub[a];
  P.X = c->dim[0]; P.Y = c->dim[1];
  int rank = 0;
  for (int col = 0; col < 8; ++col) P.rank[col] = (col < (1 << c->d) && c->n_act_col[col] > 0) ? rank++ : -1;
  P.E_per_rep = rank;
  P.mcs0 = c->mcs_host; P.n_mcs = n_mcs; P.key0 = (uint32_t)c->seed; P.key1 = (uint32_t)(c->seed >> 32); P.bin = wait_bin;
  P.n_freq = n_freq; P.n_wait = n_wait;
  const long long nsub_total = (long long)c->nsub[0] * c->nsub[1] * c->nsub[2];
  const size_t nh = (size_t)n_freq + (size_t)n_wait;
  // the array keeps the last call's contents: the histograms and both per-site words must start at zero
  CK(cudaMemsetAsync(hist, 0, nh * 8, c->stream));
  CK(cudaMemsetAsync(last, 0, (size_t)c->N * 8, c->stream));
  const unsigned blocks = (unsigned)((nsub_total + 127) / 128);
  if (c->d == 2) update_stats_kernel<2><<<blocks, 128, nh * 8, c->stream>>>(P, nsub_total, last, cnt, hist);
  else update_stats_kernel<3><<<blocks, 128, nh * 8, c->stream>>>(P, nsub_total, last, cnt, hist);
  c->launches++;
  CK(cudaGetLastError());
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  CK(cudaMemcpyAsync(freq, hist, (size_t)n_freq * 8, kind, c->stream));
  CK(cudaMemcpyAsync(wait, hist + n_freq, (size_t)n_wait * 8, kind, c->stream));
  if (!on_device) CK(cudaStreamSynchronize(c->stream));
  return CPM_OK;
}

int64_t cpm_get_threshold_table(cpm_ctx *c, uint32_t *thr, uint64_t cap) {
  if (!c) return CPM_ERR_ARG;
  for (uint64_t h = 0; thr && h < cap && h < c->thr.size(); ++h) thr[h] = c->thr[(size_t)h];
  return (int64_t)c->Hmax;
}

int cpm_get_launch_info(cpm_ctx *c, uint64_t out[6]) {
  if (!c || !out) return CPM_ERR_ARG;
  out[0] = c->launches; out[1] = c->sweep_launches; out[2] = (uint64_t)c->wpc; out[3] = (uint64_t)c->cta_smem;
  out[4] = c->use_tma ? 1 : 0; out[5] = c->pooled ? 1 : 0;
  return CPM_OK;
}

int cpm_set_kernel_timing(cpm_ctx *c, int enabled) {
  if (!c) return CPM_ERR_ARG;
  c->timing = enabled != 0;
  return CPM_OK;
}

int cpm_get_kernel_timing(cpm_ctx *c, double *ms_total, uint64_t *n, int reset) {
  if (!c) return CPM_ERR_ARG;
  CK(cudaSetDevice(c->device));
  CK(cudaStreamSynchronize(c->stream));
  double tot = 0;
  for (size_t i = 0; i + 1 < c->ev_used; i += 2) {
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, c->ev_pool[i], c->ev_pool[i + 1]));
    tot += ms;
  }
  if (ms_total) *ms_total = tot;
  if (n) *n = c->ev_used / 2;
  if (reset) c->ev_used = 0;
  return CPM_OK;
}

const char *cpm_last_error(const cpm_ctx *c) { return c ? c->err.c_str() : "null context"; }

int cpm_debug_philox(int device, const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n) {
  if (!ctr || !key || !out) return CPM_ERR_ARG;
  if (cudaSetDevice(device) != cudaSuccess) return CPM_ERR_CUDA;
  uint32_t *dc = nullptr, *dk = nullptr, *dout = nullptr;
  int rc = CPM_OK;
  if (cudaMalloc(&dc, n * 16) != cudaSuccess || cudaMalloc(&dk, n * 8) != cudaSuccess || cudaMalloc(&dout, n * 16) != cudaSuccess) rc = CPM_ERR_OOM;
  if (rc == CPM_OK) {
    cudaMemcpy(dc, ctr, n * 16, cudaMemcpyHostToDevice);
    cudaMemcpy(dk, key, n * 8, cudaMemcpyHostToDevice);
    philox_debug_kernel<<<(unsigned)((n + 255) / 256), 256>>>(dc, dk, dout, (long long)n);
    if (cudaMemcpy(out, dout, n * 16, cudaMemcpyDeviceToHost) != cudaSuccess) rc = CPM_ERR_CUDA;
  }
  cudaFree(dc); cudaFree(dk); cudaFree(dout);
  return rc;
}

}  // extern "C"
