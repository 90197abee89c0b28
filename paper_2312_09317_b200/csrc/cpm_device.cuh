// cpm_device.cuh -- sm_100a device code of the checkerboard CPM sweep: parameter blocks, PTX wrappers (mbarrier, TMA),
// Philox4x32-10, the pieces both sweep kernels share (Act side, vector-term bias, periodic image), the
// WARP-PER-SUBSECTION kernel (larger or non-power-of-two subsections, > 8 cell types) and the auxiliary kernels
// (Act decay, snapshot, pack / unpack / recount of the row-major layout, persistence, centroid tracking).  The
// pooled kernel for small subsections lives in cpm_pool_kernel.cuh, the instrumentation in cpm_stats_kernels.cuh.
//
// Warp-per-subsection kernel: one WARP owns one active checkerboard subsection for one activation:
//   a2  id tile + halo staged into shared memory by TMA (cp.async.bulk.tensor, OOB zero-fill =
//       "outside is medium"), completion on a per-warp mbarrier.  TMA needs the innermost start
//       coordinate at a 16-byte boundary (measured on B200: a 4-byte-aligned start raises
//       "illegal instruction"), so the tile starts at x0-4 words; the 1-byte Act tile is staged
//       with plain 32-bit loads while the TMA is in flight;
//   a3  Philox4x32-10: every lane draws one 128-bit block = 4 consecutive proposals -> 128 / batch;
//   a4  all 128 proposals are screened in parallel against the tile (same cell / frozen);
//   a5-a9 the surviving ("interesting") proposals are processed strictly in attempt order, one at
//       a time, with lanes = Moore neighbours: ballot/popc for n_A, n_B, REDUX for the adhesion sum;
//       after an accepted copy the not-yet-processed proposals are re-screened, so the result is
//       exactly that of k sequential attempts; acceptance words are drawn up front with the proposals;
//   a10 tile written back with 128-bit stores, integer deltas flushed with 64-bit atomics.
// Nothing here is shared with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace cpm {

constexpr uint32_t ID_MASK = 0x00FFFFFFu;   // lattice word = [frozen:1 | type:7 | id:24]
constexpr uint32_t FULL = 0xFFFFFFFFu;
constexpr int COUNTER_SLOTS = 256;

struct __align__(16) TypeParams {  // per cell type, Tables 1-3 of the paper
  int32_t lamV, tgtV, lamP, tgtP;
  int32_t lamA, maxA;
  int32_t cap;   // bound on this type's side of the Act bias: lamA * (largest Act value in the field) / maxA + 1
  int32_t pad1;
};

// Tiled lattice layout of the pooled kernel (cpm_pool_kernel.cuh): every subsection owns a tile of (S+2)^d
// words (its sites + a halo replicated from its neighbours); the tiles of 8 same-colour subsections
// (consecutive in the active-subsection order w) are interleaved: word j of subsection w of colour col at
// base[col] + (((w >> 3) * TW + j) << 3) + (w & 7) (or chain-major, see PK_CHAIN_MAJOR in cpm_pool_kernel.cuh).
struct TileLayout {
  uint32_t *tiles;
  unsigned long long base[8];   // word offset of the first group of each colour
  int nact[8][3];               // subsections of that colour per axis
  int S, TW;
};

struct SweepParams {
  uint32_t *lat;            // pitched lattice words (warp kernel; null with the tiled layout)
  uint8_t *act;             // pitched Act bytes (may be null)
  long long pitch;          // words per lattice row
  long long apitch;         // bytes per Act row
  int X, Y, Z;
  int per[3];
  int S, log2S, sites, k;   // subsection edge, log2 (or -1), S^d, attempts per activation
  int nsub[3];              // subsections per axis
  int nact[3];              // active subsections per axis for this colour
  uint32_t nact_mul[2], nact_shr[2];   // w / nact[a] = umulhi(w, mul) >> shr for w < 2^31 (host-built; mul = 0: nact[a] = 1)
  int col[3];               // colour bits of this phase-step
  unsigned long long n_active;
  uint32_t p;               // phase-step index rep*2^d + colour
  const uint32_t *mcs_ptr;  // device MCS counter
  uint32_t key0, key1;      // Philox key = seed
  int h;                    // halo (1; 2 with Act) in y and z
  int hx;                   // x offset of the subsection inside the tile (4: TMA start alignment)
  int TX, TY, TZ;           // tile extents in words (TX = S + 2*hx rounded up to 4)
  int AX;                   // Act tile row pitch in bytes (same x origin as the id tile)
  int tile_bytes, act_tile_bytes, warp_smem_bytes;
  int use_tma;
  const int32_t *J; int nT;
  const int32_t *D;         // pooled kernel: [nT][nT][nT][2] J(a,n) - J(b,n), then [nT] J(t,t)
  const TypeParams *types;
  const uint32_t *thr; long long Hmax; int accept_all;
  const int32_t *logq16;    // [256]
  const int32_t *expq16;    // [1024]
  const unsigned long long *snapVP;  // {V:hi32, P:lo32} per cell, phase-start snapshot
  unsigned long long *liveVP;
  unsigned long long *sumx, *sumy, *sumz;
  unsigned long long *cell_arr[4];   // {liveVP, sumx, sumy, sumz}: the commit lanes index it by their role
  unsigned long long *counters;      // [COUNTER_SLOTS][2] evaluated, accepted
  int *error_flag;
  // pooled kernel
  TileLayout tl;
  unsigned long long grp_base;       // word offset of this colour's first group
  uint32_t *ovf_keys;                // spill slots of the own-delta tables: [ovf_cap][PK_SPILL]
  unsigned long long *ovf_dvp;
  int *ovf_count; int ovf_cap;
  // vector terms (Eq 4-7, readings S21/S22); all in Q14
  int vec_on;                        // any lambda_pers / lambda_chem != 0
  const int2 *vec_types;             // [nT + 1] {lambda_pers, lambda_chem}; row nT (medium) is zero
  const short4 *pq;                  // [max_cells + 1] persistence direction of the cell (null: persistence off)
  const short4 *chem;                // [N] chemotaxis field, row-major x fastest (null: no field loaded)
  int xq_len[3];                     // llround(16384 / sqrt(n)), n = 1, 2, 3: component of the unit copy direction
  const int4 *lane_tab;              // pooled kernel: [32] {tile offset, dx, dy, dz} of Moore neighbour `lane` (zeros beyond nNb)
  const unsigned char *img; int img_bytes;   // pooled kernel: per-type records + adhesion table as they sit in shared memory (one bulk copy)
  const int *anc;                    // [max_cells + 1][3] anchors of the periodic centroid tracking (reading S23); null: off
};

// ------------------------------------------------------------------ PTX wrappers ----------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
               : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *tm, uint64_t *bar, int x, int y, int z) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
               ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *tm, uint64_t *bar, int x, int y) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
               ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(x), "r"(y) : "memory");
}

// ------------------------------------------------------------------ Philox4x32-10 ---------
// Salmon et al. 2011; counter-based, so any schedule reproduces the same stream (north_star (d)).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c.x;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c.z;
    c = make_uint4((uint32_t)(p1 >> 32) ^ c.y ^ k0, (uint32_t)p1, (uint32_t)(p0 >> 32) ^ c.w ^ k1, (uint32_t)p0);
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return c;
}
__device__ __forceinline__ uint32_t pick(const uint4 &v, int j) { return j == 0 ? v.x : j == 1 ? v.y : j == 2 ? v.z : v.w; }

// floor(lamA * g / maxA) of the Act term (reading S8) without a 64-bit division: lamA >= 0,
// 0 < maxA <= 255 and g < 2^24 (EXP entry < 2^17, shifted by at most 7), so with lamA = q maxA + r
// the result is q g + floor(r g / maxA) and r g < 2^32
__device__ __forceinline__ long long act_side(int lamA, int maxA, int g) {
  const unsigned q = (unsigned)lamA / (unsigned)maxA, r = (unsigned)lamA - q * (unsigned)maxA;
  return (long long)((unsigned long long)q * (unsigned)g) + (long long)((r * (unsigned)g) / (unsigned)maxA);
}

// Bias of the vector terms (Eq 4, 5; reading S21) for a copy from source s = t + (dx,dy,dz) into t: the unit vector of
// the copy direction is -(dx,dy,dz)/|.|; each real cell contributes lambda_pers(tau) x^.p^ and lambda_chem(tau) x^.C_s.
// rA / rB: parameter rows of the two cells (nT for medium); sidx: lattice index of the source site or -1 when it lies
// outside a closed lattice (no field there).  Returns the integer that is subtracted from dH.
__device__ __forceinline__ long long vec_bias(const SweepParams &P, int dx, int dy, int dz, int rA, int rB, uint32_t A, uint32_t B, long long sidx) {
  const int K = P.xq_len[dx * dx + dy * dy + dz * dz - 1];
  const int x0 = -dx * K, x1 = -dy * K, x2 = -dz * K;
  const int2 la = __ldg(P.vec_types + rA), lb = __ldg(P.vec_types + rB);
  long long acc = 0;
  if (P.pq != nullptr) {
    if (la.x != 0) { const short4 v = __ldg(P.pq + A); acc += (long long)la.x * (long long)(x0 * v.x + x1 * v.y + x2 * v.z); }
    if (lb.x != 0) { const short4 v = __ldg(P.pq + B); acc += (long long)lb.x * (long long)(x0 * v.x + x1 * v.y + x2 * v.z); }
  }
  const int lc = la.y + lb.y;
  if (lc != 0 && P.chem != nullptr && sidx >= 0) {
    const short4 v = __ldg(P.chem + sidx);
    acc += (long long)lc * (long long)(x0 * v.x + x1 * v.y + x2 * v.z);
  }
  return (acc + (1ll << 27)) >> 28;
}

// Reading S23 (L297): on a periodic axis a site's coordinate enters a cell's sum as the image nearest to the cell's anchor
__device__ __forceinline__ int image_near(int x, int anchor, int dim) {
  const int r = x - anchor;
  return (2 * r >= dim) ? x - dim : (2 * r < -dim) ? x + dim : x;
}
// coordinate of axis a (0..2) of a site as it enters the sums of `cell`
__device__ __forceinline__ int sum_coord(const SweepParams &P, uint32_t cell, int a, int x) {
  if (P.anc == nullptr || !P.per[a]) return x;
  return image_near(x, __ldg(P.anc + 3 * (size_t)cell + a), a == 0 ? P.X : a == 1 ? P.Y : P.Z);
}

// neighbour index (0..nNb-1, centre skipped) -> (dx,dy,dz); order: (dz,dy,dx) lexicographic, dx fastest
template <int DIM>
__device__ __forceinline__ void nb_delta(int nb, int &dx, int &dy, int &dz) {
  constexpr int half = (DIM == 2) ? 4 : 13;
  const int i = nb + (nb >= half ? 1 : 0);
  dx = i % 3 - 1;
  dy = (i / 3) % 3 - 1;
  dz = (DIM == 3) ? (i / 9 - 1) : 0;
}

// per-warp table of the cells this activation touched (own deltas, deterministic mode):
// entry e lives in lane e%32 of set e/32.
template <int NSETS>
struct CellTable {
  uint32_t key[NSETS];
  unsigned long long cur[NSETS];   // snapshot {V,P} + own composite delta
  unsigned long long dvp[NSETS];   // own composite delta: dV*2^32 + dP (mod 2^64)
  int dsx[NSETS], dsy[NSETS], dsz[NSETS];
};

template <int DIM, bool ACT, bool LIVE, int NSETS>
struct Sweep {
  static constexpr int NNB = (DIM == 2) ? 8 : 26;

  const SweepParams &P;
  uint32_t *tile;
  uint8_t *atile;
  const int32_t *sJ;        // shared copies of the small tables
  const TypeParams *sT;
  const int *sOff, *sAOff;  // neighbour index -> offset in the id tile / Act tile
  int lane;
  int doff, adoff;     // this lane's neighbour offset in the tile / Act tile (lane < NNB)
  int ox, oy, oz;      // lattice origin of the subsection
  uint32_t b;          // subsection index
  CellTable<NSETS> tab;
  int n_entries;
  bool dirty;
  bool overflow;

  __device__ Sweep(const SweepParams &p) : P(p) {}

  __device__ __forceinline__ void local_coords(int l, int &lx, int &ly, int &lz) const {
    if (P.log2S >= 0) {
      lx = l & (P.S - 1);
      ly = (l >> P.log2S) & (P.S - 1);
      lz = (DIM == 3) ? (l >> (2 * P.log2S)) : 0;
    } else {
      lx = l % P.S;
      const int r = l / P.S;
      ly = r % P.S;
      lz = (DIM == 3) ? (r / P.S) : 0;
    }
  }
  __device__ __forceinline__ int tile_pos(int lx, int ly, int lz) const {
    return ((DIM == 3 ? (lz + P.h) * P.TY : 0) + (ly + P.h)) * P.TX + lx + P.hx;
  }
  __device__ __forceinline__ int atile_pos(int lx, int ly, int lz) const {
    return ((DIM == 3 ? (lz + P.h) * P.TY : 0) + (ly + P.h)) * P.AX + lx + P.hx;
  }

  // ---- per-cell state as this attempt sees it (a6) ----
  // deterministic: snapshot + own deltas.  e = index of the cell's entry in the own-delta table, -1 when the cell has
  // not been CHANGED in this activation yet (looking at a cell does not take an entry, reading R2)
  __device__ __forceinline__ unsigned long long lookup(uint32_t cell, int &e) {
    e = -1;
    if (LIVE) return __ldcg(P.liveVP + cell);  // live, possibly stale (L53)
    unsigned long long cur = 0;
    bool found = false;
#pragma unroll
    for (int s = 0; s < NSETS; ++s) {
      const unsigned m = __ballot_sync(FULL, tab.key[s] == cell);
      if (m != 0 && !found) {
        const int src = __ffs(m) - 1;
        cur = __shfl_sync(FULL, tab.cur[s], src);
        e = s * 32 + src;
        found = true;
      }
    }
    return found ? cur : __ldg(P.snapVP + cell);
  }

  // vp: the value lookup() returned for this cell (its snapshot value when e < 0)
  __device__ __forceinline__ void add_delta(uint32_t cell, int e, unsigned long long vp, int dV, int dP, int x, int y, int z, int sgn) {
    // composite delta dV*2^32 + dP, mod 2^64 (the paper's interleaved pair, L297, updated by one add)
    const unsigned long long d = ((unsigned long long)(long long)dV << 32) + (unsigned long long)(long long)dP;
    if (LIVE) {
      if (lane == 0) {
        atomicAdd(P.liveVP + cell, d);
        atomicAdd(P.sumx + cell, (unsigned long long)(long long)(sgn * x));
        atomicAdd(P.sumy + cell, (unsigned long long)(long long)(sgn * y));
        if (DIM == 3) atomicAdd(P.sumz + cell, (unsigned long long)(long long)(sgn * z));
      }
      return;
    }
    if (e < 0) {   // first change of this cell in this activation: it takes an entry now
      if (n_entries >= 32 * NSETS) { overflow = true; return; }   // table full: reported, not computed approximately
      e = n_entries++;
#pragma unroll
      for (int s = 0; s < NSETS; ++s)
        if ((e >> 5) == s && lane == (e & 31)) {
          tab.key[s] = cell; tab.cur[s] = vp; tab.dvp[s] = 0ull; tab.dsx[s] = 0; tab.dsy[s] = 0; tab.dsz[s] = 0;
        }
    }
#pragma unroll
    for (int s = 0; s < NSETS; ++s)
      if ((e >> 5) == s && lane == (e & 31)) {
        tab.cur[s] += d; tab.dvp[s] += d; tab.dsx[s] += sgn * x; tab.dsy[s] += sgn * y; tab.dsz[s] += sgn * z;
      }
  }

  // fixed-point geometric mean of Act over {x} + same-cell Moore neighbours of x (Eq 9, reading S8)
  __device__ __forceinline__ int gm_q16(int pos, int apos, uint32_t id) {
    const bool in = lane <= NNB;
    const int mypos = pos + (lane < NNB ? doff : 0);
    const int myapos = apos + (lane < NNB ? adoff : 0);
    bool same = false;
    int a = 1;
    if (in) {
      same = (lane == NNB) || ((tile[mypos] & ID_MASK) == id);
      if (same) a = atile[myapos];
    }
    const unsigned msame = __ballot_sync(FULL, same);
    const unsigned mzero = __ballot_sync(FULL, same && a == 0);
    if (mzero) return 0;
    const int lg = same ? __ldg(P.logq16 + a) : 0;
    const int ssum = __reduce_add_sync(FULL, lg);
    const int n = __popc(msame);
    const int m = ssum / n;
    return __ldg(P.expq16 + ((m >> 6) & 1023)) << (m >> 16);
  }

  // One evaluated copy attempt (a5-a9) on tile positions tpos (target) / spos (source).
  // Warp-uniform control flow.  ureg / preg are THIS lane's acceptance word and packed (l | nb<<24)
  // of the current slot; the attempt's own values live in lane src and are fetched only when needed.
  // Returns true if the copy was committed.
  __device__ __forceinline__ bool evaluate(int tpos, int spos, int src, uint32_t ureg, int preg) {
    const uint32_t wA = tile[spos], wB = tile[tpos];
    const uint32_t A = wA & ID_MASK, B = wB & ID_MASK;
    // medium (id 0) has no constraints (reading S3): it reads the all-zero parameter row nT
    const int tA = (wA >> 24) & 127, tB = (wB >> 24) & 127;
    const int rA = (A != 0) ? tA : P.nT, rB = (B != 0) ? tB : P.nT;

    // neighbour census, lanes = Moore neighbours of t
    const bool nl = lane < NNB;
    const uint32_t wn = nl ? tile[tpos + doff] : 0u;
    const uint32_t idn = wn & ID_MASK;
    const int tn = (wn >> 24) & 127;
    const bool eA = nl && idn == A, eB = nl && idn == B;
    const int nA = __popc(__ballot_sync(FULL, eA));
    const int nB = __popc(__ballot_sync(FULL, eB));
    int adh_l = 0;
    if (nl) {
      const int ja = sJ[tA * P.nT + tn], jb = sJ[tB * P.nT + tn];
      adh_l = (eA ? 0 : ja) - (eB ? 0 : jb);
    }
    long long dH = __reduce_add_sync(FULL, adh_l);

    int entA = -1, entB = -1;
    unsigned long long vpA = 0, vpB = 0;
    if (A != 0) vpA = lookup(A, entA);
    if (B != 0) {
      vpB = lookup(B, entB);
      if ((uint32_t)(vpB >> 32) <= 1u) return false;  // a cell is never erased (reading S13)
    }

    // dH assembly (a7): every product is 32x32 -> 64 or 64x32 (ranges validated by cpm_create)
    const TypeParams pa = sT[rA], pb = sT[rB];
    const int dPA = NNB - 2 * nA, dPB = 2 * nB - NNB;
    {
      const int dva = (int)(uint32_t)(vpA >> 32) - pa.tgtV, dvb = (int)(uint32_t)(vpB >> 32) - pb.tgtV;
      dH += 2 * ((long long)pa.lamV * dva - (long long)pb.lamV * dvb) + (pa.lamV + pb.lamV);
      const long long dpa = (long long)(uint32_t)vpA - pa.tgtP, dpb = (long long)(uint32_t)vpB - pb.tgtP;
      dH += (long long)(pa.lamP * dPA) * (2 * dpa + dPA) + (long long)(pb.lamP * dPB) * (2 * dpb + dPB);
    }
    if (P.vec_on) {   // warp-uniform
      const int pr = __shfl_sync(FULL, preg, src);
      int lx, ly, lz, dx, dy, dz;
      local_coords(pr & 0xFFFFFF, lx, ly, lz);
      nb_delta<DIM>((pr >> 24) & 31, dx, dy, dz);
      int g[3] = {ox + lx + dx, oy + ly + dy, (DIM == 3) ? oz + lz + dz : 0};
      const int dimv[3] = {P.X, P.Y, P.Z};
      bool inside = true;
#pragma unroll
      for (int ax = 0; ax < DIM; ++ax)
        if (g[ax] < 0 || g[ax] >= dimv[ax]) { if (P.per[ax]) g[ax] += (g[ax] < 0) ? dimv[ax] : -dimv[ax]; else inside = false; }
      const long long sidx = inside ? (long long)g[0] + (long long)P.X * ((long long)g[1] + (long long)P.Y * g[2]) : -1ll;
      dH -= vec_bias(P, dx, dy, dz, rA, rB, A, B, sidx);
    }
    if (ACT) {
      if ((pa.lamA | pb.lamA) != 0) {  // lamA is stored as 0 when the type's Max_act is 0
        const int pr = __shfl_sync(FULL, preg, src);
        int lx, ly, lz;
        local_coords(pr & 0xFFFFFF, lx, ly, lz);
        const int atpos = atile_pos(lx, ly, lz);
        long long sideA = 0, sideB = 0;
        if (pa.lamA != 0) {
          const int g = gm_q16(spos, atpos + sAOff[(pr >> 24) & 31], A);
          if (g != 0) sideA = act_side(pa.lamA, pa.maxA, g);
        }
        if (pb.lamA != 0) {
          const int g = gm_q16(tpos, atpos, B);
          if (g != 0) sideB = act_side(pb.lamA, pb.maxA, g);
        }
        dH -= (sideA - sideB + 32768) >> 16;  // copies FROM active areas are favoured (L259)
      }
    }

    // Metropolis (Eq 2) with the integer threshold table
    if (dH > 0 && !P.accept_all) {
      if (dH > P.Hmax) return false;
      if (__shfl_sync(FULL, ureg, src) >= __ldg(P.thr + dH)) return false;
    }

    // commit (a9)
    const int l = __shfl_sync(FULL, preg, src) & 0xFFFFFF;
    int lx, ly, lz;
    local_coords(l, lx, ly, lz);
    if (lane == 0) {
      tile[tpos] = wA;  // id and type of the source; neither site is frozen
      if (ACT) atile[atile_pos(lx, ly, lz)] = (uint8_t)pa.maxA;   // Max_act of the new owner; 0 for medium
    }
    __syncwarp();
    dirty = true;
    const int gx = ox + lx, gy = oy + ly, gz = oz + lz;
    if (A != 0) add_delta(A, entA, vpA, 1, dPA, sum_coord(P, A, 0, gx), sum_coord(P, A, 1, gy), sum_coord(P, A, 2, gz), +1);
    if (B != 0) add_delta(B, entB, vpB, -1, dPB, sum_coord(P, B, 0, gx), sum_coord(P, B, 1, gy), sum_coord(P, B, 2, gz), -1);
    return true;
  }

  // lattice coordinate of tile element (lx,ly,lz) under the boundary rule; false = outside (medium)
  __device__ __forceinline__ bool resolve(int lx, int ly, int lz, int &gx, int &gy, int &gz) const {
    int g[3] = {ox - P.hx + lx, oy - P.h + ly, (DIM == 3) ? oz - P.h + lz : 0};
    const int dimv[3] = {P.X, P.Y, P.Z};
    bool inside = true;
#pragma unroll
    for (int ax = 0; ax < DIM; ++ax) {
      if (g[ax] < 0 || g[ax] >= dimv[ax]) {
        if (P.per[ax]) g[ax] = (g[ax] % dimv[ax] + dimv[ax]) % dimv[ax];
        else inside = false;
      }
    }
    gx = g[0]; gy = g[1]; gz = g[2];
    return inside;
  }

  // ---- id tile staging without TMA (periodic wrap across the lattice border, S % 4 != 0, or TMA off) ----
  __device__ void load_tile_manual() {
    const int n = P.TX * P.TY * P.TZ;
    for (int i = lane; i < n; i += 32) {
      const int lx = i % P.TX;
      const int r = i / P.TX;
      int gx, gy, gz;
      const bool inside = resolve(lx, r % P.TY, r / P.TY, gx, gy, gz);
      tile[i] = inside ? P.lat[(long long)gx + P.pitch * ((long long)gy + (long long)P.Y * gz)] : 0u;
    }
  }

  // ---- Act tile staging: 32-bit loads (4 voxels) when rows are word aligned, bytes otherwise ----
  __device__ void load_act_tile() {
    const int rows = P.TY * P.TZ;
    if ((P.S & 3) == 0) {
      const int wpr = P.AX >> 2;   // words per tile row
      uint32_t *at32 = reinterpret_cast<uint32_t *>(atile);
      // lanes walk the (row, word) grid without divisions: lane -> (r0, q0), then fixed strides
      int q = lane % wpr, r = lane / wpr;
      const int dq = 32 % wpr, dr = 32 / wpr;
      int ly = r % P.TY, lz = r / P.TY;
      while (r < rows) {
        int gx, gy, gz;
        // X is a multiple of S (hence of 4): a word never straddles the lattice border
        const bool inside = resolve(4 * q, ly, lz, gx, gy, gz);
        at32[r * wpr + q] = inside ? *reinterpret_cast<const uint32_t *>(P.act + (long long)gx + P.apitch * ((long long)gy + (long long)P.Y * gz)) : 0u;
        q += dq; int adv = dr;
        if (q >= wpr) { q -= wpr; ++adv; }
        r += adv; ly += adv;
        while (ly >= P.TY) { ly -= P.TY; ++lz; }
      }
    } else {
      const int n = P.AX * rows;
      for (int i = lane; i < n; i += 32) {
        const int lx = i % P.AX;
        const int r = i / P.AX;
        int gx, gy, gz;
        const bool inside = resolve(lx, r % P.TY, r / P.TY, gx, gy, gz);
        atile[i] = inside ? P.act[(long long)gx + P.apitch * ((long long)gy + (long long)P.Y * gz)] : (uint8_t)0;
      }
    }
  }

  // ---- write the interior of the tile back (a10) ----
  __device__ void store_tile() {
    const int S = P.S;
    const int rows = (DIM == 3) ? S * S : S;
    if (P.log2S >= 2) {  // 128-bit stores: x0 is a multiple of S, the pitch a multiple of 4 words
      const int lq = P.log2S - 2;  // log2(quads per row)
      for (int i = lane; i < (rows << lq); i += 32) {
        const int q = i & ((1 << lq) - 1), r = i >> lq;
        const int ly = r & (S - 1), lz = r >> P.log2S;
        const int tp = tile_pos(4 * q, ly, lz);
        const uint4 v = make_uint4(tile[tp], tile[tp + 1], tile[tp + 2], tile[tp + 3]);
        const long long gi = (long long)(ox + 4 * q) + P.pitch * ((long long)(oy + ly) + (long long)P.Y * (oz + lz));
        *reinterpret_cast<uint4 *>(P.lat + gi) = v;
        if (ACT) {
          const long long ga = (long long)(ox + 4 * q) + P.apitch * ((long long)(oy + ly) + (long long)P.Y * (oz + lz));
          *reinterpret_cast<uint32_t *>(P.act + ga) = *reinterpret_cast<const uint32_t *>(atile + atile_pos(4 * q, ly, lz));
        }
      }
    } else {
      for (int i = lane; i < rows * S; i += 32) {
        const int lx = i % S, r = i / S;
        const int ly = r % S, lz = r / S;
        const long long gi = (long long)(ox + lx) + P.pitch * ((long long)(oy + ly) + (long long)P.Y * (oz + lz));
        P.lat[gi] = tile[tile_pos(lx, ly, lz)];
        if (ACT) {
          const long long ga = (long long)(ox + lx) + P.apitch * ((long long)(oy + ly) + (long long)P.Y * (oz + lz));
          P.act[ga] = atile[atile_pos(lx, ly, lz)];
        }
      }
    }
  }

  __device__ void flush_table() {
    if constexpr (!LIVE) {
#pragma unroll
      for (int s = 0; s < NSETS; ++s) {
        if (s * 32 + lane < n_entries) {
          const uint32_t c = tab.key[s];
          if (tab.dvp[s] != 0ull) atomicAdd(P.liveVP + c, tab.dvp[s]);
          if (tab.dsx[s] != 0) atomicAdd(P.sumx + c, (unsigned long long)(long long)tab.dsx[s]);
          if (tab.dsy[s] != 0) atomicAdd(P.sumy + c, (unsigned long long)(long long)tab.dsy[s]);
          if (DIM == 3 && tab.dsz[s] != 0) atomicAdd(P.sumz + c, (unsigned long long)(long long)tab.dsz[s]);
        }
      }
    }
  }

  // ---- the whole activation of one subsection ----
  __device__ void run(unsigned long long w, uint32_t *tile_, uint8_t *atile_, uint64_t *bar,
                      const CUtensorMap *tm_lat) {
    tile = tile_; atile = atile_;
    lane = threadIdx.x & 31;
    dirty = false; overflow = false; n_entries = 0;
#pragma unroll
    for (int s = 0; s < NSETS; ++s) { tab.key[s] = 0xFFFFFFFFu; tab.cur[s] = 0; tab.dvp[s] = 0; tab.dsx[s] = tab.dsy[s] = tab.dsz[s] = 0; }
    const uint32_t mcs = *P.mcs_ptr;

    // active subsection -> lattice origin
    const int ax = (int)(w % (unsigned)P.nact[0]);
    const unsigned long long r1 = w / (unsigned)P.nact[0];
    const int ay = (int)(r1 % (unsigned)P.nact[1]);
    const int az = (int)(r1 / (unsigned)P.nact[1]);
    const int bx = 2 * ax + P.col[0], by = 2 * ay + P.col[1], bz = (DIM == 3) ? 2 * az + P.col[2] : 0;
    b = (uint32_t)(bx + P.nsub[0] * (by + P.nsub[1] * bz));
    ox = bx * P.S; oy = by * P.S; oz = (DIM == 3) ? bz * P.S : 0;
    doff = (lane < NNB) ? sOff[lane] : 0;
    adoff = (lane < NNB) ? sAOff[lane] : 0;

    // a2: stage tile + halo
    bool tma = P.use_tma != 0;
    if (tma) {
      const int lo[3] = {ox - P.hx, oy - P.h, oz - P.h};
      const int ext[3] = {P.TX, P.TY, P.TZ};
      const int dimv[3] = {P.X, P.Y, P.Z};
#pragma unroll
      for (int a2 = 0; a2 < DIM; ++a2)
        if (P.per[a2] && (lo[a2] < 0 || lo[a2] + ext[a2] > dimv[a2])) tma = false;  // wrap: manual path
    }
    if (tma) {
      if (lane == 0) {
        mbar_expect_tx(bar, (uint32_t)P.tile_bytes);
        if (DIM == 3) tma_load_3d(tile, tm_lat, bar, ox - P.hx, oy - P.h, oz - P.h);
        else tma_load_2d(tile, tm_lat, bar, ox - P.hx, oy - P.h);
      }
      if (ACT) load_act_tile();  // overlaps the TMA
    } else {
      load_tile_manual();
      if (ACT) load_act_tile();
    }

    // a3-a9: k sequential attempts in blocks of 128: lane L draws Philox call (a0>>2) + L, whose four
    // words are attempts a0 + 4L + j, j = 0..3 (reading S15); the sequential order is (L, j) lexicographic.
    const uint32_t k = (uint32_t)P.k;
    uint32_t n_eval = 0, n_acc = 0;
    bool staged = false;
    for (uint32_t a0 = 0; a0 < k; a0 += 128) {
      const uint32_t q = (a0 >> 2) + lane;
      int prop[4];       // l | nb << 24
      int ts[4];         // tpos | spos << 16
      uint32_t u[4];     // acceptance words (Philox stream 1), drawn with the proposals so that the
                         // sequential part below never waits for a Philox
      {
        const uint4 r = philox4x32_10(make_uint4(q, b, 2u * P.p, mcs), P.key0, P.key1);
        const uint4 ua = philox4x32_10(make_uint4(q, b, 2u * P.p + 1u, mcs), P.key0, P.key1);
        u[0] = ua.x; u[1] = ua.y; u[2] = ua.z; u[3] = ua.w;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const uint32_t wj = pick(r, j);
          const uint64_t prod = (uint64_t)wj * (uint32_t)P.sites;
          const int l = (int)(prod >> 32);
          const int nb = (int)(((uint64_t)(uint32_t)prod * (uint32_t)NNB) >> 32);
          int lx, ly, lz;
          local_coords(l, lx, ly, lz);
          const int tp = tile_pos(lx, ly, lz);
          const int sp = tp + sOff[nb];
          prop[j] = l | (nb << 24);
          ts[j] = tp | (sp << 16);
        }
      }
      if (!staged) {  // first use of the tile: wait for the TMA (the Philox above overlapped it)
        if (tma) { while (!mbar_try_wait(bar, 0)) {} }
        __syncwarp();
        staged = true;
      }
      // a4: screen all 128 proposals against the current tile; m[j] = lanes whose slot j is interesting
      auto screen = [&](int tsj, bool valid) -> unsigned {
        const uint32_t wt = tile[tsj & 0xFFFF], ws = tile[(uint32_t)tsj >> 16];
        return __ballot_sync(FULL, valid && (((wt ^ ws) & ID_MASK) != 0u) && ((int)(wt | ws) >= 0));
      };
      unsigned m[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) m[j] = screen(ts[j], a0 + 4u * lane + j < k);
      while (true) {
        const unsigned any = m[0] | m[1] | m[2] | m[3];
        if (any == 0u) break;
        const int src = __ffs(any) - 1;            // first lane with an interesting slot ...
        const unsigned bit = 1u << src;
        const int j = (m[0] & bit) ? 0 : (m[1] & bit) ? 1 : (m[2] & bit) ? 2 : 3;   // ... and its first such slot
        const int tsv = j == 0 ? ts[0] : j == 1 ? ts[1] : j == 2 ? ts[2] : ts[3];
        const uint32_t uv = j == 0 ? u[0] : j == 1 ? u[1] : j == 2 ? u[2] : u[3];
        const int pv = j == 0 ? prop[0] : j == 1 ? prop[1] : j == 2 ? prop[2] : prop[3];
        const int tsel = __shfl_sync(FULL, tsv, src);
        ++n_eval;
        const bool acc = evaluate(tsel & 0xFFFF, (int)((uint32_t)tsel >> 16), src, uv, pv);
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) if (jj == j) m[jj] &= ~bit;   // attempt (src, j) is done
        if (acc) {                                                    // later attempts see the new tile
          ++n_acc;
          const unsigned after = ~((2u << src) - 1u);
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) {
            const unsigned r = screen(ts[jj], a0 + 4u * lane + jj < k);
            m[jj] = r & (after | (jj > j ? bit : 0u));
          }
        }
      }
    }

    // a10: write back, flush deltas
    if (dirty) store_tile();
    flush_table();
    if (lane == 0) {
      const int slot = (int)(blockIdx.x % COUNTER_SLOTS);
      if (n_eval) atomicAdd(P.counters + 2 * slot, (unsigned long long)n_eval);
      if (n_acc) atomicAdd(P.counters + 2 * slot + 1, (unsigned long long)n_acc);
      if (overflow) atomicOr(P.error_flag, 1);
    }
  }
};

// One warp per active subsection.  Dynamic smem: per warp [id tile | Act tile], then the mbarriers,
// then the CTA's copies of the small tables (J, per-type parameters, neighbour offsets).
template <int DIM, bool ACT, bool LIVE, int NSETS>
__global__ void __launch_bounds__(128) sweep_kernel(const __grid_constant__ CUtensorMap tm_lat,
                                                    const __grid_constant__ SweepParams P) {
  extern __shared__ __align__(128) unsigned char smem[];
  constexpr int NNB = (DIM == 2) ? 8 : 26;
  const int warp = threadIdx.x >> 5;
  const int nwarps = blockDim.x >> 5;
  const unsigned long long w = (unsigned long long)blockIdx.x * nwarps + warp;
  unsigned char *tabs = smem + (size_t)nwarps * P.warp_smem_bytes;
  uint64_t *bars = reinterpret_cast<uint64_t *>(tabs);
  int *sOff = reinterpret_cast<int *>(tabs + 64);
  int *sAOff = sOff + 32;
  TypeParams *sT = reinterpret_cast<TypeParams *>(tabs + 64 + 256);
  int32_t *sJ = reinterpret_cast<int32_t *>(tabs + 64 + 256 + (size_t)(P.nT + 1) * sizeof(TypeParams));
  for (int i = threadIdx.x; i < P.nT * P.nT; i += blockDim.x) sJ[i] = P.J[i];
  for (int i = threadIdx.x; i < (P.nT + 1) * 8; i += blockDim.x)   // P.types has nT + 1 rows, the last all zero
    reinterpret_cast<int32_t *>(sT)[i] = reinterpret_cast<const int32_t *>(P.types)[i];
  if (threadIdx.x < 32) {
    int dx = 0, dy = 0, dz = 0;
    if (threadIdx.x < NNB) nb_delta<DIM>(threadIdx.x, dx, dy, dz);
    sOff[threadIdx.x] = (dz * P.TY + dy) * P.TX + dx;
    sAOff[threadIdx.x] = (dz * P.TY + dy) * P.AX + dx;
  }
  if ((threadIdx.x & 31) == 0) {
    mbar_init(&bars[warp], 1);
    fence_mbar_init();
  }
  __syncthreads();
  if (w >= P.n_active) return;
  unsigned char *mine = smem + (size_t)warp * P.warp_smem_bytes;
  uint32_t *tile = reinterpret_cast<uint32_t *>(mine);
  uint8_t *atile = mine + ((P.tile_bytes + 127) & ~127);
  Sweep<DIM, ACT, LIVE, NSETS> sw(P);
  sw.sJ = sJ; sw.sT = sT; sw.sOff = sOff; sw.sAOff = sAOff;
  sw.run(w, tile, atile, &bars[warp], &tm_lat);
}

// ------------------------------------------------------------------ auxiliary kernels ------
// a11: Act decays by 1 per MCS down to 0 (L255); 16 bytes per thread, saturating byte subtract.
__global__ void act_decay_kernel(uint4 *act, long long n_vec, uint32_t *mcs_ptr, uint32_t *pers_n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) { *mcs_ptr += 1; if (pers_n) *pers_n += 1; }
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long j = i; j < n_vec; j += stride) {
    uint4 v = act[j];
    v.x = __vsubus4(v.x, 0x01010101u); v.y = __vsubus4(v.y, 0x01010101u);
    v.z = __vsubus4(v.z, 0x01010101u); v.w = __vsubus4(v.w, 0x01010101u);
    act[j] = v;
  }
}
// deterministic mode, after every phase-step: snapshot := live (reading S12) and the spill-slot counter of the pooled kernel
// back to 0 for the next phase-step -- one launch instead of a copy node and a memset node
__global__ void snapshot_kernel(const ulonglong2 *live, ulonglong2 *snap, long long n_pairs, int *ovf_count) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0 && ovf_count) *ovf_count = 0;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long j = i; j < n_pairs; j += stride) snap[j] = live[j];
}
__global__ void mcs_increment_kernel(uint32_t *mcs_ptr, uint32_t *pers_n) { *mcs_ptr += 1; if (pers_n) *pers_n += 1; }

// ---- periodic centroid tracking (L297, reading S23) ----
// set_lattice: the first site of every cell in scan order (lowest linear index) ...
__global__ void anchor_first_site_kernel(const uint32_t *ids, long long N, uint32_t max_cells, unsigned long long *first) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
    const uint32_t id = ids[i];
    if (id != 0 && id <= max_cells) atomicMin(first + id, (unsigned long long)i);
  }
}
// ... becomes its anchor
__global__ void anchor_from_first_kernel(long long ncell, const unsigned long long *first, int X, int Y, int *anc) {
  const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cell >= ncell) return;
  const unsigned long long f = first[cell];
  const bool have = cell != 0 && f != ~0ull;
  anc[3 * cell] = have ? (int)(f % (unsigned)X) : 0;
  anc[3 * cell + 1] = have ? (int)((f / (unsigned)X) % (unsigned)Y) : 0;
  anc[3 * cell + 2] = have ? (int)(f / ((unsigned long long)X * (unsigned)Y)) : 0;
}
// after the recount and after every MCS: centroid back into [0, dim) on periodic axes, the anchor follows the centroid
__global__ void centroid_normalise_kernel(long long ncell, const unsigned long long *liveVP, unsigned long long *sumx,
                                          unsigned long long *sumy, unsigned long long *sumz, int *anc, int X, int Y, int Z,
                                          int perx, int pery, int perz) {
  const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cell < 1 || cell >= ncell) return;
  const long long v = (long long)(uint32_t)(liveVP[cell] >> 32);
  if (v <= 0) return;
  unsigned long long *S[3] = {sumx, sumy, sumz};
  const int dimv[3] = {X, Y, Z}, per[3] = {perx, pery, perz};
  for (int a = 0; a < 3; ++a) {
    if (!per[a]) continue;
    const long long span = (long long)dimv[a] * v;
    long long s = (long long)S[a][cell] % span;
    if (s < 0) s += span;
    S[a][cell] = (unsigned long long)s;
    anc[3 * cell + a] = (int)(s / v);
  }
}

// ---- persistence (Eq 5-7, reading S22) ----
// Q14 of a direction: what the sweep reads
__device__ __forceinline__ short4 quantise_q14(double x, double y, double z) {
  return make_short4((short)__double2ll_rn(__dmul_rn(16384.0, x)), (short)__double2ll_rn(__dmul_rn(16384.0, y)),
                     (short)__double2ll_rn(__dmul_rn(16384.0, z)), 0);
}
// centroid, Eq 10: coordinate sums over volume, one IEEE division each
__device__ __forceinline__ void centroid_of(unsigned long long vp, unsigned long long sx, unsigned long long sy, unsigned long long sz, double X[3]) {
  const double v = (double)(uint32_t)(vp >> 32);
  X[0] = __ddiv_rn((double)(long long)sx, v); X[1] = __ddiv_rn((double)(long long)sy, v); X[2] = __ddiv_rn((double)(long long)sz, v);
}
// cpm_set_lattice: p^ = 0 for every cell, every slot of the look-back ring = the present centroid
__global__ void persistence_init_kernel(long long ncell, int slots, const unsigned long long *liveVP, const unsigned long long *sumx,
                                        const unsigned long long *sumy, const unsigned long long *sumz, double *phat, short4 *pq,
                                        double *ring, uint32_t *pers_n) {
  const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cell == 0) *pers_n = 0;
  if (cell >= ncell) return;
  double X[3] = {0.0, 0.0, 0.0};
  const unsigned long long vp = liveVP[cell];
  if (cell != 0 && (uint32_t)(vp >> 32) != 0u) centroid_of(vp, sumx[cell], sumy[cell], sumz[cell], X);
  for (int a = 0; a < 3; ++a) phat[3 * cell + a] = 0.0;
  pq[cell] = make_short4(0, 0, 0, 0);
  for (int sl = 0; sl < slots; ++sl)
    for (int a = 0; a < 3; ++a) ring[((long long)sl * ncell + cell) * 3 + a] = X[a];
}
// Once per MCS, one thread per cell: p = (1 - mu) (X_t - X_{t-dt}) / |X_t - X_{t-dt}| + mu p^_{t-1}; p^_t = p / |p| (Eq 6-7).
// Every step is one IEEE double operation (no fused multiply-add), so the result is the same on any conforming machine.
__global__ void persistence_update_kernel(long long ncell, int slots, const unsigned long long *liveVP, const unsigned long long *sumx,
                                          const unsigned long long *sumy, const unsigned long long *sumz, const uint8_t *ctype,
                                          const double *mu_of_type, double *phat, short4 *pq, double *ring, const uint32_t *pers_n,
                                          int wrapx, int wrapy, int wrapz) {
  const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cell < 1 || cell >= ncell) return;
  const unsigned long long vp = liveVP[cell];
  if ((uint32_t)(vp >> 32) == 0u) return;
  const unsigned long long n = (unsigned long long)*pers_n + 1ull;    // this is the n-th update
  const double *old_slot = ring + (long long)((n + 1ull) % (unsigned long long)slots) * ncell * 3;   // (n - dt) mod (dt + 1)
  double *new_slot = ring + (long long)(n % (unsigned long long)slots) * ncell * 3;
  double X[3], d[3], p[3];
  centroid_of(vp, sumx[cell], sumy[cell], sumz[cell], X);
  const double mu = mu_of_type[ctype[cell]];
  const double one_minus_mu = __dsub_rn(1.0, mu);
  const int wrap[3] = {wrapx, wrapy, wrapz};   // dim of the axes whose centroids are tracked through the periodic border, else 0
  for (int a = 0; a < 3; ++a) {
    d[a] = __dsub_rn(X[a], old_slot[3 * cell + a]);
    if (wrap[a] != 0) {   // shortest displacement through the border (reading S23)
      const double half = __dmul_rn(0.5, (double)wrap[a]);
      if (d[a] > half) d[a] = __dsub_rn(d[a], (double)wrap[a]);
      else if (d[a] < -half) d[a] = __dadd_rn(d[a], (double)wrap[a]);
    }
  }
  const double dn = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2])));
  for (int a = 0; a < 3; ++a) {
    const double keep = __dmul_rn(mu, phat[3 * cell + a]);
    p[a] = (dn > 0.0) ? __dadd_rn(__dmul_rn(one_minus_mu, __ddiv_rn(d[a], dn)), keep) : keep;
  }
  const double pn = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(p[0], p[0]), __dmul_rn(p[1], p[1])), __dmul_rn(p[2], p[2])));
  for (int a = 0; a < 3; ++a) p[a] = (pn > 0.0) ? __ddiv_rn(p[a], pn) : 0.0;
  for (int a = 0; a < 3; ++a) { phat[3 * cell + a] = p[a]; new_slot[3 * cell + a] = X[a]; }
  pq[cell] = quantise_q14(p[0], p[1], p[2]);
}
// cpm_set_persistence: p^ from the caller (components in [-1,1]) and its Q14 copy
// commit == 0: only validate (nothing is written when any component is out of range)
__global__ void persistence_set_kernel(long long ncell, const double *src, double *phat, short4 *pq, int *error_flag, int commit) {
  const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cell >= ncell) return;
  double v[3];
  for (int a = 0; a < 3; ++a) {
    v[a] = src[3 * cell + a];
    if (!(v[a] >= -1.0 && v[a] <= 1.0)) { atomicOr(error_flag, 8); return; }
  }
  if (!commit) return;
  for (int a = 0; a < 3; ++a) phat[3 * cell + a] = v[a];
  pq[cell] = (cell == 0) ? make_short4(0, 0, 0, 0) : quantise_q14(v[0], v[1], v[2]);
}
// cpm_set_chemotaxis_field: float components in [-1,1] -> Q14 (round to nearest even), one short4 per site
// commit == 0: only validate
__global__ void chem_set_kernel(const float *src, short4 *chem, long long N, int ndim, int *error_flag, int commit) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
    short q[3] = {0, 0, 0};
    bool ok = true;
    for (int a = 0; a < ndim; ++a) {
      const float v = src[i * ndim + a];
      if (!(v >= -1.0f && v <= 1.0f)) { ok = false; break; }
      q[a] = (short)__float2int_rn(__fmul_rn(v, 16384.0f));
    }
    if (!ok) { atomicOr(error_flag, 8); continue; }
    if (commit) chem[i] = make_short4(q[0], q[1], q[2], 0);
  }
}

// set_lattice: ids (+frozen, cell types) -> packed pitched words; flags ids above max_cells
__global__ void pack_kernel(const uint32_t *ids, const uint8_t *frozen, const uint8_t *ctype, uint32_t max_cells,
                            uint32_t *lat, long long pitch, int X, int Y, int Z, int *error_flag) {
  const long long N = (long long)X * Y * Z;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
    const int x = (int)(i % X);
    const long long r = i / X;
    uint32_t id = ids[i];
    if (id > max_cells) { atomicOr(error_flag, 2); id = 0; }
    const uint32_t w = id | ((uint32_t)ctype[id] << 24) | ((frozen && frozen[i]) ? 0x80000000u : 0u);
    lat[(long long)x + pitch * r] = w;
  }
}
__global__ void unpack_kernel(const uint32_t *lat, long long pitch, int X, int Y, int Z, uint32_t *ids) {
  const long long N = (long long)X * Y * Z;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
    const int x = (int)(i % X);
    const long long r = i / X;
    ids[i] = lat[(long long)x + pitch * r] & ID_MASK;
  }
}
__global__ void act_set_kernel(const float *src, uint8_t *act, long long apitch, int X, int Y, int Z, int *error_flag) {
  const long long N = (long long)X * Y * Z;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
    const int x = (int)(i % X);
    const long long r = i / X;
    const float v = src[i];
    if (!(v >= 0.f) || v > 255.f || v != floorf(v)) atomicOr(error_flag, 4);
    act[(long long)x + apitch * r] = (uint8_t)fminf(fmaxf(v, 0.f), 255.f);
  }
}
__global__ void act_get_kernel(const uint8_t *act, long long apitch, int X, int Y, int Z, float *dst) {
  const long long N = (long long)X * Y * Z;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
    const int x = (int)(i % X);
    const long long r = i / X;
    dst[i] = act ? (float)act[(long long)x + apitch * r] : 0.f;
  }
}

// recount of the per-cell globals from the lattice: V (L225), A = Moore interfaces with sites not
// of the same cell (L234; outside-medium counts as foreign), coordinate sums (L288).
// Lanes of a warp that hold the same cell id (runs along x) are combined with match_any + REDUX so
// that one lane issues the atomics for the whole group.
template <int DIM>
__global__ void recount_kernel(const uint32_t *lat, long long pitch, int X, int Y, int Z, int perx, int pery, int perz,
                               unsigned long long *liveVP, unsigned long long *sumx, unsigned long long *sumy,
                               unsigned long long *sumz, const int *anc) {
  const long long N = (long long)X * Y * Z;
  const long long stride = (long long)gridDim.x * blockDim.x;
  const int per[3] = {perx, pery, perz};
  const int dimv[3] = {X, Y, Z};
  constexpr int NNB = (DIM == 2) ? 8 : 26;
  const long long first = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long n_iter = (N + stride - 1) / stride;   // same trip count for every lane of a warp
  for (long long it = 0; it < n_iter; ++it) {
    const long long i = first + it * stride;
    uint32_t me = 0;
    int x = 0, y = 0, z = 0, foreign = 0;
    if (i < N) {
      x = (int)(i % X);
      const long long r = i / X;
      y = (int)(r % Y); z = (int)(r / Y);
      me = lat[(long long)x + pitch * r] & ID_MASK;
      if (me != 0) {
        for (int nb = 0; nb < NNB; ++nb) {
          int dx, dy, dz;
          nb_delta<DIM>(nb, dx, dy, dz);
          int g[3] = {x + dx, y + dy, z + dz};
          bool inside = true;
#pragma unroll
          for (int a = 0; a < DIM; ++a) {
            if (g[a] < 0 || g[a] >= dimv[a]) {
              if (per[a]) g[a] = (g[a] + dimv[a]) % dimv[a];
              else inside = false;
            }
          }
          const uint32_t other = inside ? (lat[(long long)g[0] + pitch * ((long long)g[1] + (long long)Y * g[2])] & ID_MASK) : 0u;
          foreign += (other != me);
        }
      }
    }
    if (anc != nullptr && me != 0) {   // reading S23: the image of the site nearest to the cell's anchor
      if (perx) x = image_near(x, anc[3 * (size_t)me], X);
      if (pery) y = image_near(y, anc[3 * (size_t)me + 1], Y);
      if (perz) z = image_near(z, anc[3 * (size_t)me + 2], Z);
    }
    const unsigned peers = __match_any_sync(FULL, me);
    const unsigned cnt = __popc(peers);
    const unsigned f = __reduce_add_sync(peers, (unsigned)foreign);
    const unsigned sx = __reduce_add_sync(peers, (unsigned)x);
    const unsigned sy = __reduce_add_sync(peers, (unsigned)y);
    const unsigned sz = (DIM == 3) ? __reduce_add_sync(peers, (unsigned)z) : 0u;
    if (me != 0 && (int)(threadIdx.x & 31) == __ffs(peers) - 1) {
      atomicAdd(liveVP + me, ((unsigned long long)cnt << 32) + (unsigned long long)f);
      atomicAdd(sumx + me, (unsigned long long)(long long)(int)sx);   // images may be negative
      atomicAdd(sumy + me, (unsigned long long)(long long)(int)sy);
      if (DIM == 3) atomicAdd(sumz + me, (unsigned long long)(long long)(int)sz);
    }
  }
}
__global__ void stats_unpack_kernel(const unsigned long long *liveVP, long long n, uint32_t *V, uint32_t *Pm) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const unsigned long long v = (i == 0) ? 0ull : liveVP[i];
  if (V) V[i] = (uint32_t)(v >> 32);
  if (Pm) Pm[i] = (uint32_t)v;
}
__global__ void philox_debug_kernel(const uint32_t *ctr, const uint32_t *key, uint32_t *out, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 r = philox4x32_10(make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]), key[2 * i], key[2 * i + 1]);
  out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

}  // namespace cpm
