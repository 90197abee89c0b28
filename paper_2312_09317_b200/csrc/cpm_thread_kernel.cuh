// cpm_thread_kernel.cuh -- sm_100a sweep kernel with one THREAD per active checkerboard subsection
// (the paper's own granularity: "a 4x4 area per thread", Fig 4; thread = local simulation, L47).
//
// Used for small power-of-two subsections (3D S = 2, 4; 2D S = 2..16).  Same algorithm, same RNG
// counters and same results as the warp-per-subsection kernel of cpm_device.cuh:
//   a2  every lane stages its own (S+2)^d tile into shared memory, INTERLEAVED across the 32 lanes of
//       the warp (word j of lane L at [j][L]): every later shared-memory access of a warp is
//       bank-conflict free whatever sites the lanes picked; global loads are 128-bit for the interior
//       of a row plus the two halo words;
//   a3  Philox4x32-10, one call = four consecutive attempts of this lane's subsection;
//   a4  each lane screens its own attempts (same cell / frozen) until it finds one that needs a dH,
//       at most SCREEN_BUDGET per round, then the warp reconverges and
//   a5-a9 all lanes that found one evaluate it together, each serially over its 26 (8) neighbours:
//       n_A, n_B by compares, adhesion through the difference table D[tA][tB][tn] = J(tA,tn) - J(tB,tn);
//       acceptance words (Philox stream 1) are drawn only for uphill moves inside the table range;
//   a10 dirty interiors are written back with 128-bit stores, own deltas flushed with 64-bit atomics.
// With Act the tile keeps halo 1; the geometric mean around a source that lies in the halo reads the
// few voxels of ring 2 straight from global memory (they belong to inactive subsections, so they are
// stable during the phase-step).
// Nothing here is shared with oracle/.
#pragma once
#include "cpm_device.cuh"

namespace cpm {

constexpr int TK_CAP = 32;          // own-delta entries per thread (cells changed in one activation)
constexpr int SCREEN_BUDGET = 8;    // screened attempts per lane between two evaluation rounds

template <int DIM, int S>
struct TGeom {
  static constexpr int T = S + 2;
  static constexpr int ROWS = (DIM == 3) ? T * T : T;
  static constexpr int WORDS = ROWS * T;
  static constexpr int SITES = (DIM == 3) ? S * S * S : S * S;
  static constexpr int NNB = (DIM == 3) ? 26 : 8;
  static constexpr int LOG2S = (S == 2) ? 1 : (S == 4) ? 2 : (S == 8) ? 3 : 4;
  static constexpr int LOG2SITES = DIM * LOG2S;
  static_assert(S == 2 || S == 4 || S == 8 || S == 16, "power-of-two subsection edge");
};

// compile-time neighbour offsets, same enumeration as nb_delta
template <int DIM>
__host__ __device__ constexpr int nbc_dx(int nb) { return (nb + (nb >= ((DIM == 2) ? 4 : 13) ? 1 : 0)) % 3 - 1; }
template <int DIM>
__host__ __device__ constexpr int nbc_dy(int nb) { return ((nb + (nb >= ((DIM == 2) ? 4 : 13) ? 1 : 0)) / 3) % 3 - 1; }
template <int DIM>
__host__ __device__ constexpr int nbc_dz(int nb) { return (DIM == 3) ? (nb + (nb >= 13 ? 1 : 0)) / 9 - 1 : 0; }

template <int DIM, int S, bool ACT, bool LIVE>
struct ThreadSweep {
  using G = TGeom<DIM, S>;
  static constexpr int T = G::T;
  static constexpr int NNB = G::NNB;
  static constexpr uint32_t CELL_MASK = 0x7FFFFFFFu;   // type + id: equal iff same cell

  const SweepParams &P;
  uint32_t *tile;          // this lane's word 0; word j at tile[32 * j]
  uint8_t *atile;          // this lane's Act byte 0; byte j at atile[32 * j]
  const int *sOff;         // neighbour index -> 32 * tile offset
  const int32_t *sD;       // [nT][nT][nT] adhesion difference table
  const int32_t *sDiag;    // [nT] J(t,t)
  const TypeParams *sT;    // [nT + 1], row nT all zero (medium)
  int ox, oy, oz;
  uint32_t b;
  uint32_t mcs;
  // own deltas of this activation (deterministic mode), in local memory
  uint32_t key[TK_CAP];
  unsigned long long dvp[TK_CAP];
  int dsx[TK_CAP], dsy[TK_CAP], dsz[TK_CAP];
  int n_entries;
  bool dirty, overflow;

  __device__ ThreadSweep(const SweepParams &p) : P(p) {}

  static __device__ __forceinline__ int off32(int dx, int dy, int dz) { return 32 * ((dz * T + dy) * T + dx); }

  // ---- boundary rule for one axis (reading S5): false = outside a closed lattice ----
  static __device__ __forceinline__ bool wrap(int &g, int n, int per) {
    if (g < 0) { if (!per) return false; g += n; }
    else if (g >= n) { if (!per) return false; g -= n; }
    return true;
  }

  // ---- a2: stage this lane's tile ----
  __device__ __forceinline__ void load_tile() {
#pragma unroll
    for (int r = 0; r < G::ROWS; ++r) {
      const int ty = r % T, tz = r / T;
      int gy = oy - 1 + ty, gz = (DIM == 3) ? oz - 1 + tz : 0;
      bool ok = wrap(gy, P.Y, P.per[1]);
      if (DIM == 3) ok = wrap(gz, P.Z, P.per[2]) && ok;
      const long long rowi = (long long)gy + (long long)P.Y * gz;
      const uint32_t *rowp = P.lat + P.pitch * rowi;
      uint32_t *dst = tile + 32 * (r * T);
      int xl = ox - 1, xr = ox + S;
      const bool okl = ok && wrap(xl, P.X, P.per[0]);
      const bool okr = ok && wrap(xr, P.X, P.per[0]);
      dst[0] = okl ? __ldg(rowp + xl) : 0u;
      dst[32 * (S + 1)] = okr ? __ldg(rowp + xr) : 0u;
      if constexpr (S % 4 == 0) {
#pragma unroll
        for (int q = 0; q < S / 4; ++q) {
          uint4 v = make_uint4(0u, 0u, 0u, 0u);
          if (ok) v = __ldg(reinterpret_cast<const uint4 *>(rowp + ox + 4 * q));
          dst[32 * (1 + 4 * q)] = v.x; dst[32 * (2 + 4 * q)] = v.y; dst[32 * (3 + 4 * q)] = v.z; dst[32 * (4 + 4 * q)] = v.w;
        }
      } else {
        uint2 v = make_uint2(0u, 0u);
        if (ok) v = __ldg(reinterpret_cast<const uint2 *>(rowp + ox));
        dst[32] = v.x; dst[64] = v.y;
      }
      if constexpr (ACT) {
        const uint8_t *arow = P.act + P.apitch * rowi;
        uint8_t *ad = atile + 32 * (r * T);
        ad[0] = okl ? __ldg(arow + xl) : (uint8_t)0;
        ad[32 * (S + 1)] = okr ? __ldg(arow + xr) : (uint8_t)0;
        if constexpr (S % 4 == 0) {
#pragma unroll
          for (int q = 0; q < S / 4; ++q) {
            const uint32_t v = ok ? __ldg(reinterpret_cast<const uint32_t *>(arow + ox + 4 * q)) : 0u;
            ad[32 * (1 + 4 * q)] = (uint8_t)v; ad[32 * (2 + 4 * q)] = (uint8_t)(v >> 8);
            ad[32 * (3 + 4 * q)] = (uint8_t)(v >> 16); ad[32 * (4 + 4 * q)] = (uint8_t)(v >> 24);
          }
        } else {
          const uint32_t v = ok ? (uint32_t)__ldg(reinterpret_cast<const unsigned short *>(arow + ox)) : 0u;
          ad[32] = (uint8_t)v; ad[64] = (uint8_t)(v >> 8);
        }
      }
    }
  }

  // ---- a10: write the interior back ----
  __device__ __forceinline__ void store_tile() {
    constexpr int NR = (DIM == 3) ? S * S : S;
#pragma unroll
    for (int r = 0; r < NR; ++r) {
      const int ly = r % S, lz = r / S;
      const long long rowi = (long long)(oy + ly) + (long long)P.Y * ((DIM == 3) ? oz + lz : 0);
      uint32_t *rowp = P.lat + P.pitch * rowi + ox;
      const uint32_t *src = tile + 32 * ((((DIM == 3) ? (lz + 1) * T : 0) + ly + 1) * T + 1);
      if constexpr (S % 4 == 0) {
#pragma unroll
        for (int q = 0; q < S / 4; ++q)
          *reinterpret_cast<uint4 *>(rowp + 4 * q) = make_uint4(src[32 * (4 * q)], src[32 * (4 * q + 1)], src[32 * (4 * q + 2)], src[32 * (4 * q + 3)]);
      } else {
        *reinterpret_cast<uint2 *>(rowp) = make_uint2(src[0], src[32]);
      }
      if constexpr (ACT) {
        uint8_t *arow = P.act + P.apitch * rowi + ox;
        const uint8_t *as = atile + 32 * ((((DIM == 3) ? (lz + 1) * T : 0) + ly + 1) * T + 1);
        if constexpr (S % 4 == 0) {
#pragma unroll
          for (int q = 0; q < S / 4; ++q)
            *reinterpret_cast<uint32_t *>(arow + 4 * q) = (uint32_t)as[32 * (4 * q)] | ((uint32_t)as[32 * (4 * q + 1)] << 8) |
                                                         ((uint32_t)as[32 * (4 * q + 2)] << 16) | ((uint32_t)as[32 * (4 * q + 3)] << 24);
        } else {
          *reinterpret_cast<unsigned short *>(arow) = (unsigned short)((uint32_t)as[0] | ((uint32_t)as[32] << 8));
        }
      }
    }
  }

  // ---- a6: per-cell {V,P} as this attempt sees it ----
  __device__ __forceinline__ unsigned long long view(uint32_t cell, unsigned long long base) const {
    if constexpr (LIVE) {
      return base;
    } else {
      for (int e = 0; e < n_entries; ++e)
        if (key[e] == cell) return base + dvp[e];
      return base;
    }
  }
  __device__ __forceinline__ void add_delta(uint32_t cell, int dV, int dP, int x, int y, int z, int sgn) {
    const unsigned long long d = ((unsigned long long)(long long)dV << 32) + (unsigned long long)(long long)dP;
    if (LIVE) {
      atomicAdd(P.liveVP + cell, d);
      atomicAdd(P.sumx + cell, (unsigned long long)(long long)(sgn * x));
      atomicAdd(P.sumy + cell, (unsigned long long)(long long)(sgn * y));
      if (DIM == 3) atomicAdd(P.sumz + cell, (unsigned long long)(long long)(sgn * z));
      return;
    }
    int e = 0;
    while (e < n_entries && key[e] != cell) ++e;
    if (e == n_entries) {
      if (n_entries == TK_CAP) { overflow = true; return; }
      key[e] = cell; dvp[e] = 0ull; dsx[e] = 0; dsy[e] = 0; dsz[e] = 0;
      ++n_entries;
    }
    dvp[e] += d; dsx[e] += sgn * x; dsy[e] += sgn * y; dsz[e] += sgn * z;
  }
  __device__ __forceinline__ void flush_table() {
    if constexpr (!LIVE) {
      for (int e = 0; e < n_entries; ++e) {
        const uint32_t c = key[e];
        if (dvp[e] != 0ull) atomicAdd(P.liveVP + c, dvp[e]);
        if (dsx[e] != 0) atomicAdd(P.sumx + c, (unsigned long long)(long long)dsx[e]);
        if (dsy[e] != 0) atomicAdd(P.sumy + c, (unsigned long long)(long long)dsy[e]);
        if (DIM == 3 && dsz[e] != 0) atomicAdd(P.sumz + c, (unsigned long long)(long long)dsz[e]);
      }
    }
  }

  // ---- Act: fixed-point geometric mean over {x} + same-cell Moore neighbours (Eq 9, reading S8) ----
  __device__ __forceinline__ int gm_finish(int ssum, int n, bool zero) const {
    if (zero) return 0;
    const int m = ssum / n;
    return __ldg(P.expq16 + ((m >> 6) & 1023)) << (m >> 16);
  }
  // centre inside the subsection: the whole neighbourhood is in the tile
  __device__ __forceinline__ int gm_inner(int c32, uint32_t mC) const {
    int a = atile[c32];
    bool zero = (a == 0);
    int ssum = __ldg(P.logq16 + a), n = 1;
#pragma unroll
    for (int nb = 0; nb < NNB; ++nb) {
      const int o = off32(nbc_dx<DIM>(nb), nbc_dy<DIM>(nb), nbc_dz<DIM>(nb));
      if ((tile[c32 + o] & CELL_MASK) == mC) {
        a = atile[c32 + o];
        zero |= (a == 0);
        ssum += __ldg(P.logq16 + a);
        ++n;
      }
    }
    return gm_finish(ssum, n, zero);
  }
  // centre in the halo: neighbours outside the tile are read from global memory
  __device__ int gm_outer(int cx, int cy, int cz, uint32_t mC) const {   // tile coordinates in [0, T)
    const int c32 = 32 * ((cz * T + cy) * T + cx);
    int a = atile[c32];
    bool zero = (a == 0);
    int ssum = __ldg(P.logq16 + a), n = 1;
#pragma unroll 1
    for (int nb = 0; nb < NNB; ++nb) {
      int dx, dy, dz;
      nb_delta<DIM>(nb, dx, dy, dz);
      const int px = cx + dx, py = cy + dy, pz = cz + dz;
      uint32_t w; int av;
      const bool in = px >= 0 && px < T && py >= 0 && py < T && (DIM == 2 || (pz >= 0 && pz < T));
      if (in) {
        const int p32 = 32 * ((pz * T + py) * T + px);
        w = tile[p32]; av = atile[p32];
      } else {
        int gx = ox - 1 + px, gy = oy - 1 + py, gz = (DIM == 3) ? oz - 1 + pz : 0;
        bool ok = wrap(gx, P.X, P.per[0]);
        ok = wrap(gy, P.Y, P.per[1]) && ok;
        if (DIM == 3) ok = wrap(gz, P.Z, P.per[2]) && ok;
        if (!ok) continue;   // outside a closed lattice: medium, never the same cell
        const long long rowi = (long long)gy + (long long)P.Y * gz;
        w = __ldg(P.lat + P.pitch * rowi + gx);
        av = __ldg(P.act + P.apitch * rowi + gx);
      }
      if ((w & CELL_MASK) == mC) { zero |= (av == 0); ssum += __ldg(P.logq16 + av); ++n; }
    }
    return gm_finish(ssum, n, zero);
  }

  // ---- a5-a9: one evaluated copy attempt; l = site index, nb = neighbour index, a = attempt index ----
  __device__ __forceinline__ bool evaluate(int t32, int s32, int l, int nb, int a) {
    const uint32_t wA = tile[s32], wB = tile[t32];
    const uint32_t A = wA & ID_MASK, B = wB & ID_MASK;
    const uint32_t mA = wA & CELL_MASK, mB = wB & CELL_MASK;
    const int tA = (int)(mA >> 24), tB = (int)(mB >> 24);
    // per-cell state: issue the loads first, they are consumed after the census
    unsigned long long baseA = 0ull, baseB = 0ull;
    if (A != 0) baseA = LIVE ? __ldcg(P.liveVP + A) : __ldg(P.snapVP + A);
    if (B != 0) baseB = LIVE ? __ldcg(P.liveVP + B) : __ldg(P.snapVP + B);

    // neighbour census of t: n_A, n_B and sum_n [J(tA,tn) - J(tB,tn)]
    const int32_t *Drow = sD + (tA * P.nT + tB) * P.nT;
    int nA = 0, nB = 0, adh = 0;
#pragma unroll
    for (int n = 0; n < NNB; ++n) {
      const uint32_t m = tile[t32 + off32(nbc_dx<DIM>(n), nbc_dy<DIM>(n), nbc_dz<DIM>(n))] & CELL_MASK;
      nA += (m == mA);
      nB += (m == mB);
      adh += Drow[m >> 24];
    }
    // a neighbour of cell A has type tA: its J(tA,tA) term drops out (sigma_n == A); same for B
    adh += nB * sDiag[tB] - nA * sDiag[tA];
    long long dH = adh;

    const unsigned long long vpA = (A != 0) ? view(A, baseA) : 0ull;
    const unsigned long long vpB = (B != 0) ? view(B, baseB) : 0ull;
    if (B != 0 && (uint32_t)(vpB >> 32) <= 1u) return false;   // a cell is never erased (reading S13)

    const int rA = (A != 0) ? tA : P.nT, rB = (B != 0) ? tB : P.nT;   // medium reads the all-zero row (S3)
    const TypeParams pa = sT[rA], pb = sT[rB];
    const int dPA = NNB - 2 * nA, dPB = 2 * nB - NNB;
    {
      const int dva = (int)(uint32_t)(vpA >> 32) - pa.tgtV, dvb = (int)(uint32_t)(vpB >> 32) - pb.tgtV;
      dH += 2 * ((long long)pa.lamV * dva - (long long)pb.lamV * dvb) + (pa.lamV + pb.lamV);
      const long long dpa = (long long)(uint32_t)vpA - pa.tgtP, dpb = (long long)(uint32_t)vpB - pb.tgtP;
      dH += (long long)(pa.lamP * dPA) * (2 * dpa + dPA) + (long long)(pb.lamP * dPB) * (2 * dpb + dPB);
    }
    int lx = l & (S - 1), ly = (l >> G::LOG2S) & (S - 1), lz = (DIM == 3) ? (l >> (2 * G::LOG2S)) : 0;
    if constexpr (ACT) {
      if ((pa.lamA | pb.lamA) != 0) {   // lamA is stored as 0 when the type's Max_act is 0
        long long sideA = 0, sideB = 0;
        if (pa.lamA != 0) {
          int dx, dy, dz;
          nb_delta<DIM>(nb, dx, dy, dz);
          const int sx = lx + dx, sy = ly + dy, sz = lz + dz;
          const bool inner = sx >= 0 && sx < S && sy >= 0 && sy < S && (DIM == 2 || (sz >= 0 && sz < S));
          const int g = inner ? gm_inner(s32, mA) : gm_outer(sx + 1, sy + 1, (DIM == 3) ? sz + 1 : 0, mA);
          if (g != 0) sideA = ((long long)pa.lamA * g) / pa.maxA;
        }
        if (pb.lamA != 0) {
          const int g = gm_inner(t32, mB);
          if (g != 0) sideB = ((long long)pb.lamA * g) / pb.maxA;
        }
        dH -= (sideA - sideB + 32768) >> 16;   // copies FROM active areas are favoured (L259)
      }
    }

    // a8: Metropolis (Eq 2) against the integer threshold table; the word comes from stream 1
    if (dH > 0 && !P.accept_all) {
      if (dH > P.Hmax) return false;
      const uint4 ua = philox4x32_10(make_uint4((uint32_t)a >> 2, b, 2u * P.p + 1u, mcs), P.key0, P.key1);
      if (pick(ua, a & 3) >= __ldg(P.thr + dH)) return false;
    }

    // a9: commit
    tile[t32] = wA;
    if constexpr (ACT) atile[t32] = (uint8_t)pa.maxA;   // Max_act of the new owner; 0 for medium
    dirty = true;
    const int gx = ox + lx, gy = oy + ly, gz = oz + lz;
    if (A != 0) add_delta(A, 1, dPA, gx, gy, gz, +1);
    if (B != 0) add_delta(B, -1, dPB, gx, gy, gz, -1);
    return true;
  }

  // ---- the whole activation of this lane's subsection ----
  __device__ void run(bool active, unsigned long long w, int lane) {
    n_entries = 0; dirty = false; overflow = false;
    mcs = *P.mcs_ptr;
    ox = oy = oz = 0; b = 0;
    if (active) {
      const int ax = (int)(w % (unsigned)P.nact[0]);
      const unsigned long long r1 = w / (unsigned)P.nact[0];
      const int ay = (int)(r1 % (unsigned)P.nact[1]);
      const int az = (int)(r1 / (unsigned)P.nact[1]);
      const int bx = 2 * ax + P.col[0], by = 2 * ay + P.col[1], bz = (DIM == 3) ? 2 * az + P.col[2] : 0;
      b = (uint32_t)(bx + P.nsub[0] * (by + P.nsub[1] * bz));
      ox = bx * S; oy = by * S; oz = (DIM == 3) ? bz * S : 0;
      load_tile();
    }
    const int k = active ? P.k : 0;
    int a = 0, rq = -1;
    uint4 r = make_uint4(0u, 0u, 0u, 0u);
    uint32_t n_eval = 0, n_acc = 0;
    while (true) {
      bool found = false;
      int t32 = 0, s32 = 0, l = 0, nb = 0;
      int budget = SCREEN_BUDGET;
      while (a < k && budget > 0) {
        if ((a >> 2) != rq) {
          rq = a >> 2;
          r = philox4x32_10(make_uint4((uint32_t)rq, b, 2u * P.p, mcs), P.key0, P.key1);
        }
        const uint32_t wd = pick(r, a & 3);
        l = (int)(wd >> (32 - G::LOG2SITES));                     // = (wd * S^d) >> 32
        nb = (int)__umulhi(wd << G::LOG2SITES, (uint32_t)NNB);    // = (u32(wd * S^d) * nNb) >> 32
        const int lx = l & (S - 1), ly = (l >> G::LOG2S) & (S - 1), lz = (DIM == 3) ? (l >> (2 * G::LOG2S)) : 0;
        t32 = 32 * ((((DIM == 3) ? (lz + 1) * T : 0) + ly + 1) * T + lx + 1);
        s32 = t32 + sOff[nb];
        const uint32_t wt = tile[t32], ws = tile[s32];
        if ((((wt ^ ws) & ID_MASK) != 0u) && ((int)(wt | ws) >= 0)) { found = true; break; }
        ++a; --budget;
      }
      if (!__any_sync(FULL, a < k)) break;
      if (found) {
        ++n_eval;
        if (evaluate(t32, s32, l, nb, a)) ++n_acc;
        ++a;
      }
    }
    if (dirty) store_tile();
    flush_table();
    n_eval = __reduce_add_sync(FULL, n_eval);
    n_acc = __reduce_add_sync(FULL, n_acc);
    const bool any_over = __any_sync(FULL, overflow);
    if (lane == 0) {
      const int slot = (int)(blockIdx.x % COUNTER_SLOTS);
      if (n_eval) atomicAdd(P.counters + 2 * slot, (unsigned long long)n_eval);
      if (n_acc) atomicAdd(P.counters + 2 * slot + 1, (unsigned long long)n_acc);
      if (any_over) atomicOr(P.error_flag, 1);
    }
  }
};

// One warp per CTA, one lane per active subsection.  Dynamic smem: [id tiles: WORDS x 32 words]
// [Act tiles: WORDS x 32 bytes] [neighbour offsets: 32 ints] [type records: nT+1] [D: nT^3, then J(t,t): nT].
template <int DIM, int S, bool ACT, bool LIVE>
__global__ void __launch_bounds__(32) sweep_thread_kernel(const __grid_constant__ SweepParams P) {
  extern __shared__ __align__(128) unsigned char smem[];
  using G = TGeom<DIM, S>;
  const int lane = threadIdx.x;
  uint32_t *tiles = reinterpret_cast<uint32_t *>(smem);
  uint8_t *atiles = smem + (size_t)G::WORDS * 128;
  unsigned char *tabs = atiles + (ACT ? (size_t)G::WORDS * 32 : 0);
  int *sOff = reinterpret_cast<int *>(tabs);
  TypeParams *sT = reinterpret_cast<TypeParams *>(tabs + 128);
  int32_t *sD = reinterpret_cast<int32_t *>(tabs + 128 + (size_t)(P.nT + 1) * sizeof(TypeParams));
  {
    int dx = 0, dy = 0, dz = 0;
    if (lane < G::NNB) nb_delta<DIM>(lane, dx, dy, dz);
    sOff[lane] = 32 * ((dz * G::T + dy) * G::T + dx);
    for (int i = lane; i < (P.nT + 1) * 8; i += 32)
      reinterpret_cast<int32_t *>(sT)[i] = reinterpret_cast<const int32_t *>(P.types)[i];
    const int nD = P.nT * P.nT * P.nT + P.nT;
    for (int i = lane; i < nD; i += 32) sD[i] = P.D[i];
  }
  __syncwarp();
  const unsigned long long w = (unsigned long long)blockIdx.x * 32 + lane;
  ThreadSweep<DIM, S, ACT, LIVE> sw(P);
  sw.tile = tiles + lane; sw.atile = atiles + lane;
  sw.sOff = sOff; sw.sD = sD; sw.sDiag = sD + P.nT * P.nT * P.nT; sw.sT = sT;
  sw.run(w < P.n_active, w, lane);
}

}  // namespace cpm
