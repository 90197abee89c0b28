// cpm_thread_kernel.cuh -- sm_100a sweep kernel with one lane PAIR per active checkerboard subsection
// (the paper's own granularity: "a 4x4 area per thread", Fig 4; one local simulation per
// worker, L47).
//
// Used for small power-of-two subsections (3D S = 2, 4; 2D S = 2..16).  Same algorithm, same RNG
// counters and same results as the warp-per-subsection kernel of cpm_device.cuh.
// The attempts of a subsection are a sequential chain, so the time of a phase-step is set by how many
// chains an SM holds (shared memory) and by the latency of one link; two lanes per chain halve the
// work on that critical path and leave room for twice as many warps:
//   a2  the pair stages the (S+2)^d tile of its subsection (rows split by parity), INTERLEAVED across
//       the 16 subsections of the warp (word j of subsection c at [j][c]); global loads are 128-bit for
//       the interior of a row plus the two halo words;
//   a3  Philox4x32-10, one call = four consecutive attempts; each lane of the pair draws one call, so a
//       draw covers eight consecutive attempts ("oct");
//   a4  the warp works in rounds.  Step 1 (converged): every pair without a pending attempt draws its
//       next oct and screens the eight proposals against its tile (same cell / frozen) -> 8-bit mask;
//   a5-a9 step 2 (converged): every pair with a pending attempt evaluates the first one: each lane
//       visits 13 (4) of the 26 (8) neighbours -- n_A, n_B by compares, adhesion through the difference
//       table D[tA][tB][tn] = J(tA,tn) - J(tB,tn) -- and a shuffle adds the halves; dH, Metropolis and
//       the own-delta table are computed by both lanes alike, memory is written by the even lane; after
//       an accepted copy the rest of the oct is re-screened, so the result is exactly that of k
//       sequential attempts; acceptance words (Philox stream 1) are drawn only for uphill moves inside
//       the table range;
//   Act the geometric means (Eq 9) are needed by few pairs at a time, so they are computed by the
//       WHOLE warp for one pair after the other (lanes = the 27 sites, ballot / REDUX).  The Act bytes
//       are not staged: the geometric means read them from global memory (L2) and accepted copies
//       store Max_act there directly.  The id tile keeps halo 1; the few ids of ring 2 around a source
//       that lies in the halo are read from global memory too (they belong to inactive subsections, so
//       they are stable during the phase-step);
//   a10 dirty interiors are written back with 128-bit stores; the integer deltas of every accepted
//       copy go out at once as 64-bit reductions (RED) on the live per-cell arrays.
// Nothing here is shared with oracle/.
#pragma once
#include "cpm_device.cuh"

namespace cpm {

constexpr int TK_CAP = 32;     // own-delta entries per subsection (cells changed in one activation)
constexpr int TK_REG = 4;      // of which the first are held in registers
constexpr int GM_BATCH = 2;    // Act geometric means computed per batch (their global loads overlap)
constexpr int TK_CH = 16;      // subsections (chains) per warp: one lane pair each
constexpr int TK_WARPS = 4;    // warps per CTA: 4 CTAs of 4 x 13.5 KB tiles fill the 228 KB of an SM (3D, S = 4)

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

// dynamically indexed part of the own-delta table: kept apart from ThreadSweep so that everything
// else in there stays in registers
struct OwnTable {
  uint32_t key[TK_CAP];
  unsigned long long dvp[TK_CAP];
};

template <int DIM, int S, bool ACT, bool LIVE>
struct ThreadSweep {
  using G = TGeom<DIM, S>;
  static constexpr int T = G::T;
  static constexpr int NNB = G::NNB;
  static constexpr int HNB = NNB / 2;                  // neighbours per lane of the pair
  static constexpr int CH = TK_CH;
  static constexpr uint32_t CELL_MASK = 0x7FFFFFFFu;   // type + id: equal iff same cell

  const SweepParams &P;
  // Shared-memory layout of the CTA (TK_WARPS warps), all offsets compile-time so that every access is a
  // plain LDS/STS: [id tiles: TK_WARPS x WORDS x CH words][neighbour offsets: 32 ints][neighbour codes: 32
  // ints][site offsets: 256 shorts][type records: 9][D: nT^3, then J(t,t): nT]
  static constexpr int OFF_TAB = TK_WARPS * G::WORDS * CH * 4;
  static constexpr int OFF_SITE = OFF_TAB + 256;
  static constexpr int OFF_TYPES = OFF_SITE + 512;
  static constexpr int OFF_D = OFF_TYPES + 9 * (int)sizeof(TypeParams);
  static __device__ __forceinline__ unsigned char *sm() { extern __shared__ __align__(128) unsigned char smem[]; return smem; }
  static __device__ __forceinline__ uint32_t *tl0() {   // tile of subsection 0 of this warp
    return reinterpret_cast<uint32_t *>(sm()) + (threadIdx.x >> 5) * (G::WORDS * CH);
  }
  static __device__ __forceinline__ uint32_t *tl() { return tl0() + ((threadIdx.x & 31) >> 1); }   // this pair's word j at [CH * j]
  static __device__ __forceinline__ int *so() { return reinterpret_cast<int *>(sm() + OFF_TAB); }             // nbr -> CH * tile offset
  static __device__ __forceinline__ int *sn() { return so() + 32; }   // nbr -> (dx+1) | (dy+1) << 2 | (dz+1) << 4; entry NNB = centre
  static __device__ __forceinline__ unsigned short *ssite() { return reinterpret_cast<unsigned short *>(sm() + OFF_SITE); }   // site -> CH * tile offset
  static __device__ __forceinline__ TypeParams *st() { return reinterpret_cast<TypeParams *>(sm() + OFF_TYPES); }   // [nT + 1], row nT zero
  static __device__ __forceinline__ int32_t *sd() { return reinterpret_cast<int32_t *>(sm() + OFF_D); }       // [nT][nT][nT] adhesion differences
  __device__ __forceinline__ const int32_t *sdiag() const { return sd() + P.nT * P.nT * P.nT; }                // [nT] J(t,t)
  int lane, half;          // half = lane & 1: which lane of the pair
  int noff[HNB];           // CH * tile offsets of this lane's neighbours: n = 2 i + half
  int ox, oy, oz;
  uint32_t b;
  uint32_t mcs;
  // own deltas of this activation (deterministic mode): cell -> composite {dV, dP}; the first TK_REG
  // entries in registers, the rest in local memory; both lanes of the pair keep the same copy
  uint32_t rk[TK_REG];
  unsigned long long rdv[TK_REG];
  OwnTable &tb;
  int n_entries;
  bool dirty, overflow;

  __device__ __forceinline__ ThreadSweep(const SweepParams &p, OwnTable &t) : P(p), tb(t) {}

  static __device__ __forceinline__ int siteoff(int l) {   // site index -> CH * tile offset
    const int lx = l & (S - 1), ly = (l >> G::LOG2S) & (S - 1), lz = (DIM == 3) ? (l >> (2 * G::LOG2S)) : 0;
    return CH * ((((DIM == 3) ? (lz + 1) * T : 0) + ly + 1) * T + lx + 1);
  }

  // ---- boundary rule for one axis (reading S5): false = outside a closed lattice ----
  static __device__ __forceinline__ bool wrap(int &g, int n, int per) {
    if (g < 0) { if (!per) return false; g += n; }
    else if (g >= n) { if (!per) return false; g -= n; }
    return true;
  }

  // ---- a2: stage this pair's tile; this lane takes the rows r = 2 i + half ----
  __device__ __forceinline__ void load_tile() {
    int xl = ox - 1, xr = ox + S;
    const bool okxl = wrap(xl, P.X, P.per[0]);
    const bool okxr = wrap(xr, P.X, P.per[0]);
    const int hrow = half * (CH * T);
#pragma unroll
    for (int i = 0; i < G::ROWS / 2; ++i) {
      // T is even: row 2 i + half lies in plane (2 i) / T at y = (2 i) % T + half
      const int ty0 = (2 * i) % T, tz = (2 * i) / T;
      int gy = oy - 1 + ty0 + half, gz = (DIM == 3) ? oz - 1 + tz : 0;
      bool ok = true;
      if (ty0 == 0 || ty0 == T - 2) ok = wrap(gy, P.Y, P.per[1]);        // only the outermost rows can be outside
      if (DIM == 3 && (tz == 0 || tz == T - 1)) ok = wrap(gz, P.Z, P.per[2]) && ok;
      const long long rowi = (long long)gy + (long long)P.Y * gz;
      const uint32_t *rowp = P.lat + P.pitch * rowi;
      uint32_t *dst = tl() + CH * T * (2 * i) + hrow;
      const bool okl = ok && okxl, okr = ok && okxr;
      dst[0] = okl ? __ldg(rowp + xl) : 0u;
      dst[CH * (S + 1)] = okr ? __ldg(rowp + xr) : 0u;
      if constexpr (S % 4 == 0) {
#pragma unroll
        for (int q = 0; q < S / 4; ++q) {
          uint4 v = make_uint4(0u, 0u, 0u, 0u);
          if (ok) v = __ldg(reinterpret_cast<const uint4 *>(rowp + ox + 4 * q));
          dst[CH * (1 + 4 * q)] = v.x; dst[CH * (2 + 4 * q)] = v.y; dst[CH * (3 + 4 * q)] = v.z; dst[CH * (4 + 4 * q)] = v.w;
        }
      } else {
        uint2 v = make_uint2(0u, 0u);
        if (ok) v = __ldg(reinterpret_cast<const uint2 *>(rowp + ox));
        dst[CH] = v.x; dst[2 * CH] = v.y;
      }
    }
  }

  // ---- a10: write the interior back; this lane takes the interior rows r = 2 i + half ----
  __device__ __forceinline__ void store_tile() {
    constexpr int NR = (DIM == 3) ? S * S : S;
#pragma unroll
    for (int i = 0; i < NR / 2; ++i) {
      const int ly0 = (2 * i) % S, lz = (2 * i) / S;   // S is even
      const long long rowi = (long long)(oy + ly0 + half) + (long long)P.Y * ((DIM == 3) ? oz + lz : 0);
      uint32_t *rowp = P.lat + P.pitch * rowi + ox;
      const uint32_t *src = tl() + CH * ((((DIM == 3) ? (lz + 1) * T : 0) + ly0 + 1) * T + 1) + half * (CH * T);
      if constexpr (S % 4 == 0) {
#pragma unroll
        for (int q = 0; q < S / 4; ++q)
          *reinterpret_cast<uint4 *>(rowp + 4 * q) = make_uint4(src[CH * (4 * q)], src[CH * (4 * q + 1)], src[CH * (4 * q + 2)], src[CH * (4 * q + 3)]);
      } else {
        *reinterpret_cast<uint2 *>(rowp) = make_uint2(src[0], src[CH]);
      }
    }
  }

  // ---- a6: per-cell {V,P} as this attempt sees it: snapshot + own deltas (deterministic) / live ----
  __device__ __forceinline__ unsigned long long view(uint32_t cell, unsigned long long base) const {
    if constexpr (LIVE) {
      return base;
    } else {
      unsigned long long d = 0ull;
#pragma unroll
      for (int i = 0; i < TK_REG; ++i)
        if (rk[i] == cell) d = rdv[i];
      if (n_entries > TK_REG)
        for (int i = TK_REG; i < n_entries; ++i)
          if (tb.key[i] == cell) { d = tb.dvp[i]; break; }
      return base + d;
    }
  }
  // a9/a10: the integer deltas of an accepted copy go to the live per-cell arrays at once (fire-and-forget
  // reductions by the even lane; nobody reads them before the next phase-step in deterministic mode)
  // and, in deterministic mode, into the own-delta table (both lanes)
  __device__ __forceinline__ void add_delta(uint32_t cell, int dV, int dP, int x, int y, int z, int sgn) {
    const unsigned long long d = ((unsigned long long)(long long)dV << 32) + (unsigned long long)(long long)dP;
    if (half == 0) {
      atomicAdd(P.liveVP + cell, d);
      atomicAdd(P.sumx + cell, (unsigned long long)(long long)(sgn * x));
      atomicAdd(P.sumy + cell, (unsigned long long)(long long)(sgn * y));
      if (DIM == 3) atomicAdd(P.sumz + cell, (unsigned long long)(long long)(sgn * z));
    }
    if constexpr (!LIVE) {
      bool hit = false;
#pragma unroll
      for (int i = 0; i < TK_REG; ++i)
        if (rk[i] == cell) { rdv[i] += d; hit = true; }
      if (!hit) {
        for (int i = TK_REG; i < n_entries; ++i)
          if (tb.key[i] == cell) { tb.dvp[i] += d; hit = true; break; }
        if (!hit) {
          const int e = n_entries;
          if (e == TK_CAP) { overflow = true; return; }
#pragma unroll
          for (int i = 0; i < TK_REG; ++i)
            if (i == e) { rk[i] = cell; rdv[i] = d; }
          if (e >= TK_REG) { tb.key[e] = cell; tb.dvp[e] = d; }
          n_entries = e + 1;
        }
      }
    }
  }

  // ---- Act: fixed-point geometric mean over {x} + same-cell Moore neighbours (Eq 9, reading S8) ----
  // Computed by the whole warp for subsection c of the warp: lane n < NNB takes neighbour n of the
  // centre (cx, cy, cz) (tile coordinates packed in ctr), lane NNB the centre itself.  Ids outside the
  // halo-1 tile (ring 2 around the subsection) and all Act bytes are read from global memory.
  // Warp-uniform arguments.  gm_site: this lane's site -> (same cell?, Act value); gm_value: the reduction.
  __device__ __forceinline__ bool gm_site(int c, int ctr, uint32_t mC, int oxL, int oyL, int ozL, int &av_out) const {
    const bool part = lane <= NNB;
    const int code = sn()[part ? lane : NNB];
    const int px = (ctr & 255) + (code & 3) - 1, py = ((ctr >> 8) & 255) + ((code >> 2) & 3) - 1;
    const int pz = (DIM == 3) ? ((ctr >> 16) & 255) + ((code >> 4) & 3) - 1 : 0;
    uint32_t w = 0u;
    int av = 1;
    bool have = false;
    long long gidx = 0;
    if (part) {
      const bool in = px >= 0 && px < T && py >= 0 && py < T && (DIM == 2 || (pz >= 0 && pz < T));
      int gx = oxL - 1 + px, gy = oyL - 1 + py, gz = (DIM == 3) ? ozL - 1 + pz : 0;
      bool ok = wrap(gx, P.X, P.per[0]);
      ok = wrap(gy, P.Y, P.per[1]) && ok;
      if (DIM == 3) ok = wrap(gz, P.Z, P.per[2]) && ok;
      const long long rowi = (long long)gy + (long long)P.Y * gz;
      gidx = P.apitch * rowi + gx;
      if (in) w = tl0()[CH * ((pz * T + py) * T + px) + c];
      else if (ok) w = __ldg(P.lat + P.pitch * rowi + gx);
      have = ok;   // outside a closed lattice: medium, never the same cell
    }
    const bool same = have && (lane == NNB || (w & CELL_MASK) == mC);
    if (same) av = __ldcg(P.act + gidx);   // L2: sees the Act bytes this warp stored on earlier commits
    av_out = av;
    return same;
  }
  __device__ __forceinline__ int gm_value(bool same, int av) const {
    const unsigned msame = __ballot_sync(FULL, same);
    const unsigned mzero = __ballot_sync(FULL, same && av == 0);
    const int ssum = __reduce_add_sync(FULL, same ? __ldg(P.logq16 + av) : 0);
    if (mzero) return 0;
    const int m = ssum / __popc(msame);
    return __ldg(P.expq16 + ((m >> 6) & 1023)) << (m >> 16);
  }

  // ---- a5-a7 for this pair's attempt: census of t, per-cell state, dH without the Act term ----
  struct Eval {
    int toff, soff, l, nb, a;
    uint32_t wA, mA, mB;
    long long dH;
    int dPA, dPB;
    int lamA_a, maxA_a, lamA_b, maxA_b;   // Act parameters of the source / target cell's type
    bool go;                              // false: refused before Metropolis (reading S13)
  };
  __device__ __forceinline__ void census(Eval &e, unsigned evmask) {
    const uint32_t wA = tl()[e.soff], wB = tl()[e.toff];
    const uint32_t A = wA & ID_MASK, B = wB & ID_MASK;
    const uint32_t mA = wA & CELL_MASK, mB = wB & CELL_MASK;
    const int tA = (int)(mA >> 24), tB = (int)(mB >> 24);
    e.wA = wA; e.mA = mA; e.mB = mB;
    // per-cell state: issue the loads first, they are consumed after the census
    unsigned long long baseA = 0ull, baseB = 0ull;
    if (A != 0) baseA = LIVE ? __ldcg(P.liveVP + A) : __ldg(P.snapVP + A);
    if (B != 0) baseB = LIVE ? __ldcg(P.liveVP + B) : __ldg(P.snapVP + B);

    // neighbour census of t, this lane's half: n_A, n_B and sum_n [J(tA,tn) - J(tB,tn)]
    const int32_t *Drow = sd() + (tA * P.nT + tB) * P.nT;
    int nAB = 0, adh = 0;   // n_A in the low half-word, n_B in the high one
#pragma unroll
    for (int i = 0; i < HNB; ++i) {
      const uint32_t m = tl()[e.toff + noff[i]] & CELL_MASK;
      nAB += (m == mA) ? 1 : 0;
      nAB += (m == mB) ? 0x10000 : 0;
      adh += Drow[m >> 24];
    }
    nAB += __shfl_xor_sync(evmask, nAB, 1);   // the other lane's half of the neighbourhood
    adh += __shfl_xor_sync(evmask, adh, 1);
    const int nA = nAB & 0xFFFF, nB = nAB >> 16;
    // a neighbour of cell A has type tA: its J(tA,tA) term drops out (sigma_n == A); same for B
    adh += nB * sdiag()[tB] - nA * sdiag()[tA];
    long long dH = adh;

    const unsigned long long vpA = (A != 0) ? view(A, baseA) : 0ull;
    const unsigned long long vpB = (B != 0) ? view(B, baseB) : 0ull;
    e.go = !(B != 0 && (uint32_t)(vpB >> 32) <= 1u);   // a cell is never erased (reading S13)

    const int rA = (A != 0) ? tA : P.nT, rB = (B != 0) ? tB : P.nT;   // medium reads the all-zero row (S3)
    const TypeParams pa = st()[rA], pb = st()[rB];
    const int dPA = NNB - 2 * nA, dPB = 2 * nB - NNB;
    {
      const int dva = (int)(uint32_t)(vpA >> 32) - pa.tgtV, dvb = (int)(uint32_t)(vpB >> 32) - pb.tgtV;
      dH += 2 * ((long long)pa.lamV * dva - (long long)pb.lamV * dvb) + (pa.lamV + pb.lamV);
      const long long dpa = (long long)(uint32_t)vpA - pa.tgtP, dpb = (long long)(uint32_t)vpB - pb.tgtP;
      dH += (long long)(pa.lamP * dPA) * (2 * dpa + dPA) + (long long)(pb.lamP * dPB) * (2 * dpb + dPB);
    }
    e.dH = dH; e.dPA = dPA; e.dPB = dPB;
    e.lamA_a = pa.lamA; e.maxA_a = pa.maxA; e.lamA_b = pb.lamA; e.maxA_b = pb.maxA;
  }

  // ---- a8-a9: Metropolis and commit (both lanes alike; the even lane writes memory) ----
  __device__ __forceinline__ bool decide(const Eval &e) {
    const long long dH = e.dH;
    if (dH > 0 && !P.accept_all) {
      if (dH > P.Hmax) return false;
      const uint4 ua = philox4x32_10(make_uint4((uint32_t)e.a >> 2, b, 2u * P.p + 1u, mcs), P.key0, P.key1);
      if (pick(ua, e.a & 3) >= __ldg(P.thr + dH)) return false;
    }
    if (half == 0) tl()[e.toff] = e.wA;
    dirty = true;
    const int l = e.l;
    const int lx = l & (S - 1), ly = (l >> G::LOG2S) & (S - 1), lz = (DIM == 3) ? (l >> (2 * G::LOG2S)) : 0;
    const int gx = ox + lx, gy = oy + ly, gz = oz + lz;
    if constexpr (ACT)   // Max_act of the new owner; 0 for medium
      if (half == 0) P.act[P.apitch * ((long long)gy + (long long)P.Y * gz) + gx] = (uint8_t)e.maxA_a;
    const uint32_t A = e.mA & ID_MASK, B = e.mB & ID_MASK;
    if (A != 0) add_delta(A, 1, e.dPA, gx, gy, gz, +1);
    if (B != 0) add_delta(B, -1, e.dPB, gx, gy, gz, -1);
    return true;
  }

  // screen one proposal against the current tile (a4): true = it needs a dH
  // a proposal is kept as toff | nb << 13 | l << 18 (toff = CH * tile offset of the target site)
  static __device__ __forceinline__ int pack_prop(int l, int nb) { return (int)ssite()[l] | (nb << 13) | (l << 18); }
  __device__ __forceinline__ bool interesting(int prop) const {
    const int toff = prop & 0x1FFF;
    const uint32_t wt = tl()[toff], ws = tl()[toff + so()[(prop >> 13) & 31]];
    return (((wt ^ ws) & ID_MASK) != 0u) && ((int)(wt | ws) >= 0);
  }

  // ---- the whole activation of this pair's subsection ----
  __device__ __forceinline__ void run(bool active, unsigned long long w) {
    n_entries = 0; dirty = false; overflow = false;
#pragma unroll
    for (int i = 0; i < TK_REG; ++i) { rk[i] = 0xFFFFFFFFu; rdv[i] = 0ull; }
#pragma unroll
    for (int i = 0; i < HNB; ++i) noff[i] = so()[2 * i + half];
    const unsigned pairmask = 3u << (lane & ~1);
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
    const int noct = (k + 7) >> 3;   // octs of this activation
    int oq = 0;                      // next oct to draw
    unsigned mask8 = 0u;             // attempts of the current oct (bit jj) that still need a dH
    int prop[4] = {0, 0, 0, 0};      // this lane's four attempts 4 half + j of the oct (pack_prop)
    uint32_t n_eval = 0, n_acc = 0;
    while (true) {
      __syncwarp();   // tile words written by the other lane of the pair (staging, commits) are visible
      // step 1: pairs without a pending attempt draw and screen their next oct
      unsigned my = 0u;
      const bool draw = mask8 == 0u && oq < noct;
      if (draw) {
        const uint4 r = philox4x32_10(make_uint4((uint32_t)(2 * oq + half), b, 2u * P.p, mcs), P.key0, P.key1);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const uint32_t wd = pick(r, j);
          const int l = (int)(wd >> (32 - G::LOG2SITES));                          // = (wd * S^d) >> 32
          const int nb = (int)__umulhi(wd << G::LOG2SITES, (uint32_t)NNB);         // = (u32(wd * S^d) * nNb) >> 32
          prop[j] = pack_prop(l, nb);
          if (8 * oq + 4 * half + j < k && interesting(prop[j])) my |= 1u << j;
        }
        ++oq;
      }
      {
        const unsigned other = __shfl_xor_sync(FULL, my, 1);
        if (draw) mask8 = half ? (other | (my << 4)) : (my | (other << 4));
      }
      const bool ev = mask8 != 0u;
      const unsigned evmask = __ballot_sync(FULL, ev);
      if (evmask == 0u && !__any_sync(FULL, oq < noct)) break;

      // step 2: pairs with a pending attempt evaluate the first one
      Eval e;
      e.go = false; e.lamA_a = 0; e.lamA_b = 0; e.maxA_a = 0; e.maxA_b = 0; e.mA = 0u; e.mB = 0u; e.l = 0; e.nb = 0;
      int jj = 0;
      if (ev) {
        jj = __ffs(mask8) - 1;
        const int j = jj & 3;
        const int cand = j == 0 ? prop[0] : j == 1 ? prop[1] : j == 2 ? prop[2] : prop[3];
        const int pj = __shfl_sync(evmask, cand, (lane & ~1) | (jj >> 2));   // the attempt lives in lane jj / 4 of the pair
        e.l = pj >> 18; e.nb = (pj >> 13) & 31;
        e.toff = pj & 0x1FFF; e.soff = e.toff + so()[e.nb];
        e.a = 8 * (oq - 1) + jj;
        if (half == 0) ++n_eval;
        census(e, evmask);
      }
      if constexpr (ACT) {
        // geometric means for the pairs whose source / target cell has an Act bias, by the whole warp
        // (the Act bytes stored by earlier commits are visible after the __syncwarp above)
        unsigned needA = __ballot_sync(FULL, ev && half == 0 && e.go && e.lamA_a != 0);
        unsigned needB = __ballot_sync(FULL, ev && half == 0 && e.go && e.lamA_b != 0);
        long long sideA = 0, sideB = 0;
        int ct = 0, cs = 0;   // tile coordinates of the target / the source site, packed
        if (needA | needB) {
          const int lx = e.l & (S - 1), ly = (e.l >> G::LOG2S) & (S - 1), lz = (DIM == 3) ? (e.l >> (2 * G::LOG2S)) : 0;
          const int code = sn()[e.nb];
          ct = (lx + 1) | ((ly + 1) << 8) | ((lz + 1) << 16);
          cs = (lx + (code & 3)) | ((ly + ((code >> 2) & 3)) << 8) | ((DIM == 3 ? lz + ((code >> 4) & 3) : 1) << 16);
        }
        while (needA | needB) {
          // up to GM_BATCH neighbourhoods at a time: all their global Act loads are in flight together
          int Ls[GM_BATCH], av[GM_BATCH];
          bool isAs[GM_BATCH], same[GM_BATCH];
#pragma unroll
          for (int i = 0; i < GM_BATCH; ++i) {
            Ls[i] = -1; isAs[i] = false; same[i] = false; av[i] = 1;
            if (needA | needB) {
              isAs[i] = needA != 0u;
              Ls[i] = __ffs(isAs[i] ? needA : needB) - 1;
              if (isAs[i]) needA &= needA - 1; else needB &= needB - 1;
              const int ctr = __shfl_sync(FULL, isAs[i] ? cs : ct, Ls[i]);
              const uint32_t mC = __shfl_sync(FULL, isAs[i] ? e.mA : e.mB, Ls[i]);
              const int oxL = __shfl_sync(FULL, ox, Ls[i]), oyL = __shfl_sync(FULL, oy, Ls[i]), ozL = __shfl_sync(FULL, oz, Ls[i]);
              same[i] = gm_site(Ls[i] >> 1, ctr, mC, oxL, oyL, ozL, av[i]);
            }
          }
#pragma unroll
          for (int i = 0; i < GM_BATCH; ++i) {
            if (Ls[i] >= 0) {
              const int g = gm_value(same[i], av[i]);
              if ((lane >> 1) == (Ls[i] >> 1) && g != 0) {   // both lanes of the pair
                if (isAs[i]) sideA = act_side(e.lamA_a, e.maxA_a, g);
                else sideB = act_side(e.lamA_b, e.maxA_b, g);
              }
            }
          }
        }
        if ((e.lamA_a | e.lamA_b) != 0) e.dH -= (sideA - sideB + 32768) >> 16;   // copies FROM active areas are favoured (L259)
      }
      if (ev) {
        mask8 &= mask8 - 1u;               // attempt jj is done
        if (e.go && decide(e)) {
          if (half == 0) ++n_acc;
          // later attempts of the oct see the new tile: screen them again
          __syncwarp(pairmask);
          unsigned m2 = 0u;
#pragma unroll
          for (int j = 0; j < 4; ++j)
            if (4 * half + j > jj && 8 * (oq - 1) + 4 * half + j < k && interesting(prop[j])) m2 |= 1u << j;
          const unsigned o2 = __shfl_xor_sync(pairmask, m2, 1);
          mask8 = half ? (o2 | (m2 << 4)) : (m2 | (o2 << 4));
        }
      }
    }
    __syncwarp();
    if (dirty) store_tile();
    n_eval = __reduce_add_sync(FULL, n_eval);
    n_acc = __reduce_add_sync(FULL, n_acc);
    const bool any_over = __any_sync(FULL, overflow);
    if (lane == 0) {
      const int slot = (int)((blockIdx.x * TK_WARPS + (threadIdx.x >> 5)) % COUNTER_SLOTS);
      if (n_eval) atomicAdd(P.counters + 2 * slot, (unsigned long long)n_eval);
      if (n_acc) atomicAdd(P.counters + 2 * slot + 1, (unsigned long long)n_acc);
      if (any_over) atomicOr(P.error_flag, 1);
    }
  }
};

// TK_WARPS warps per CTA (they share only the small tables), one lane pair per active subsection;
// dynamic smem laid out as in ThreadSweep.
template <int DIM, int S, bool ACT, bool LIVE>
__global__ void __launch_bounds__(32 * TK_WARPS) sweep_thread_kernel(const __grid_constant__ SweepParams P) {
  using TS = ThreadSweep<DIM, S, ACT, LIVE>;
  using G = TGeom<DIM, S>;
  const int tid = threadIdx.x;
  if (tid < 32) {
    int dx = 0, dy = 0, dz = 0;
    if (tid < G::NNB) nb_delta<DIM>(tid, dx, dy, dz);
    TS::so()[tid] = TK_CH * ((dz * G::T + dy) * G::T + dx);
    TS::sn()[tid] = (dx + 1) | ((dy + 1) << 2) | ((dz + 1) << 4);
  }
  for (int i = tid; i < G::SITES; i += 32 * TK_WARPS) TS::ssite()[i] = (unsigned short)TS::siteoff(i);
  for (int i = tid; i < (P.nT + 1) * 8; i += 32 * TK_WARPS)
    reinterpret_cast<int32_t *>(TS::st())[i] = reinterpret_cast<const int32_t *>(P.types)[i];
  const int nD = P.nT * P.nT * P.nT + P.nT;
  for (int i = tid; i < nD; i += 32 * TK_WARPS) TS::sd()[i] = P.D[i];
  __syncthreads();
  const unsigned long long w = (unsigned long long)blockIdx.x * (TK_CH * TK_WARPS) + (tid >> 5) * TK_CH + ((tid & 31) >> 1);
  OwnTable tab;
  TS sw(P, tab);
  sw.lane = tid & 31;
  sw.half = tid & 1;
  sw.run(w < P.n_active, w);
}

}  // namespace cpm
