// cpm_pool_kernel.cuh -- sm_100a sweep kernel for small power-of-two subsections (3D S = 2, 4, 8; 2D S = 2..16):
// one WARP owns a GROUP of 8 active checkerboard subsections ("chains") and evaluates their copy attempts
// SPECULATIVELY IN PARALLEL, pooled over the 8 chains, while keeping the exact sequential semantics of every
// chain (the attempts of one subsection are applied in order).  Warps never wait for one
// another: a CTA is one warp, all synchronisation is __syncwarp().
//
// Data layout in HBM: the lattice is stored as per-subsection TILES WITH HALO
// ((S+2)^d words each, the halo replicated from the neighbouring subsections), 8 same-colour tiles
// interleaved: word j of chain c of group g at  base[colour] + ((g * TW + j) << 3) + c.  A group is one
// contiguous block of TW * 32 bytes, so
//   a2  ONE bulk asynchronous copy (TMA, cp.async.bulk -> SASS UBLKCP) stages the tiles of the 8 chains, already
//       in the order the kernel wants (bank = chain + 8 (j mod 4)); completion on an mbarrier while the warp
//       draws its random numbers;
//   a10 there is no tile write-back: an accepted copy stores its word to the home tile and to the (at most
//       2^d - 1) halo replicas in the neighbouring subsections' tiles, which are inactive in this phase-step.
// Lane (q, c) = (lane >> 3, lane & 7) serves chain c:
//   a3  all proposals of (up to) 64 attempts per chain are drawn up front: one Philox4x32-10 block (counter
//       (a>>2, b, 2p, mcs), reading S15) = 4 attempts, quads q, q+4, ... per lane; decoded proposals go to shared
//       memory;
//   a4  every chain has its own position (attempts before it are final).  Per round the lanes of a chain screen
//       the next 4 NJ attempts behind its position against its tile (same cell / frozen); ballot + popc compact
//       the surviving attempts of all 8 chains into one queue, ordered by distance from the chain's position; at
//       most 32 are taken per round (a chain's window ends at its first attempt left out);
//   a5-a7 the queue is evaluated one item per lane whatever chain it belongs to: neighbour census from the
//       chain's tile column, per-cell state (snapshot + the chain's own deltas / live), dH in int64;
//   Act the geometric means (Eq 9) the items need are computed by the whole warp, one request after the other
//       (lanes = the sites of the neighbourhood);
//   a8  Metropolis; an accepted item enters a shared-memory atomicMin on its chain's slot, keyed by the attempt
//       index, so the FIRST accepted attempt of every chain wins;
//   a9  nothing is committed before every item of the round is decided: all of them saw the state at the start
//       of the round, what lies before a chain's winner is final, the winner is committed (8 lanes per winner:
//       home word and halo replicas, the reductions of both cells), the chain continues behind its winner on the
//       new state and the others behind their window, so the result equals k sequential attempts per subsection
//       exactly;
//   a10 the integer deltas of a committed copy go to the live per-cell arrays at once as 64-bit reductions.
// Nothing here is shared with oracle/.
#pragma once
#include "cpm_device.cuh"

namespace cpm {

constexpr int PK_GS = 3;                     // log2 of the chains per group
constexpr int PK_GC = 1 << PK_GS;            // chains per warp = per group
constexpr int PK_THREADS = 32;               // one warp per CTA
constexpr int PK_SUPER = 64;                 // attempts per chain whose proposals are drawn up front
#ifndef PK_TARGET_VALUE
#define PK_TARGET_VALUE 12
#endif
#ifndef PK_NJ_VALUE
#define PK_NJ_VALUE 6
#endif
#ifndef PK_MINB
#define PK_MINB 20
#endif
#ifndef PK_MINB_2D
#define PK_MINB_2D 28   // 2D tiles are small: shared memory allows 28 CTAs per SM at S = 8, so the registers are held to 73 (measured: C5 16384^2 2.53 -> 2.26 ms per MCS, C7 0.147 -> 0.137; the 3D instantiations lose 3 % at 28)
#endif
constexpr int PK_TARGET = PK_TARGET_VALUE;   // a round's window grows until it holds this many items
constexpr int PK_NJ = PK_NJ_VALUE;                     // a chain's window per round: 4 NJ attempts behind its position
constexpr int PK_CAP = 32;                   // own-delta entries per chain and activation (reading R2)
constexpr int PK_DCAP = 3;                   // of which the first live in shared memory, the rest in a spill slot
constexpr int PK_SPILL = PK_CAP - PK_DCAP;
constexpr int PK_NOWIN = PK_SUPER << 10;     // "no accepted attempt": a chain's winner slot holds a << 10 | n_A << 5 | n_B
// lattice word of the tiled layout: [type:5 | frozen:1 | 00 | id:24]: the top byte is the byte offset type * 8 +
// frozen * 4 into a row of the adhesion table, so a neighbour's adhesion term costs one multiply-high, one load
// and one add
// Order of a group's 8 tiles, in HBM and (the bulk copy keeps it) in shared memory: chain-major = the tile of chain c
// is the contiguous block [c * TW, (c + 1) * TW); else word j of chain c at j * 8 + c.
#ifndef PK_CHAIN_MAJOR
#define PK_CHAIN_MAJOR 0   // measured on C4 1024^3: the sweep takes the same time either way (11.14 vs 11.16 ms per MCS: shared-memory bank conflicts are not what bounds it), pack and recount are slower chain-major (51 vs 33 ms)
#endif
constexpr int PK_TS = PK_CHAIN_MAJOR ? 1 : PK_GC;   // distance (words) between consecutive words of one chain's tile
__host__ __device__ __forceinline__ constexpr int pk_tbase(int c, int TW) { return PK_CHAIN_MAJOR ? c * TW : c; }   // first word of chain c's tile
constexpr uint32_t PK_FROZEN = 1u << 26;
constexpr uint32_t PK_CELL = ~PK_FROZEN;        // type + id: equal iff same cell
constexpr int PK_TYPE_SHIFT = 27;
constexpr uint32_t CELL_MASK31 = PK_CELL;

template <int DIM, int S>
struct PGeom {
  static constexpr int T = S + 2;
  static constexpr int TW = (DIM == 3) ? T * T * T : T * T;
  static constexpr int SITES = (DIM == 3) ? S * S * S : S * S;
  static constexpr int NNB = (DIM == 3) ? 26 : 8;
  static constexpr int LOG2S = (S == 2) ? 1 : (S == 4) ? 2 : (S == 8) ? 3 : 4;
  static constexpr int LOG2SITES = DIM * LOG2S;
  static_assert(S == 2 || S == 4 || S == 8 || S == 16, "power-of-two subsection edge");
  static_assert(TW * 4 * 8 < 65536, "byte offsets into a group's tiles are kept in 16 bits");
  // neighbour n (0..NNB-1, centre skipped; n = NNB is the centre itself) -> offsets
  static __host__ __device__ constexpr int idx27(int n) { return n == NNB ? NNB / 2 : n + (n >= NNB / 2 ? 1 : 0); }
  static __host__ __device__ constexpr int dx(int n) { return idx27(n) % 3 - 1; }
  static __host__ __device__ constexpr int dy(int n) { return (idx27(n) / 3) % 3 - 1; }
  static __host__ __device__ constexpr int dz(int n) { return DIM == 3 ? idx27(n) / 9 - 1 : 0; }
  static __host__ __device__ constexpr int noff(int n) { return (dz(n) * T + dy(n)) * T + dx(n); }   // in tile words
};

// shared-memory carve-up of one warp; D (2 nT^3 + nT words) comes last
template <int DIM, int S>
struct PSmem {
  using G = PGeom<DIM, S>;
  static constexpr int TILE = 0;                                   // uint32 [TW][8]
  static constexpr int DDVP = TILE + G::TW * 4 * PK_GC;            // uint64 [DCAP][8]
  static constexpr int MBAR = DDVP + PK_DCAP * 8 * PK_GC;          // uint64
  static constexpr int DKEY = MBAR + 8;                            // uint32 [DCAP][8]
  static constexpr int PROP = DKEY + PK_DCAP * 4 * PK_GC;          // uint32 [64][8]   byte offsets into the chain's tile column: target | source << 16
  static constexpr int QUEUE = PROP + PK_SUPER * 4 * PK_GC;        // uint16 [32]   chain | a << 3
  static constexpr int DN = QUEUE + 32 * PK_NJ * 2;                        // int [8] own-delta table of the chain: entries | (spill slot + 1) << 8
  static constexpr int FIRST = DN + 4 * PK_GC;                     // int [8] first accepted attempt of the round
  static constexpr int ORIG = FIRST + 4 * PK_GC;                   // int [3][8] lattice origin of the chain
  static constexpr int NOFF = ORIG + 12 * PK_GC;                   // int [32] neighbour -> tile offset (entry NNB = centre = 0)
  static constexpr int TYPES = (NOFF + 128 + 15) / 16 * 16;        // TypeParams [nT + 1], then int32 [nT][nT][nT][2] adhesion
                                                                   // differences, then [nT] J(t,t)
  static constexpr size_t img_bytes(int nT) { return (((size_t)(nT + 1) * 32 + ((size_t)2 * nT * nT * nT + nT) * 4) + 15) / 16 * 16; }   // the bulk-copied part
  static constexpr size_t bytes(int nT) { return (size_t)TYPES + img_bytes(nT); }
};

// n += ((raw ^ w) & PK_CELL) == 0, as one logic op with a predicate result and one predicated add
__device__ __forceinline__ void count_same(int &n, uint32_t raw, uint32_t w) {
  asm("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\tlop3.b32 t, %1, %2, %3, 0x28;\n\tsetp.eq.u32 p, t, 0;\n\t@p add.s32 %0, %0, 1;\n\t}"
      : "+r"(n) : "r"(raw), "r"(w), "r"(PK_CELL));
}

__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// tile offset (non-negative) -> tile coordinates, with unsigned divisions by the compile-time edge
template <int DIM, int T>
__device__ __forceinline__ void tile_xyz(int off, int &x, int &y, int &z) {
  const unsigned u = (unsigned)off;
  const unsigned r = u / (unsigned)T;
  x = (int)(u - r * (unsigned)T);
  if (DIM == 3) { const unsigned r2 = r / (unsigned)T; y = (int)(r - r2 * (unsigned)T); z = (int)r2; }
  else { y = (int)r; z = 0; }
}

// byte offset of site (x,y,z) in the Act field: y + Y z fits 32 bits (fewer than 2^31 rows), one widening multiply-add
__device__ __forceinline__ long long act_index(const SweepParams &P, int x, int y, int z) {
  return (long long)(y + P.Y * z) * P.apitch + x;
}

// word offset of tile element j of the subsection (bx,by,bz) in the tiled lattice
__device__ __forceinline__ unsigned long long tile_word(const TileLayout &L, int bx, int by, int bz, int j) {
  const int col = (bx & 1) | ((by & 1) << 1) | ((bz & 1) << 2);
  const unsigned long long w = (unsigned long long)(bx >> 1) + (unsigned long long)L.nact[col][0] * ((unsigned long long)(by >> 1) + (unsigned long long)L.nact[col][1] * (unsigned long long)(bz >> 1));
  return L.base[col] + (w >> PK_GS) * (unsigned long long)(L.TW * PK_GC) + (unsigned long long)(pk_tbase((int)(w & (unsigned long long)(PK_GC - 1)), L.TW) + j * PK_TS);
}
// home word of lattice site (x,y,z), all inside the lattice; S = L.S
template <int DIM>
__device__ __forceinline__ unsigned long long home_word(const TileLayout &L, int S, int x, int y, int z) {
  const int T = S + 2;
  const int bx = x / S, by = y / S, bz = (DIM == 3) ? z / S : 0;
  const int j = (((DIM == 3) ? (z - bz * S + 1) * T : 0) + (y - by * S + 1)) * T + (x - bx * S + 1);
  return tile_word(L, bx, by, bz, j);
}

template <int DIM, int S, bool ACT, bool LIVE, bool VEC>
__global__ void __launch_bounds__(PK_THREADS, (DIM == 2) ? PK_MINB_2D : PK_MINB) sweep_pool_kernel(const __grid_constant__ SweepParams P) {
  using G = PGeom<DIM, S>;
  using M = PSmem<DIM, S>;
  constexpr int T = G::T, TW = G::TW, NNB = G::NNB, GC = PK_GC, NJ = PK_NJ, TS = PK_TS;
  extern __shared__ __align__(128) unsigned char smem[];
  uint32_t *tile = reinterpret_cast<uint32_t *>(smem + M::TILE);
  uint32_t *prop = reinterpret_cast<uint32_t *>(smem + M::PROP);
  unsigned short *queue = reinterpret_cast<unsigned short *>(smem + M::QUEUE);
  uint32_t *dkey = reinterpret_cast<uint32_t *>(smem + M::DKEY);
  unsigned long long *ddvp = reinterpret_cast<unsigned long long *>(smem + M::DDVP);
  int *dn = reinterpret_cast<int *>(smem + M::DN);
  int *first = reinterpret_cast<int *>(smem + M::FIRST);
  int *orig = reinterpret_cast<int *>(smem + M::ORIG);
  int *snoff = reinterpret_cast<int *>(smem + M::NOFF);
  uint64_t *mbar = reinterpret_cast<uint64_t *>(smem + M::MBAR);
  TypeParams *st = reinterpret_cast<TypeParams *>(smem + M::TYPES);
  int32_t *sd = reinterpret_cast<int32_t *>(smem + M::TYPES + (P.nT + 1) * 32);
  const int32_t *sdiag = sd + 2 * P.nT * P.nT * P.nT;

  const uint32_t mcs = __ldg(P.mcs_ptr);   // first: the only global load the Philox counters wait for
  const int lane = threadIdx.x;
  const int c = lane & (GC - 1), q = lane >> PK_GS;   // this lane serves chain c; q = its slot among the chain's 4 lanes
  const unsigned lt = (1u << lane) - 1u;
  uint32_t *const gtile = P.tl.tiles + P.grp_base + (unsigned long long)blockIdx.x * (unsigned long long)(TW * GC);   // this group's tiles in HBM

  // ---- a2: one bulk copy stages the 8 tiles; it overlaps the set-up and the Philox blocks ----
  if (lane == 0) {
    mbar_init(mbar, 1); fence_mbar_init();
    mbar_expect_tx(mbar, (uint32_t)(TW * 4 * GC) + (uint32_t)P.img_bytes);
    bulk_load(tile, gtile, (uint32_t)(TW * 4 * GC), mbar);
    bulk_load(st, P.img, (uint32_t)P.img_bytes, mbar);   // per-type records and the adhesion table, first used after the wait below
  }
  // small tables
  // per-lane constants: tile offset and (dx, dy, dz) of Moore neighbour `lane` (zeros for lanes >= NNB: the centre), one
  // coalesced 16-byte load from a host-built table instead of divisions by 3 and 9
  const int4 lane_nb = __ldg(P.lane_tab + lane);
  // neighbour -> what it adds to a packed proposal (target | source << 16, byte offsets): its tile offset in the source half
  snoff[lane] = (int)((uint32_t)(lane_nb.x * (4 * TS)) << 16);
  // geometry of the chains (the host limits n_active to 31 bits for this kernel)
  if (lane < GC) {
    const uint32_t w = blockIdx.x * (uint32_t)GC + (uint32_t)lane;
    int ox = -1, oy = 0, oz = 0;    // ox < 0: no such chain (ragged last group)
    if (w < (uint32_t)P.n_active) {
      // w -> (ax, ay, az) with the host-built reciprocals of the launch parameters (exact for w < 2^31)
      const uint32_t r1 = P.nact_mul[0] ? __umulhi(w, P.nact_mul[0]) >> P.nact_shr[0] : w, ax = w - r1 * (uint32_t)P.nact[0];
      const uint32_t az = P.nact_mul[1] ? __umulhi(r1, P.nact_mul[1]) >> P.nact_shr[1] : r1, ay = r1 - az * (uint32_t)P.nact[1];
      ox = (2 * (int)ax + P.col[0]) * S; oy = (2 * (int)ay + P.col[1]) * S; oz = (DIM == 3) ? (2 * (int)az + P.col[2]) * S : 0;
    }
    orig[lane] = ox; orig[GC + lane] = oy; orig[2 * GC + lane] = oz;
    dn[lane] = 0; first[lane] = PK_NOWIN;
  }
  __syncwarp();
  const bool active = orig[c] >= 0;
  // origins of active chains are non-negative multiples of S: a shift divides them
  const uint32_t b = active ? (uint32_t)((orig[c] >> G::LOG2S) + P.nsub[0] * ((orig[GC + c] >> G::LOG2S) + P.nsub[1] * (orig[2 * GC + c] >> G::LOG2S))) : 0u;
  const int k = P.k;
  uint32_t n_eval = 0, n_acc = 0;
  bool overflow = false;
  bool staged = false;
  static_assert(PK_CHAIN_MAJOR == 0, "packed proposals carry the chain's byte offset below 4 TS: interleaved tiles only");
  const uint32_t cbase2 = (uint32_t)(pk_tbase(c, TW) * 4) * 0x10001u;   // byte offset of this lane's chain inside the group's tiles, in both halves

  for (int sc = 0; sc < k; sc += PK_SUPER) {
    const int kk = min(PK_SUPER, k - sc);   // attempts of this stretch
    // ---- a3: the proposals of the stretch, quads q, q + 4, ... of chain c ----
#pragma unroll 1
    for (int qq = q; 4 * qq < kk; qq += 4) {
      const uint4 r = philox4x32_10(make_uint4((uint32_t)((sc >> 2) + qq), b, 2u * P.p, mcs), P.key0, P.key1);
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint32_t wd = pick(r, j);
        const int l = (int)(wd >> (32 - G::LOG2SITES));                          // = (wd * S^d) >> 32
        const int nb = (int)__umulhi(wd << G::LOG2SITES, (uint32_t)NNB);         // = (u32(wd * S^d) * nNb) >> 32
        const int lx = l & (S - 1), ly = (l >> G::LOG2S) & (S - 1), lz = (DIM == 3) ? (l >> (2 * G::LOG2S)) : 0;
        const int toff = (((DIM == 3) ? (lz + 1) * T : 0) + ly + 1) * T + lx + 1;
        // both halves carry the byte offset of the chain's tile inside the group (4 c < 4 TS with interleaved tiles, so offset / (4 TS) is
        // still the tile word): a screen or a census load then needs no address arithmetic beyond the shared-memory base
        prop[(4 * qq + j) * GC + c] = (uint32_t)toff * (uint32_t)((4 * TS) * 0x10001) + (uint32_t)snoff[nb] + cbase2;
      }
    }
    int pos = active ? 0 : kk;   // attempts < pos of this stretch are final (same value in the 4 lanes of a chain)
    if (!staged) {   // first use of the tiles
      while (!mbar_try_wait(mbar, 0)) {}
      staged = true;
    }
    __syncwarp();

    while (true) {
      // ---- a4: screen the window of this lane's chain: relative attempts q, q + 4, ... behind its position;
      //      the queue is ordered by (relative attempt, chain) ----
      bool in[NJ];
      unsigned m[NJ];
#pragma unroll
      for (int j = 0; j < NJ; ++j) {
        const int a = pos + q + 4 * j;
        const bool ok = a < kk;
        uint32_t wt = 0u, ws = 0u;
        if (ok) {
          const uint32_t prc = prop[a * GC + c];
          wt = *reinterpret_cast<const uint32_t *>(reinterpret_cast<const char *>(tile) + (prc & 0xffffu));
          ws = *reinterpret_cast<const uint32_t *>(reinterpret_cast<const char *>(tile) + (prc >> 16));
        }
        in[j] = ok && (((wt ^ ws) & ID_MASK) != 0u) && (((wt | ws) & PK_FROZEN) == 0u);
        m[j] = __ballot_sync(FULL, in[j]);
      }
      int W = 0;
#pragma unroll
      for (int j = 0; j < NJ; ++j) {
        if (in[j]) queue[W + __popc(m[j] & lt)] = (unsigned short)(c | ((pos + q + 4 * j) << PK_GS));
        W += __popc(m[j]);
      }
      int lim = 4 * NJ;   // the window of this lane's chain covered by this round
      if (W > 32) {       // warp-uniform, rare: a round takes the first 32 items; a chain's window ends at its first item left out
        int fu = 4 * NJ, base = 0;
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
          if (in[j] && base + __popc(m[j] & lt) >= 32) fu = min(fu, q + 4 * j);
          base += __popc(m[j]);
        }
        fu = min(fu, __shfl_xor_sync(FULL, fu, 8));
        fu = min(fu, __shfl_xor_sync(FULL, fu, 16));
        lim = fu; W = 32;
      }
      __syncwarp();

      // ---- a5-a7: one item per lane ----
      const bool have = lane < W;
      int ci = 0, a = 0;
      if (W > 0) {   // warp-uniform
      const int item = have ? (int)queue[lane] : 0;
      ci = item & (GC - 1); a = item >> PK_GS;
      const uint32_t prc = prop[a * GC + ci];
      const int toff = (int)((prc & 0xffffu) / (unsigned)(4 * TS)), soff = (int)((prc >> 16) / (unsigned)(4 * TS));
      int nA = 0, nB = 0;
      const uint32_t *const tc = tile + pk_tbase(ci, TW);
      const uint32_t wA = tc[soff * TS], wB = tc[toff * TS];
      const uint32_t A = wA & ID_MASK, Bc = wB & ID_MASK;
      const uint32_t mA = wA & CELL_MASK31, mB = wB & CELL_MASK31;
      const int tA = (int)(wA >> PK_TYPE_SHIFT), tB = (int)(wB >> PK_TYPE_SHIFT);
      long long dH = 0;
      bool go = false;
      TypeParams pa = st[P.nT], pb = st[P.nT];
      bool wantA = false, wantB = false;
      if (have) {
        unsigned long long baseA = 0ull, baseB = 0ull;
        if (A != 0) baseA = LIVE ? __ldcg(P.liveVP + A) : __ldg(P.snapVP + A);
        if (Bc != 0) baseB = LIVE ? __ldcg(P.liveVP + Bc) : __ldg(P.snapVP + Bc);
        const char *Drow = reinterpret_cast<const char *>(sd + (tA * P.nT + tB) * P.nT * 2);   // [type][frozen] -> J(tA,type) - J(tB,type)
        int adh = 0;
#pragma unroll
        for (int n = 0; n < NNB; ++n) {
          const uint32_t raw = tc[(toff + G::noff(n)) * TS];
          count_same(nA, raw, wA);
          count_same(nB, raw, wB);
          adh += *reinterpret_cast<const int32_t *>(Drow + (raw >> 24));
        }
        // a neighbour of cell A has type tA: its J(tA,tA) term drops out (sigma_n == A); same for B
        adh += nB * sdiag[tB] - nA * sdiag[tA];
        dH = adh;
        // a6: per-cell {V,P} as this attempt sees it: snapshot + the chain's own deltas / live
        unsigned long long vpA = baseA, vpB = baseB;
        if constexpr (!LIVE) {
          const int di = dn[ci];
          const int ne = di & 255;
          if (ne > 0) {
            unsigned long long dA = 0ull, dB = 0ull;
#pragma unroll
            for (int i = 0; i < PK_DCAP; ++i) {   // the shared-memory entries, without a loop (entries beyond ne hold stale keys: masked)
              const uint32_t key = (i < ne) ? dkey[i * GC + ci] : 0xffffffffu;
              const unsigned long long v = ddvp[i * GC + ci];
              if (key == A) dA = v;
              if (key == Bc) dB = v;
            }
            if (ne > PK_DCAP) {
              const long long sl = (long long)((di >> 8) - 1) * PK_SPILL;
              for (int i = 0; i < ne - PK_DCAP; ++i) {
                const uint32_t key = __ldcg(P.ovf_keys + sl + i);
                const unsigned long long v = __ldcg(P.ovf_dvp + sl + i);
                if (key == A) dA = v;
                if (key == Bc) dB = v;
              }
            }
            if (A != 0) vpA += dA;
            if (Bc != 0) vpB += dB;
          }
        }
        go = !(Bc != 0 && (uint32_t)(vpB >> 32) <= 1u);   // a cell is never erased (reading S13)
        if (A != 0) pa = st[tA];
        if (Bc != 0) pb = st[tB];                          // medium reads the all-zero row (S3)
        const int dPA = NNB - 2 * nA, dPB = 2 * nB - NNB;
        const int dva = (int)(uint32_t)(vpA >> 32) - pa.tgtV, dvb = (int)(uint32_t)(vpB >> 32) - pb.tgtV;
        dH += 2 * ((long long)pa.lamV * dva - (long long)pb.lamV * dvb) + (pa.lamV + pb.lamV);
        const long long dpa = (long long)(uint32_t)vpA - pa.tgtP, dpb = (long long)(uint32_t)vpB - pb.tgtP;
        dH += (long long)(pa.lamP * dPA) * (2 * dpa + dPA) + (long long)(pb.lamP * dPB) * (2 * dpb + dPB);
        if constexpr (VEC) {
          // chemotaxis / persistence bias (Eq 4, 5; reading S21), only for the specialisation that has these terms (L282)
          if (go && P.vec_on) {   // (the specialisation also serves periodic centroid tracking alone)
            constexpr int CEN = (DIM == 3) ? (T * T + T + 1) : (T + 1);
            const int dd = soff - toff + CEN;   // = ((dz + 1) T + dy + 1) T + dx + 1 of the source's offset
            int ddx, ddy, ddz, sx0, sy0, sz0;
            tile_xyz<DIM, T>(dd, ddx, ddy, ddz); ddx -= 1; ddy -= 1; ddz = (DIM == 3) ? ddz - 1 : 0;
            tile_xyz<DIM, T>(soff, sx0, sy0, sz0);
            int gx = orig[ci] - 1 + sx0, gy = orig[GC + ci] - 1 + sy0, gz = (DIM == 3) ? orig[2 * GC + ci] - 1 + sz0 : 0;
            bool inside = true;   // false: the source lies outside a closed lattice (no field there)
            if (gx < 0) { gx += P.X; inside = P.per[0] != 0; } else if (gx >= P.X) { gx -= P.X; inside = P.per[0] != 0; }
            if (gy < 0) { gy += P.Y; inside = inside && P.per[1] != 0; } else if (gy >= P.Y) { gy -= P.Y; inside = inside && P.per[1] != 0; }
            if (DIM == 3) { if (gz < 0) { gz += P.Z; inside = inside && P.per[2] != 0; } else if (gz >= P.Z) { gz -= P.Z; inside = inside && P.per[2] != 0; } }
            const long long sidx = inside ? (long long)gx + (long long)P.X * ((long long)gy + (long long)P.Y * gz) : -1ll;
            dH -= vec_bias(P, ddx, ddy, ddz, A != 0 ? tA : P.nT, Bc != 0 ? tB : P.nT, A, Bc, sidx);
          }
        }
        if constexpr (ACT) {
          // The Act bias lies in [-capB, +capA] (cap = lamA * largest Act value in the field / maxA, host-built):
          // it is only worked out when it can change the outcome.
          const long long capA = pa.lamA != 0 ? pa.cap : 0, capB = pb.lamA != 0 ? pb.cap : 0;
          const bool matters = go && !P.accept_all && dH + capB > 0 && dH - capA <= P.Hmax;
          wantA = matters && pa.lamA != 0; wantB = matters && pb.lamA != 0;
        }
      }

      // ---- Act: the geometric means (Eq 9) the items of this warp need, one after the other, by the whole warp ----
      if constexpr (ACT) {
        // any zero makes the mean zero, and the centre belongs to its own neighbourhood: look at it first
        if (wantA | wantB) {
          const int ox = orig[ci], oy = orig[GC + ci], oz = orig[2 * GC + ci];
          if (wantA) {
            int sx3, sy3, sz3;
            tile_xyz<DIM, T>(soff, sx3, sy3, sz3);
            int gx = ox - 1 + sx3, gy = oy - 1 + sy3, gz = (DIM == 3) ? oz - 1 + sz3 : 0;
            gx += (gx < 0) ? P.X : (gx >= P.X) ? -P.X : 0;   // the source holds a cell: it lies inside the lattice, possibly through the wrap
            gy += (gy < 0) ? P.Y : (gy >= P.Y) ? -P.Y : 0;
            if (DIM == 3) gz += (gz < 0) ? P.Z : (gz >= P.Z) ? -P.Z : 0;
            wantA = __ldcg(P.act + act_index(P, gx, gy, gz)) != 0;
          }
          if (wantB) {
            int tx3, ty3, tz3;
            tile_xyz<DIM, T>(toff, tx3, ty3, tz3);
            wantB = __ldcg(P.act + act_index(P, ox - 1 + tx3, oy - 1 + ty3, (DIM == 3) ? oz - 1 + tz3 : 0)) != 0;
          }
        }
        unsigned mwA = __ballot_sync(FULL, wantA), mwB = __ballot_sync(FULL, wantB);
        if (mwA | mwB) {   // warp-uniform
          // lanes = the sites of the neighbourhood (lane NNB = the centre): all loads of a request are in flight together
          int ddx = 0, ddy = 0, ddz = 0;
          ddx = lane_nb.y; ddy = lane_nb.z; ddz = lane_nb.w;
          const int mynoff = lane_nb.x;
          int gA = 0, gB = 0;
          while (mwA | mwB) {
            const bool sideB = mwA == 0u;
            const int src = __ffs(sideB ? mwB : mwA) - 1;
            if (sideB) mwB &= mwB - 1; else mwA &= mwA - 1;
            const int ctr = __shfl_sync(FULL, sideB ? toff : soff, src);
            const int cc = __shfl_sync(FULL, ci, src);
            const uint32_t mC = __shfl_sync(FULL, sideB ? mB : mA, src);
            int px, py, pz;
            tile_xyz<DIM, T>(ctr, px, py, pz);
            // the centre is inside the lattice (its cell is not medium), possibly through the wrap
            int cx = orig[cc] - 1 + px, cy = orig[GC + cc] - 1 + py, cz = (DIM == 3) ? orig[2 * GC + cc] - 1 + pz : 0;
            cx += (cx < 0) ? P.X : (cx >= P.X) ? -P.X : 0;
            cy += (cy < 0) ? P.Y : (cy >= P.Y) ? -P.Y : 0;
            if (DIM == 3) cz += (cz < 0) ? P.Z : (cz >= P.Z) ? -P.Z : 0;
            int gx = cx + ddx, gy = cy + ddy, gz = cz + ddz;
            bool ok = lane <= NNB;   // false = outside a closed lattice: medium, never the same cell (S5)
            if (cx < 1 || cx > P.X - 2 || cy < 1 || cy > P.Y - 2 || (DIM == 3 && (cz < 1 || cz > P.Z - 2))) {   // warp-uniform
              if (gx < 0) { gx += P.X; ok = ok && P.per[0] != 0; } else if (gx >= P.X) { gx -= P.X; ok = ok && P.per[0] != 0; }
              if (gy < 0) { gy += P.Y; ok = ok && P.per[1] != 0; } else if (gy >= P.Y) { gy -= P.Y; ok = ok && P.per[1] != 0; }
              if (DIM == 3) { if (gz < 0) { gz += P.Z; ok = ok && P.per[2] != 0; } else if (gz >= P.Z) { gz -= P.Z; ok = ok && P.per[2] != 0; } }
            }
            bool same = ok && lane == NNB;
            if (ok && lane < NNB) {
              const int qx = px + ddx, qy = py + ddy, qz = pz + ddz;
              const bool intile = qx >= 0 && qx < T && qy >= 0 && qy < T && (DIM == 2 || (qz >= 0 && qz < T));
              // ids two sites away from the subsection belong to inactive subsections: stable during this phase-step
              const uint32_t wq = intile ? tile[pk_tbase(cc, TW) + (ctr + mynoff) * TS] : __ldg(P.tl.tiles + home_word<DIM>(P.tl, S, gx, gy, gz));
              same = (wq & CELL_MASK31) == mC;
            }
            int av = 1;
            // L2: sees the Act bytes stored by earlier commits of this warp
            if (same) av = __ldcg(P.act + act_index(P, gx, gy, gz));
            const unsigned msame = __ballot_sync(FULL, same);
            const unsigned mzero = __ballot_sync(FULL, same && av == 0);
            const int ssum = __reduce_add_sync(FULL, same ? __ldg(P.logq16 + av) : 0);
            int g = 0;
            if (!mzero) { const int mm = ssum / __popc(msame); g = __ldg(P.expq16 + ((mm >> 6) & 1023)) << (mm >> 16); }
            if (lane == src) { if (sideB) gB = g; else gA = g; }
          }
          long long sideA = 0, sideB2 = 0;
          if (wantA && gA != 0) sideA = act_side(pa.lamA, pa.maxA, gA);
          if (wantB && gB != 0) sideB2 = act_side(pb.lamA, pb.maxA, gB);
          if (wantA || wantB) dH -= (sideA - sideB2 + 32768) >> 16;   // copies FROM active areas are favoured (L259)
        }
      }

      // ---- a8: Metropolis (Eq 2) against the integer threshold table; the acceptance word (Philox stream 1)
      //      is drawn only for uphill moves inside the table ----
      bool acc = have && go;
      const bool uphill = acc && dH > 0 && !P.accept_all;
      if (uphill && dH > P.Hmax) acc = false;
      const bool draw = uphill && acc;
      if (__any_sync(FULL, draw)) {
        if (draw) {
          const int ag = sc + a;
          const uint32_t th = __ldg(P.thr + dH);   // issued before the ten Philox rounds, which hide its latency
          const uint4 ua = philox4x32_10(make_uint4((uint32_t)ag >> 2, (uint32_t)((orig[ci] >> G::LOG2S) + P.nsub[0] * ((orig[GC + ci] >> G::LOG2S) + P.nsub[1] * (orig[2 * GC + ci] >> G::LOG2S))), 2u * P.p + 1u, mcs), P.key0, P.key1);
          if (pick(ua, ag & 3) >= th) acc = false;
        }
      }
      // ---- a9: the first accepted attempt of every chain wins ----
      if (acc) atomicMin(first + ci, (a << 10) | (nA << 5) | nB);
      __syncwarp();
      if (have && a <= (first[ci] >> 10)) ++n_eval;   // what lies before a chain's winner (and the winner) is final
      }

      // ---- a9/a10: the winners are committed, 8 lanes per winner, 4 winners at a time.  Lane r of a winner's
      //      8: r = 0 the home word (shared memory, HBM) and the Act byte, r = 1 .. 2^d - 1 the halo replica towards
      //      the face / edge / corner r (bit 0: x, 1: y, 2: z); r = 0..3 the reductions of the source's cell (V and
      //      P, sum x, sum y, sum z), r = 4..7 those of the target's cell ----
      const int fwc = first[c];   // winner slot of this lane's own chain (for its position)
      unsigned rem = __ballot_sync(FULL, lane < GC && first[lane] < PK_NOWIN);
      while (rem) {   // warp-uniform
        unsigned mm = rem;
        if (q > 0) mm &= mm - 1;   // drop the q lowest winners: this lane's group of 8 serves the (q + 1)-th
        if (q > 1) mm &= mm - 1;
        if (q > 2) mm &= mm - 1;
        const bool on = mm != 0u;
        const int cw = on ? __ffs(mm) - 1 : 0;
        const int r = c;
        const int fw = first[cw];
        const int nA = (fw >> 5) & 31, nB = fw & 31;
        const uint32_t prc = prop[(on ? (fw >> 10) : 0) * GC + cw];
        const int toff = (int)((prc & 0xffffu) / (unsigned)(4 * TS));
        const uint32_t wA = tile[pk_tbase(cw, TW) + (int)((prc >> 16) / (unsigned)(4 * TS)) * TS], wB = tile[pk_tbase(cw, TW) + toff * TS];
        const uint32_t A = wA & ID_MASK, Bc = wB & ID_MASK;
        __syncwarp();   // every lane has read the state of the round's start
        if (on) {
          int px, py, pz;   // tile coordinates 1..S
          tile_xyz<DIM, T>(toff, px, py, pz);
          const int ox = orig[cw], oy = orig[GC + cw], oz = orig[2 * GC + cw];
          const int gx = ox + px - 1, gy = oy + py - 1, gz = (DIM == 3) ? oz + pz - 1 : 0;
          if (r == 0) {
            tile[pk_tbase(cw, TW) + toff * TS] = wA;                                  // id and type of the source; neither site is frozen
            gtile[pk_tbase(cw, TW) + toff * TS] = wA;                                 // home word in HBM
            if constexpr (ACT)   // Max_act of the new owner; 0 for medium
              P.act[act_index(P, gx, gy, gz)] = (uint8_t)((A != 0) ? st[wA >> PK_TYPE_SHIFT].maxA : 0);
            ++n_acc;
          } else if (r < (1 << DIM)) {
            // halo replica of this site in the tile of the adjacent (inactive) subsection towards r
            const int fx = (px == 1) ? -1 : (px == S) ? 1 : 0, fy = (py == 1) ? -1 : (py == S) ? 1 : 0;
            const int fz = (DIM == 3) ? ((pz == 1) ? -1 : (pz == S) ? 1 : 0) : 0;
            const int avail = (fx != 0 ? 1 : 0) | (fy != 0 ? 2 : 0) | (fz != 0 ? 4 : 0);
            if ((r & ~avail) == 0) {
              const int dx = (r & 1) ? fx : 0, dy = (r & 2) ? fy : 0, dz = (r & 4) ? fz : 0;
              int nx = (ox >> G::LOG2S) + dx, ny = (oy >> G::LOG2S) + dy, nz = (oz >> G::LOG2S) + dz;
              bool ok = true;
              if (nx < 0) { nx += P.nsub[0]; ok = P.per[0] != 0; } else if (nx >= P.nsub[0]) { nx -= P.nsub[0]; ok = P.per[0] != 0; }
              if (ny < 0) { ny += P.nsub[1]; ok = ok && P.per[1] != 0; } else if (ny >= P.nsub[1]) { ny -= P.nsub[1]; ok = ok && P.per[1] != 0; }
              if (DIM == 3) { if (nz < 0) { nz += P.nsub[2]; ok = ok && P.per[2] != 0; } else if (nz >= P.nsub[2]) { nz -= P.nsub[2]; ok = ok && P.per[2] != 0; } }
              if (ok) {
                const int jj = (((DIM == 3) ? (pz - dz * S) * T : 0) + (py - dy * S)) * T + (px - dx * S);
                P.tl.tiles[tile_word(P.tl, nx, ny, nz, jj)] = wA;
              }
            }
          }
          // a10: integer deltas -> live per-cell arrays (64-bit reductions on the composite {V,P} word, L297)
          {
            const int side = r >> 2, which = r & 3;
            const uint32_t cell = side ? Bc : A;
            if (cell != 0 && (which < 3 || DIM == 3)) {
              const int sgn = side ? -1 : 1;
              const int dP = side ? 2 * nB - NNB : NNB - 2 * nA;
              unsigned long long *const arr = P.cell_arr[which];   // {V,P}, sum x, sum y, sum z
              const unsigned long long v = which == 0 ? ((unsigned long long)(long long)sgn << 32) + (unsigned long long)(long long)dP
                                                      : (unsigned long long)(long long)(sgn * (VEC ? sum_coord(P, cell, which - 1, which == 1 ? gx : which == 2 ? gy : gz)
                                                                                                   : (which == 1 ? gx : which == 2 ? gy : gz)));   // periodic tracking (S23) rides on the VEC specialisation
              atomicAdd(arr + cell, v);
            }
          }
        }
        // deterministic mode: the chain's own-delta table.  Lanes r = 0 (the source's cell) and r = 4 (the target's
        // cell) of a winner's 8 update it together when what they add fits the shared-memory part
        if constexpr (!LIVE) {
          const int side = r >> 2;
          const uint32_t cell = side ? Bc : A;
          const int sgn = side ? -1 : 1;
          const int dP = side ? 2 * nB - NNB : NNB - 2 * nA;
          const unsigned long long d = ((unsigned long long)(long long)sgn << 32) + (unsigned long long)(long long)dP;
          const bool mine = on && (r & 3) == 0 && cell != 0;
          const int di = dn[cw];
          const int ne = di & 255;
          int hit = -1;
          if (mine) {
#pragma unroll
            for (int i = 0; i < PK_DCAP; ++i)
              if (i < ne && dkey[i * GC + cw] == cell) hit = i;
          }
          const int need = (mine && hit < 0) ? 1 : 0;
          const int needA = __shfl_sync(FULL, need, lane & ~7), needB = __shfl_sync(FULL, need, (lane & ~7) | 4);
          const bool fast = ne + needA + needB <= PK_DCAP;   // then every entry is in shared memory and so are the new ones
          __syncwarp();   // dn, dkey read by both lanes before either writes
          if (mine && fast) {
            if (hit >= 0) ddvp[hit * GC + cw] += d;
            else { const int sl = ne + (side ? needA : 0); dkey[sl * GC + cw] = cell; ddvp[sl * GC + cw] = d; }
            if (side == (A != 0 ? 0 : 1)) dn[cw] = di + needA + needB;
          }
          if (on && !fast && r == 0) {
#pragma unroll 1
            for (int side2 = 0; side2 < 2; ++side2) {
              const uint32_t cell2 = side2 ? Bc : A;
              if (cell2 == 0) continue;
              const int sgn2 = side2 ? -1 : 1;
              const int dP2 = side2 ? 2 * nB - NNB : NNB - 2 * nA;
              const unsigned long long d2 = ((unsigned long long)(long long)sgn2 << 32) + (unsigned long long)(long long)dP2;
              const int di2 = dn[cw];
              const int ne2 = di2 & 255;
              int slot = (di2 >> 8) - 1;
              bool hit2 = false;
              const int ns = min(ne2, PK_DCAP);
              for (int i = 0; i < ns; ++i)
                if (dkey[i * GC + cw] == cell2) { ddvp[i * GC + cw] += d2; hit2 = true; }
              if (!hit2 && ne2 > PK_DCAP) {
                const long long sl = (long long)slot * PK_SPILL;
                for (int i = 0; i < ne2 - PK_DCAP; ++i)
                  if (__ldcg(P.ovf_keys + sl + i) == cell2) { P.ovf_dvp[sl + i] = __ldcg(P.ovf_dvp + sl + i) + d2; hit2 = true; }
              }
              if (!hit2) {
                if (ne2 < PK_DCAP) { dkey[ne2 * GC + cw] = cell2; ddvp[ne2 * GC + cw] = d2; dn[cw] = di2 + 1; }
                else if (ne2 < PK_CAP) {
                  if (slot < 0) {
                    slot = atomicAdd(P.ovf_count, 1);
                    if (slot >= P.ovf_cap) { slot = -1; overflow = true; }
                  }
                  if (slot >= 0) {
                    const long long sl = (long long)slot * PK_SPILL;
                    P.ovf_keys[sl + ne2 - PK_DCAP] = cell2; P.ovf_dvp[sl + ne2 - PK_DCAP] = d2;
                    dn[cw] = (ne2 + 1) | ((slot + 1) << 8);
                  }
                } else overflow = true;
              }
            }
          }
        }
        // the four lowest winners are done
        for (int i = 0; i < 4; ++i) rem &= rem - 1;
      }
      // chains with an accepted copy continue behind it on the new state, the others behind their window
      pos = (fwc < PK_NOWIN) ? (fwc >> 10) + 1 : min(pos + lim, kk);
      if (lane < GC) first[lane] = PK_NOWIN;
      __syncwarp();
      if (__all_sync(FULL, pos >= kk)) break;
    }
  }
  if (!staged) { while (!mbar_try_wait(mbar, 0)) {} }   // never leave a bulk copy in flight
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

// ------------------------------------------------------------ tiled-layout helpers ----------
// set_lattice: ids (+frozen, cell types) -> tiles with halo.  A block takes whole groups; thread t writes the words
// j = t >> 3, t >> 3 + blockDim / 8, ... of chain t & 7, so the chain's geometry is worked out once per group and the
// stores of a warp are contiguous (no 64-bit division per word).  Groups [g_begin, g_end) of the colour: the host packs
// a large lattice slab by slab while the next slab is still on its way from the host.
template <int DIM>
__global__ void tile_pack_kernel(const uint32_t *ids, const uint8_t *frozen, const uint8_t *ctype, uint32_t max_cells, TileLayout L,
                                 int col, unsigned long long n_active, unsigned long long g_begin, unsigned long long g_end,
                                 int X, int Y, int Z, int perx, int pery, int perz, int *error_flag) {
  const int S = L.S, T = S + 2, TW = L.TW;
  // chain-major tiles: a warp writes one chain's contiguous tile; interleaved tiles: 8 consecutive threads = the 8 chains
  const int c = PK_CHAIN_MAJOR ? (int)((threadIdx.x >> 5) & (PK_GC - 1)) : (int)(threadIdx.x & (PK_GC - 1));
  const int j0 = PK_CHAIN_MAJOR ? (int)(threadIdx.x & 31) + 32 * (int)(threadIdx.x >> 8) : (int)(threadIdx.x >> PK_GS);
  const int jstep = PK_CHAIN_MAJOR ? 32 * (int)(blockDim.x >> 8) : (int)(blockDim.x >> PK_GS);   // blockDim is a multiple of 256
  for (unsigned long long grp = g_begin + blockIdx.x; grp < g_end; grp += gridDim.x) {
    const unsigned long long w = grp * (unsigned long long)PK_GC + (unsigned long long)c;
    const bool live = w < n_active;   // the host keeps n_active below 2^31 for this layout
    const uint32_t w32 = (uint32_t)w;
    const int ax = (int)(w32 % (unsigned)L.nact[col][0]);
    const uint32_t r1 = w32 / (unsigned)L.nact[col][0];
    const int ay = (int)(r1 % (unsigned)L.nact[col][1]);
    const int az = (int)(r1 / (unsigned)L.nact[col][1]);
    const int x0 = (2 * ax + (col & 1)) * S - 1, y0 = (2 * ay + ((col >> 1) & 1)) * S - 1, z0 = (DIM == 3) ? (2 * az + ((col >> 2) & 1)) * S - 1 : 0;
    uint32_t *out = L.tiles + L.base[col] + grp * (unsigned long long)TW * (unsigned long long)PK_GC + (unsigned long long)pk_tbase(c, TW);
    for (int j = j0; j < TW; j += jstep) {
      uint32_t word = 0u;
      if (live) {
        int x = x0 + j % T, y = y0 + (j / T) % T, z = (DIM == 3) ? z0 + j / (T * T) : 0;
        bool ok = true;
        if (x < 0) { if (perx) x += X; else ok = false; } else if (x >= X) { if (perx) x -= X; else ok = false; }
        if (y < 0) { if (pery) y += Y; else ok = false; } else if (y >= Y) { if (pery) y -= Y; else ok = false; }
        if (DIM == 3) { if (z < 0) { if (perz) z += Z; else ok = false; } else if (z >= Z) { if (perz) z -= Z; else ok = false; } }
        if (ok) {
          const long long gi = (long long)x + (long long)X * ((long long)y + (long long)Y * z);
          uint32_t id = ids[gi];
          if (id > max_cells) { atomicOr(error_flag, 2); id = 0; }
          word = id | ((uint32_t)ctype[id] << PK_TYPE_SHIFT) | ((frozen && frozen[gi]) ? PK_FROZEN : 0u);
        }
      }
      out[j * PK_TS] = word;
    }
  }
}
// sites [i_begin, i_end) in row-major order (the host reads a large lattice back slab by slab)
template <int DIM>
__global__ void tile_unpack_kernel(TileLayout L, int X, int Y, int Z, uint32_t *ids, long long i_begin, long long i_end) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = i_begin + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < i_end; i += stride) {
    const int x = (int)(i % X);
    const long long r = i / X;
    ids[i] = L.tiles[home_word<DIM>(L, L.S, x, (int)(r % Y), (int)(r / Y))] & ID_MASK;
  }
}
// recount of V, A (Moore interfaces with sites not of the same cell, L234) and the coordinate sums (L288) from the
// tiles: a thread takes one chain and walks its S^d interior sites; every neighbour is inside the chain's own
// tile, the loads of the 8 lanes of a group are one 32-byte sector; runs of equal ids are flushed with one atomic
// per array.  blockIdx.y = the colour, of which the chains [w_begin, w_end) are taken: a thread's walk over its chain is a
// long serial affair (~0.3 ms whatever the size of the launch), so all colours go into ONE launch.
struct RecountRanges { unsigned long long w_begin[8], w_end[8]; };
template <int DIM>
__global__ void tile_recount_kernel(TileLayout L, RecountRanges R, unsigned long long *liveVP,
                                    unsigned long long *sumx, unsigned long long *sumy, unsigned long long *sumz,
                                    const int *anc, int X, int Y, int Z, int perx, int pery, int perz) {
  const int S = L.S, T = S + 2, TW = L.TW;
  constexpr int NNB = (DIM == 2) ? 8 : 26;
  const int col = (int)blockIdx.y;
  const unsigned long long w_begin = R.w_begin[col], w_end = R.w_end[col];
  if (w_end <= w_begin) return;   // the whole block: nothing of this colour in the range
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  const unsigned long long first = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long n_iter = (w_end - w_begin + stride - 1) / stride;   // same trip count for every lane of a warp
  for (unsigned long long it = 0; it < n_iter; ++it) {
    const unsigned long long w = w_begin + first + it * stride;
    // frozen voxels (one obstacle id can own a fifth of the lattice, L139) are tallied apart and combined over the warp
    // before they reach the per-cell arrays: their atomics would all hit the same few addresses
    uint32_t fid = 0;
    int fcnt = 0, ffor = 0, fsx = 0, fsy = 0, fsz = 0;
    if (w < w_end) {
      const uint32_t *tc = L.tiles + L.base[col] + (w >> PK_GS) * (unsigned long long)TW * (unsigned long long)PK_GC + (unsigned long long)pk_tbase((int)(w & (unsigned long long)(PK_GC - 1)), TW);
      const uint32_t w32 = (uint32_t)w;   // the host keeps n_active below 2^31 for this layout
      const int ax = (int)(w32 % (unsigned)L.nact[col][0]);
      const uint32_t r1 = w32 / (unsigned)L.nact[col][0];
      const int ay = (int)(r1 % (unsigned)L.nact[col][1]);
      const int az = (int)(r1 / (unsigned)L.nact[col][1]);
      const int ox = (2 * ax + (col & 1)) * S, oy = (2 * ay + ((col >> 1) & 1)) * S, oz = (DIM == 3) ? (2 * az + ((col >> 2) & 1)) * S : 0;
      uint32_t cur = 0;
      unsigned long long cv = 0, cx = 0, cy = 0, cz = 0;
      auto flush = [&](uint32_t id, unsigned long long v, unsigned long long x, unsigned long long y, unsigned long long z) {
        if (id != 0) {
          atomicAdd(liveVP + id, v);
          atomicAdd(sumx + id, x); atomicAdd(sumy + id, y);
          if (DIM == 3) atomicAdd(sumz + id, z);
        }
      };
      for (int lz = 0; lz < (DIM == 3 ? S : 1); ++lz)
        for (int ly = 0; ly < S; ++ly)
          for (int lx = 0; lx < S; ++lx) {
            const int j = (((DIM == 3) ? (lz + 1) * T : 0) + ly + 1) * T + lx + 1;
            const uint32_t word = tc[j * PK_TS];
            const uint32_t me = word & ID_MASK;
            const bool frozen = (word & PK_FROZEN) != 0u;
            if (!frozen && me != cur) { flush(cur, cv, cx, cy, cz); cur = me; cv = cx = cy = cz = 0; }
            if (me == 0) continue;
            int foreign = 0;
            for (int nb = 0; nb < NNB; ++nb) {
              int dx, dy, dz;
              nb_delta<DIM>(nb, dx, dy, dz);
              foreign += ((tc[(j + (dz * T + dy) * T + dx) * PK_TS] & ID_MASK) != me);
            }
            int qx = ox + lx, qy = oy + ly, qz = oz + lz;
            if (anc != nullptr) {   // reading S23: the image of the site nearest to the cell's anchor
              if (perx) qx = image_near(qx, anc[3 * (size_t)me], X);
              if (pery) qy = image_near(qy, anc[3 * (size_t)me + 1], Y);
              if (perz) qz = image_near(qz, anc[3 * (size_t)me + 2], Z);
            }
            if (frozen) {
              if (me != fid) {   // a second obstacle id in one subsection: rare, flushed directly
                flush(fid, ((unsigned long long)fcnt << 32) + (unsigned long long)ffor, (unsigned long long)(long long)fsx,
                      (unsigned long long)(long long)fsy, (unsigned long long)(long long)fsz);
                fid = me; fcnt = ffor = fsx = fsy = fsz = 0;
              }
              fcnt += 1; ffor += foreign; fsx += qx; fsy += qy; fsz += qz;
            } else {
              cv += (1ull << 32) + (unsigned long long)foreign;
              cx += (unsigned long long)(long long)qx; cy += (unsigned long long)(long long)qy; cz += (unsigned long long)(long long)qz;
            }
          }
      flush(cur, cv, cx, cy, cz);
    }
    // lanes holding the same obstacle id add up first; one lane issues the atomics (<= 64 sites per lane: 32-bit sums)
    const unsigned peers = __match_any_sync(FULL, fid);
    const int tcnt = (int)__reduce_add_sync(peers, (unsigned)fcnt), tfor = (int)__reduce_add_sync(peers, (unsigned)ffor);
    const int tsx = (int)__reduce_add_sync(peers, (unsigned)fsx), tsy = (int)__reduce_add_sync(peers, (unsigned)fsy);
    const int tsz = (int)__reduce_add_sync(peers, (unsigned)fsz);
    if (fid != 0 && (int)(threadIdx.x & 31) == __ffs(peers) - 1) {
      atomicAdd(liveVP + fid, ((unsigned long long)(unsigned)tcnt << 32) + (unsigned long long)(unsigned)tfor);
      atomicAdd(sumx + fid, (unsigned long long)(long long)tsx); atomicAdd(sumy + fid, (unsigned long long)(long long)tsy);
      if (DIM == 3) atomicAdd(sumz + fid, (unsigned long long)(long long)tsz);
    }
  }
}

}  // namespace cpm
