/*
 * cpm_oracle.cpp -- plain, slow, single-threaded CPU ORACLE of the checkerboard-partitioned
 * Metropolis copy-attempt sweep of the parallel Cellular Potts Model (arXiv 2312.09317).
 *
 * TEST INFRASTRUCTURE ONLY.  Shares no code with the CUDA path.  Its own Philox4x32-10, its
 * own table builders, its own schedule.  Everything is written in the order and notation of
 * the paper / of DESIGN.md's readings so that it can be checked against them by eye:
 *
 *   - state: lattice of cell ids, per-cell type, per-cell globals
 *   - a copy attempt picks a random site and a random neighbour             L49, L220
 *   - Hamiltonian: adhesion + volume (Eq 1), perimeter (Eq 3)
 *   - Metropolis acceptance (Eq 2)
 *   - Act model (Eq 8-9)
 *   - chemotaxis along a vector field (Eq 4), persistence along one vector per cell
 *     (Eq 5-7), readings S21-S22 of DESIGN.md
 *   - checkerboard of active subsections, cycling periodically              L49, L77
 *   - atomics = no update of a global is ever lost                           L51, L57
 *   - stale reads of globals are tolerated                                   L53
 *   - integer centroid sums                                                  L288-290 (Eq 10)
 *   - one MCS = one attempt per lattice site                                 L65
 *
 * Points where the paper is silent are resolved by the readings S1..S20 of SURVEY.md 8(c),
 * restated in DESIGN.md; the ones used here are quoted at the place they are used.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force H(after)-H(before) == dH (P1),
 * tallies == recount (P2), T->0 / T->inf limits (P3), acceptance frequency vs Eq 2 (P4),
 * conservation (P5), order independence inside a phase-step (P6), proposal statistics (P7),
 * Philox known answers (P8), resume (P10), fixed-point GM vs pow() (P11), threshold table
 * (P12), DETERMINISTIC == LIVE when no cell is shared (P13); round 2: P13b (cells straddling
 * subsection borders, lambda_P != 0: pins the per-phase-step snapshot refresh and the own dP view),
 * P11b (each side of the Act bias uses its own cell's type), Act decay after the last phase-step;
 * P14 (direction table, dH of Eq 4-5 against the formula in double, sign by drift), P15 (the
 * recurrence of Eq 6-7 against a numpy restatement on recorded centroids).
 * Parity unpinned: nothing in this file (the LIVE-mode *GPU* ensemble is only statistical).
 */
#include "cpm_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <map>
#include <string>
#include <vector>

namespace {

/* ---------------------------------------------------------------- Philox4x32-10 ----------
 * Salmon et al. 2011; 10 rounds of: two 32x32->64 multiplies, xor with the other counter
 * words and the key; the key is bumped by the Weyl constants between rounds.  Reading S15. */
const uint32_t PHILOX_MUL_A = 0xD2511F53u, PHILOX_MUL_B = 0xCD9E8D57u;
const uint32_t PHILOX_WEYL_A = 0x9E3779B9u, PHILOX_WEYL_B = 0xBB67AE85u;

void philox(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  uint32_t c[4] = {ctr_in[0], ctr_in[1], ctr_in[2], ctr_in[3]};
  uint32_t k[2] = {key_in[0], key_in[1]};
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k[0] += PHILOX_WEYL_A; k[1] += PHILOX_WEYL_B; }
    uint64_t p0 = (uint64_t)PHILOX_MUL_A * c[0];
    uint64_t p1 = (uint64_t)PHILOX_MUL_B * c[2];
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c[1] ^ k[0];
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c[3] ^ k[1];
    uint32_t n3 = lo0;
    c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
  }
  out[0] = c[0]; out[1] = c[1]; out[2] = c[2]; out[3] = c[3];
}

struct Delta { int64_t dV = 0, dP = 0, dSX = 0, dSY = 0, dSZ = 0; };

}  // namespace

struct oracle_ctx {
  int d = 0;
  int dim[3] = {1, 1, 1};
  int per[3] = {0, 0, 0};
  int nT = 0;
  std::vector<int64_t> J, lamV, tgtV, lamP, tgtP, lamA, maxA;
  /* vector terms (Eq 4-7): strengths per type, persistence memory mu per type, look-back dt in MCS */
  std::vector<int64_t> lamPers, lamChem;
  std::vector<double> mu;
  int dt = 0;
  bool pers_on = false, chem_on = false;
  int64_t xq[26][3];                 /* Q14 unit vector of the copy direction source -> target, per neighbour index */
  std::vector<int32_t> cq;           /* Q14 chemotaxis field, [N][3] */
  std::vector<double> phat;          /* persistence direction per cell, [max_cells+1][3] */
  std::vector<double> ring;          /* centroids of the last dt+1 MCS, [dt+1][max_cells+1][3] */
  uint64_t n_updates = 0;            /* persistence updates since set_lattice */
  /* periodic centroid tracking (L297, reading S23): per-cell anchor = floor of the centroid at the last MCS boundary */
  bool unwrap = false;
  std::vector<int64_t> anc;          /* [max_cells+1][3] */
  double T = 0;
  bool accept_all = false;
  uint64_t seed = 0;
  int S = 0;
  int64_t sites = 0;  /* S^d */
  int64_t k = 0, R = 0;
  int mode = 0;
  uint32_t max_cells = 0;
  int nNb = 0;
  int off[26][3];
  int nsub[3] = {1, 1, 1};

  std::vector<uint32_t> id;
  std::vector<uint8_t> frozen;
  std::vector<uint8_t> type;
  std::vector<int32_t> act;
  bool have_lattice = false;

  /* per-cell globals: live, and the phase-start snapshot (reading S12) */
  std::vector<int64_t> V, P, SX, SY, SZ, snapV, snapP;

  uint32_t mcs = 0;
  uint64_t attempts = 0, evaluated = 0, accepted = 0;

  std::vector<uint32_t> thr;
  int64_t Hmax = 0;

  int order = 0;
  uint64_t order_seed = 0;

  int64_t *trace = nullptr;
  uint64_t trace_cap = 0;
  uint64_t *trace_count = nullptr;

  std::string err;
};

namespace {

int64_t LOG_Q16[256];
int64_t EXP_Q16[1024];
bool tables_built = false;

/* Reading S8(iv): LOG[a] = llround(65536*log2 a); EXP[f] = llround(65536*2^(f/1024)). */
void build_act_tables() {
  if (tables_built) return;
  LOG_Q16[0] = 0;
  for (int a = 1; a < 256; ++a) LOG_Q16[a] = std::llround(65536.0 * std::log2((double)a));
  for (int f = 0; f < 1024; ++f) EXP_Q16[f] = std::llround(65536.0 * std::exp2((double)f / 1024.0));
  tables_built = true;
}

/* Reading S8(iv): fixed-point geometric mean, Q16.  Any zero -> 0. */
int64_t gm_q16(const int32_t *a, int n) {
  build_act_tables();
  if (n <= 0) return 0;
  int64_t ssum = 0;
  for (int i = 0; i < n; ++i) {
    if (a[i] <= 0) return 0;
    ssum += LOG_Q16[a[i]];
  }
  int64_t m = ssum / n; /* ssum >= 0: floor */
  return EXP_Q16[(m >> 6) & 1023] << (m >> 16);
}

/* Reading S7: thr[h] = floor(exp(-h/T) * 2^32) for h = 1..Hmax, Hmax = floor(T*32*ln 2). */
int64_t threshold_hmax(double T) {
  if (!(T > 0) || std::isinf(T)) return 0;
  return (int64_t)std::floor(T * 32.0 * std::log(2.0));
}
uint32_t threshold_value(double T, int64_t h) {
  double v = std::floor(std::exp(-(double)h / T) * 4294967296.0);
  if (v >= 4294967295.0) return 0xffffffffu;
  if (v < 0) return 0;
  return (uint32_t)v;
}

/* Reading S16: neighbour enumeration: (dz,dy,dx) lexicographic over {-1,0,1}^d, dx fastest,
 * the all-zero offset skipped.  2D: (dy,dx). */
int build_offsets(int d, int off[26][3]) {
  int n = 0;
  if (d == 2) {
    for (int dy = -1; dy <= 1; ++dy)
      for (int dx = -1; dx <= 1; ++dx) {
        if (dx == 0 && dy == 0) continue;
        off[n][0] = dx; off[n][1] = dy; off[n][2] = 0; ++n;
      }
  } else {
    for (int dz = -1; dz <= 1; ++dz)
      for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
          if (dx == 0 && dy == 0 && dz == 0) continue;
          off[n][0] = dx; off[n][1] = dy; off[n][2] = dz; ++n;
        }
  }
  return n;
}

/* Reading S16: multiply-shift cascade.  l = floor(w * sites / 2^32); the low 32 bits of that
 * product give the neighbour index the same way. */
void decode_proposal(uint32_t w, uint32_t sites, uint32_t n_nb, uint32_t *l, uint32_t *nb) {
  uint64_t prod = (uint64_t)w * (uint64_t)sites;
  *l = (uint32_t)(prod >> 32);
  uint32_t rem = (uint32_t)prod;
  *nb = (uint32_t)(((uint64_t)rem * (uint64_t)n_nb) >> 32);
}

inline int64_t lin(const oracle_ctx *c, int x, int y, int z) {
  return (int64_t)x + (int64_t)c->dim[0] * ((int64_t)y + (int64_t)c->dim[1] * (int64_t)z);
}

/* Reading S5: closed lattice = embedded in immutable medium; periodic axes wrap.
 * Returns false if (x,y,z) is outside after applying the boundary rule. */
inline bool resolve(const oracle_ctx *c, int &x, int &y, int &z) {
  int *v[3] = {&x, &y, &z};
  for (int a = 0; a < 3; ++a) {
    if (*v[a] < 0 || *v[a] >= c->dim[a]) {
      if (!c->per[a]) return false;
      *v[a] = (*v[a] % c->dim[a] + c->dim[a]) % c->dim[a];
    }
  }
  return true;
}

struct SiteView { uint32_t id; int tau; bool frozen; bool inside; int32_t act; };

inline SiteView view(const oracle_ctx *c, int x, int y, int z) {
  SiteView s;
  if (!resolve(c, x, y, z)) { s.id = 0; s.tau = 0; s.frozen = false; s.inside = false; s.act = 0; return s; }
  int64_t i = lin(c, x, y, z);
  s.id = c->id[i]; s.tau = c->type[s.id]; s.frozen = c->frozen[i] != 0; s.inside = true; s.act = c->act[i];
  return s;
}

/* Reading S8(ii): N(x) = {x} + Moore neighbours of x holding the same cell id; GM = 0 for medium. */
int64_t gm_at(const oracle_ctx *c, int x, int y, int z) {
  SiteView me = view(c, x, y, z);
  if (!me.inside || me.id == 0) return 0;
  int32_t vals[27];
  int n = 0;
  vals[n++] = me.act;
  for (int q = 0; q < c->nNb; ++q) {
    SiteView nb = view(c, x + c->off[q][0], y + c->off[q][1], z + c->off[q][2]);
    if (nb.inside && nb.id == me.id) vals[n++] = nb.act;
  }
  return gm_q16(vals, n);
}

struct Eval {
  int status;      /* 0 early-out, 1 evaluated, 2 extinction-refused */
  uint32_t A, B;
  int tauA, tauB;
  int nA, nB;
  int64_t dH_ham;  /* adhesion + volume + perimeter (Eq 1, 3) */
  int64_t dH_act;  /* Act bias, subtracted (reading S8(i)) */
  int64_t dH_dir;  /* chemotaxis + persistence bias, subtracted (reading S21) */
};

/* dH of copying the state of the neighbour (sx,sy,sz) into the target (tx,ty,tz), given the
 * values VA,PA,VB,PB the attempt "sees" for the two cells (live, or snapshot+own deltas). */
template <class Lookup>
Eval evaluate(const oracle_ctx *c, int tx, int ty, int tz, int nb, Lookup seen) {
  Eval e{};
  const int sx = tx + c->off[nb][0], sy = ty + c->off[nb][1], sz = tz + c->off[nb][2];
  SiteView t = view(c, tx, ty, tz);
  SiteView s = view(c, sx, sy, sz);
  e.A = s.id; e.B = t.id; e.tauA = s.tau; e.tauB = t.tau;
  /* early-outs (a4): same cell, frozen target, frozen source (reading S14) */
  if (e.A == e.B || t.frozen || (s.inside && s.frozen)) { e.status = 0; return e; }

  int64_t VA = 0, PA = 0, VB = 0, PB = 0;
  if (e.A != 0) seen(e.A, VA, PA);
  if (e.B != 0) seen(e.B, VB, PB);
  /* reading S13: a cell is never erased */
  if (e.B != 0 && VB <= 1) { e.status = 2; return e; }
  e.status = 1;

  /* neighbour census of t (a5): Eq 1 summed over the unordered pairs that contain t (S2) */
  int64_t adh = 0;
  int nA = 0, nB = 0;
  for (int q = 0; q < c->nNb; ++q) {
    SiteView n = view(c, tx + c->off[q][0], ty + c->off[q][1], tz + c->off[q][2]);
    if (n.id == e.A) ++nA;
    if (n.id == e.B) ++nB;
    int64_t after  = (n.id != e.A) ? c->J[e.tauA * c->nT + n.tau] : 0;
    int64_t before = (n.id != e.B) ? c->J[e.tauB * c->nT + n.tau] : 0;
    adh += after - before;
  }
  e.nA = nA; e.nB = nB;

  /* volume term of Eq 1; medium has no constraint (S3) */
  int64_t vol = 0;
  if (e.A != 0) vol += c->lamV[e.tauA] * (2 * (VA - c->tgtV[e.tauA]) + 1);
  if (e.B != 0) vol += c->lamV[e.tauB] * (1 - 2 * (VB - c->tgtV[e.tauB]));

  /* perimeter term, Eq 3 with the closed form of reading S4 */
  int64_t per = 0;
  if (e.A != 0) { int64_t dP = c->nNb - 2 * nA; per += c->lamP[e.tauA] * dP * (2 * (PA - c->tgtP[e.tauA]) + dP); }
  if (e.B != 0) { int64_t dP = 2 * nB - c->nNb; per += c->lamP[e.tauB] * dP * (2 * (PB - c->tgtP[e.tauB]) + dP); }

  e.dH_ham = adh + vol + per;

  /* Act bias, Eq 8-9 with reading S8: source side uses A's type, target side B's type;
   * evaluated before the copy */
  int64_t sideA = 0, sideB = 0;
  if (e.A != 0 && c->lamA[e.tauA] != 0 && c->maxA[e.tauA] != 0)
    sideA = (c->lamA[e.tauA] * gm_at(c, sx, sy, sz)) / c->maxA[e.tauA];
  if (e.B != 0 && c->lamA[e.tauB] != 0 && c->maxA[e.tauB] != 0)
    sideB = (c->lamA[e.tauB] * gm_at(c, tx, ty, tz)) / c->maxA[e.tauB];
  e.dH_act = (sideA - sideB + 32768) >> 16;

  /* Vector terms, Eq 4 and Eq 5 with reading S21: x^ = unit vector of the copy direction, from the source
   * site i = s to the target site j = t; a copy ALONG the field / the cell's persistence direction is favoured,
   * so the bias is subtracted (same argument as L259 for Act); both the extending cell A and the retracting
   * cell B are pushed along x^ by this copy, each with the strength of its own type; medium has none (S3);
   * the field value is the one at the source site (Eq 4: C_i), zero outside a closed lattice.
   * Fixed point: x^, p^ and C in Q14, the products summed in Q28 and rounded once. */
  e.dH_dir = 0;
  if (c->pers_on || c->chem_on) {
    const int64_t *x = c->xq[nb];
    int64_t acc = 0;
    if (c->pers_on) {
      if (e.A != 0 && c->lamPers[e.tauA] != 0) {
        int64_t dot = 0;
        for (int a = 0; a < 3; ++a) dot += x[a] * (int64_t)std::llrint(16384.0 * c->phat[3 * (size_t)e.A + a]);
        acc += c->lamPers[e.tauA] * dot;
      }
      if (e.B != 0 && c->lamPers[e.tauB] != 0) {
        int64_t dot = 0;
        for (int a = 0; a < 3; ++a) dot += x[a] * (int64_t)std::llrint(16384.0 * c->phat[3 * (size_t)e.B + a]);
        acc += c->lamPers[e.tauB] * dot;
      }
    }
    if (c->chem_on && s.inside && !c->cq.empty()) {
      int rx = sx, ry = sy, rz = sz;
      resolve(c, rx, ry, rz);
      const int32_t *C = &c->cq[3 * (size_t)lin(c, rx, ry, rz)];
      int64_t dot = 0;
      for (int a = 0; a < 3; ++a) dot += x[a] * (int64_t)C[a];
      int64_t lam = 0;
      if (e.A != 0) lam += c->lamChem[e.tauA];
      if (e.B != 0) lam += c->lamChem[e.tauB];
      acc += lam * dot;
    }
    e.dH_dir = (acc + ((int64_t)1 << 27)) >> 28;
  }
  return e;
}

/* Reading S23 (L297: "adding or subtracting dimension x |cell| to the sum values ... to keep centroids within
 * simulation bounds"): on a periodic axis a site's coordinate enters a cell's sum as its periodic image nearest to
 * the cell's anchor, x' = x + m dim with x' - anchor in [-dim/2, dim/2). */
inline int64_t image_near(int64_t x, int64_t anchor, int64_t dim) {
  int64_t r = x - anchor;
  if (2 * r >= dim) return x - dim;
  if (2 * r < -dim) return x + dim;
  return x;
}
inline void site_coords(const oracle_ctx *c, uint32_t cell, int x, int y, int z, int64_t out[3]) {
  const int64_t v[3] = {x, y, z};
  for (int a = 0; a < 3; ++a)
    out[a] = (c->unwrap && c->per[a]) ? image_near(v[a], c->anc[3 * (size_t)cell + a], c->dim[a]) : v[a];
}
/* keep the centroid inside [0, dim) on periodic axes by shifting the sum by dim x V; the anchor follows the centroid */
void normalise_centroid(oracle_ctx *c, uint32_t cell) {
  if (c->V[cell] <= 0) return;
  int64_t *S[3] = {&c->SX[cell], &c->SY[cell], &c->SZ[cell]};
  for (int a = 0; a < 3; ++a) {
    if (!c->per[a]) continue;
    const int64_t span = (int64_t)c->dim[a] * c->V[cell];
    while (*S[a] < 0) *S[a] += span;
    while (*S[a] >= span) *S[a] -= span;
    c->anc[3 * (size_t)cell + a] = *S[a] / c->V[cell];
  }
}

/* commit (a9): the lattice site takes the source's state; Act(t) = Max_act of the new owner;
 * returns the changes of the globals.  Medium (id 0) is not tallied (S3). */
void commit(oracle_ctx *c, int tx, int ty, int tz, const Eval &e, Delta &dA, Delta &dB) {
  int64_t ti = lin(c, tx, ty, tz);
  c->id[ti] = e.A;
  c->act[ti] = (e.A != 0) ? (int32_t)c->maxA[e.tauA] : 0;
  int64_t q[3];
  if (e.A != 0) { site_coords(c, e.A, tx, ty, tz, q); dA.dV += 1; dA.dP += c->nNb - 2 * e.nA; dA.dSX += q[0]; dA.dSY += q[1]; dA.dSZ += q[2]; }
  if (e.B != 0) { site_coords(c, e.B, tx, ty, tz, q); dB.dV -= 1; dB.dP += 2 * e.nB - c->nNb; dB.dSX -= q[0]; dB.dSY -= q[1]; dB.dSZ -= q[2]; }
}

void apply(oracle_ctx *c, uint32_t cell, const Delta &dl) {
  c->V[cell] += dl.dV; c->P[cell] += dl.dP; c->SX[cell] += dl.dSX; c->SY[cell] += dl.dSY; c->SZ[cell] += dl.dSZ;
}

/* recount of all globals from the lattice: definition of V (L225), A (L234, reading S4), sums (L288) */
void recount(oracle_ctx *c) {
  size_t n = (size_t)c->max_cells + 1;
  c->V.assign(n, 0); c->P.assign(n, 0); c->SX.assign(n, 0); c->SY.assign(n, 0); c->SZ.assign(n, 0);
  if (c->unwrap) {   /* reading S23: the first site of a cell in scan order anchors the images of its other sites */
    c->anc.assign(3 * n, 0);
    std::vector<uint8_t> seen(n, 0);
    for (int z = 0; z < c->dim[2]; ++z)
      for (int y = 0; y < c->dim[1]; ++y)
        for (int x = 0; x < c->dim[0]; ++x) {
          uint32_t me = c->id[lin(c, x, y, z)];
          if (me == 0 || seen[me]) continue;
          seen[me] = 1; c->anc[3 * (size_t)me] = x; c->anc[3 * (size_t)me + 1] = y; c->anc[3 * (size_t)me + 2] = z;
        }
  }
  for (int z = 0; z < c->dim[2]; ++z)
    for (int y = 0; y < c->dim[1]; ++y)
      for (int x = 0; x < c->dim[0]; ++x) {
        uint32_t me = c->id[lin(c, x, y, z)];
        if (me == 0) continue;
        int64_t q[3];
        site_coords(c, me, x, y, z, q);
        c->V[me] += 1; c->SX[me] += q[0]; c->SY[me] += q[1]; c->SZ[me] += q[2];
        for (int q = 0; q < c->nNb; ++q) {
          SiteView nb = view(c, x + c->off[q][0], y + c->off[q][1], z + c->off[q][2]);
          if (nb.id != me) c->P[me] += 1;
        }
      }
  if (c->unwrap) for (size_t cell = 1; cell < n; ++cell) normalise_centroid(c, (uint32_t)cell);
}

/* one activation of subsection b in phase-step p (the inner loop of SURVEY 8(c)) */
void run_subsection(oracle_ctx *c, int64_t b, uint32_t p) {
  const int S = c->S;
  const int bx = (int)(b % c->nsub[0]);
  const int by = (int)((b / c->nsub[0]) % c->nsub[1]);
  const int bz = (int)(b / ((int64_t)c->nsub[0] * c->nsub[1]));
  const int ox = bx * S, oy = by * S, oz = (c->d == 3) ? bz * S : 0;
  const uint32_t key[2] = {(uint32_t)c->seed, (uint32_t)(c->seed >> 32)};
  std::map<uint32_t, Delta> loc; /* own deltas of this activation (reading S12) */

  /* Reading S15: attempt a uses word a&3 of the Philox call with counter
   * (a>>2, b, 2p+stream, mcs): one call serves four consecutive attempts.  (The paper is silent on
   * the generator's indexing, L284.) */
  uint32_t w4[4] = {0, 0, 0, 0};
  for (int64_t a = 0; a < c->k; ++a) {
    const uint32_t call = (uint32_t)(a >> 2);
    const int word = (int)(a & 3);
    if (word == 0) {
      uint32_t ctr[4] = {call, (uint32_t)b, 2 * p + 0, c->mcs};
      philox(ctr, key, w4);
    }
    uint32_t w = w4[word];
    uint32_t l, nb;
    decode_proposal(w, (uint32_t)c->sites, (uint32_t)c->nNb, &l, &nb);
    const int tx = ox + (int)(l % S);
    const int ty = oy + (int)((l / S) % S);
    const int tz = (c->d == 3) ? oz + (int)(l / (S * S)) : 0;
    c->attempts++;

    Eval e;
    if (c->mode == ORACLE_MODE_LIVE) {
      e = evaluate(c, tx, ty, tz, (int)nb, [&](uint32_t cell, int64_t &Vv, int64_t &Pp) {
        Vv = c->V[cell]; Pp = c->P[cell]; });
    } else {
      e = evaluate(c, tx, ty, tz, (int)nb, [&](uint32_t cell, int64_t &Vv, int64_t &Pp) {
        Vv = c->snapV[cell]; Pp = c->snapP[cell];
        auto it = loc.find(cell);
        if (it != loc.end()) { Vv += it->second.dV; Pp += it->second.dP; } });
    }
    int64_t rec_dH = 0; int rec_acc = 0; uint32_t rec_u = 0;
    if (e.status != 0) c->evaluated++;
    if (e.status == 1) {
      const int64_t dH = e.dH_ham - e.dH_act - e.dH_dir;
      rec_dH = dH;
      bool acc;
      if (dH <= 0 || c->accept_all) acc = true;          /* Eq 2, reading S6 */
      else if (dH > c->Hmax) acc = false;                /* exp(-dH/T) < 2^-32, reading S7 */
      else {
        uint32_t ctr[4] = {call, (uint32_t)b, 2 * p + 1, c->mcs};
        uint32_t u4[4];
        philox(ctr, key, u4);
        rec_u = u4[word];
        acc = rec_u < c->thr[(size_t)dH];
      }
      if (acc) {
        rec_acc = 1;
        c->accepted++;
        Delta dA, dB;
        commit(c, tx, ty, tz, e, dA, dB);
        if (c->mode == ORACLE_MODE_LIVE) {
          if (e.A != 0) apply(c, e.A, dA);
          if (e.B != 0) apply(c, e.B, dB);
        } else {
          if (e.A != 0) { Delta &t = loc[e.A]; t.dV += dA.dV; t.dP += dA.dP; t.dSX += dA.dSX; t.dSY += dA.dSY; t.dSZ += dA.dSZ; }
          if (e.B != 0) { Delta &t = loc[e.B]; t.dV += dB.dV; t.dP += dB.dP; t.dSX += dB.dSX; t.dSY += dB.dSY; t.dSZ += dB.dSZ; }
        }
      }
    }
    if (c->trace && c->trace_count && *c->trace_count < c->trace_cap) {
      int64_t *r = c->trace + 6 * (*c->trace_count);
      r[0] = lin(c, tx, ty, tz); r[1] = nb; r[2] = e.status; r[3] = rec_dH; r[4] = rec_acc; r[5] = rec_u;
      (*c->trace_count)++;
    }
  }
  /* "live += loc": what the atomics of the parallel scheme add up to (L51, L57) */
  if (c->mode != ORACLE_MODE_LIVE)
    for (auto &kv : loc) apply(c, kv.first, kv.second);
}

/* centroid of a cell, Eq 10: coordinate sums over volume, in double */
inline void centroid(const oracle_ctx *c, size_t cell, double X[3]) {
  const double v = (double)c->V[cell];
  X[0] = (double)c->SX[cell] / v; X[1] = (double)c->SY[cell] / v; X[2] = (double)c->SZ[cell] / v;
}

/* Eq 6-7, once per MCS for every cell that exists (reading S22):
 *   p = (1 - mu) (X_t - X_{t-dt}) / |X_t - X_{t-dt}| + mu p^_{t-1};   p^_t = p / |p|.
 * X_{t-dt} is the centroid dt MCS ago (the one at set_lattice while fewer than dt MCS have passed).  A cell that
 * has not moved contributes no direction (the first term is dropped); a zero p keeps p^ = 0 (no bias).
 * Every operation is a single IEEE double operation in the order written (no fused multiply-add). */
void persistence_update(oracle_ctx *c) {
  const size_t ncell = (size_t)c->max_cells + 1;
  const uint64_t n = c->n_updates + 1;                 /* this is the n-th update */
  const size_t slots = (size_t)c->dt + 1;
  double *old_slot = &c->ring[((n + 1) % slots) * ncell * 3];   /* (n - dt) mod (dt + 1) */
  double *new_slot = &c->ring[(n % slots) * ncell * 3];
  for (size_t cell = 1; cell < ncell; ++cell) {
    if (c->V[cell] <= 0) continue;
    double X[3];
    centroid(c, cell, X);
    const double mu = c->mu[c->type[cell]];
    const double one_minus_mu = 1.0 - mu;
    double d[3], p[3];
    for (int a = 0; a < 3; ++a) {
      d[a] = X[a] - old_slot[3 * cell + a];
      if (c->unwrap && c->per[a]) {   /* shortest displacement through the periodic border (S23) */
        const double half = 0.5 * (double)c->dim[a];
        if (d[a] > half) d[a] = d[a] - (double)c->dim[a];
        else if (d[a] < -half) d[a] = d[a] + (double)c->dim[a];
      }
    }
    const double dn = std::sqrt((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]);
    for (int a = 0; a < 3; ++a) {
      const double keep = mu * c->phat[3 * cell + a];
      if (dn > 0.0) { const double u = d[a] / dn; const double turn = one_minus_mu * u; p[a] = turn + keep; }
      else p[a] = keep;
    }
    const double pn = std::sqrt((p[0] * p[0] + p[1] * p[1]) + p[2] * p[2]);
    for (int a = 0; a < 3; ++a) c->phat[3 * cell + a] = (pn > 0.0) ? p[a] / pn : 0.0;
    for (int a = 0; a < 3; ++a) new_slot[3 * cell + a] = X[a];
  }
  c->n_updates = n;
}

void one_mcs(oracle_ctx *c) {
  const int ncol = 1 << c->d;
  const int64_t nsub_total = (int64_t)c->nsub[0] * c->nsub[1] * c->nsub[2];
  std::vector<int64_t> active;
  for (int64_t rep = 0; rep < c->R; ++rep)
    for (int col = 0; col < ncol; ++col) {
      const uint32_t p = (uint32_t)(rep * ncol + col);
      if (c->mode != ORACLE_MODE_LIVE) { c->snapV = c->V; c->snapP = c->P; }
      active.clear();
      for (int64_t b = 0; b < nsub_total; ++b) {
        int bx = (int)(b % c->nsub[0]);
        int by = (int)((b / c->nsub[0]) % c->nsub[1]);
        int bz = (int)(b / ((int64_t)c->nsub[0] * c->nsub[1]));
        int colour = (bx & 1) | ((by & 1) << 1) | ((bz & 1) << 2);
        if (colour == col) active.push_back(b);
      }
      if (c->order == 1) std::reverse(active.begin(), active.end());
      if (c->order == 2) {
        uint64_t st = c->order_seed * 6364136223846793005ull + 1442695040888963407ull + p + 977ull * c->mcs;
        for (size_t i = active.size(); i > 1; --i) {
          st = st * 6364136223846793005ull + 1442695040888963407ull;
          size_t j = (size_t)((st >> 33) % i);
          std::swap(active[i - 1], active[j]);
        }
      }
      for (int64_t b : active) run_subsection(c, b, p);
    }
  /* Act decay (L255, reading S9): once per MCS, after the last phase-step */
  for (auto &a : c->act) a = std::max(a - 1, 0);
  /* centroids back into the lattice on periodic axes (L297, reading S23) */
  if (c->unwrap) for (size_t cell = 1; cell <= c->max_cells; ++cell) normalise_centroid(c, (uint32_t)cell);
  /* persistence directions (Eq 6-7): "updated iteratively at every MCS" (L246) */
  if (c->pers_on) persistence_update(c);
  c->mcs++;
}

int fail(oracle_ctx *c, int code, const char *msg) { if (c) c->err = msg; return code; }

}  // namespace

extern "C" {

int oracle_create(const oracle_params *p, oracle_ctx **out) {
  if (!p || !out) return ORACLE_ERR_ARG;
  *out = nullptr;
  if (p->ndim != 2 && p->ndim != 3) return ORACLE_ERR_DIMS;
  if (p->neighbourhood != 0) return ORACLE_ERR_UNSUPPORTED;
  if (p->n_types < 1 || p->n_types > 127 || !p->J) return ORACLE_ERR_ARG;
  if (p->T < 0 || std::isnan(p->T)) return ORACLE_ERR_ARG;
  if (p->mode != ORACLE_MODE_DETERMINISTIC && p->mode != ORACLE_MODE_LIVE) return ORACLE_ERR_ARG;
  if (p->max_cells >= (1u << 24)) return ORACLE_ERR_UNSUPPORTED;
  oracle_ctx *c = new oracle_ctx();
  c->d = p->ndim;
  for (int a = 0; a < 3; ++a) { c->dim[a] = (a < c->d) ? p->dims[a] : 1; c->per[a] = (a < c->d) ? (p->periodic[a] != 0) : 0; }
  for (int a = 0; a < c->d; ++a) if (c->dim[a] < 1) { delete c; return ORACLE_ERR_DIMS; }
  c->nT = p->n_types;
  const int nT = c->nT;
  c->J.resize((size_t)nT * nT);
  for (int i = 0; i < nT * nT; ++i) c->J[i] = p->J[i];
  for (int i = 0; i < nT; ++i)
    for (int j = 0; j < nT; ++j)
      if (c->J[i * nT + j] != c->J[j * nT + i]) { delete c; return ORACLE_ERR_ARG; }
  auto take = [&](const int32_t *src, std::vector<int64_t> &dst) {
    dst.assign(nT, 0);
    if (src) for (int i = 0; i < nT; ++i) dst[i] = src[i];
  };
  take(p->lambda_V, c->lamV); take(p->target_V, c->tgtV); take(p->lambda_P, c->lamP);
  take(p->target_P, c->tgtP); take(p->lambda_act, c->lamA); take(p->max_act, c->maxA);
  for (int i = 0; i < nT; ++i) if (c->maxA[i] < 0 || c->maxA[i] > 255 || c->lamA[i] < 0) { delete c; return ORACLE_ERR_ARG; }
  take(p->lambda_pers, c->lamPers); take(p->lambda_chem, c->lamChem);
  c->mu.assign(nT, 0.0);
  if (p->mu_pers) for (int i = 0; i < nT; ++i) c->mu[i] = p->mu_pers[i];
  c->dt = p->dt_pers;
  for (int i = 0; i < nT; ++i) {
    if (!(c->mu[i] >= 0.0 && c->mu[i] <= 1.0) || std::llabs(c->lamPers[i]) > (1 << 24) || std::llabs(c->lamChem[i]) > (1 << 24)) { delete c; return ORACLE_ERR_ARG; }
    if (c->lamPers[i] != 0) c->pers_on = true;
    if (c->lamChem[i] != 0) c->chem_on = true;
  }
  if (c->dt < 0 || (c->pers_on && c->dt < 1)) { delete c; return ORACLE_ERR_ARG; }
  c->unwrap = p->unwrap_centroids != 0 && (c->per[0] || c->per[1] || c->per[2]);
  c->T = p->T;
  c->accept_all = std::isinf(p->T);
  c->seed = p->seed;
  c->mode = p->mode;
  c->max_cells = p->max_cells;

  /* schedule (a1, readings S11): S must divide every dimension; periodic axes need an even
   * number of subsections so that same-colour subsections are never adjacent through the wrap */
  int S = p->subsection;
  if (S == 0) {
    S = (c->d == 2) ? 8 : 4;   /* a small area per worker, as in the paper's Fig 4 (4x4 per thread) */
    auto divides = [&](int s) { for (int a = 0; a < c->d; ++a) if (c->dim[a] % s) return false; return true; };
    while (S > 2 && !divides(S)) S /= 2;
  }
  if (S < 2) { delete c; return ORACLE_ERR_DIMS; }
  for (int a = 0; a < c->d; ++a) {
    if (c->dim[a] % S) { delete c; return ORACLE_ERR_DIMS; }
    c->nsub[a] = c->dim[a] / S;
    if (c->per[a] && (c->nsub[a] & 1)) { delete c; return ORACLE_ERR_DIMS; }
  }
  c->S = S;
  c->sites = 1; for (int a = 0; a < c->d; ++a) c->sites *= S;
  c->k = p->attempts_per_activation ? p->attempts_per_activation : c->sites;
  if (c->k < 1 || c->sites % c->k) { delete c; return ORACLE_ERR_ARG; }
  c->R = c->sites / c->k;

  c->nNb = build_offsets(c->d, c->off);
  /* reading S21: x^ of neighbour index nb points from the source s = t + OFF[nb] to the target t */
  for (int q = 0; q < c->nNb; ++q) {
    const double len = std::sqrt((double)(c->off[q][0] * c->off[q][0] + c->off[q][1] * c->off[q][1] + c->off[q][2] * c->off[q][2]));
    for (int a = 0; a < 3; ++a) c->xq[q][a] = std::llround(16384.0 * (double)(-c->off[q][a]) / len);
  }
  c->Hmax = threshold_hmax(c->T);
  c->thr.assign((size_t)c->Hmax + 1, 0xffffffffu);
  for (int64_t h = 1; h <= c->Hmax; ++h) c->thr[(size_t)h] = threshold_value(c->T, h);
  build_act_tables();

  size_t N = (size_t)c->dim[0] * c->dim[1] * c->dim[2];
  c->id.assign(N, 0); c->frozen.assign(N, 0); c->act.assign(N, 0);
  c->type.assign((size_t)c->max_cells + 1, 0);
  recount(c);
  *out = c;
  return ORACLE_OK;
}

int oracle_destroy(oracle_ctx *c) { delete c; return ORACLE_OK; }

int oracle_set_lattice(oracle_ctx *c, const uint32_t *ids, const uint8_t *frozen, const uint8_t *cell_type) {
  if (!c || !ids || !cell_type) return fail(c, ORACLE_ERR_ARG, "null argument");
  size_t N = c->id.size();
  for (size_t i = 0; i <= c->max_cells; ++i)
    if (cell_type[i] >= c->nT) return fail(c, ORACLE_ERR_ARG, "cell type out of range");
  if (cell_type[0] != 0) return fail(c, ORACLE_ERR_ARG, "cell 0 must have type 0 (medium)");
  for (size_t i = 0; i < N; ++i)
    if (ids[i] > c->max_cells) return fail(c, ORACLE_ERR_ARG, "cell id above max_cells");
  std::copy(ids, ids + N, c->id.begin());
  if (frozen) std::copy(frozen, frozen + N, c->frozen.begin()); else c->frozen.assign(N, 0);
  std::copy(cell_type, cell_type + c->max_cells + 1, c->type.begin());
  c->act.assign(N, 0); /* reading S9 */
  recount(c);
  if (c->pers_on) {   /* reading S22: p^ = 0 (no bias), the look-back window starts at the present centroids */
    const size_t ncell = (size_t)c->max_cells + 1;
    c->phat.assign(ncell * 3, 0.0);
    c->ring.assign(((size_t)c->dt + 1) * ncell * 3, 0.0);
    for (size_t cell = 1; cell < ncell; ++cell) {
      if (c->V[cell] <= 0) continue;
      double X[3];
      centroid(c, cell, X);
      for (size_t sl = 0; sl <= (size_t)c->dt; ++sl)
        for (int a = 0; a < 3; ++a) c->ring[(sl * ncell + cell) * 3 + a] = X[a];
    }
    c->n_updates = 0;
  }
  c->have_lattice = true;
  return ORACLE_OK;
}

int oracle_set_act(oracle_ctx *c, const float *act) {
  if (!c || !act) return fail(c, ORACLE_ERR_ARG, "null argument");
  for (size_t i = 0; i < c->act.size(); ++i) {
    float v = act[i];
    if (!(v >= 0.f) || v > 255.f || v != std::floor(v)) return fail(c, ORACLE_ERR_ARG, "act must be an integer in [0,255]");
    c->act[i] = (int32_t)v;
  }
  return ORACLE_OK;
}

int oracle_set_mcs(oracle_ctx *c, uint32_t mcs) { if (!c) return ORACLE_ERR_ARG; c->mcs = mcs; return ORACLE_OK; }

int oracle_step(oracle_ctx *c, uint32_t n_mcs) {
  if (!c) return ORACLE_ERR_ARG;
  if (!c->have_lattice) return fail(c, ORACLE_ERR_STATE, "set_lattice first");
  for (uint32_t i = 0; i < n_mcs; ++i) one_mcs(c);
  return ORACLE_OK;
}

int oracle_get_lattice(oracle_ctx *c, uint32_t *ids) {
  if (!c || !ids) return ORACLE_ERR_ARG;
  std::copy(c->id.begin(), c->id.end(), ids);
  return ORACLE_OK;
}

int oracle_get_act(oracle_ctx *c, float *act) {
  if (!c || !act) return ORACLE_ERR_ARG;
  for (size_t i = 0; i < c->act.size(); ++i) act[i] = (float)c->act[i];
  return ORACLE_OK;
}

int oracle_get_cell_stats(oracle_ctx *c, uint32_t *volume, uint32_t *perimeter, uint64_t *sx, uint64_t *sy, uint64_t *sz) {
  if (!c) return ORACLE_ERR_ARG;
  for (size_t i = 0; i <= c->max_cells; ++i) {
    if (volume) volume[i] = (uint32_t)c->V[i];
    if (perimeter) perimeter[i] = (uint32_t)c->P[i];
    if (sx) sx[i] = (uint64_t)c->SX[i];
    if (sy) sy[i] = (uint64_t)c->SY[i];
    if (sz) sz[i] = (uint64_t)c->SZ[i];
  }
  return ORACLE_OK;
}

int oracle_get_counters(oracle_ctx *c, uint64_t out[4]) {
  if (!c || !out) return ORACLE_ERR_ARG;
  out[0] = c->attempts; out[1] = c->evaluated; out[2] = c->accepted; out[3] = c->mcs;
  return ORACLE_OK;
}

int oracle_get_schedule(oracle_ctx *c, int32_t *S, int32_t *k, int32_t *steps) {
  if (!c) return ORACLE_ERR_ARG;
  if (S) *S = c->S;
  if (k) *k = (int32_t)c->k;
  if (steps) *steps = (int32_t)((1 << c->d) * c->R);
  return ORACLE_OK;
}

const char *oracle_last_error(const oracle_ctx *c) { return c ? c->err.c_str() : "null context"; }

int oracle_set_visit_order(oracle_ctx *c, int32_t order, uint64_t order_seed) {
  if (!c || order < 0 || order > 2) return ORACLE_ERR_ARG;
  c->order = order; c->order_seed = order_seed;
  return ORACLE_OK;
}

int oracle_probe(oracle_ctx *c, uint64_t t_index, int32_t nb, int32_t *status, int64_t *dH_ham, int64_t *dH_act) {
  if (!c || nb < 0 || nb >= c->nNb || t_index >= c->id.size()) return ORACLE_ERR_ARG;
  int tx = (int)(t_index % c->dim[0]);
  int ty = (int)((t_index / c->dim[0]) % c->dim[1]);
  int tz = (int)(t_index / ((uint64_t)c->dim[0] * c->dim[1]));
  Eval e = evaluate(c, tx, ty, tz, nb, [&](uint32_t cell, int64_t &Vv, int64_t &Pp) { Vv = c->V[cell]; Pp = c->P[cell]; });
  if (status) *status = e.status;
  if (dH_ham) *dH_ham = e.dH_ham;
  if (dH_act) *dH_act = e.dH_act;
  return ORACLE_OK;
}

int oracle_force_copy(oracle_ctx *c, uint64_t t_index, int32_t nb) {
  if (!c || nb < 0 || nb >= c->nNb || t_index >= c->id.size()) return ORACLE_ERR_ARG;
  int tx = (int)(t_index % c->dim[0]);
  int ty = (int)((t_index / c->dim[0]) % c->dim[1]);
  int tz = (int)(t_index / ((uint64_t)c->dim[0] * c->dim[1]));
  Eval e = evaluate(c, tx, ty, tz, nb, [&](uint32_t cell, int64_t &Vv, int64_t &Pp) { Vv = c->V[cell]; Pp = c->P[cell]; });
  if (e.status != 1) return fail(c, ORACLE_ERR_STATE, "copy is an early-out or refused");
  Delta dA, dB;
  commit(c, tx, ty, tz, e, dA, dB);
  if (e.A != 0) apply(c, e.A, dA);
  if (e.B != 0) apply(c, e.B, dB);
  return ORACLE_OK;
}

int oracle_set_trace(oracle_ctx *c, int64_t *buf, uint64_t cap, uint64_t *count) {
  if (!c) return ORACLE_ERR_ARG;
  c->trace = buf; c->trace_cap = cap; c->trace_count = count;
  if (count) *count = 0;
  return ORACLE_OK;
}

int oracle_set_chemotaxis_field(oracle_ctx *c, const float *field) {
  if (!c || !field) return fail(c, ORACLE_ERR_ARG, "null argument");
  if (!c->chem_on) return fail(c, ORACLE_ERR_UNSUPPORTED, "no type has lambda_chem != 0");
  const size_t N = c->id.size();
  for (size_t i = 0; i < N * (size_t)c->d; ++i)
    if (!(field[i] >= -1.0f && field[i] <= 1.0f)) return fail(c, ORACLE_ERR_ARG, "field components must lie in [-1,1]");
  c->cq.assign(N * 3, 0);
  for (size_t i = 0; i < N; ++i)
    for (int a = 0; a < c->d; ++a)
      c->cq[3 * i + a] = (int32_t)std::lrintf(field[i * (size_t)c->d + a] * 16384.0f);   /* Q14, round to nearest even */
  return ORACLE_OK;
}

int oracle_set_persistence(oracle_ctx *c, const double *p) {
  if (!c || !p) return fail(c, ORACLE_ERR_ARG, "null argument");
  if (!c->pers_on || !c->have_lattice) return fail(c, ORACLE_ERR_STATE, "persistence is off or no lattice");
  const size_t n3 = 3 * ((size_t)c->max_cells + 1);
  for (size_t i = 0; i < n3; ++i)
    if (!(p[i] >= -1.0 && p[i] <= 1.0)) return fail(c, ORACLE_ERR_ARG, "components must lie in [-1,1]");
  std::copy(p, p + n3, c->phat.begin());
  return ORACLE_OK;
}

int oracle_get_persistence(oracle_ctx *c, double *p) {
  if (!c || !p) return ORACLE_ERR_ARG;
  if (!c->pers_on || !c->have_lattice) return fail(c, ORACLE_ERR_STATE, "persistence is off or no lattice");
  std::copy(c->phat.begin(), c->phat.end(), p);
  return ORACLE_OK;
}

/* Eq 10: centroid = coordinate sums / number of sites, in double; (0,0,0) for ids that hold no site */
int oracle_get_centroids(oracle_ctx *c, double *xyz) {
  if (!c || !xyz) return ORACLE_ERR_ARG;
  for (size_t cell = 0; cell <= c->max_cells; ++cell) {
    double X[3] = {0.0, 0.0, 0.0};
    if (cell != 0 && c->V[cell] > 0) centroid(c, cell, X);
    for (int a = 0; a < 3; ++a) xyz[3 * cell + a] = X[a];
  }
  return ORACLE_OK;
}

int oracle_probe_dir(oracle_ctx *c, uint64_t t_index, int32_t nb, int64_t *dH_dir) {
  if (!c || nb < 0 || nb >= c->nNb || t_index >= c->id.size() || !dH_dir) return ORACLE_ERR_ARG;
  int tx = (int)(t_index % c->dim[0]);
  int ty = (int)((t_index / c->dim[0]) % c->dim[1]);
  int tz = (int)(t_index / ((uint64_t)c->dim[0] * c->dim[1]));
  Eval e = evaluate(c, tx, ty, tz, nb, [&](uint32_t cell, int64_t &Vv, int64_t &Pp) { Vv = c->V[cell]; Pp = c->P[cell]; });
  *dH_dir = (e.status == 1) ? e.dH_dir : 0;
  return ORACLE_OK;
}

int oracle_direction_table(int32_t ndim, int64_t *out) {
  int off[26][3];
  if (ndim != 2 && ndim != 3) return ORACLE_ERR_ARG;
  int n = build_offsets(ndim, off);
  for (int q = 0; q < n; ++q) {
    const double len = std::sqrt((double)(off[q][0] * off[q][0] + off[q][1] * off[q][1] + off[q][2] * off[q][2]));
    for (int a = 0; a < 3; ++a) out[3 * q + a] = std::llround(16384.0 * (double)(-off[q][a]) / len);
  }
  return n;
}

/* ---- instrumentation: sorting observables and update statistics ---- */

/* Number of unordered Moore pairs {i, j} of lattice positions held by DIFFERENT cells, by the types of the two cells
 * (the interfaces Eq 1 sums J over; homotypic = diagonal, heterotypic = off-diagonal: the sorting observable of
 * Fig 4, L69).  A position outside a closed lattice is medium (reading S5), so a cell site on the border forms a
 * (type, 0) pair with each of its outside neighbours.  out[a*nT + b] == out[b*nT + a]. */
int oracle_get_interface_counts(oracle_ctx *c, uint64_t *out) {
  if (!c || !out) return ORACLE_ERR_ARG;
  const int nT = c->nT;
  std::vector<uint64_t> cnt((size_t)nT * nT, 0);
  for (int z = 0; z < c->dim[2]; ++z)
    for (int y = 0; y < c->dim[1]; ++y)
      for (int x = 0; x < c->dim[0]; ++x) {
        SiteView me = view(c, x, y, z);
        for (int q = 0; q < c->nNb; ++q) {
          SiteView nb = view(c, x + c->off[q][0], y + c->off[q][1], z + c->off[q][2]);
          if (nb.id == me.id) continue;
          /* an inside pair is met from both ends: count it from the end whose offset comes first (q < nNb/2 means the
           * neighbour precedes in scan order); a pair with an outside position is met once */
          if (nb.inside && q < c->nNb / 2) continue;
          cnt[(size_t)me.tau * nT + nb.tau] += 1;
          if (me.tau != nb.tau) cnt[(size_t)nb.tau * nT + me.tau] += 1;
        }
      }
  std::copy(cnt.begin(), cnt.end(), out);
  return ORACLE_OK;
}

/* Update statistics of the schedule (Fig 3, L65-79): which positions the copy attempts of the next n_mcs MCS pick as
 * targets, without touching the lattice.  All active subsections advance in lock-step (the paper puts a barrier
 * after every update, L75), so attempt a of the e-th non-empty phase-step of the m-th MCS happens at tick
 * (m * E + e) * k + a, E = non-empty phase-steps per MCS.
 *   freq[j]: (position, MCS) pairs in which the position was picked exactly j times in that MCS (last bin: >= n_freq-1);
 *   wait[j]: consecutive picks of the same position whose ticks differ by dt with (dt-1)/bin == j (last bin: beyond). */
int oracle_update_statistics(oracle_ctx *c, uint32_t n_mcs, uint64_t *freq, int32_t n_freq, uint64_t *wait, int32_t n_wait,
                             uint32_t bin) {
  if (!c || !freq || !wait || n_freq < 1 || n_wait < 1 || bin < 1) return ORACLE_ERR_ARG;
  const size_t N = c->id.size();
  std::vector<uint64_t> last(N, 0);       /* tick + 1 of the last pick; 0 = never */
  std::vector<uint32_t> cnt(N, 0);
  std::fill(freq, freq + n_freq, 0); std::fill(wait, wait + n_wait, 0);
  const int ncol = 1 << c->d;
  const int64_t nsub_total = (int64_t)c->nsub[0] * c->nsub[1] * c->nsub[2];
  const uint32_t key[2] = {(uint32_t)c->seed, (uint32_t)(c->seed >> 32)};
  std::vector<int> occurs(ncol, 0);
  for (int64_t b = 0; b < nsub_total; ++b) {
    int bx = (int)(b % c->nsub[0]), by = (int)((b / c->nsub[0]) % c->nsub[1]), bz = (int)(b / ((int64_t)c->nsub[0] * c->nsub[1]));
    occurs[(bx & 1) | ((by & 1) << 1) | ((bz & 1) << 2)] = 1;
  }
  int E_per_rep = 0;
  for (int col = 0; col < ncol; ++col) E_per_rep += occurs[col];
  const uint64_t E = (uint64_t)E_per_rep * (uint64_t)c->R;
  for (uint32_t m = 0; m < n_mcs; ++m) {
    uint64_t e = 0;
    for (int64_t rep = 0; rep < c->R; ++rep)
      for (int col = 0; col < ncol; ++col) {
        if (!occurs[col]) continue;
        const uint32_t p = (uint32_t)(rep * ncol + col);
        for (int64_t b = 0; b < nsub_total; ++b) {
          int bx = (int)(b % c->nsub[0]), by = (int)((b / c->nsub[0]) % c->nsub[1]), bz = (int)(b / ((int64_t)c->nsub[0] * c->nsub[1]));
          if (((bx & 1) | ((by & 1) << 1) | ((bz & 1) << 2)) != col) continue;
          uint32_t w4[4] = {0, 0, 0, 0};
          for (int64_t a = 0; a < c->k; ++a) {
            if ((a & 3) == 0) { uint32_t ctr[4] = {(uint32_t)(a >> 2), (uint32_t)b, 2 * p + 0, c->mcs + m}; philox(ctr, key, w4); }
            uint32_t l, nb;
            decode_proposal(w4[a & 3], (uint32_t)c->sites, (uint32_t)c->nNb, &l, &nb);
            const int S = c->S;
            const int tx = bx * S + (int)(l % S), ty = by * S + (int)((l / S) % S), tz = (c->d == 3) ? bz * S + (int)(l / (S * S)) : 0;
            const size_t i = (size_t)lin(c, tx, ty, tz);
            const uint64_t tick = ((uint64_t)m * E + e) * (uint64_t)c->k + (uint64_t)a;
            if (last[i] != 0) {
              const uint64_t dt = tick + 1 - last[i];
              wait[std::min<uint64_t>((dt - 1) / bin, (uint64_t)n_wait - 1)] += 1;
            }
            last[i] = tick + 1;
            cnt[i] += 1;
          }
        }
        ++e;
      }
    for (size_t i = 0; i < N; ++i) { freq[std::min<uint32_t>(cnt[i], (uint32_t)n_freq - 1)] += 1; cnt[i] = 0; }
  }
  return ORACLE_OK;
}

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox(ctr, key, out); }

void oracle_decode_proposal(uint32_t w, uint32_t sites, uint32_t n_nb, uint32_t *l, uint32_t *nb) {
  decode_proposal(w, sites, n_nb, l, nb);
}

int64_t oracle_threshold_table(double T, uint32_t *thr, uint64_t cap) {
  int64_t hmax = threshold_hmax(T);
  if (thr && cap > 0) thr[0] = 0xffffffffu;
  for (int64_t h = 1; h <= hmax && (uint64_t)h < cap; ++h) thr[h] = threshold_value(T, h);
  return hmax;
}

int64_t oracle_gm_q16(const int32_t *act, int32_t n) { return gm_q16(act, n); }

int oracle_neighbour_offsets(int32_t ndim, int32_t *out) {
  int off[26][3];
  if (ndim != 2 && ndim != 3) return ORACLE_ERR_ARG;
  int n = build_offsets(ndim, off);
  for (int i = 0; i < n; ++i) { out[3 * i] = off[i][0]; out[3 * i + 1] = off[i][1]; out[3 * i + 2] = off[i][2]; }
  return n;
}

}  // extern "C"
