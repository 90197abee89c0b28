// cpm_stats_kernels.cuh -- instrumentation kernels: interface counts by cell type (the sorting
// observable of PAPER.md Fig 4, L69) and the update statistics of the checkerboard schedule (Fig 3, L65-79).
// Neither is on the sweep's hot path; both read the state the sweep kernels keep.  Nothing here is shared with oracle/.
#pragma once
#include "cpm_device.cuh"
#include "cpm_pool_kernel.cuh"

namespace cpm {

// the lattice under either layout: row-major words [frozen:1 | type:7 | id:24] or tiles [type:5 | frozen:1 | 00 | id:24]
struct LatView {
  const uint32_t *lat; long long pitch;
  TileLayout tl; int pooled;
  int X, Y, Z, per[3];
};
template <int DIM>
__device__ __forceinline__ void site_at(const LatView &V, int x, int y, int z, uint32_t &id, int &type) {
  if (V.pooled) {
    const uint32_t w = V.tl.tiles[home_word<DIM>(V.tl, V.tl.S, x, y, z)];
    id = w & ID_MASK; type = (int)(w >> PK_TYPE_SHIFT);
  } else {
    const uint32_t w = V.lat[(long long)x + V.pitch * ((long long)y + (long long)V.Y * z)];
    id = w & ID_MASK; type = (int)((w >> 24) & 127u);
  }
}

// Unordered Moore pairs of positions held by different cells, by the two cells' types (Eq 1's interfaces).  A position
// outside a closed lattice is medium (reading S5).  An inside pair is met from both ends and counted from the end
// whose offset index is in the upper half; equal (type, type) keys of a warp are combined before the atomics.
template <int DIM>
__global__ void interface_count_kernel(LatView V, int nT, unsigned long long *out, int use_smem) {
  constexpr int NNB = (DIM == 2) ? 8 : 26;
  extern __shared__ unsigned long long hist[];   // block-local counts [nT][nT] (use_smem), flushed once per block
  if (use_smem) {
    for (int i = threadIdx.x; i < nT * nT; i += blockDim.x) hist[i] = 0ull;
    __syncthreads();
  }
  unsigned long long *const acc = use_smem ? hist : out;
  const long long N = (long long)V.X * V.Y * V.Z;
  const long long stride = (long long)gridDim.x * blockDim.x;
  const long long first = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long n_iter = (N + stride - 1) / stride;
  for (long long it = 0; it < n_iter; ++it) {
    const long long i = first + it * stride;
    const bool live = i < N;
    int x = 0, y = 0, z = 0, tm = 0;
    uint32_t me = 0;
    if (live) {
      x = (int)(i % V.X);
      const long long r = i / V.X;
      y = (int)(r % V.Y); z = (int)(r / V.Y);
      site_at<DIM>(V, x, y, z, me, tm);
    }
#pragma unroll 1
    for (int q = 0; q < NNB; ++q) {
      int key = -1;
      if (live) {
        int dx, dy, dz;
        nb_delta<DIM>(q, dx, dy, dz);
        int g[3] = {x + dx, y + dy, z + dz};
        const int dimv[3] = {V.X, V.Y, V.Z};
        bool inside = true;
#pragma unroll
        for (int a = 0; a < DIM; ++a)
          if (g[a] < 0 || g[a] >= dimv[a]) { if (V.per[a]) g[a] += (g[a] < 0) ? dimv[a] : -dimv[a]; else inside = false; }
        if (!(inside && q < NNB / 2)) {
          uint32_t other = 0; int tn = 0;
          if (inside) site_at<DIM>(V, g[0], g[1], g[2], other, tn);
          if (other != me) key = tm * nT + tn;
        }
      }
      const unsigned peers = __match_any_sync(FULL, key);
      if (key >= 0 && (int)(threadIdx.x & 31) == __ffs(peers) - 1) {
        const unsigned long long n = (unsigned long long)__popc(peers);
        atomicAdd(acc + key, n);
        const int a = key / nT, b = key % nT;
        if (a != b) atomicAdd(acc + b * nT + a, n);
      }
    }
  }
  if (use_smem) {
    __syncthreads();
    for (int i = threadIdx.x; i < nT * nT; i += blockDim.x)
      if (hist[i] != 0ull) atomicAdd(out + i, hist[i]);
  }
}

// Eq 10: centroid = coordinate sums / volume (one IEEE division per component)
__global__ void centroid_kernel(long long ncell, const unsigned long long *liveVP, const unsigned long long *sumx,
                                const unsigned long long *sumy, const unsigned long long *sumz, double *xyz) {
  const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cell >= ncell) return;
  double X[3] = {0.0, 0.0, 0.0};
  const unsigned long long vp = liveVP[cell];
  if (cell != 0 && (uint32_t)(vp >> 32) != 0u) centroid_of(vp, sumx[cell], sumy[cell], sumz[cell], X);
  xyz[3 * cell] = X[0]; xyz[3 * cell + 1] = X[1]; xyz[3 * cell + 2] = X[2];
}

// Update statistics: one thread per subsection walks the target picks of its own activations over n_mcs MCS (proposal
// stream of the sweep: Philox counter (a>>2, b, 2p, mcs), word a&3, multiply-shift decode), in lock-step ticks
// (m E + e) k + a, E = non-empty phase-steps per MCS.  last / cnt: per-site scratch (N words each), only ever touched
// by the thread that owns the site's subsection.  hist = [n_freq | n_wait] counters.
struct StatParams {
  int S, sites, k, R, nNb;
  int nsub[3]; int X, Y;
  int rank[8];          // colour -> its rank among the colours that occur (or -1)
  int E_per_rep;
  uint32_t mcs0, n_mcs, key0, key1, bin;
  int n_freq, n_wait;
};
template <int DIM>
__global__ void update_stats_kernel(StatParams P, long long nsub_total, uint32_t *last, uint32_t *cnt, unsigned long long *hist) {
  extern __shared__ unsigned long long sh[];   // block-local copy of the histograms
  const int nh = P.n_freq + P.n_wait;
  for (int i = threadIdx.x; i < nh; i += blockDim.x) sh[i] = 0ull;
  __syncthreads();
  const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (b < nsub_total) {
    const int bx = (int)(b % P.nsub[0]), by = (int)((b / P.nsub[0]) % P.nsub[1]), bz = (int)(b / ((long long)P.nsub[0] * P.nsub[1]));
    const int col = (bx & 1) | ((by & 1) << 1) | ((bz & 1) << 2);
    const int ncol = 1 << DIM;
    const unsigned long long E = (unsigned long long)P.E_per_rep * (unsigned long long)P.R;
    for (uint32_t m = 0; m < P.n_mcs; ++m) {
      for (int rep = 0; rep < P.R; ++rep) {
        const uint32_t p = (uint32_t)(rep * ncol + col);
        const unsigned long long e = (unsigned long long)rep * P.E_per_rep + (unsigned long long)P.rank[col];
        uint4 r = make_uint4(0, 0, 0, 0);
        for (int a = 0; a < P.k; ++a) {
          if ((a & 3) == 0) r = philox4x32_10(make_uint4((uint32_t)a >> 2, (uint32_t)b, 2u * p, P.mcs0 + m), P.key0, P.key1);
          const int l = (int)(((unsigned long long)pick(r, a & 3) * (unsigned)P.sites) >> 32);
          const int tx = bx * P.S + l % P.S, ty = by * P.S + (l / P.S) % P.S, tz = (DIM == 3) ? bz * P.S + l / (P.S * P.S) : 0;
          const long long i = (long long)tx + (long long)P.X * ((long long)ty + (long long)P.Y * tz);
          const uint32_t tick1 = (uint32_t)(((unsigned long long)m * E + e) * (unsigned long long)P.k + (unsigned long long)a) + 1u;
          const uint32_t lst = last[i];
          if (lst != 0u) {
            const uint32_t j = (tick1 - lst - 1u) / P.bin;
            atomicAdd(sh + P.n_freq + min(j, (uint32_t)P.n_wait - 1u), 1ull);
          }
          last[i] = tick1;
          cnt[i] += 1u;
        }
      }
      // picks per position in this MCS
      for (int l = 0; l < P.sites; ++l) {
        const int tx = bx * P.S + l % P.S, ty = by * P.S + (l / P.S) % P.S, tz = (DIM == 3) ? bz * P.S + l / (P.S * P.S) : 0;
        const long long i = (long long)tx + (long long)P.X * ((long long)ty + (long long)P.Y * tz);
        atomicAdd(sh + min(cnt[i], (uint32_t)P.n_freq - 1u), 1ull);
        cnt[i] = 0u;
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < nh; i += blockDim.x)
    if (sh[i] != 0ull) atomicAdd(hist + i, sh[i]);
}

}  // namespace cpm
