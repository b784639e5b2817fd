// a3_seeds.cu -- stage a3: cellular-automaton link cleaner, chain starts, seed extraction (SURVEY 8(c)
// "Stage 3", P11-P14).  Integer only -> bit-exact.
//
// One synchronous cleaning step from the raw tables: up'[h] = up[h] if dn[up[h]] == h else -1 (dn' likewise).
// Chain start: dn'[h] < 0 and up'[h] >= 0; a chain is a seed iff it has >= l_min clusters, which a walk of at
// most l_min - 1 steps decides; seeds are ranked by ascending start id (P14).
// Thread per cluster id, so the seed flags come out in id order and one single-pass look-back scan turns
// them into ranks: clean + start test + bounded walk + rank + compaction are one kernel.
// For a4 the kernel also packs (y, z, up', dn') of every cluster into one 16-byte record (a4 then needs one
// gather per followed hit instead of three) and looks up the (sector,row) of every seed start.
#include "tpc_internal.cuh"

namespace {

constexpr int A3_THREADS = 256;
constexpr int A3_ITEMS = A3_TILE / A3_THREADS;

__global__ void __launch_bounds__(A3_THREADS)
a3_seeds_kernel(const DevGeom g, int64_t n, const int32_t* __restrict__ y, const int32_t* __restrict__ z,
                const uint32_t* __restrict__ ro, const int32_t* __restrict__ up, const int32_t* __restrict__ dn,
                int4* __restrict__ rec, int32_t* __restrict__ seed_start, int32_t* __restrict__ seed_sr,
                DevCtl* __restrict__ ctl, uint64_t* __restrict__ status, uint32_t n_tiles) {
  __shared__ uint32_t wsum[33];
  __shared__ uint32_t sh_tile;
  __shared__ uint64_t sh_excl;
  if (threadIdx.x == 0) sh_tile = atomicAdd(&ctl->ticket_a3, 1u);
  __syncthreads();
  const uint32_t tile = sh_tile;
  const int64_t base = (int64_t)tile * A3_TILE;

  bool seed[A3_ITEMS];
  uint32_t pos[A3_ITEMS];
  uint32_t running = 0;
#pragma unroll
  for (int k = 0; k < A3_ITEMS; ++k) {
    const int64_t h = base + k * A3_THREADS + threadIdx.x;
    seed[k] = false;
    if (h < n) {
      const int u = up[h], d = dn[h];
      const int uc = (u >= 0 && dn[u] == (int)h) ? u : -1;   // P11
      const int dc = (d >= 0 && up[d] == (int)h) ? d : -1;
      rec[h] = make_int4(y[h], z[h], uc, dc);
      if (dc < 0 && uc >= 0) {   // P12 chain start; the walk uses raw links + the mutual test (= cleaned links)
        int len = 2, c = uc;
        while (len < g.l_min) {
          const int nx = up[c];
          if (nx < 0 || dn[nx] != c) break;
          c = nx;
          ++len;
        }
        seed[k] = len >= g.l_min;   // P13
      }
    }
    uint32_t tot;
    pos[k] = running + block_excl_scan(seed[k] ? 1u : 0u, wsum, &tot);
    running += tot;
  }
  const uint32_t excl = (uint32_t)lookback_scan(status, tile, running, &sh_excl);
#pragma unroll
  for (int k = 0; k < A3_ITEMS; ++k)
    if (seed[k]) {
      const uint32_t h = (uint32_t)(base + k * A3_THREADS + threadIdx.x);
      int lo = 0, hi = g.n_sectors * g.n_rows;   // (sector,row) of the start: largest sr with ro[sr] <= h
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (ro[mid] <= h) lo = mid; else hi = mid;
      }
      seed_start[excl + pos[k]] = (int32_t)h;
      seed_sr[excl + pos[k]] = lo;
    }
  if (tile == n_tiles - 1 && threadIdx.x == 0) ctl->n_seeds = excl + running;
}

}  // namespace

cudaError_t launch_a3_seeds(const tpc_tracker* t, const int32_t* y, const int32_t* z, const uint32_t* ro, int64_t n,
                            cudaStream_t st) {
  if (t->tiles_a3 == 0 || n == 0) return cudaSuccess;
  const uint32_t tiles = (uint32_t)((n + A3_TILE - 1) / A3_TILE);
  a3_seeds_kernel<<<tiles, A3_THREADS, 0, st>>>(t->g, n, y, z, ro, t->s.link_up, t->s.link_dn, t->s.rec,
                                               t->s.seed_start, t->s.seed_sr, t->s.ctl, t->s.scan_a3, tiles);
  return cudaGetLastError();
}
