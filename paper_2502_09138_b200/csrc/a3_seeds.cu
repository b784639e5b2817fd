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

// Latency-bound (gathers, look-back): full occupancy (8 CTAs, 32 registers, 24 B of spill) beats 6 CTAs at 40
// registers, 0.297 against 0.347 ms.
__global__ void __launch_bounds__(A3_THREADS, 8)
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

  // Each thread owns A3_ITEMS consecutive ids: every load level is issued for all items before any is used, so
  // the gathers of one level are in flight together (the kernel is bound by their latency, not by bandwidth).
  const int64_t h0 = base + (int64_t)threadIdx.x * A3_ITEMS;
  int u[A3_ITEMS], d[A3_ITEMS], yy[A3_ITEMS], zz[A3_ITEMS];
  static_assert(A3_ITEMS == 4, "one 16-byte load per array and thread");
  const bool vec = h0 + A3_ITEMS <= n && ((((uintptr_t)y | (uintptr_t)z) & 15) == 0);   // up, dn: arena, 256-B aligned
  if (vec) {
    const int4 vu = *(const int4*)(up + h0), vd = *(const int4*)(dn + h0);
    const int4 vy = *(const int4*)(y + h0), vz = *(const int4*)(z + h0);
    u[0] = vu.x; u[1] = vu.y; u[2] = vu.z; u[3] = vu.w;
    d[0] = vd.x; d[1] = vd.y; d[2] = vd.z; d[3] = vd.w;
    yy[0] = vy.x; yy[1] = vy.y; yy[2] = vy.z; yy[3] = vy.w;
    zz[0] = vz.x; zz[1] = vz.y; zz[2] = vz.z; zz[3] = vz.w;
  } else {
#pragma unroll
    for (int k = 0; k < A3_ITEMS; ++k) {
      const bool in = h0 + k < n;
      u[k] = in ? up[h0 + k] : -1;
      d[k] = in ? dn[h0 + k] : -1;
      yy[k] = in ? y[h0 + k] : 0;
      zz[k] = in ? z[h0 + k] : 0;
    }
  }
  int du[A3_ITEMS], ud[A3_ITEMS];
#pragma unroll
  for (int k = 0; k < A3_ITEMS; ++k) {
    du[k] = u[k] >= 0 ? dn[u[k]] : -1;
    ud[k] = d[k] >= 0 ? up[d[k]] : -1;
  }
  int c[A3_ITEMS], len[A3_ITEMS];
  bool walk[A3_ITEMS];
#pragma unroll
  for (int k = 0; k < A3_ITEMS; ++k) {
    const int h = (int)(h0 + k);
    const int uc = (u[k] >= 0 && du[k] == h) ? u[k] : -1;   // P11
    const int dc = (d[k] >= 0 && ud[k] == h) ? d[k] : -1;
    if (h0 + k < n) rec[h0 + k] = make_int4(yy[k], zz[k], uc, dc);
    walk[k] = dc < 0 && uc >= 0;   // P12 chain start; the walk uses raw links + the mutual test (= cleaned links)
    c[k] = uc;
    len[k] = 2;
  }
  for (int step = 2; step < g.l_min; ++step) {   // all walks of the thread advance together
    int nx[A3_ITEMS], back[A3_ITEMS];
#pragma unroll
    for (int k = 0; k < A3_ITEMS; ++k) nx[k] = (walk[k] && len[k] == step) ? up[c[k]] : -1;
#pragma unroll
    for (int k = 0; k < A3_ITEMS; ++k) back[k] = nx[k] >= 0 ? dn[nx[k]] : -1;
#pragma unroll
    for (int k = 0; k < A3_ITEMS; ++k)
      if (nx[k] >= 0 && back[k] == c[k]) {
        c[k] = nx[k];
        ++len[k];
      }
  }
  bool seed[A3_ITEMS];
  uint32_t mine = 0;
#pragma unroll
  for (int k = 0; k < A3_ITEMS; ++k) {
    seed[k] = walk[k] && len[k] >= g.l_min;   // P13
    mine += seed[k] ? 1u : 0u;
  }
  uint32_t running;
  uint32_t pos = block_excl_scan(mine, wsum, &running);   // ids ascend with (thread, item): ranks follow (P14)
  const uint32_t excl = (uint32_t)lookback_scan(status, tile, running, &sh_excl);
#pragma unroll
  for (int k = 0; k < A3_ITEMS; ++k)
    if (seed[k]) {
      const uint32_t h = (uint32_t)(h0 + k);
      int lo = 0, hi = g.n_sectors * g.n_rows;   // (sector,row) of the start: largest sr with ro[sr] <= h
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (ro[mid] <= h) lo = mid; else hi = mid;
      }
      seed_start[excl + pos] = (int32_t)h;
      seed_sr[excl + pos] = lo;
      ++pos;
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
