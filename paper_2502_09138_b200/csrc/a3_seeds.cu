// a3_seeds.cu -- stage a3: cellular-automaton link cleaner, chain starts, seed extraction (SURVEY 8(c)
// "Stage 3", P11-P14).  Integer only -> bit-exact.
//
// Everything here runs in SORTED space: a2 wrote link_up[p] / link_dn[p] as positions in srt (the bin-ordered cluster
// array of a1), at position p.  One synchronous cleaning step from the raw tables: up'[p] = up[p] if dn[up[p]] == p
// else -1 (dn' likewise).  Chain start: dn'[p] < 0 and up'[p] >= 0; a chain is a seed iff it has >= l_min clusters,
// which a walk of at most l_min - 1 steps decides.
// Thread per sorted position: loads and stores of the link tables are coalesced; the cleaned up links go to a table of
// their own (clean_up, whole sectors per warp), which a4 reads next to the srt record of every chain hit it follows.
// Seeds come out in sorted-position order (block scan + single-pass look-back scan); P14 ranks them by ascending
// start *id*.  Positions and ids of a (sector,row) fill the same index range, so the two orders differ only inside
// a row: a3_rank_kernel moves every seed to its id-order rank by counting, among the seeds of its own row (which
// are adjacent in the position-ordered list), those with a smaller start id.
#include "tpc_internal.cuh"

namespace {

constexpr int A3_THREADS = 256;
constexpr int A3_ITEMS = A3_TILE / A3_THREADS;

// Latency-bound (gathers, look-back): full occupancy (8 CTAs, 32 registers) beats 6 CTAs at 40 registers.
__global__ void __launch_bounds__(A3_THREADS, 8)
a3_seeds_kernel(const DevGeom g, int64_t n, const uint32_t* __restrict__ ro, const int32_t* __restrict__ up,
                const int32_t* __restrict__ dn, int32_t* __restrict__ clean_up, const int4* __restrict__ srt,
                int4* __restrict__ seed_tmp, uint32_t* __restrict__ seed_mask,
                DevCtl* __restrict__ ctl, uint64_t* __restrict__ status, uint32_t n_tiles, uint32_t s_cap) {
  __shared__ uint32_t wsum[33];
  __shared__ uint32_t sh_tile;
  __shared__ uint64_t sh_excl;
  if (ctl->bad_offsets) return;   // a0_check: nothing was sorted, no seeds
  if (threadIdx.x == 0) sh_tile = atomicAdd(&ctl->ticket_a3, 1u);
  __syncthreads();
  const uint32_t tile = sh_tile;
  const int64_t base = (int64_t)tile * A3_TILE;

  // Each thread owns A3_ITEMS consecutive positions: every load level is issued for all items before any is used,
  // so the gathers of one level are in flight together (the kernel is bound by their latency, not by bandwidth).
  const int64_t p0 = base + (int64_t)threadIdx.x * A3_ITEMS;
  int u[A3_ITEMS], d[A3_ITEMS];
  static_assert(A3_ITEMS == 4, "one 16-byte load per array and thread");
  const bool vec = p0 + A3_ITEMS <= n;   // up, dn: arena, 256-B aligned
  if (vec) {
    const int4 vu = *(const int4*)(up + p0), vd = *(const int4*)(dn + p0);
    u[0] = vu.x; u[1] = vu.y; u[2] = vu.z; u[3] = vu.w;
    d[0] = vd.x; d[1] = vd.y; d[2] = vd.z; d[3] = vd.w;
  } else {
#pragma unroll
    for (int k = 0; k < A3_ITEMS; ++k) {
      const bool in = p0 + k < n;
      u[k] = in ? up[p0 + k] : -1;
      d[k] = in ? dn[p0 + k] : -1;
    }
  }
  int du[A3_ITEMS], ud[A3_ITEMS];
#pragma unroll
  for (int k = 0; k < A3_ITEMS; ++k) {
    du[k] = u[k] >= 0 ? dn[u[k]] : -1;
    ud[k] = d[k] >= 0 ? up[d[k]] : -1;
  }
  int c[A3_ITEMS], len[A3_ITEMS], cl[A3_ITEMS];
  bool walk[A3_ITEMS];
#pragma unroll
  for (int k = 0; k < A3_ITEMS; ++k) {
    const int p = (int)(p0 + k);
    const int uc = (u[k] >= 0 && du[k] == p) ? u[k] : -1;   // P11
    const int dc = (d[k] >= 0 && ud[k] == p) ? d[k] : -1;
    cl[k] = uc;
    walk[k] = dc < 0 && uc >= 0;   // P12 chain start; the walk uses raw links + the mutual test (= cleaned links)
    c[k] = uc;
    len[k] = 2;
  }
  // the cleaned up links go to a table of their own, 16 bytes per thread, whole sectors per warp (as the fourth word
  // of the srt records every 4-byte store dirtied a sector that DRAM had to fill first: 0.6 GB of traffic per step)
  if (vec) {
    *(int4*)(clean_up + p0) = make_int4(cl[0], cl[1], cl[2], cl[3]);
  } else {
#pragma unroll
    for (int k = 0; k < A3_ITEMS; ++k)
      if (p0 + k < n) clean_up[p0 + k] = cl[k];
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
  uint32_t pos = block_excl_scan(mine, wsum, &running);
  const uint32_t excl = (uint32_t)lookback_scan(status, tile, running, &sh_excl);
#pragma unroll
  for (int k = 0; k < A3_ITEMS; ++k)
    if (seed[k]) {
      const uint32_t p = (uint32_t)(p0 + k);
      int lo = 0, hi = g.n_sectors * g.n_rows;   // (sector,row) of the start: largest sr with ro[sr] <= p
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (ro[mid] <= p) lo = mid; else hi = mid;
      }
      if (excl + pos < s_cap) {
        const int id = srt[p].z;
        seed_tmp[excl + pos] = make_int4((int)p, id, lo, 0);
        atomicOr(&seed_mask[id >> 5], 1u << (id & 31));   // for a3_rank_kernel's long rows
      }
      ++pos;
    }
  if (tile == n_tiles - 1 && threadIdx.x == 0) {
    const uint32_t found = excl + running;
    ctl->n_seeds_found = found;
    ctl->n_seeds = found < s_cap ? found : s_cap;   // a5 raises TPC_FLAG_SEED_OVERFLOW when they differ
  }
}

// P14: seed rank = ascending start id.  seed_tmp is in position order; the seeds of one (sector,row) are adjacent in
// it and fill the same rank range in both orders: rank = seeds of earlier rows + seeds of the own row with a smaller
// id.  Rows with a few seeds (central events: two per row): both counts by walking the neighbours in seed_tmp.  A
// walk that does not reach the row's ends within A3_RANK_WALK seeds (pile-up: a thousand seeds in a row, and the walk
// is quadratic) is replaced by a binary search for the row's first seed and a population count over the row's part
// of the seed bit mask (bit = cluster id).  Both give the same number.
constexpr int A3_RANK_WALK = 24;

__global__ void __launch_bounds__(256)
a3_rank_kernel(const DevCtl* __restrict__ ctl, const uint32_t* __restrict__ ro, const int4* __restrict__ seed_tmp,
               const uint32_t* __restrict__ seed_mask, const int4* __restrict__ srt,
               const int32_t* __restrict__ clean_up,
               int32_t* __restrict__ seed_start, int32_t* __restrict__ seed_pos, int32_t* __restrict__ seed_sr,
               int4* __restrict__ seed_rec) {
  const int64_t ns = ctl->n_seeds;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < ns; k += (int64_t)gridDim.x * blockDim.x) {
    const int4 me = seed_tmp[k];
    const int up0 = clean_up[me.x];
    const int4 c0 = srt[me.x];     // the seed's first cluster and (requested before the counting loops) its second
    const int4 c1 = srt[up0];
    int64_t left = 0, smaller = 0;
    bool whole = true;   // both walks reached the ends of the row
    for (int64_t j = k - 1; j >= 0; --j) {
      const int4 o = seed_tmp[j];
      if (o.z != me.z) break;
      if (left == A3_RANK_WALK) { whole = false; break; }
      ++left;
      smaller += o.y < me.y;
    }
    if (whole) {
      int steps = 0;
      for (int64_t j = k + 1; j < ns; ++j) {
        const int4 o = seed_tmp[j];
        if (o.z != me.z) break;
        if (steps == A3_RANK_WALK) { whole = false; break; }
        ++steps;
        smaller += o.y < me.y;
      }
    }
    int64_t rank = k - left + smaller;
    if (!whole) {
      int64_t lo = -1, hi = k;   // first seed of the row: smallest index whose (sector,row) is this one
      while (hi - lo > 1) {
        const int64_t mid = (lo + hi) >> 1;
        if (seed_tmp[mid].z < me.z) lo = mid; else hi = mid;
      }
      const uint32_t a = ro[me.z], id = (uint32_t)me.y;   // ids of the row: a .. ; seeds with an id in [a, id)
      uint32_t cnt = 0;
      for (uint32_t w = a >> 5; w <= id >> 5; ++w) {
        uint32_t m = seed_mask[w];
        if (w == a >> 5) m &= ~0u << (a & 31);
        if (w == id >> 5) m &= (1u << (id & 31)) - 1u;
        cnt += __popc(m);
      }
      rank = hi + cnt;
    }
    seed_start[rank] = me.y;
    seed_pos[rank] = me.x;
    seed_sr[rank] = me.z;
    // everything a4 needs to start the tracklet, in one 32-byte record: (sr, y0, z0, id0) (up0, y1, z1, -)
    seed_rec[2 * rank] = make_int4(me.z, c0.x, c0.y, c0.z);
    seed_rec[2 * rank + 1] = make_int4(up0, c1.x, c1.y, 0);
  }
}

}  // namespace

cudaError_t launch_a3_seeds(const tpc_tracker* t, const uint32_t* ro, int64_t n, cudaStream_t st) {
  if (t->tiles_a3 == 0 || n == 0) return cudaSuccess;
  const uint32_t tiles = (uint32_t)((n + A3_TILE - 1) / A3_TILE);
  a3_seeds_kernel<<<tiles, A3_THREADS, 0, st>>>(t->g, n, ro, t->s.link_up, t->s.link_dn, t->s.clean_up, t->s.srt, t->s.seed_tmp, t->s.seed_mask,
                                               t->s.ctl, t->s.scan_a3, tiles, (uint32_t)t->s_cap);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  // the seed count stays on the device: a grid-stride kernel sized for the device, not for the capacity
  a3_rank_kernel<<<t->a4_sms * 8, 256, 0, st>>>(t->s.ctl, ro, t->s.seed_tmp, t->s.seed_mask, t->s.srt, t->s.clean_up, t->s.seed_start, t->s.seed_pos,
                                               t->s.seed_sr, t->s.seed_rec);
  return cudaGetLastError();
}
