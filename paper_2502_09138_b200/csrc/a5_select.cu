// a5_select.cu -- stage a5: hit-ownership selection and output compaction (SURVEY 8(c) "Stage 5", P24-P29;
// north_star "hit-ownership resolution with atomicMax on packed (quality, track-id) words").
//
// The votes (atomicMax of (n_hits << 24 | 0xFFFFFF - rank) per tracklet hit) were cast at the end of a4.
// Here: thread per tracklet counts the hits it owns, keeps the tracklet iff owned >= n_min_owned (P27), and a
// single-pass look-back scan over (kept, owned) gives each kept tracklet its output slot and hit offset in
// ascending seed order (P29).  Track parameters are the a4 fit over all tracklet hits (P28).
#include "tpc_internal.cuh"

namespace {

__global__ void __launch_bounds__(A5_TILE)
a5_select_kernel(const DevGeom g, int64_t s_cap, DevCtl* __restrict__ ctl, const int32_t* __restrict__ seed_start,
                 const float* __restrict__ tl_par, const float* __restrict__ tl_cov, const float* __restrict__ tl_chi2,
                 const int32_t* __restrict__ tl_nhits, const int32_t* __restrict__ tl_sr0,
                 const int32_t* __restrict__ tl_hits, const uint32_t* __restrict__ owner,
                 uint64_t* __restrict__ status, tpc_track_rec_t* __restrict__ tracks, int32_t track_capacity,
                 int32_t* __restrict__ hit_ids, int32_t hit_capacity, int32_t* __restrict__ counts) {
  __shared__ uint32_t wsum[33];
  __shared__ uint32_t sh_tile;
  __shared__ uint64_t sh_excl;
  const uint32_t n_seeds = ctl->n_seeds;
  const uint32_t n_tiles = (n_seeds + A5_TILE - 1) / A5_TILE;
  if (n_seeds == 0) {
    if (blockIdx.x == 0 && threadIdx.x == 0) {
      counts[0] = 0;
      counts[1] = 0;
      counts[2] = 0;
      counts[3] = 0;
    }
    return;
  }
  if (blockIdx.x >= n_tiles) return;   // the grid is sized by the seed capacity
  if (threadIdx.x == 0) sh_tile = atomicAdd(&ctl->ticket_a5, 1u);
  __syncthreads();
  const uint32_t tile = sh_tile;
  const int64_t i = (int64_t)tile * A5_TILE + threadIdx.x;
  const int nr = g.n_rows;

  uint32_t owned = 0;
  int first = -1, last = -1;
  uint32_t word = 0;
  if (i < n_seeds) {
    const int nh = tl_nhits[i];
    if (nh >= g.n_min_tracklet) {
      word = ((uint32_t)nh << 24) | (0xFFFFFFu - (uint32_t)i);
      for (int r = 0; r < nr; ++r) {
        const int h = tl_hits[(int64_t)r * s_cap + i];
        if (h >= 0 && owner[h] == word) {
          ++owned;
          if (first < 0) first = r;
          last = r;
        }
      }
    }
  }
  const bool keep = word != 0 && owned >= (uint32_t)g.n_min_owned;
  if (!keep) owned = 0;
  uint32_t tot_k, tot_h;
  const uint32_t pos_k = block_excl_scan(keep ? 1u : 0u, wsum, &tot_k);
  const uint32_t pos_h = block_excl_scan(owned, wsum, &tot_h);
  // payload: tracks in bits 61..38 (s_cap < 2^24), hits in bits 37..0 (n < 2^31)
  const uint64_t ex = lookback_scan(status, tile, ((uint64_t)tot_k << 38) | tot_h, &sh_excl);
  const uint32_t excl[2] = {(uint32_t)(ex >> 38), (uint32_t)(ex & ((1ull << 38) - 1))};

  if (keep) {
    const uint32_t slot = excl[0] + pos_k;
    const uint32_t off = excl[1] + pos_h;
    if (slot < (uint32_t)track_capacity) {
      tpc_track_rec_t rec;
      rec.x = tl_par[0 * s_cap + i];
      rec.y = tl_par[1 * s_cap + i];
      rec.z = tl_par[2 * s_cap + i];
      rec.sinphi = tl_par[3 * s_cap + i];
      rec.tanl = tl_par[4 * s_cap + i];
      rec.qpt = tl_par[5 * s_cap + i];
#pragma unroll
      for (int k = 0; k < 15; ++k) rec.cov[k] = tl_cov[k * s_cap + i];
      rec.chi2 = tl_chi2[i];
      rec.sector = tl_sr0[i] / nr;
      rec.first_row = first;
      rec.last_row = last;
      rec.n_hits = (int32_t)owned;
      rec.hit_offset = (int32_t)off;
      rec.seed_cluster = seed_start[i];
      tracks[slot] = rec;
    }
    if ((uint64_t)off + owned <= (uint64_t)hit_capacity) {
      uint32_t w = off;
      for (int r = first; r <= last; ++r) {
        const int h = tl_hits[(int64_t)r * s_cap + i];
        if (h >= 0 && owner[h] == word) hit_ids[w++] = h;
      }
    }
  }
  if (tile == n_tiles - 1 && threadIdx.x == 0) {
    const uint32_t nt = excl[0] + tot_k, nhits = excl[1] + tot_h;
    counts[0] = (int32_t)nt;
    counts[1] = (int32_t)nhits;
    counts[2] = (nt > (uint32_t)track_capacity ? TPC_FLAG_TRACK_OVERFLOW : 0u) |
                (nhits > (uint32_t)hit_capacity ? TPC_FLAG_HIT_OVERFLOW : 0u);
    counts[3] = (int32_t)n_seeds;
  }
}

__global__ void a5_empty_kernel(int32_t* counts) {
  counts[0] = counts[1] = counts[2] = counts[3] = 0;
}

}  // namespace

cudaError_t launch_a5_select(const tpc_tracker* t, const tpc_tracks_out_t* out, cudaStream_t st) {
  if (t->s_cap == 0 || t->last_n == 0) {
    a5_empty_kernel<<<1, 1, 0, st>>>(out->counts);
    return cudaGetLastError();
  }
  const unsigned blocks = (unsigned)((t->s_cap + A5_TILE - 1) / A5_TILE);
  a5_select_kernel<<<blocks, A5_TILE, 0, st>>>(t->g, t->s_cap, t->s.ctl, t->s.seed_start, t->s.tl_par, t->s.tl_cov,
                                              t->s.tl_chi2, t->s.tl_nhits, t->s.tl_sr0, t->s.tl_hits, t->s.owner,
                                              t->s.scan_a5, out->tracks, out->track_capacity, out->hit_ids,
                                              out->hit_capacity, out->counts);
  return cudaGetLastError();
}
