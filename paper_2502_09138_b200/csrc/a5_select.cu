// a5_select.cu -- stage a5: hit-ownership selection and output compaction (SURVEY 8(c) "Stage 5", P24-P29;
// north_star "hit-ownership resolution with atomicMax on packed (quality, track-id) words").
//
// The votes (atomicMax of (n_hits << 24 | 0xFFFFFF - rank) per tracklet hit) were cast at the end of a4.
// Here: the hits each tracklet owns are counted, a tracklet is kept iff owned >= n_min_owned (P27), and a
// single-pass look-back scan over (kept, owned) gives each kept tracklet its output slot and hit offset in
// ascending seed order (P29).  Track parameters are the a4 fit over all tracklet hits (P28).
#include "tpc_internal.cuh"

namespace {

constexpr int A5_MASK_WORDS = 8;   // n_rows <= 255 (checked at create) -> at most 8 ballot words per tracklet
constexpr int A5_UNROLL = 8;       // tracklets whose loads one warp keeps in flight

// Block = max(A5_TILE, 32 * ceil(n_rows / 32)) threads, tile = A5_TILE tracklets.
// Pass 1: warp w owns rows 32w .. 32w+31 and walks the tile's tracklets, A5_UNROLL at a time: one coalesced load of
// the [seed][row] hit table and one owner gather per lane, ballot -> the tracklet's owned-hit mask word w in shared
// memory.  Then thread k of the block holds the count of tracklet k, the block scan + look-back scan place it, and
// pass 2 writes the hit lists, one warp per tracklet.
// Two resident CTAs asked for: the compiler then keeps all A5_UNROLL x 2 loads of pass 1 in flight (78 registers);
// with its default register target (48) it serialised them, 0.295 against 0.264 ms.
__global__ void __launch_bounds__(256, 2)
a5_select_kernel(const DevGeom g, DevCtl* __restrict__ ctl, const int32_t* __restrict__ seed_start,
                 const float4* __restrict__ tl_rec, const int32_t* __restrict__ tl_hits,
                 const uint32_t* __restrict__ tl_span, const uint32_t* __restrict__ owner, uint64_t* __restrict__ status,
                 uint8_t* __restrict__ hit_row, tpc_track_rec_t* __restrict__ tracks, int32_t track_capacity,
                 int32_t* __restrict__ hit_ids,
                 int32_t hit_capacity, int32_t* __restrict__ counts) {
  __shared__ uint32_t wsum[33];
  __shared__ uint32_t sh_tile;
  __shared__ uint64_t sh_excl;
  __shared__ uint32_t own_mask[A5_TILE][A5_MASK_WORDS];
  __shared__ uint32_t s_word[A5_TILE];   // packed vote word of a surviving tracklet, 0 = discarded (P24)
  __shared__ uint32_t s_span[A5_TILE];   // first | last << 8 row the tracklet visited: only those table entries exist
  __shared__ uint32_t sh_off[A5_TILE];   // output hit offset of a kept tracklet, 0xFFFFFFFF = no hit list to write
  const unsigned FULL = 0xffffffffu;
  const uint32_t n_seeds = ctl->n_seeds;
  const uint32_t n_tiles = (n_seeds + A5_TILE - 1) / A5_TILE;
  const uint32_t seed_flags = (ctl->n_seeds_found > n_seeds ? TPC_FLAG_SEED_OVERFLOW : 0u) |
                              (ctl->bad_offsets ? TPC_FLAG_BAD_OFFSETS : 0u);
  if (n_seeds == 0) {
    if (blockIdx.x == 0 && threadIdx.x == 0) {
      counts[0] = 0;
      counts[1] = 0;
      counts[2] = (int32_t)seed_flags;
      counts[3] = 0;
    }
    return;
  }
  if (blockIdx.x >= n_tiles) return;   // the grid is sized by the seed capacity
  if (threadIdx.x == 0) sh_tile = atomicAdd(&ctl->ticket_a5, 1u);
  __syncthreads();
  const uint32_t tile = sh_tile;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
  const int nr = g.n_rows;
  const int n_words = (nr + 31) >> 5;
  const int64_t t0 = (int64_t)tile * A5_TILE;
  const int n_here = (int)min((int64_t)A5_TILE, (int64_t)n_seeds - t0);
  const int64_t i = t0 + threadIdx.x;   // this thread's tracklet in the scans and the record

  if (threadIdx.x < A5_TILE) {
    uint32_t w = 0, sp = 1u;   // span 1 .. 0: empty
    if (threadIdx.x < n_here) {
      const int nh = __float_as_int(tl_rec[i * TL_REC_V4 + 1].w);
      if (nh >= g.n_min_tracklet) {   // a discarded tracklet owns nothing: none of its table is read
        w = ((uint32_t)nh << 24) | (0xFFFFFFu - (uint32_t)i);
        sp = tl_span[i];
      }
    }
    s_word[threadIdx.x] = w;
    s_span[threadIdx.x] = sp;
  }
  __syncthreads();

  // pass 1
  if (wid < n_words) {
    const int r = wid * 32 + lane;
    const bool in_row = r < nr;
    const int32_t* col = tl_hits + t0 * nr + r;
    // the table entries of the next batch are requested while the owner words of this one are in flight
    auto load_batch = [&](int tb, int* h) {
#pragma unroll
      for (int u = 0; u < A5_UNROLL; ++u) {   // rows outside the tracklet's span hold nothing
        const uint32_t sp = s_span[min(tb + u, A5_TILE - 1)];
        const bool in_span = in_row && tb + u < n_here && r >= (int)(sp & 0xffu) && r <= (int)((sp >> 8) & 0xffu);
        h[u] = in_span ? col[(int64_t)(tb + u) * nr] : -1;
      }
    };
    int hn[A5_UNROLL];
    load_batch(0, hn);
    for (int tb = 0; tb < n_here; tb += A5_UNROLL) {
      int h[A5_UNROLL];
      uint32_t ow[A5_UNROLL];
#pragma unroll
      for (int u = 0; u < A5_UNROLL; ++u) h[u] = hn[u];
#pragma unroll
      for (int u = 0; u < A5_UNROLL; ++u) ow[u] = h[u] >= 0 ? owner[h[u]] : 0u;
      load_batch(tb + A5_UNROLL, hn);   // beyond the tile: all -1, no loads
#pragma unroll
      for (int u = 0; u < A5_UNROLL; ++u) {
        if (tb + u < n_here) {   // warp-uniform
          const uint32_t w = s_word[tb + u];
          const unsigned m = __ballot_sync(FULL, w != 0u && ow[u] == w);
          if (lane == 0) own_mask[tb + u][wid] = m;
        }
      }
    }
  }
  __syncthreads();
  uint32_t owned = 0;
  int first = -1, last = -1;
  if (threadIdx.x < n_here) {
    for (int k = 0; k < n_words; ++k) {
      const unsigned m = own_mask[threadIdx.x][k];
      if (m) {
        if (first < 0) first = k * 32 + __ffs(m) - 1;
        last = k * 32 + 31 - __clz(m);
        owned += __popc(m);
      }
    }
  }
  const bool keep = owned >= (uint32_t)g.n_min_owned && owned > 0;   // P27
  if (!keep) owned = 0;
  uint32_t tot_k, tot_h;
  const uint32_t pos_k = block_excl_scan(keep ? 1u : 0u, wsum, &tot_k);
  const uint32_t pos_h = block_excl_scan(owned, wsum, &tot_h);
  // payload: tracks in bits 61..38 (s_cap < 2^24), hits in bits 37..0 (n < 2^31)
  const uint64_t ex = lookback_scan(status, tile, ((uint64_t)tot_k << 38) | tot_h, &sh_excl);
  const uint32_t excl[2] = {(uint32_t)(ex >> 38), (uint32_t)(ex & ((1ull << 38) - 1))};

  uint32_t my_off = 0xFFFFFFFFu;
  if (keep) {
    const uint32_t slot = excl[0] + pos_k;
    const uint32_t off = excl[1] + pos_h;
    if (slot < (uint32_t)track_capacity) {
      const float4* q = tl_rec + i * TL_REC_V4;
      const float4 q0 = q[0], q1 = q[1], q2 = q[2], q3 = q[3], q4 = q[4], q5 = q[5];
      tpc_track_rec_t rec;
      rec.x = q0.x; rec.y = q0.y; rec.z = q0.z; rec.sinphi = q0.w;
      rec.tanl = q1.x; rec.qpt = q1.y;
      rec.cov[0] = q2.x; rec.cov[1] = q2.y; rec.cov[2] = q2.z; rec.cov[3] = q2.w;
      rec.cov[4] = q3.x; rec.cov[5] = q3.y; rec.cov[6] = q3.z; rec.cov[7] = q3.w;
      rec.cov[8] = q4.x; rec.cov[9] = q4.y; rec.cov[10] = q4.z; rec.cov[11] = q4.w;
      rec.cov[12] = q5.x; rec.cov[13] = q5.y; rec.cov[14] = q5.z;
      rec.chi2 = q1.z;
      rec.sector = __float_as_int(q5.w) / nr;
      rec.first_row = first;
      rec.last_row = last;
      rec.n_hits = (int32_t)owned;
      rec.hit_offset = (int32_t)off;
      rec.seed_cluster = seed_start[i];
      tracks[slot] = rec;
    }
    if ((uint64_t)off + owned <= (uint64_t)hit_capacity) my_off = off;
  }
  if (threadIdx.x < A5_TILE) sh_off[threadIdx.x] = my_off;
  __syncthreads();

  // pass 2: hit lists, ascending row, one warp per tracklet
  for (int t = wid; t < n_here; t += n_warps) {
    uint32_t w = sh_off[t];
    if (w == 0xFFFFFFFFu) continue;
    const int32_t* src = tl_hits + (t0 + t) * nr;
    int v[A5_MASK_WORDS];   // all loads of the tracklet first, then the stores
    unsigned mk[A5_MASK_WORDS];
#pragma unroll
    for (int k = 0; k < A5_MASK_WORDS; ++k) {
      mk[k] = k < n_words ? own_mask[t][k] : 0u;
      v[k] = ((mk[k] >> lane) & 1u) ? src[k * 32 + lane] : -1;
    }
#pragma unroll
    for (int k = 0; k < A5_MASK_WORDS; ++k) {
      if ((mk[k] >> lane) & 1u) {
        const uint32_t at = w + __popc(mk[k] & ((1u << lane) - 1u));
        hit_ids[at] = v[k];
        hit_row[at] = (uint8_t)(k * 32 + lane);   // for a6 (tpc_refit): the row of every output hit
      }
      w += __popc(mk[k]);
    }
  }
  if (tile == n_tiles - 1 && threadIdx.x == 0) {
    const uint32_t nt = excl[0] + tot_k, nhits = excl[1] + tot_h;
    counts[0] = (int32_t)nt;
    counts[1] = (int32_t)nhits;
    counts[2] = (int32_t)((nt > (uint32_t)track_capacity ? TPC_FLAG_TRACK_OVERFLOW : 0u) |
                          (nhits > (uint32_t)hit_capacity ? TPC_FLAG_HIT_OVERFLOW : 0u) | seed_flags);
    counts[3] = (int32_t)ctl->n_seeds_found;
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
  const int row_threads = 32 * ((t->g.n_rows + 31) / 32);
  a5_select_kernel<<<blocks, row_threads > A5_TILE ? row_threads : A5_TILE, 0, st>>>(t->g, t->s.ctl, t->s.seed_start, t->s.tl_rec, t->s.tl_hits, t->s.tl_span, t->s.owner,
                                              t->s.scan_a5, t->s.hit_row, out->tracks, out->track_capacity, out->hit_ids,
                                              out->hit_capacity, out->counts);
  return cudaGetLastError();
}
