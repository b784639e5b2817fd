// tpc_internal.cuh -- shared declarations of the CUDA path (handle, device-side geometry, launchers).
// Product code: shares nothing with oracle/.  Stage definitions: SURVEY.md 8(c) / DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <limits.h>

#include "../../include/tpc_track.h"

// Device view of geometry + parameters, passed by value to every kernel.
struct DevGeom {
  int32_t n_sectors, n_rows;
  // a1 grid shape: bin = iz * ny + iy, iy = (y - org_y) >> shift_y clamped to [0, ny-1],
  // iz = (z - org_z[sector]) >> shift_z clamped to [0, nz-1].  org_y comes from the geometry (minus the widest row's
  // half width), org_z is the smallest z of the sector's clusters (a0), so drift offsets cost no bins.
  int32_t shift_y, shift_z, ny, nz, nb_stride, org_y;
  const double* row_x;     // [n_rows] cm
  const float* row_dx;     // [n_rows] row_x[r+1] - row_x[r], rounded once from double (last entry repeats)
  const int32_t* gap_w;    // [n_rows - 1] P48 pitch weights nearbyint(64 * pitch / cm), or NULL when all are equal
  // a2 / a3
  int32_t w_y, w_z, cost_wy, cost_wz, c_max, l_min;
  // a4 / a5
  int32_t max_miss, n_min_tracklet, n_min_owned;
  float sy2, sz2, sinphi_max, gate_d, gate_y, gate_z, inv_units, units, cq;
  float c_reset[5];
  double inv_units_d;
};

// Counters living in device memory, zeroed at the start of every call.
constexpr int A4_Q_BUCKETS = 8;   // a4 phase queues are split by expected tracklet length, longest served first
struct CtlLine {         // one hot counter per 128-byte line
  uint32_t v;
  uint32_t pad[31];
};
struct DevCtl {
  uint32_t n_seeds;      // written by a3: seeds kept = min(seeds found, seed capacity)
  uint32_t ticket_a3;    // dynamic tile ids for the a3 look-back scan
  uint32_t ticket_a5;
  uint32_t next_seed;    // a4 work queue: next seed rank to hand to a free lane
  uint32_t next_track;   // a6 work queue
  uint32_t n_seeds_found; // a3: seeds the call holds (> n_seeds iff the seed capacity was too small)
  uint32_t bad_offsets;  // a0: row_offsets are not a CSR over n clusters -> every later stage does nothing
  uint32_t pad[25];
  CtlLine q_alloc[3 * A4_Q_BUCKETS];   // a4 phase queues B, C, D x length bucket: items pushed by earlier phases ...
  CtlLine q_head[3 * A4_Q_BUCKETS];    // ... and items claimed by the consuming phase
};

struct Scratch {
  // a1
  int4* srt;                // clusters in bin order inside each row: (y, z, cluster id, 0) -- one 16-B load per search
                            // candidate and per followed chain hit
  uint32_t* sec_key;        // [n_sectors] a0: order-preserving key of the sector's smallest z (zeroed per call)
  uint32_t* bin_start;      // [R * nb_stride] global sorted index of the first cluster of each bin (+ sentinel)
  // a2 / a3: raw links in SORTED space (position of the linked cluster in srt, -1 = none), written coalesced
  int32_t *link_up, *link_dn;
  int32_t* clean_up;        // [n, sorted space] a3: the cleaned up link (P11: the raw one where it is mutual, else -1)
  uint32_t* owner;          // [n, id space] packed (n_hits << 24 | 0xFFFFFF - rank), 0 = none (zeroed per call)
  uint8_t* hit_row;         // [n] a5: row of the hit at each position of the output hit list (for a6)
  uint32_t* q_items;        // [3 * A4_Q_BUCKETS][s_cap] a4 phase queues: seed ranks
  int4* tl_state;           // [s_cap][A4_STATE_V4] a4 filter state of a tracklet between two phases
  uint32_t* tl_span;        // [s_cap] first | last << 8 row a tracklet visited (rows outside hold no hit)
  // a3 -> a4
  int4* seed_tmp;           // [s_cap] a3: seeds in sorted-position order (position, start id, sector*n_rows+row, 0)
  int32_t* seed_start;      // [s_cap] start cluster id, ascending (P14)
  int32_t* seed_pos;        // [s_cap] sorted position of the start cluster
  int32_t* seed_sr;         // [s_cap] sector * n_rows + row of the start cluster
  int4* seed_rec;           // [s_cap][2] (sr, y0, z0, id0) (up0, y1, z1, -): a tracklet's start in one 32-byte load
  // a4 tracklets, one 96-B record + one row table per seed
  float4* tl_rec;           // [s_cap][6]: (x_ref,y,z,sinphi) (tanl,qpt,chi2,n_hits as int bits) cov[0..3] cov[4..7]
                            //             cov[8..11] (cov[12],cov[13],cov[14],sector*n_rows+first seed row as int bits)
  int32_t* tl_hits;         // [s_cap][n_rows] cluster id or -1
  int2* tl_yz;              // [s_cap][n_rows] (y, z) of the hit the upward pass recorded in that row (y = INT32_MIN:
                            // none): the downward refit streams these instead of gathering clusters by id
  // control
  DevCtl* ctl;
  uint32_t* seed_mask;      // [n/32 + 1] a3: bit id set iff cluster id starts a kept seed (zeroed per call)
  uint64_t* scan_a3;        // look-back status words
  uint64_t* scan_a5;        // two channels per tile
  // host-buffer path staging
  int32_t *st_y, *st_z; uint32_t* st_ro;
  tpc_track_rec_t* st_tracks; int32_t* st_hits; int32_t* st_counts;
};

constexpr int32_t YZ_NONE = INT32_MIN;   // tl_yz[..].x of a row without a hit

constexpr int TIMING_SETS = 64;   // ring of per-call stage-event sets (tpc_get_stage_ms_mean averages over them)

struct tpc_tracker {
  int device;
  DevGeom g;                 // device pointers inside point at geom_blob
  void* geom_blob;
  tpc_params_t params;
  double bz;
  // scratch arena
  void* arena; size_t arena_bytes;
  void* host_arena; size_t host_arena_bytes;   // staging for tpc_track_host
  int64_t cap_n, cap_rows;   // sizes the arena was laid out for
  int base_shift_y, base_shift_z;   // coarsest grid (bins >= 2 x the widest window); dense calls refine it
  int64_t y_units, z_units;         // grid extents in fixed-point units
  int64_t s_cap;             // seed capacity of the current layout (api.cu: seed_capacity)
  int64_t seed_reserve;      // tpc_reserve_seeds: lower bound on s_cap
  int64_t tiles_a3, tiles_a5;
  int a4_phased;             // the most recent call ran a4 as phase kernels (api.cu)
  int concurrency;           // tpc_set_concurrency: calls the caller keeps in flight on the device (0 / 1: this one alone)
  int a2_variant;            // tpc_debug_set_a2_variant: 0 = direct kernels, 1 = shared-memory staged rows (sparse calls)
  int a4_variant;            // tpc_debug_set_a4_variant: 0 = by call size, 1 = uniform kernel, 2 = phase kernels
  int a4_sms;              // SMs of the device (phase kernels size their own persistent grids)
  int a4_blocks, a4_warps;   // persistent a4 grid: blocks x warps per block = resident warps of the device (set at create)
  size_t ctl_bytes;          // bytes zeroed per call
  Scratch s;
  // a7 (tpc_merge) scratch, grown on demand: per-sector track ranges, best partner and its chi2 for both directions
  int32_t* merge_sec; int32_t* merge_best; double* merge_chi2; int64_t merge_cap;
  // a9 (tpc_clusterize) scratch, grown on demand: sorted keys of rows too long for shared memory, peak flags and
  // parked clusters per digit, clusters per row
  uint32_t* cl_keys; uint8_t* cl_flag; int4* cl_parked; uint32_t* cl_row_count; int64_t cl_cap;
  // a10 (tpc_rans_encode) scratch, grown on demand: chunk slots, histogram, cumulative table, per-chunk counts
  void* rans_scratch; size_t rans_scratch_cap;
  int64_t last_n; const uint32_t* last_ro; const int32_t* last_y; const int32_t* last_z;
  // stage timing
  int timing; int64_t timed_calls; cudaEvent_t ev[TIMING_SETS * 6];
  cudaError_t last_err; char err_buf[256];
};

constexpr int64_t A4_PHASED_MIN_CLUSTERS = 5000000;   // calls at least this large run a4 as phase kernels
constexpr int GRID_MAX_BINS = 48 * 1024;   // bins per row: one row's histogram fits a CTA's shared memory
constexpr int GRID_MIN_SHIFT = 9;          // finest bins: 512 units = 0.8 cm
constexpr int A3_TILE = 1024;   // ids per a3 block (256 threads x 4)
constexpr int A5_TILE = 128;    // tracklets per a5 block
// a0 keeps the smallest z of a sector as max over key(z) = ~(z ^ 0x80000000): zero-initialised memory then means
// "no cluster yet" and atomicMax does the reduction.
__host__ __device__ __forceinline__ uint32_t zmin_key(int32_t z) { return ~((uint32_t)z ^ 0x80000000u); }
__host__ __device__ __forceinline__ int32_t zmin_from_key(uint32_t k) { return k ? (int32_t)(~k ^ 0x80000000u) : 0; }

constexpr int A4_STATE_V4 = 8;  // 16-byte words of a parked a4 state: 15 U D U^T factors, 5 state, bookkeeping, origin
constexpr int TL_REC_V4 = 6;    // float4 words per tracklet record

// launchers (each in its own .cu)
cudaError_t launch_a0_check(const tpc_tracker* t, const uint32_t* ro, int64_t n, cudaStream_t st);
cudaError_t launch_a0_origin(const tpc_tracker* t, const int32_t* z, const uint32_t* ro, int64_t n, cudaStream_t st);
cudaError_t launch_a1_grid(const tpc_tracker* t, const int32_t* y, const int32_t* z, const uint32_t* ro, int64_t n, cudaStream_t st);
cudaError_t launch_a2_neighbours(const tpc_tracker* t, const uint32_t* ro, int64_t n, cudaStream_t st);
cudaError_t launch_a3_seeds(const tpc_tracker* t, const uint32_t* ro, int64_t n, cudaStream_t st);
cudaError_t launch_a4_follow(const tpc_tracker* t, int64_t n, cudaStream_t st);
cudaError_t setup_a4_attributes(tpc_tracker* t);
cudaError_t launch_a4_phases(const tpc_tracker* t, int64_t n, cudaStream_t st);
cudaError_t launch_a5_select(const tpc_tracker* t, const tpc_tracks_out_t* out, cudaStream_t st);
cudaError_t launch_a6_refit(const tpc_tracker* t, const int32_t* y, const int32_t* z, const tpc_tracks_out_t* tracks,
                            tpc_track_rec_t* refit_out, cudaStream_t st);
cudaError_t launch_a6_refit_merged(const tpc_tracker* t, const tpc_merge_params_t* mp, const int32_t* y,
                                   const int32_t* z, const tpc_tracks_out_t* tracks, const int32_t* succ,
                                   const int32_t* pred, tpc_track_rec_t* refit_out, cudaStream_t st);
cudaError_t launch_a8_compress(const tpc_tracker* t, const int32_t* y, const int32_t* z, const tpc_tracks_out_t* tracks,
                               const tpc_compressed_t* c, cudaStream_t st);
cudaError_t launch_a8_decompress(const tpc_tracker* t, const tpc_tracks_out_t* tracks, const tpc_compressed_t* c,
                                 int32_t* row, int32_t* y, int32_t* z, cudaStream_t st);
cudaError_t setup_a9_attributes();
cudaError_t setup_a2_attributes();
size_t rans_scratch_bytes(int64_t n, int32_t chunk, int32_t bits);
cudaError_t launch_a10_rans_encode(const tpc_tracker* t, const void* values, int32_t value_bytes, int64_t n,
                                   int32_t bits, int32_t chunk, const tpc_rans_stream_t* out, cudaStream_t st);
cudaError_t launch_a10_rans_decode(const tpc_tracker* t, const tpc_rans_stream_t* in, int64_t n, int32_t bits,
                                   int32_t chunk, void* values, int32_t value_bytes, cudaStream_t st);
cudaError_t launch_a9_clusterize(const tpc_tracker* t, const tpc_cluster_params_t* cp, const tpc_digits_t* d,
                                 int64_t n_digits, const tpc_clusters_out_t* out, cudaStream_t st);
cudaError_t launch_a7_merge(const tpc_tracker* t, const tpc_merge_params_t* mp, const tpc_track_rec_t* tracks,
                            const int32_t* counts, int32_t cap, int32_t* succ, int32_t* pred, float* link_chi2,
                            int32_t* merge_counts, cudaStream_t st);
cudaError_t setup_a1_attributes(const tpc_tracker* t);
size_t a1_smem_bytes(const DevGeom& g);

// debug.cu
cudaError_t launch_dbg_links(const tpc_tracker* t, int64_t n, int which, int32_t* up, int32_t* dn, cudaStream_t st);
cudaError_t launch_dbg_seed_len(const tpc_tracker* t, int32_t* start, int32_t* len, cudaStream_t st);
cudaError_t launch_dbg_tracklets(const tpc_tracker* t, float* par, float* cov, float* chi2, int32_t* n_hits, int32_t* hits, cudaStream_t st);
cudaError_t launch_dbg_owner(const tpc_tracker* t, int64_t n, int32_t* owner, cudaStream_t st);

// ------------------------------------------------------------------------------------------------
// Single-pass device-wide exclusive scan (decoupled look-back).  One 64-bit status word per tile:
// bits 63..62 = state (0 not ready, 1 tile aggregate, 2 inclusive prefix), bits 61..0 = payload, so state and
// value always change together.  The payload may pack several counters in disjoint bit fields as long as no
// field can overflow into the next (a5 packs tracks and hits).  Tiles take their index from an atomic ticket,
// so every predecessor of a tile is already running.
// Called by all threads of the block; `tile_sum` must be valid in thread 0.  Returns the exclusive prefix
// (sum over tiles < tile) to every thread through shared memory.
// ------------------------------------------------------------------------------------------------
constexpr uint64_t LB_PAYLOAD = (1ull << 62) - 1;

__device__ __forceinline__ uint64_t lookback_scan(volatile uint64_t* status, uint32_t tile, uint64_t tile_sum,
                                                  uint64_t* sh /* one word of shared memory */) {
  if (threadIdx.x < 32) {
    const unsigned lane = threadIdx.x;
    const uint64_t sum = __shfl_sync(0xffffffffu, tile_sum, 0);
    if (tile == 0) {
      if (lane == 0) {
        status[0] = (2ull << 62) | sum;
        *sh = 0;
      }
    } else {
      if (lane == 0) status[tile] = (1ull << 62) | sum;
      uint64_t run = 0;
      int64_t base = (int64_t)tile - 1;   // lane l looks at tile base - l
      while (true) {
        const int64_t idx = base - lane;
        uint64_t w;
        do {
          w = idx >= 0 ? status[idx] : (2ull << 62);
        } while (!__all_sync(0xffffffffu, (w >> 62) != 0));
        // nearest predecessor that already holds an inclusive prefix ends the walk
        const unsigned mask = __ballot_sync(0xffffffffu, (w >> 62) == 2);
        const int stop = mask ? __ffs(mask) - 1 : 31;
        uint64_t v = lane <= (unsigned)stop ? (w & LB_PAYLOAD) : 0ull;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        run += v;
        if (mask) break;
        base -= 32;
      }
      if (lane == 0) {
        status[tile] = (2ull << 62) | (run + sum);
        *sh = run;
      }
    }
  }
  __syncthreads();
  return *sh;
}

// Block-wide exclusive scan of one uint32 per thread (blockDim.x multiple of 32, <= 1024).
// Returns the exclusive prefix; *total (same in all threads) is the block sum.  `wsum` = 33 words of smem.
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* wsum, uint32_t* total) {
  const unsigned lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= (unsigned)o) inc += t;
  }
  __syncthreads();   // protect wsum reuse
  if (lane == 31) wsum[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    uint32_t s = lane < nw ? wsum[lane] : 0u;
    uint32_t si = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t t = __shfl_up_sync(0xffffffffu, si, o);
      if (lane >= (unsigned)o) si += t;
    }
    wsum[lane] = si - s;            // exclusive warp offsets
    if (lane == 31) wsum[32] = si;  // block total
  }
  __syncthreads();
  *total = wsum[32];
  return wsum[wid] + inc - v;
}
