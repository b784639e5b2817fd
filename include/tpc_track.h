/* tpc_track.h -- C ABI of libtpctrack.so: TPC sector track finding on one B200 (sm_100a).
 *
 * What it computes: the "TPC tracking" part of the line "TPC Processing (Tracking, Clustering, Compression)
 * 99.37 %" of the paper's Table 1 ("fully dominated by the TPC tracking which can run on GPUs",
 * PAPER.md:40), in the five stages BASELINE.json's north_star names:
 *   a1 per-pad-row (y,z) grid binning, a2 neighbour finding (best up/down pair in the adjacent rows),
 *   a3 cellular-automaton link cleaner + chain/seed extraction, a4 Kalman-filter tracklet following (helix,
 *   constant Bz), a5 hit-ownership selection + output compaction.
 * The paper gives no algorithm; every stage is defined in SURVEY.md section 8(c) (readings P1..P40, restated in
 * DESIGN.md).  The three entry points are the ones north_star lists; the handle argument of tpc_track and the
 * host-buffer / debug entry points are additions.
 *
 * Conventions
 *  - Every function returns an int status: TPC_OK (0) or a negative TPC_ERR_* code.  Nothing throws or aborts.
 *  - Pointers are tagged [host] or [device] below.  The caller owns every buffer it passes; the handle owns
 *    all scratch memory (grown on demand, released by tpc_tracker_destroy).
 *  - tpc_track is asynchronous on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream);
 *    results are valid after the caller synchronises that stream.  One handle serves one stream at a time.
 *  - Cluster ids are indices into the input arrays.  Clusters of one (sector,row) are contiguous:
 *    row_offsets[s*n_rows + r] .. row_offsets[s*n_rows + r + 1]; the order inside a row is arbitrary.
 *  - Coordinates are int32 fixed point, units_per_cm units per cm (640 = 1/64 mm, BASELINE.json configs[0]).
 *    Sector-local frame: x along the sector's central radius (pad row r is the plane x = row_x[r]),
 *    y across the sector, z along the beam.  Track state at x: (y, z, sin phi, tan lambda, q/pT [1/GeV]).
 */
#ifndef TPC_TRACK_H
#define TPC_TRACK_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TPC_OK 0
#define TPC_ERR_ARG (-1)       /* NULL pointer, negative size, parameter out of range */
#define TPC_ERR_GEOMETRY (-2)  /* n_rows < 3, rows not ascending, pitch outside 1/64 .. 512 cm, non-positive extents */
#define TPC_ERR_CUDA (-3)      /* a CUDA runtime call failed (tpc_last_cuda_error() tells which) */
#define TPC_ERR_NOMEM (-4)     /* scratch allocation failed */
#define TPC_ERR_CAPACITY (-5)  /* n too large for the packed ownership word (n/l_min >= 2^24) */
#define TPC_ERR_STATIC_SCRATCH (-6) /* tpc_rans_encode_static: the input needs more than its fixed scratch array */

/* device-side flags OR-ed into counts[2] */
#define TPC_FLAG_TRACK_OVERFLOW 1u /* more output tracks than track_capacity: tracks beyond it not written */
#define TPC_FLAG_HIT_OVERFLOW 2u   /* more output hits than hit_capacity: those tracks' hit lists not written */
#define TPC_FLAG_SEED_OVERFLOW 4u  /* more seeds than the handle's seed capacity (n/16 + 4096 unless reserved): the
                                      seeds beyond it (in bin order of their start cluster) were not followed, so
                                      tracks are missing; counts[3] holds the number of seeds the call needs --
                                      pass it to tpc_reserve_seeds and repeat the call */
#define TPC_FLAG_BAD_OFFSETS 8u    /* row_offsets not ascending or row_offsets[last] != n: nothing was tracked */

/* Free constants of the method.  tpc_default_params fills the defaults. */
typedef struct {
  int32_t w_y, w_z;          /* a2 window half-widths, fixed-point units, inclusive (P7): 1280, 1600 */
  int32_t cost_wy, cost_wz;  /* a2 cost = cost_wy*(y_u+y_d-2y_h)^2 + cost_wz*(z_u+z_d-2z_h)^2 (P8): 9, 4 */
  int32_t c_max;             /* a2 accept iff cost <= c_max (P10): 3538944 */
  int32_t l_min;             /* a3 seed iff chain length >= l_min clusters (P13): 5 */
  int32_t max_miss;          /* a4 stop after this many consecutive rows without a hit (P20): 5; >= 1 */
  int32_t n_min_tracklet;    /* a4/a5 tracklets with fewer hits are discarded (P24): 10 */
  int32_t n_min_owned;       /* a5 output iff owned hits >= this (P27): 10 */
  int32_t reserved;          /* must be 0 */
  double sigma_y, sigma_z;   /* a4 hit errors in cm (P15): 0.1, 0.15 */
  double sinphi_max;         /* a4 transport fails iff |sin phi| >= this before or after a step (P18): 0.95 */
  double gate_d;             /* a4 accept a searched hit iff d < gate_d (P21): 15 */
  double gate_y_cm, gate_z_cm; /* a4 search restricted to |dy| <= 2.0, |dz| <= 2.5 cm (P21) */
  double c_reset[5];         /* a4 covariance reset, variances (P22): 0.25, 0.25, 0.05, 0.05, 25 */
  double cq_per_tesla;       /* a4 curvature k = cq_per_tesla * Bz * q/pT, 1/cm (P4): -0.00299792458 */
} tpc_params_t;

typedef struct {
  int32_t n_sectors;       /* independent sectors in one call (36; 1 for configs[0]; B*36 for a batch of B events) */
  int32_t n_rows;          /* pad rows per sector (152), >= 3 */
  const double* row_x;     /* [host] n_rows local x of the pad rows in cm, ascending; pitches may differ (P48) */
  double units_per_cm;     /* fixed-point scale (640) */
  double y_half_tan;       /* |y| <= row_x[r]*y_half_tan (tan 10 deg); used for grid sizing only */
  double y_half_cm;        /* if > 0: |y| extent in cm for every row instead (open sector, configs[0]); grid sizing only */
  double z_extent_cm;      /* z-length covered by one sector's clusters incl. drift offsets; grid sizing only */
  const tpc_params_t* params; /* [host] NULL = defaults */
} tpc_geometry_t;
/* "grid sizing only": clusters outside these extents are still handled exactly (edge bins absorb them). */

typedef struct {
  double bz_tesla; /* constant field along z (0.5) */
} tpc_field_t;

typedef struct {
  const int32_t* y;            /* [device] n fixed-point y */
  const int32_t* z;            /* [device] n fixed-point z */
  const uint32_t* row_offsets; /* [device] n_sectors*n_rows + 1 CSR offsets; row_offsets[last] == n */
} tpc_clusters_t;

/* One output track (112 bytes).  Parameters are the a4 fit over all the tracklet's hits at x (P23, P28). */
typedef struct {
  float x, y, z, sinphi, tanl, qpt;
  float cov[15];       /* packed lower triangle 00,10,11,20,21,22,30,... in (y,z,sinphi,tanl,qpt) order */
  float chi2;          /* accumulated over the downward pass (P22) */
  int32_t sector;
  int32_t first_row, last_row; /* of the owned hits */
  int32_t n_hits;      /* owned hits = length of this track's hit list */
  int32_t hit_offset;  /* start of the hit list in hit_ids */
  int32_t seed_cluster; /* start cluster id of the seed; tracks ascend by it (P29) */
} tpc_track_rec_t;

typedef struct {
  tpc_track_rec_t* tracks; /* [device] track_capacity records */
  int32_t track_capacity;
  int32_t hit_capacity;
  int32_t* hit_ids;        /* [device] hit_capacity cluster ids; per track ascending row */
  int32_t* counts;         /* [device] 4 x int32: [0] tracks found, [1] hits found (both may exceed the
                              capacities: then the matching TPC_FLAG_* is set and the excess is not written),
                              [2] flags, [3] number of seeds the call holds (= tracklets followed, unless
                              TPC_FLAG_SEED_OVERFLOW is set) */
} tpc_tracks_out_t;

typedef struct tpc_tracker tpc_tracker_t;

void tpc_default_params(tpc_params_t* p);

/* Copies geometry, field and parameters into a new handle for the current CUDA device.  No cluster-sized
 * allocation happens here.  Errors: TPC_ERR_ARG, TPC_ERR_GEOMETRY, TPC_ERR_CUDA, TPC_ERR_NOMEM. */
int tpc_tracker_create(const tpc_geometry_t* geometry, const tpc_field_t* field, tpc_tracker_t** out);

/* Runs a1..a5 on n clusters, enqueued on `stream`; no host synchronisation unless scratch must grow.
 * clusters and out are [host] structs holding [device] pointers.  n may be 0.
 * The call only enqueues memsets and kernels whose launch parameters depend on (n, the handle) alone: once an earlier
 * call of at least this size has sized the scratch (and with stage timing off) it can be captured into a CUDA graph
 * (stream capture on `stream`) and replayed on new data in the same buffers.
 * Errors: TPC_ERR_ARG, TPC_ERR_CAPACITY, TPC_ERR_NOMEM, TPC_ERR_CUDA. */
int tpc_track(tpc_tracker_t* t, const tpc_clusters_t* clusters, int64_t n, void* stream, tpc_tracks_out_t* out);

/* Seed capacity of the handle.  Scratch per seed is ~2.2 KB (hit table, measurement stream, filter state), so the
 * default bound is n/16 + 4096 seeds per call instead of the worst case n/l_min; events with more seeds set
 * TPC_FLAG_SEED_OVERFLOW.  tpc_reserve_seeds raises the bound for all later calls (never lowers it).  The
 * synthetic configs of BASELINE.json need n/50 (central Pb-Pb) to n/20 (stress).  Errors: TPC_ERR_ARG. */
int tpc_reserve_seeds(tpc_tracker_t* t, int64_t n_seeds);

/* How many tpc_track calls the caller keeps in flight on the device at the same time (this handle's and those of other
 * handles on other streams).  1 (the default): the persistent grids of the tracklet follower fill the GPU, which is
 * fastest for a call that runs alone.  >= 2: they leave a quarter of the SMs' CTA slots to the other calls (three
 * instead of four resident CTAs per SM, four instead of seven in the refit phase); measured with three handles on three
 * streams: 3.4 % more clusters/s in aggregate, and 6 % fewer for a call that then runs alone after all.  The results do
 * not depend on it.  Errors: TPC_ERR_ARG (k < 1). */
int tpc_set_concurrency(tpc_tracker_t* t, int32_t k);

/* Same computation with HOST buffers: copies y, z, row_offsets to device staging owned by the handle, runs
 * tpc_track, copies counts, tracks and hit_ids back into the [host] buffers of `out_host`, and synchronises
 * `stream` before returning.  Pinned host memory makes the copies asynchronous but is not required.
 * On TPC_FLAG_SEED_OVERFLOW it reserves the seeds the call asked for and runs it once more before returning.
 * Hit ids are copied for min(counts[1], hit_capacity) entries (the lists of the tracks that fitted). */
int tpc_track_host(tpc_tracker_t* t, const tpc_clusters_t* clusters_host, int64_t n, void* stream,
                   tpc_tracks_out_t* out_host);

/* NEXT-1 (reading P41 in DESIGN.md): refit of the tracks the most recent tpc_track call on this handle
 * wrote, over their owned hits only (the parameters tpc_track reports are the fit over all hits of the tracklet,
 * P28).  `clusters` and `n` must be those of that call, `tracks` its output (all [device]); refit_out: [device]
 * track_capacity records, written for the first min(counts[0], track_capacity) tracks: x .. chi2 hold the refit at
 * the row where its downward pass ended, n_hits the hits used on the way down, the other fields are copied.
 * Asynchronous on `stream` (the same stream, or one ordered after the tpc_track call).  Not part of tpc_track.
 * Errors: TPC_ERR_ARG (also when `clusters` is not the input of the handle's last call), TPC_ERR_CUDA. */
int tpc_refit(tpc_tracker_t* t, const tpc_clusters_t* clusters, int64_t n, void* stream, const tpc_tracks_out_t* tracks,
              tpc_track_rec_t* refit_out);

/* NEXT-1 (readings P42..P46 in DESIGN.md): links between sector tracks that are pieces of one particle
 * -- across a sector edge, across the central membrane, or inside one sector.  a -> b is a candidate iff b's first row
 * lies 1..gap_max rows above a's last row and the sectors are equal, azimuthal neighbours on one z side, or face each
 * other across the membrane (sectors come in groups of 2*n_per_side = one event; side = (s / n_per_side) % 2).
 * a's record is rotated into b's frame, transported to b's x, and chi2 = D^T (C_a' + C_b)^-1 D over the five
 * parameters; succ(a) / pred(b) = candidate of smallest (chi2, index) with chi2 < chi2_max; a link stands iff
 * succ(a) == b and pred(b) == a. */
typedef struct {
  int32_t gap_max;      /* P43: 25 rows */
  int32_t n_per_side;   /* sectors per z side: 18 */
  double chi2_max;      /* P44: 50 */
  double sector_angle;  /* radians between the frames of neighbouring sectors: 20 degrees */
} tpc_merge_params_t;
void tpc_default_merge_params(tpc_merge_params_t* p);
/* tracks: [device] records as written by tpc_track or tpc_refit (ascending sector), counts: [device] the int32[4] of
 * that call (counts[0] tracks), track_capacity: records readable.  params: [host], NULL = defaults.
 * Outputs, all [device]: succ[track_capacity], pred[track_capacity] (track index or -1), link_chi2[track_capacity]
 * (chi2 of a's link, -1 without), merge_counts int32[4]: [0] links, [1] merged tracks (= tracks - links), [2] tracks.
 * Asynchronous on `stream`.  Errors: TPC_ERR_ARG, TPC_ERR_NOMEM, TPC_ERR_CUDA. */
int tpc_merge(tpc_tracker_t* t, const tpc_track_rec_t* tracks, const int32_t* counts, int32_t track_capacity,
              const tpc_merge_params_t* params, void* stream, int32_t* succ, int32_t* pred, float* link_chi2,
              int32_t* merge_counts);

/* P47: refit over the hits of every chain of linked tracks.  `clusters`, `n`, `tracks` as for tpc_refit
 * (the tpc_track output of the handle's last call, whose hit lists are used); succ / pred: [device] links from
 * tpc_merge.  For every chain head (pred < 0) the P41 schedule runs over the owned hits of the head, its successor,
 * ...; before a hit of another sector the state is rotated into that sector's frame (P42).  refit_out: [device]
 * track_capacity records: heads get x .. chi2 at the row where the downward pass ended, `sector` = the frame of that
 * state, n_hits = hits used on the way down; other tracks get n_hits = 0; the remaining fields are copied.
 * Asynchronous on `stream`.  Errors: TPC_ERR_ARG, TPC_ERR_CUDA. */
int tpc_refit_merged(tpc_tracker_t* t, const tpc_clusters_t* clusters, int64_t n, void* stream,
                     const tpc_tracks_out_t* tracks, const int32_t* succ, const int32_t* pred,
                     const tpc_merge_params_t* params, tpc_track_rec_t* refit_out);

/* NEXT-3 (readings P50..P52 in DESIGN.md): track-model cluster compression, the residual transform.
 * Every hit an output track owns is replaced by (row step, y residual, z residual) against an integer predictor
 * built from the track's previous hits: j = 0 absolute; j = 1 first difference; j >= 2 the least-squares line
 * through the last four hits when those and the hit sit in five consecutive rows, pred = floor((2 c1 + c2 - c4) / 2),
 * else the two-point line with the row gaps, pred = c1 + floor((c1 - c2) g2 / g1).  Integer, lossless.
 * All pointers [device]; drow, ry, rz: hit_capacity entries in hit-list order; hist_ry / hist_rz: 65536 uint32 bins of
 * the residuals of the hits with j >= 2 (bin = residual + 32768, edge bins collect the rest), hist_drow: 256 bins of
 * the row steps of the hits with j >= 1.  The histograms are what an entropy coder (the paper's rANS stage) needs. */
typedef struct {
  uint8_t* drow;
  int32_t* ry;
  int32_t* rz;
  uint32_t* hist_ry;
  uint32_t* hist_rz;
  uint32_t* hist_drow;
} tpc_compressed_t;
/* clusters / n / tracks: the input and output of the handle's most recent tpc_track call (as for tpc_refit).
 * Asynchronous on `stream`.  Errors: TPC_ERR_ARG, TPC_ERR_CUDA. */
int tpc_compress(tpc_tracker_t* t, const tpc_clusters_t* clusters, int64_t n, void* stream,
                 const tpc_tracks_out_t* tracks, const tpc_compressed_t* out);
/* The inverse: row, y, z ([device], hit_capacity int32 each, hit-list order) from the residual streams and the tracks'
 * hit_offset / n_hits.  Needs no cluster input. */
int tpc_decompress(tpc_tracker_t* t, void* stream, const tpc_tracks_out_t* tracks, const tpc_compressed_t* in,
                   int32_t* row, int32_t* y, int32_t* z);

/* NEXT-3, the entropy stage ("TPC rANS Encoding"; readings P57..P60 in DESIGN.md): static range-variant
 * asymmetric numeral system over independent chunks of a value stream.  State in [2^16, 2^32), 16-bit words,
 * probabilities in units of 1/65536.
 * P57: alphabet A = 2^alphabet_bits; a value v with -A/2 < v < A/2 is the symbol v + A/2, any other value is the
 *      escape symbol 0 and is kept as it is in the escape list (stream order).
 * P58: frequencies from the stream's own histogram n_s (N values, K symbols occur): f_s = 1 + floor(n_s (65536 - K) / N)
 *      for the symbols that occur, the remainder 65536 - sum f_s goes to the most frequent (smallest among equals).
 * P59: a chunk (`chunk` consecutive values, the last one shorter) is coded backwards from x = 2^16: if x >= f_s 2^16
 *      the low 16 bits of x are emitted and x >>= 16; x = floor(x / f_s) 2^16 + x mod f_s + c_s (c_s = sum of f below s).
 * P60: chunk c is payload[chunk_off[c] .. chunk_off[c+1]): the final x (uint32, little endian), then the emitted
 *      words, last emitted first (uint16, little endian); its escapes are escapes[esc_off[c] .. esc_off[c+1]).
 * All pointers [device] and caller-owned.  counts: int64[4] = payload bytes, escapes, chunks, flags (bit 0: the
 * payload did not fit payload_capacity, bit 1: the escapes did not fit; nothing is written out of bounds, the sizes
 * reported are the needed ones).  payload_capacity >= 4 * n_chunks + 2 * n and escape_capacity >= n always fit. */
typedef struct {
  uint32_t* freq;        /* 2^alphabet_bits normalised frequencies */
  uint32_t* chunk_off;   /* n_chunks + 1 byte offsets, n_chunks = ceil(n / chunk) */
  uint32_t* esc_off;     /* n_chunks + 1 */
  uint8_t* payload;      /* payload_capacity bytes, 2-byte aligned */
  int32_t* escapes;      /* escape_capacity values */
  int64_t* counts;       /* int64[4] */
  int64_t payload_capacity;
  int64_t escape_capacity;
} tpc_rans_stream_t;
/* values: [device] n values of value_bytes = 4 (int32) or 1 (uint8, e.g. the row steps); 1 <= alphabet_bits <= 12,
 * 1 <= chunk <= 65535 (512 is what bench.py uses).  Asynchronous on `stream` (the handle's scratch grows on demand,
 * which synchronises once).  Errors: TPC_ERR_ARG, TPC_ERR_NOMEM, TPC_ERR_CUDA. */
int tpc_rans_encode(tpc_tracker_t* t, const void* values, int32_t value_bytes, int64_t n, int32_t alphabet_bits,
                    int32_t chunk, void* stream, const tpc_rans_stream_t* out);
/* The inverse: n values from a stream written with the same alphabet_bits and chunk. */
int tpc_rans_decode(tpc_tracker_t* t, const tpc_rans_stream_t* in, int64_t n, int32_t alphabet_bits, int32_t chunk,
                    void* stream, void* values, int32_t value_bytes);

/* tpc_rans_encode for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): the same kernels, the same stream layout and bytes as tpc_rans_encode, but the scratch (chunk
 * slots, histogram, cumulative table, per-chunk counts) is a fixed array in device memory that belongs to the library
 * image, not to a handle -- TPC_RANS_STATIC_SCRATCH_BYTES on every GPU that loads the library, until the process
 * exits.  No handle; the call makes no cudaMalloc / cudaFree and calls no allocating library routine (the first call
 * on a device looks the array's address up once, cudaGetSymbolAddress, with that device current).
 * Limit: the scratch a call needs is
 *     ceil(n / chunk) * (4 + 2 * chunk)  +  4 * 2^alphabet_bits  +  4 * (2^alphabet_bits + 1)  +  8 * (ceil(n / chunk) + 1)
 * bytes (each of the four parts rounded up to 16); an input that needs more than TPC_RANS_STATIC_SCRATCH_BYTES is
 * rejected with TPC_ERR_STATIC_SCRATCH before anything is enqueued.  2 000 000 values at chunk = 512, alphabet_bits = 12
 * fit (one central Pb-Pb event has ~560 000 owned clusters per residual stream).
 * All calls on a device share the one array and it keeps the last call's contents: every call clears what must start
 * at zero itself, but two calls that overlap on the GPU (different streams, or graphs replayed concurrently) race --
 * serialise them.  Arguments, outputs and the other errors as for tpc_rans_encode; after TPC_ERR_CUDA there is no handle
 * whose tpc_last_cuda_error could be asked. */
#define TPC_RANS_STATIC_SCRATCH_BYTES (4u << 20)
int tpc_rans_encode_static(const void* values, int32_t value_bytes, int64_t n, int32_t alphabet_bits, int32_t chunk,
                           void* stream, const tpc_rans_stream_t* out);

/* NEXT-2 (readings P53..P56 in DESIGN.md): clusterizer in front of the path, digits -> clusters.
 * Digits of a (sector,row): cells (pad, time bin) with an ADC value >= 1, unique, ascending by (time, pad).
 * Peak (P53): adc >= q_peak_min, greater than each of its 8 neighbours that precede it in (time, pad) order and
 * greater or equal to the others (absent cells count 0).  Cluster (P54): over the peak's 3 x 3 block Q = sum a,
 * Sy = sum a dp, St = sum a dt; y = p * pad_units - floor((n_pads - 1) * pad_units / 2) + rdiv(pad_units * Sy, Q),
 * |z| = t * time_units + rdiv(time_units * St, Q), negative on the C side ((sector / n_per_side) % 2 == 1),
 * rdiv(a, b) = floor((2a + b) / (2b)).  Clusters of a (sector,row) ascend by (time, pad) of their peak (P55). */
typedef struct {
  const uint16_t* pad;       /* [device] n_digits */
  const uint16_t* time;      /* [device] n_digits */
  const uint16_t* adc;       /* [device] n_digits, 1..1023 */
  const uint32_t* offsets;   /* [device] n_sectors*n_rows + 1 CSR offsets into the digit arrays */
} tpc_digits_t;
typedef struct {
  int32_t n_pads;            /* pads per row (<= 32768); pad p is y = (p - (n_pads-1)/2) * pad pitch */
  int32_t n_per_side;        /* sectors per z side: 18 */
  int32_t pad_units;         /* pad pitch in fixed-point units: 256 = 0.4 cm */
  int32_t time_units;        /* time-bin width in fixed-point units of z: 330 */
  int32_t q_peak_min;        /* P53: 6 */
} tpc_cluster_params_t;
void tpc_default_cluster_params(tpc_cluster_params_t* p);
typedef struct {
  int32_t* y;                /* [device] capacity; with z and row_offsets the input format of tpc_track */
  int32_t* z;
  int32_t* qtot;             /* [device] capacity: charge of the 3 x 3 block */
  int32_t* qmax;             /* [device] capacity: ADC value of the peak */
  uint32_t* row_offsets;     /* [device] n_sectors*n_rows + 1 */
  int32_t* counts;           /* [device] int32[2]: [0] clusters found, [1] 1 iff that exceeds capacity (the excess is
                                not written; row_offsets still describe the full result) */
  int32_t capacity;
} tpc_clusters_out_t;
/* Geometry (n_sectors, n_rows) from the handle.  Asynchronous on `stream`.  Errors: TPC_ERR_ARG, TPC_ERR_NOMEM,
 * TPC_ERR_CUDA. */
int tpc_clusterize(tpc_tracker_t* t, const tpc_digits_t* digits, int64_t n_digits, const tpc_cluster_params_t* params,
                   void* stream, const tpc_clusters_out_t* out);

int tpc_tracker_destroy(tpc_tracker_t* t);

const char* tpc_status_string(int status);
const char* tpc_last_cuda_error(const tpc_tracker_t* t);

/* Scratch bytes currently owned by the handle. */
int64_t tpc_scratch_bytes(const tpc_tracker_t* t);

/* Number of kernel launches one tpc_track call enqueues (for launch accounting in the bench). */
int tpc_launches_per_call(const tpc_tracker_t* t);

/* Per-stage device times in ms of the most recent tpc_track call made while stage timing was enabled
 * (tpc_set_stage_timing(t, 1) inserts CUDA events between the stages).  ms[0..4] = a1..a5.  Synchronises. */
int tpc_set_stage_timing(tpc_tracker_t* t, int enable);
int tpc_get_stage_ms(tpc_tracker_t* t, float ms[5]);
/* Mean per-stage device times over the (up to 64) most recent calls made since stage timing was enabled;
 * *n_calls (may be NULL) receives how many calls were averaged.  Synchronises on those calls' events. */
int tpc_get_stage_ms_mean(tpc_tracker_t* t, float ms[5], int32_t* n_calls);

/* ---- test-only: a4 has two variants that compute the same thing (phase kernels for large calls, one uniform
 * kernel for small ones).  0 = choose by call size (default), 1 = uniform, 2 = phased. */
int tpc_debug_set_a4_variant(tpc_tracker_t* t, int variant);
/* a2 on sparse calls: 0 = rows read through L1/L2 (default), 1 = rows staged in shared memory by TMA bulk copies, a
 * CTA sliding a three-row window over 19 rows (north_star's sketch; same links; profiles/r02_a2_staged.md). */
int tpc_debug_set_a2_variant(tpc_tracker_t* t, int variant);

/* ---- test-only exports: intermediate results of the most recent tpc_track call on this handle ----
 * All outputs are [device] buffers in id space (-1 = none), written asynchronously on `stream`. */
/* which = 0: raw a2 link tables; 1: cleaned links as a3 stored them (the up link per cluster; the down links are
 * the inverse of those, a3 keeps no down table).  Internally links are sorted positions; the export translates
 * them to cluster ids.  up, dn: n int32 each. */
int tpc_debug_copy_links(tpc_tracker_t* t, int which, int32_t* up, int32_t* dn, void* stream);
/* start, len: counts[3] entries each (seeds ascend by start id, P14). */
int tpc_debug_copy_seeds(tpc_tracker_t* t, int32_t* start, int32_t* len, void* stream);
/* Tracklets of all seeds, seed-major: par[s*6 + 0..5] = (x_ref, y, z, sin phi, tan lambda, q/pT),
 * cov[s*15 + ..], chi2[s], n_hits[s], hits[s*n_rows + r] = cluster id in row r or -1.
 * Any pointer may be NULL to skip it.  Sizes from counts[3]. */
int tpc_debug_copy_tracklets(tpc_tracker_t* t, float* par, float* cov, float* chi2, int32_t* n_hits, int32_t* hits,
                             void* stream);
/* owner[h] = rank of the owning seed or -1; n int32. */
int tpc_debug_copy_owner(tpc_tracker_t* t, int32_t* owner, void* stream);
/* Sorted-grid view of a1 for the most recent call (the grid resolution is chosen per call from the cluster
 * density): ids_sorted[n] (cluster id at each sorted position), bin_start [n_sectors*n_rows *
 * bins_per_row_stride] ; returns the stride and per-row bin shape through the scalars (host). */
int tpc_debug_grid_info(const tpc_tracker_t* t, int32_t* bins_stride, int32_t* nz, int32_t* shift_y, int32_t* shift_z);
int tpc_debug_copy_grid(tpc_tracker_t* t, int32_t* ids_sorted, uint32_t* bin_start, void* stream);

#ifdef __cplusplus
}
#endif
#endif
