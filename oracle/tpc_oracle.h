/* tpc_oracle.h -- CPU oracle for TPC sector track finding.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, fp64, obviously-correct restatement of the five-stage path that BASELINE.json's
 * north_star names (the paper, Table 1 / PAPER.md:40, only says "TPC tracking"; it gives no
 * algorithm).  Every stage follows SURVEY.md section 8(c) step by step, in that order and notation;
 * readings P1..P40 are listed in DESIGN.md.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this library.  It shares no code, header, table or
 * constant generator with paper_2502_09138_b200/ (the CUDA path); neither includes the other.
 *
 * All pointers are host pointers.  Cluster ids are indices into the event arrays; -1 = none.
 * Clusters of one (sector,row) are contiguous: row_offsets[s*n_rows + r] .. row_offsets[s*n_rows+r+1].
 */
#ifndef TPC_ORACLE_H
#define TPC_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  /* stage 2 (integer) -- SURVEY 8(c) P7, P8, P10 */
  int32_t w_y, w_z;            /* search window half-widths in fixed-point units, inclusive: 1280, 1600 */
  int32_t cost_wy, cost_wz;    /* cost = cost_wy*ddy^2 + cost_wz*ddz^2 : 9, 4 */
  int32_t c_max;               /* accept iff cost <= c_max : 3538944 */
  /* stage 3 -- P13 */
  int32_t l_min;               /* seed iff chain length >= l_min : 5 */
  /* stage 4 -- P15..P24 */
  double units_per_cm;         /* 640 */
  double sigma_y, sigma_z;     /* 0.1, 0.15 cm */
  double sinphi_max;           /* 0.95 */
  int32_t max_miss;            /* 5 consecutive rows */
  int32_t n_min_tracklet;      /* 10 */
  double gate_d;               /* accept iff d < 15 */
  double gate_y_cm, gate_z_cm; /* |dy| <= 2.0, |dz| <= 2.5 */
  double c_reset[5];           /* variances 0.25, 0.25, 0.05, 0.05, 25 */
  double cq_per_tesla;         /* k = cq_per_tesla * Bz * q/pT : -0.00299792458 (P4) */
  /* stage 5 -- P27 */
  int32_t n_min_owned;         /* 10 */
} orc_params_t;

void orc_default_params(orc_params_t* p);

/* ---- stage 1-2: neighbour finding (integer, bit-exact) -- SURVEY 8(c) "Stage 1-2" ---- */
/* definition: all pairs over the two adjacent rows */
void orc_neighbours_brute(const orc_params_t* p, int32_t n_sectors, int32_t n_rows, const int32_t* y,
                          const int32_t* z, const uint32_t* row_offsets, int32_t* link_up, int32_t* link_dn);
/* same result through the oracle's own pruning structure (per-row z-sorted index + binary search) */
void orc_neighbours_pruned(const orc_params_t* p, int32_t n_sectors, int32_t n_rows, const int32_t* y,
                           const int32_t* z, const uint32_t* row_offsets, int32_t* link_up, int32_t* link_dn);

/* P48 (NEXT-4: rows that are not equidistant).  gap_w[r], r = 0..n_rows-2: integer pitch weight of the gap between
 * rows r and r+1 (nearbyint(64 * pitch in cm), oracle.py: pitch_weights); NULL = all equal.  For cluster h in row r
 * with wa = gap_w[r-1], wb = gap_w[r]: cost = cost_wy*(wa y_u + wb y_d - (wa+wb) y_h)^2 + cost_wz*(...z...)^2,
 * minimised as before, accepted iff 4 cost <= c_max (wa + wb)^2.  With equal weights this is P8 / P10 exactly. */
void orc_neighbours_brute_w(const orc_params_t* p, int32_t n_sectors, int32_t n_rows, const int32_t* gap_w,
                            const int32_t* y, const int32_t* z, const uint32_t* row_offsets, int32_t* link_up,
                            int32_t* link_dn);
void orc_neighbours_pruned_w(const orc_params_t* p, int32_t n_sectors, int32_t n_rows, const int32_t* gap_w,
                             const int32_t* y, const int32_t* z, const uint32_t* row_offsets, int32_t* link_up,
                             int32_t* link_dn);

/* ---- stage 3: cleaner, chains, seeds (integer, bit-exact) -- SURVEY 8(c) "Stage 3" ---- */
void orc_clean_links(int64_t n, const int32_t* up, const int32_t* dn, int32_t* up_c, int32_t* dn_c);
/* returns number of seeds; seeds ascend by start id; seed_start/seed_len need capacity n / l_min + 1 */
int64_t orc_find_seeds(const orc_params_t* p, int64_t n, const int32_t* up_c, const int32_t* dn_c,
                       int32_t* seed_start, int32_t* seed_len);

/* ---- stage 4 building blocks (exported for the pins) -- SURVEY Appendix C ---- */
/* state = (y, z, sin phi, tan lambda, q/pT); cov = full 5x5 row-major (may be NULL); k = cq*q/pT.
 * Returns 1 on success, 0 on transport failure (|sin phi| >= sinphi_max before or after). */
int orc_transport(double cq, double sinphi_max, double dx, double* state, double* cov);
void orc_jacobian(double cq, double dx, const double* state, double* F /* 5x5 row-major */);
/* joint (y,z) Kalman update, V = diag(sy2, sz2); returns the chi2 increment */
double orc_update(double* state, double* cov, double ym, double zm, double sy2, double sz2);

/* ---- stage 4: follower ---- */
/* Inputs: y_cm/z_cm are cluster coordinates in cm as doubles (normally int/units_per_cm; tests may pass
 * exact doubles).  search_mode 0 = full-row scan (the definition, P17), 1 = z-sorted pruning (same result).
 * Outputs per seed i: par[i*6 + 0..5] = (x_ref, y, z, sin phi, tan lambda, q/pT); cov[i*15 ..] packed lower
 * triangle (00,10,11,20,21,22,...); chi2[i]; n_hits[i]; hits[i*n_rows + r] = cluster id in row r or -1. */
void orc_follow(const orc_params_t* p, double bz, int32_t n_sectors, int32_t n_rows, const double* row_x,
                const double* y_cm, const double* z_cm, const uint32_t* row_offsets, const int32_t* up_c,
                int64_t n_seeds, const int32_t* seed_start, const int32_t* seed_len, int search_mode,
                double* par, double* cov, double* chi2, int32_t* n_hits, int32_t* hits);

/* ---- stage 5: ownership, selection, output -- SURVEY 8(c) "Stage 5" ---- */
/* owner[h] = seed rank owning cluster h or -1.  Outputs tracks in ascending seed start id:
 * trk_seed[t] = seed rank; trk_n_owned[t]; trk_hit_offset[t]; hit_ids = owned hits ascending row.
 * Returns number of output tracks; *n_out_hits = total hits written. */
int64_t orc_select(const orc_params_t* p, int64_t n, int32_t n_rows, int64_t n_seeds, const int32_t* seed_start,
                   const int32_t* n_hits, const int32_t* hits, int32_t* owner, int32_t* trk_seed,
                   int32_t* trk_n_owned, int32_t* trk_hit_offset, int32_t* hit_ids, int64_t* n_out_hits);

/* ---- NEXT-1: refit of an output track over its owned hits only (reading P41) ----
 * Hits h_0..h_{m-1} of track t = hit_ids[trk_hit_offset[t] .. + trk_n_owned[t]), ascending row.
 * State from h_0, h_1 as in P19 (dx = x(row h_1) - x(row h_0)), C = C_reset, update h_0; up: one transport per
 * hit over the row gap + update, stop at the first failed transport; C = C_reset, chi2 = 0, update with the last
 * hit reached; down: transport + update back to h_0, stop at a failed transport.
 * Outputs per track: par[t*6..] = (x_ref, y, z, sin phi, tan lambda, q/pT) at the row where the down pass ended,
 * cov[t*15..] packed lower triangle, chi2[t] of the down pass, n_used[t] = hits updated in the down pass. */
void orc_refit(const orc_params_t* p, double bz, int32_t n_sectors, int32_t n_rows, const double* row_x,
               const double* y_cm, const double* z_cm, const uint32_t* row_offsets, int64_t n_tracks,
               const int32_t* trk_hit_offset, const int32_t* trk_n_owned, const int32_t* hit_ids, double* par,
               double* cov, double* chi2, int32_t* n_used);

/* ---- NEXT-1: merging of sector tracks (readings P42..P46) ----
 * orc_rotate: state (y, z, sin phi, tan lambda, q/pT) at the plane x of a sector frame -> the frame turned by alpha
 * (radians, positive = towards larger azimuth): *x and state are replaced by the same point and direction in the new
 * frame, cov (full 5x5 row-major, may be NULL) by R C R^T for the state taken at the new plane x = *x.  Returns 0
 * (nothing changed) iff the track does not move along +x' in the new frame or |sin phi'| >= sinphi_max. */
int orc_rotate(double cq, double sinphi_max, double alpha, double* x, double* state, double* cov);
/* chi2 of "track a continues as track b": a's record (x_ref, state, packed covariance) is rotated by alpha into b's
 * frame, transported to b's x_ref, D = p_b - p_a', S = C_b + C_a', chi2 = D^T S^-1 D.  Negative iff the rotation or
 * the transport fails. */
double orc_match_chi2(double cq, double sinphi_max, double alpha, const double* par_a, const double* cov_a,
                      const double* par_b, const double* cov_b);
/* Links between the n_tracks records (par[t*6..] = x_ref + state, cov[t*15..] packed lower triangle, sector,
 * first_row, last_row of the owned hits).  Candidate a -> b (P43): 1 <= first_row[b] - last_row[a] <= gap_max and the
 * sectors are the same, azimuthal neighbours on the same side ((s' - s) mod n_per_side in {1, n_per_side - 1},
 * alpha = +-sector_angle), or face each other across the central membrane (s' = s +- n_per_side inside one group of
 * 2 n_per_side sectors -- a batch of events is laid out as such groups --, alpha = 0).
 * succ[a] = candidate b minimising (chi2, b) among those with 0 <= chi2 < chi2_max; pred[b] likewise over a; a link
 * a -> b stands iff succ[a] == b and pred[b] == a (P45).  Outputs: succ, pred (-1 = none, only standing links),
 * link_chi2[a] of a's standing link (else -1).  Returns the number of links. */
int64_t orc_merge(double cq, double sinphi_max, int32_t n_per_side, double sector_angle, int32_t gap_max,
                  double chi2_max, int64_t n_tracks, const double* par, const double* cov, const int32_t* sector,
                  const int32_t* first_row, const int32_t* last_row, int32_t* succ, int32_t* pred, double* link_chi2);

/* P47: refit over the hits of a whole chain of linked tracks.  For every chain head a (pred[a] < 0): hits = owned hits
 * of a, succ[a], succ[succ[a]], ... in that order (rows ascend along a chain, P43); the P41 schedule runs over that
 * list, the state living in the frame of the sector of the hit it was last moved to: before a transport to a hit of
 * another sector the state and covariance are rotated into that sector's frame (P42; a failed rotation ends the pass
 * like a failed transport).  Outputs per track index: heads get (x_ref, state) at the row where the down pass ended
 * in the frame of that hit's sector (out_sector), packed covariance, chi2 and the hits used on the way down; tracks
 * that are not heads get n_used = 0 and nothing else. */
void orc_refit_merged(const orc_params_t* p, double bz, int32_t n_sectors, int32_t n_rows, const double* row_x,
                      const double* y_cm, const double* z_cm, const uint32_t* row_offsets, int32_t n_per_side,
                      double sector_angle, int64_t n_tracks, const int32_t* trk_hit_offset,
                      const int32_t* trk_n_owned, const int32_t* hit_ids, const int32_t* succ, const int32_t* pred,
                      double* par, double* cov, double* chi2, int32_t* n_used, int32_t* out_sector);

/* ---- NEXT-3: track-model cluster compression, the residual transform (readings P50..P52) ----
 * Lossless integer transform of the clusters an output track owns into small residuals against a predictor built
 * from the track's previous hits (the entropy coder that follows is a separate 0.10 % line of the paper's Table 1).
 * For track t with hits h_0..h_{m-1} (ascending rows r_j), for coordinate c in {y, z} (fixed-point ints), P50:
 *   j = 0: drow = r_0, residual = c_0 (absolute);  j = 1: drow = r_1 - r_0, residual = c_1 - c_0;
 *   j >= 2, the four previous hits in four consecutive rows and r_j = r_{j-1} + 1 (least-squares line through the last
 *           four hits, extrapolated one row): pred = floor((2 c_{j-1} + c_{j-2} - c_{j-4}) / 2);
 *   j >= 2 otherwise (two-point line with the row gaps g1 = r_{j-1} - r_{j-2}, g2 = r_j - r_{j-1}):
 *           pred = c_{j-1} + floor((c_{j-1} - c_{j-2}) * g2 / g1);   residual = c_j - pred, drow = g2.
 * floor = rounding towards minus infinity.  Outputs in hit-list order: drow[k], ry[k], rz[k], k = hit_offset + j. */
void orc_compress(int32_t n_rows, const int32_t* y, const int32_t* z, const uint32_t* row_offsets, int64_t n_sr,
                  int64_t n_tracks, const int32_t* trk_hit_offset, const int32_t* trk_n_owned, const int32_t* hit_ids,
                  uint8_t* drow, int32_t* ry, int32_t* rz);
/* Inverse (P51): rebuilds row, y, z of every hit from the residual streams, track by track. */
void orc_decompress(int64_t n_tracks, const int32_t* trk_hit_offset, const int32_t* trk_n_owned, const uint8_t* drow,
                    const int32_t* ry, const int32_t* rz, int32_t* row, int32_t* y, int32_t* z);
/* P52: histogram of the residuals of the hits with j >= `j_min` of every track, clamped to [-32768, 32767]
 * (bin = residual + 32768; the two edge bins collect everything beyond), 65536 bins. */
void orc_residual_histogram(int64_t n_tracks, const int32_t* trk_hit_offset, const int32_t* trk_n_owned,
                            const int32_t* res, int32_t j_min, int64_t* hist);

/* ---- NEXT-3, entropy stage (the paper's "TPC rANS Encoding"; readings P57..P60) ----
 * Static range-variant asymmetric numeral system (Duda 2013) over independent chunks of a symbol stream, state
 * in [2^16, 2^32), 16-bit renormalisation, probabilities in units of 1/M, M = 2^16.
 * P57 symbols: alphabet A = 2^alphabet_bits; a value v with -A/2 < v < A/2 is the symbol v + A/2; any other value is
 *   the escape symbol 0 and goes, as it is, to the escape list (stream order).
 * P58 frequencies: n_s = occurrences of s, N = their sum, K = symbols that occur; f_s = 0 if n_s = 0, else
 *   f_s = 1 + floor(n_s (M - K) / N); the remainder M - sum f_s (0 <= . < K) goes to the most frequent symbol (the
 *   smallest one among equals).  c_s = sum_{u<s} f_u.  N = 0: all f_s = 0.
 * P59 coding of a chunk (symbols i0 .. i1-1 of the stream, `chunk` symbols, the last chunk shorter): x = 2^16; for
 *   i = i1-1 down to i0, s = symbol i: if x >= f_s 2^16, the low 16 bits of x are emitted and x >>= 16; then
 *   x = floor(x / f_s) 2^16 + (x mod f_s) + c_s.  Decoding runs forwards: slot = x mod 2^16, s = the symbol with
 *   c_s <= slot < c_s + f_s, x = f_s floor(x / 2^16) + slot - c_s; if x < 2^16, x = x 2^16 + the next 16-bit word.
 * P60 layout: the bytes of a chunk are the final x (uint32, little endian) followed by the emitted words in the order
 *   the decoder consumes them (the last emitted first; uint16, little endian); chunk c occupies
 *   payload[chunk_off[c] .. chunk_off[c+1]), its escapes escapes[esc_off[c] .. esc_off[c+1]).
 * Capacities the caller provides: freq[A], chunk_off / esc_off[n_chunks + 1] with n_chunks = ceil(n / chunk),
 * payload[n_chunks * 4 + 2 n], escapes[n].  orc_rans_encode returns the payload size in bytes. */
int32_t orc_rans_symbol(int32_t v, int32_t alphabet_bits);
void orc_rans_normalise(int32_t alphabet, const int64_t* counts, uint32_t* freq);
int64_t orc_rans_encode(const int32_t* values, int64_t n, int32_t alphabet_bits, int32_t chunk, uint32_t* freq,
                        uint32_t* chunk_off, uint32_t* esc_off, uint8_t* payload, int32_t* escapes);
void orc_rans_decode(int64_t n, int32_t alphabet_bits, int32_t chunk, const uint32_t* freq, const uint32_t* chunk_off,
                     const uint32_t* esc_off, const uint8_t* payload, const int32_t* escapes, int32_t* values);

/* ---- NEXT-2: clusterizer, digits -> clusters (readings P53..P56) ----
 * Digits of a (sector,row): cells (pad, time bin) with an ADC value >= 1, unique, ascending by (time, pad) (P56).
 * P53 peak: a digit with adc >= q_peak_min that is greater than each of its 8 neighbours preceding it in (time, pad)
 *   order and greater than or equal to each of the others (absent cells count 0): a plateau yields its first cell.
 * P54 cluster of a peak at (p, t): over its 3 x 3 block Q = sum a, Sy = sum a dp, St = sum a dt;
 *   y = p * pad_units - floor((n_pads - 1) * pad_units / 2) + rdiv(pad_units * Sy, Q),
 *   |z| = t * time_units + rdiv(time_units * St, Q), z < 0 on the C side (side = (sector / n_per_side) % 2),
 *   rdiv(a, b) = floor((2 a + b) / (2 b)); qtot = Q, qmax = the peak's adc.  A digit may belong to several blocks.
 * P55 order: the clusters of a (sector,row) ascend by (time, pad) of their peak.
 * Outputs y, z, qtot, qmax (capacity = number of digits suffices), row_offsets[n_sectors * n_rows + 1].
 * Returns the number of clusters. */
int64_t orc_clusterize(int32_t n_sectors, int32_t n_rows, int32_t n_per_side, int32_t n_pads, int32_t n_time,
                       int32_t pad_units, int32_t time_units, int32_t q_peak_min, const uint16_t* pad,
                       const uint16_t* time, const uint16_t* adc, const uint32_t* digit_offsets, int32_t* y,
                       int32_t* z, int32_t* qtot, int32_t* qmax, uint32_t* row_offsets);

int orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
