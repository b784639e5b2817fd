// a6_refit.cu -- NEXT-1: refit of the output tracks over their owned hits only (reading P41,
// DESIGN.md; the a4 fit of a track runs over all hits of its tracklet, P28, including hits another track won).
//
// Per track with owned hits h_0 .. h_{m-1} (ascending row): state from h_0, h_1 as in P19 (dx = the row gap),
// C = C_reset, update h_0; up: one transport over the row gap + update per hit, stop at a failed transport;
// C = C_reset, chi2 = 0, update with the last hit reached; down: transport + update back to h_0.  Result: state,
// covariance and x at the row where the down pass ended, chi2 and the number of hits of the down pass.
//
// Same execution model as a4: persistent warps, one lane per track, lanes refill from a device counter, one
// uniform step (optional covariance reset, optional transport, update) for both passes; fp32 state relative to
// the first hit, fp32 U D U^T covariance (kalman.cuh).  The hit's (y, z) comes from the caller's cluster arrays (y[id], z[id]), requested
// one step ahead; its row from the row list a5 wrote next to the hit list.
#include "tpc_internal.cuh"
#include "kalman.cuh"

namespace {

constexpr int A6_THREADS = 128;

enum : int { R_IDLE = 0, R_FIRST, R_UP, R_TOP, R_DOWN };

// Predicated loads straight into their destination registers (see a4_follow.cu for why they are PTX).
__device__ __forceinline__ void ld_yz_if(int& y, int& z, const int32_t* py, const int32_t* pz, bool pred) {
  asm volatile("{ .reg .pred q; setp.ne.s32 q, %2, 0; @q ld.global.nc.s32 %0, [%3]; @q ld.global.nc.s32 %1, [%4]; }"
               : "+r"(y), "+r"(z) : "r"((int)pred), "l"(py), "l"(pz));
}

__global__ void __launch_bounds__(A6_THREADS, 4)
a6_refit_kernel(const DevGeom g, DevCtl* __restrict__ ctl, const int32_t* __restrict__ cy_in,
                const int32_t* __restrict__ cz_in, const uint8_t* __restrict__ hit_row, const tpc_track_rec_t* __restrict__ tracks,
                int32_t track_capacity, const int32_t* __restrict__ hit_ids, int32_t hit_capacity,
                const int32_t* __restrict__ counts, tpc_track_rec_t* __restrict__ out) {
  extern __shared__ double s_row_x[];
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int nr = g.n_rows;
  for (int r = threadIdx.x; r < nr; r += blockDim.x) s_row_x[r] = g.row_x[r];
  __syncthreads();
  // tracks whose record or hit list was not written (capacity overflow) are not refitted
  const uint32_t n_tracks = (uint32_t)min(counts[0], track_capacity);
  const bool hits_ok = counts[1] <= hit_capacity;
  if (n_tracks == 0 || !hits_ok) return;

  int phase = R_IDLE;
  bool exhausted = false;
  int k = -1, m = 0, j = 0, last = 0, used = 0, row = 0, y0 = 0, z0 = 0;
  const int32_t* hl = hit_ids;     // this track's hit ids ...
  const uint8_t* hr = hit_row;     // ... and their rows (a5)
  int pf_j = -1, pf_y = 0, pf_z = 0;   // (y, z) of hit pf_j, requested one step ahead
  float chi2 = 0.f;
  State p;
  Cov C;
  p.y = p.z = p.s = p.t = p.q = 0; p.oy = p.oz = 0;
  cov_reset(g, C);

  while (true) {
    const bool want = phase == R_IDLE && !exhausted;
    const unsigned idle = __ballot_sync(FULL, want);
    if (idle) {
      uint32_t base = 0;
      if (lane == 0) base = atomicAdd(&ctl->next_track, (uint32_t)__popc(idle));
      base = __shfl_sync(FULL, base, 0);
      if (base + (uint32_t)__popc(idle) >= n_tracks) exhausted = true;
      const uint32_t kk = base + (uint32_t)__popc(idle & ((1u << lane) - 1u));
      if (want && kk < n_tracks) {
        k = (int)kk;
        const tpc_track_rec_t* t = tracks + k;
        m = t->n_hits;
        hl = hit_ids + t->hit_offset;
        hr = hit_row + t->hit_offset;
        row = hr[0];
        y0 = cy_in[hl[0]];
        z0 = cz_in[hl[0]];
        pf_j = 0; pf_y = y0; pf_z = z0;
        p.y = 0; p.z = 0; p.s = 0; p.t = 0; p.q = 0;
        p.oy = y0; p.oz = z0;
        if (m >= 2) {   // P19 with the gap to the second owned hit
          const int y1 = cy_in[hl[1]], z1 = cz_in[hl[1]];
          const float dxr = (float)(s_row_x[hr[1]] - s_row_x[row]);
          const float dy = (float)(y1 - y0) * g.inv_units, dz = (float)(z1 - z0) * g.inv_units;
          const float ichord = rsqrtf(fmaf(dxr, dxr, dy * dy));
          p.s = dy * ichord;
          p.t = dz * ichord;
        }
        j = 0; last = 0; used = 0; chi2 = 0.f;
        phase = R_FIRST;
      }
    }
    if (!__any_sync(FULL, phase != R_IDLE)) break;

    // ---- one step: which hit, reset?, transport? ----
    if (phase == R_UP && j >= m) phase = R_TOP;
    if (phase == R_TOP) j = last;
    const int ph = phase;
    const bool active = ph != R_IDLE;
    const bool reset = ph == R_FIRST || ph == R_TOP;
    const bool tr = ph == R_UP || ph == R_DOWN;
    int trow = row, cy = pf_y, cz = pf_z;
    if (active) {
      trow = hr[j];
      ld_yz_if(cy, cz, cy_in + hl[j], cz_in + hl[j], pf_j != j);   // not requested ahead (after a pass ended early): load now
    }
    // the hit of the next step: its record is requested now and used then
    {
      int jn = -1;
      if (ph == R_FIRST) jn = 1;
      if (ph == R_UP) jn = j + 1;
      if (ph == R_TOP || ph == R_DOWN) jn = j - 1;
      const bool fetch = active && jn >= 0 && jn < m;
      int hn = 0;
      if (fetch) hn = hl[jn];
      if (fetch) pf_j = jn;
      ld_yz_if(pf_y, pf_z, cy_in + hn, cz_in + hn, fetch);
    }
    if (active && reset) cov_reset(g, C);
    if (ph == R_TOP) { chi2 = 0.f; used = 0; }
    bool ok = active;
    if (tr) ok = transport<true>(g, (float)(s_row_x[trow] - s_row_x[row]), p, C);
    if (ok) {
      row = trow;
      chi2 += update(g, p, C, resid_y(g, p, cy), resid_z(g, p, cz));
      ++used;
      if (ph == R_FIRST) { phase = R_UP; j = 1; }
      else if (ph == R_UP) { last = j; ++j; }
      else if (ph == R_TOP) { phase = R_DOWN; j = last - 1; }
      else --j;
    } else if (ph == R_UP) {
      phase = R_TOP;   // P18: the up pass stops, the hits above are not used
    }
    // the down pass is over: transport failed, or h_0 is done
    if (active && ((ph == R_DOWN && !ok) || (phase == R_DOWN && j < 0))) {
      tpc_track_rec_t r = tracks[k];
      r.x = (float)s_row_x[row];
      r.y = (float)(((double)p.y + (double)p.oy) * g.inv_units_d);
      r.z = (float)(((double)p.z + (double)p.oz) * g.inv_units_d);
      r.sinphi = (float)p.s;
      r.tanl = (float)p.t;
      r.qpt = (float)p.q;
      float cv[15];
      C.lower(cv);
#pragma unroll
      for (int q = 0; q < 15; ++q) r.cov[q] = cv[q];
      r.chi2 = chi2;
      r.n_hits = used;
      out[k] = r;
      phase = R_IDLE;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// P47: refit over a whole chain of linked tracks (tpc_refit_merged).  One thread per chain head; the hits of the
// head, its successor, ... are walked up and back down with the same filter (kalman.cuh); when the next hit lies in
// another sector the state is rotated into that sector's frame (P42).  The rotation happens once or twice per chain,
// so it is done in fp64: factors -> full covariance -> R C R^T -> factors, and the split position is rebuilt.
// ---------------------------------------------------------------------------------------------------------------
struct FrameCfg {
  double sa, ca;   // sin, cos of the angle between neighbouring sector frames
  int nps;         // sectors per z side
};

__device__ __forceinline__ bool rotate_state(const DevGeom& g, double sa, double ca, double& x, State& p, Cov& C) {
  const double s = p.s;
  if (!(fabs(s) < 1.0)) return false;
  const double c = sqrt(1.0 - s * s);
  const double s1 = s * ca - c * sa, c1 = c * ca + s * sa;
  if (!(c1 > 0.0) || !(fabs(s1) < (double)g.sinphi_max)) return false;
  float cf[15];
  C.lower(cf);
  double F[5][5];
  for (int i = 0, q = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j, ++q) F[i][j] = F[j][i] = cf[q];
  // R = I except R00 = c/c1, R10 = -sa t/c1, R20 = -sa k, R22 = c1/c
  const double r00 = c / c1, r10 = -sa * (double)p.t / c1, r20 = -sa * (double)g.cq * (double)p.q, r22 = c1 / c;
  double M[5][5];   // M = R F
  for (int j = 0; j < 5; ++j) {
    M[0][j] = r00 * F[0][j];
    M[1][j] = F[1][j] + r10 * F[0][j];
    M[2][j] = r22 * F[2][j] + r20 * F[0][j];
    M[3][j] = F[3][j];
    M[4][j] = F[4][j];
  }
  for (int i = 0; i < 5; ++i) {   // F = M R^T
    const double m0 = M[i][0], m1 = M[i][1], m2 = M[i][2];
    F[i][0] = r00 * m0;
    F[i][1] = m1 + r10 * m0;
    F[i][2] = r22 * m2 + r20 * m0;
    F[i][3] = M[i][3];
    F[i][4] = M[i][4];
  }
  // U D U^T factorisation of the symmetric F (upper unit triangular U), from the last column backwards
  double U[5][5], D[5];
  for (int j = 4; j >= 0; --j) {
    double d = F[j][j];
    for (int k = j + 1; k < 5; ++k) d -= D[k] * U[j][k] * U[j][k];
    D[j] = d;
    for (int i = 0; i < j; ++i) {
      double u = F[i][j];
      for (int k = j + 1; k < 5; ++k) u -= D[k] * U[i][k] * U[j][k];
      U[i][j] = u / d;
    }
  }
  C.d0 = (float)D[0]; C.d1 = (float)D[1]; C.d2 = (float)D[2]; C.d3 = (float)D[3]; C.d4 = (float)D[4];
  C.u01 = (float)U[0][1]; C.u02 = (float)U[0][2]; C.u03 = (float)U[0][3]; C.u04 = (float)U[0][4];
  C.u12 = (float)U[1][2]; C.u13 = (float)U[1][3]; C.u14 = (float)U[1][4];
  C.u23 = (float)U[2][3]; C.u24 = (float)U[2][4]; C.u34 = (float)U[3][4];
  // the point: (x, y) with y = (origin + fraction) / units
  const double y0 = ((double)p.oy + (double)p.y) * g.inv_units_d;
  const double x1 = x * ca + y0 * sa, y1 = (-x * sa + y0 * ca) * (double)g.units;
  x = x1;
  const double oy = rint(y1);
  p.oy = (int)oy;
  p.y = (float)(y1 - oy);
  p.s = (float)s1;
  return true;
}

__global__ void __launch_bounds__(128)
a6_refit_merged_kernel(const DevGeom g, const FrameCfg fc, const int32_t* __restrict__ cy_in,
                       const int32_t* __restrict__ cz_in, const uint8_t* __restrict__ hit_row,
                       const tpc_track_rec_t* __restrict__ tracks, int32_t track_capacity,
                       const int32_t* __restrict__ hit_ids, int32_t hit_capacity, const int32_t* __restrict__ counts,
                       const int32_t* __restrict__ succ, const int32_t* __restrict__ pred,
                       tpc_track_rec_t* __restrict__ out) {
  const int n_tracks = min(counts[0], track_capacity);
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n_tracks || counts[1] > hit_capacity) return;
  tpc_track_rec_t r = tracks[k];
  if (pred[k] >= 0) {   // not a chain head: its hits are refitted with its head
    r.n_hits = 0;
    out[k] = r;
    return;
  }
  const double* row_x = g.row_x;
  // frame angle from sector a to sector b (related by P43): 0, +angle or -angle
  auto angle_sign = [&](int a, int b) {
    if (a == b || a / fc.nps != b / fc.nps) return 0;
    const int d = ((b % fc.nps - a % fc.nps) % fc.nps + fc.nps) % fc.nps;
    return d == 1 ? 1 : -1;
  };
  int ct = k, j = 0;                                     // current track of the chain and hit index inside it
  const int32_t* hl = hit_ids + r.hit_offset;
  const uint8_t* hr = hit_row + r.hit_offset;
  int m = r.n_hits, cur_sec = r.sector;
  State p;
  Cov C;
  const int h0 = hl[0];
  p.oy = cy_in[h0]; p.oz = cz_in[h0]; p.y = 0.f; p.z = 0.f; p.s = 0.f; p.t = 0.f; p.q = 0.f;
  double x = row_x[hr[0]];
  if (m >= 2) {
    const int h1 = hl[1];
    const float dxr = (float)(row_x[hr[1]] - x);
    const float dy = (float)(cy_in[h1] - p.oy) * g.inv_units, dz = (float)(cz_in[h1] - p.oz) * g.inv_units;
    const float ichord = rsqrtf(fmaf(dxr, dxr, dy * dy));
    p.s = dy * ichord;
    p.t = dz * ichord;
  }
  cov_reset(g, C);
  update(g, p, C, resid_y(g, p, cy_in[h0]), resid_z(g, p, cz_in[h0]));
  // move the state to hit jj of track tt (sector ss): rotate if the sector changes, then transport to its row
  // (all or nothing: if the rotation works but the transport fails, the state stays in the old frame)
  auto move_to = [&](int ss, int row) -> bool {
    const double xt = row_x[row];
    if (ss != cur_sec) {
      State p2 = p;
      Cov C2 = C;
      double x2 = x;
      const int sg = angle_sign(cur_sec, ss);
      if (sg != 0 && !rotate_state(g, sg > 0 ? fc.sa : -fc.sa, fc.ca, x2, p2, C2)) return false;
      if (!transport<true>(g, (float)(xt - x2), p2, C2)) return false;
      p = p2;
      C = C2;
      cur_sec = ss;
      x = xt;
      return true;
    }
    if (!transport<true>(g, (float)(xt - x), p, C)) return false;
    x = xt;
    return true;
  };
  int last_t = k, last_j = 0, t_sec = r.sector;
  bool ok = true;
  while (ok) {   // up
    ++j;
    if (j >= m) {
      const int nt = succ[ct];
      if (nt < 0) break;
      ct = nt;
      const tpc_track_rec_t* q = tracks + ct;
      hl = hit_ids + q->hit_offset;
      hr = hit_row + q->hit_offset;
      m = q->n_hits;
      t_sec = q->sector;
      j = 0;
    }
    ok = move_to(t_sec, hr[j]);
    if (ok) {
      update(g, p, C, resid_y(g, p, cy_in[hl[j]]), resid_z(g, p, cz_in[hl[j]]));
      last_t = ct;
      last_j = j;
    }
  }
  // back to the last hit reached (the walk may have stepped onto a further track before failing)
  if (ct != last_t) {
    ct = last_t;
    const tpc_track_rec_t* q = tracks + ct;
    hl = hit_ids + q->hit_offset;
    hr = hit_row + q->hit_offset;
    m = q->n_hits;
    t_sec = q->sector;
  }
  j = last_j;
  cov_reset(g, C);
  float chi2 = update(g, p, C, resid_y(g, p, cy_in[hl[j]]), resid_z(g, p, cz_in[hl[j]]));
  int used = 1;
  ok = true;
  while (ok) {   // down
    --j;
    if (j < 0) {
      if (ct == k) break;
      ct = pred[ct];
      const tpc_track_rec_t* q = tracks + ct;
      hl = hit_ids + q->hit_offset;
      hr = hit_row + q->hit_offset;
      m = q->n_hits;
      t_sec = q->sector;
      j = m - 1;
    }
    ok = move_to(t_sec, hr[j]);
    if (ok) {
      chi2 += update(g, p, C, resid_y(g, p, cy_in[hl[j]]), resid_z(g, p, cz_in[hl[j]]));
      ++used;
    }
  }
  r.x = (float)x;
  r.y = (float)(((double)p.y + (double)p.oy) * g.inv_units_d);
  r.z = (float)(((double)p.z + (double)p.oz) * g.inv_units_d);
  r.sinphi = p.s;
  r.tanl = p.t;
  r.qpt = p.q;
  float cv[15];
  C.lower(cv);
#pragma unroll
  for (int q = 0; q < 15; ++q) r.cov[q] = cv[q];
  r.chi2 = chi2;
  r.n_hits = used;
  r.sector = cur_sec;
  out[k] = r;
}

}  // namespace

cudaError_t launch_a6_refit_merged(const tpc_tracker* t, const tpc_merge_params_t* mp, const int32_t* y,
                                   const int32_t* z, const tpc_tracks_out_t* tracks, const int32_t* succ,
                                   const int32_t* pred, tpc_track_rec_t* refit_out, cudaStream_t st) {
  if (t->last_n == 0 || tracks->track_capacity == 0) return cudaSuccess;
  FrameCfg fc;
  fc.sa = sin(mp->sector_angle);
  fc.ca = cos(mp->sector_angle);
  fc.nps = mp->n_per_side;
  a6_refit_merged_kernel<<<(unsigned)((tracks->track_capacity + 127) / 128), 128, 0, st>>>(
      t->g, fc, y, z, t->s.hit_row, tracks->tracks, tracks->track_capacity, tracks->hit_ids, tracks->hit_capacity,
      tracks->counts, succ, pred, refit_out);
  return cudaGetLastError();
}

cudaError_t launch_a6_refit(const tpc_tracker* t, const int32_t* y, const int32_t* z, const tpc_tracks_out_t* tracks,
                            tpc_track_rec_t* refit_out, cudaStream_t st) {
  if (t->last_n == 0 || t->a4_blocks == 0 || tracks->track_capacity == 0) return cudaSuccess;
  cudaError_t e = cudaMemsetAsync(&t->s.ctl->next_track, 0, sizeof(uint32_t), st);
  if (e != cudaSuccess) return e;
  a6_refit_kernel<<<t->a4_blocks, A6_THREADS, (size_t)t->g.n_rows * sizeof(double), st>>>(
      t->g, t->s.ctl, y, z, t->s.hit_row, tracks->tracks, tracks->track_capacity, tracks->hit_ids,
      tracks->hit_capacity, tracks->counts, refit_out);
  return cudaGetLastError();
}
