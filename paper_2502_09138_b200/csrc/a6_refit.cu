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

}  // namespace

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
