// a4_follow.cu -- stage a4: Kalman-filter tracklet following with a helix model in constant Bz
// (SURVEY 8(c) "Stage 4", P15-P24; Appendix C transport/Jacobian/update; north_star "one thread per seed with
// warp-level compaction of active seeds, that keeps the 5-parameter state and covariance in registers"), plus
// the a5 ownership vote (atomicMax on packed (n_hits, rank) words, P26) cast when a tracklet ends.
//
// fp32 state on the device.  To keep fp32 residuals exact for long drift offsets (configs[2]: |z| up to ~5400 cm)
// the filter runs in coordinates relative to the seed's first cluster: hit - origin is an exact integer
// difference, and the model is translation invariant in y and z.  The origin is added back in double at the end.
//
// Execution model (v1 was a plain thread-per-seed kernel that ran 3.85 of 32 lanes,
// profiles/r01_v1_a4_thread_per_seed.md):
//  * Persistent warps, one lane per tracklet.  A lane whose tracklet ends takes the next seed rank from a device
//    counter at the top of the loop, so the active lanes of a warp stay dense until the queue is empty.
//  * One uniform per-row step for every phase of the method (init, A fit up the chain, B extend up, C refit down,
//    D extend down, final transport): a phase only selects flags -- reset covariance?  transport by which dx?
//    where does the hit come from (chain link / row search / recorded hit table / none)? -- and then all lanes run
//    the same single transport and the same single update.  Lanes in different phases no longer serialise.
//  * The step is latency-bound on its gathers, so every gather whose address is known early is issued one step
//    ahead and carried in registers: the next chain hit's record (its id is in the current record), the next two
//    entries of the row -> hit table on the way down, and the bin starts of the next row's search window at the
//    extrapolated position (validated against the exact window after the transport; a wrong guess only costs the
//    direct loads).  The candidates of the current search are prefetched into L1 while the transport computes.
//  * The row -> hit table is the tracklet's final [row] array in global memory (L2-resident while in use); when a
//    tracklet ends the whole warp pads it with -1 and casts the ownership votes, 32 rows per instruction.  No
//    shared memory beyond two small geometry tables, so L1 keeps its full size for the gathers.
#include "tpc_internal.cuh"
#include "a4_search.cuh"

namespace {

enum : int { PH_IDLE = 0, PH_INIT, PH_A, PH_B, PH_CS, PH_CD, PH_FIN, PH_DONE };
enum : int { M_NONE = 0, M_LINK, M_TABLE, M_SEARCH };

constexpr int A4_THREADS = 128;   // warps never synchronise with each other after the geometry tables are loaded
constexpr int A4_MIN_BLOCKS = 4;   // 16 warps per SM: registers capped at 128 per thread (5 and 6 measured slower)

__global__ void __launch_bounds__(A4_THREADS, A4_MIN_BLOCKS)
a4_follow_kernel(const DevGeom g, DevCtl* __restrict__ ctl, const int4* __restrict__ srt,
                 const int32_t* __restrict__ clean_up,
                 const uint32_t* __restrict__ sec_key, const uint32_t* __restrict__ bin_start,
                 const int32_t* __restrict__ seed_pos, const int32_t* __restrict__ seed_sr,
                 float4* __restrict__ tl_rec, int32_t* __restrict__ tl_hits, int2* __restrict__ tl_yz,
                 uint32_t* __restrict__ tl_span, uint32_t* __restrict__ owner) {
  extern __shared__ double smem_a4[];
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int nr = g.n_rows;
  const uint32_t n_seeds = ctl->n_seeds;
  if (n_seeds == 0) return;
  // shared memory: row_x[nr] (double) | row_dx[nr]
  double* const s_row_x = smem_a4;
  float* const s_row_dx = (float*)(s_row_x + nr);
  for (int r = threadIdx.x; r < nr; r += blockDim.x) {
    s_row_x[r] = g.row_x[r];
    s_row_dx[r] = g.row_dx[r];
  }
  __syncthreads();
  // few seeds (one small event): spread them over all warps instead of filling the first warps' 32 lanes
  const uint32_t n_warps = gridDim.x * (blockDim.x >> 5);
  const int lanes_used = (int)min(32u, (n_seeds + n_warps - 1) / n_warps);

  int phase = PH_IDLE;
  bool exhausted = false;
  int i = -1, sec_base = 0, r0 = 0, row = 0, nh = 0, miss = 0, lowest = 0, rmin = 0, rmax = 0;
  bool more = false;   // the chain has a further hit (its record is in rcn)
  int org_z = 0;
  bool fail_dn = false;
  float chi2 = 0.f;
  int32_t* tab = tl_hits;   // this tracklet's row -> hit id table
  int2* yz = tl_yz;         // and its row -> (y, z) stream for the downward refit
  State p;
  Cov C;
  p.y = p.z = p.s = p.t = p.q = 0; p.oy = p.oz = 0;
  cov_reset(g, C);
  // gathers issued one step ahead (a mismatch of the tag only costs the direct load)
  Rec rcn = {0, 0, -1, -1};        // srt record of the next chain hit
  int s1_row = -1, s1_y = YZ_NONE, s1_z = 0;   // stream entries of the next two rows on the way down
  int s2_row = -1, s2_y = YZ_NONE, s2_z = 0;
  uint32_t pk_y = 0xFFFFFFFFu, pk_z = 0xFFFFFFFFu;   // bin ranges of the window keyed (pk_y, pk_z)
  BinRanges pq = {0, 0, 0, 0};

  while (true) {
    uint32_t nk_y, nk_z;   // next step's window key and bin ranges (loaded during this step)
    BinRanges npq;
    // ---- refill free lanes from the seed queue ----
    const bool want = phase == PH_IDLE && lane < lanes_used && !exhausted;
    const unsigned idle = __ballot_sync(FULL, want);
    if (idle) {
      uint32_t base = 0;
      if (lane == 0) base = atomicAdd(&ctl->next_seed, (uint32_t)__popc(idle));
      base = __shfl_sync(FULL, base, 0);
      if (base + (uint32_t)__popc(idle) >= n_seeds) exhausted = true;
      const uint32_t k = base + (uint32_t)__popc(idle & ((1u << lane) - 1u));
      if (want && k < n_seeds) {
        // P19: state from the first two chain hits; the INIT step resets C and updates with the first hit
        i = (int)k;
        const int h = seed_pos[k];
        const int sr = seed_sr[k];
        const int sec = sr / nr;
        sec_base = sec * nr;
        r0 = sr - sec_base;
        org_z = zmin_from_key(sec_key[sec]);
        tab = tl_hits + (size_t)k * nr;
        yz = tl_yz + (size_t)k * ((nr + 3) & ~3);   // groups of four rows are 32-byte aligned (a4_phases.cu)
        const int up0 = clean_up[h];
        const int4 c0 = srt[h];
        const int4 c1 = srt[up0];
        rcn.y = c0.x; rcn.z = c0.y; rcn.id = c0.z; rcn.up = up0;
        more = true;
        const int y0 = c0.x, z0 = c0.y;
        const float dxr = s_row_dx[r0];
        const float dy = (float)(c1.x - y0) * g.inv_units, dz = (float)(c1.y - z0) * g.inv_units;
        const float ichord = rsqrtf(fmaf(dxr, dxr, dy * dy));
        p.y = 0; p.z = 0; p.s = dy * ichord; p.t = dz * ichord; p.q = 0;
        p.oy = y0; p.oz = z0;
        row = rmin = rmax = lowest = r0;
        nh = 0; miss = 0; chi2 = 0.f; fail_dn = false;
        s1_row = s2_row = -1;
        pk_y = pk_z = 0xFFFFFFFFu;
        phase = PH_INIT;
      }
    }
    if (!__any_sync(FULL, phase != PH_IDLE)) break;

    // ---- phase transitions that need no work ----
    if (phase == PH_A && !more) phase = PH_B;                                                      // chain ended
    if (phase == PH_B && !(row + 1 < nr && miss < g.max_miss)) phase = PH_CS;                      // P20
    if (phase == PH_CD && (row == 0 || (row - 1 < r0 && miss >= g.max_miss))) phase = PH_FIN;      // P20
    const int ph = phase;

    // ---- what this step does ----
    if (ph == PH_CS) { chi2 = 0.f; miss = 0; lowest = r0; }
    if (ph == PH_INIT || ph == PH_CS) cov_reset(g, C);                                             // P19, P22
    const int dir = (ph == PH_A || ph == PH_B) ? 1 : (ph == PH_CD ? -1 : 0);
    int trow = row + dir;
    bool tr = dir != 0;
    float dx = 0.f;
    if (dir > 0) dx = s_row_dx[row];
    if (dir < 0) dx = -s_row_dx[row - 1];
    int mode = M_NONE;
    if (ph == PH_INIT || ph == PH_A) mode = M_LINK;
    if (ph == PH_B || (ph == PH_CD && trow < r0)) mode = M_SEARCH;
    if (ph == PH_CS || (ph == PH_CD && trow >= r0)) mode = M_TABLE;
    if (ph == PH_FIN && !fail_dn && lowest != row) {   // P23: back to the lowest-row hit, no update
      tr = true;
      trow = lowest;
      dx = (float)(s_row_x[lowest] - s_row_x[row]);
    }

    // ---- hit known before the transport (chain link or recorded hit) ----
    int hid = -1, hy = YZ_NONE, hz = 0;
    const Rec rc = rcn;
    if (mode == M_LINK) {
      hid = rc.id;
      hy = rc.y;
      hz = rc.z;
    }
    ld_rec_if(rcn, srt + rc.up, clean_up + rc.up, mode == M_LINK && rc.up >= 0);   // the next chain hit, one step ahead
    if (mode == M_TABLE) {
      // rolling two-deep pipeline over the tracklet's (y, z) stream on the way down
      ld_cg_yz_if(s1_y, s1_z, yz + trow, s1_row != trow);
      hy = s1_y;
      hz = s1_z;
      hid = hy != YZ_NONE ? 0 : -1;   // the id is not needed on the way down
      const int n1 = trow - 1, n2 = trow - 2;
      const bool have1 = s2_row == n1;
      s1_y = s2_y;
      s1_z = s2_z;
      s1_row = n1 >= r0 ? n1 : -1;
      ld_cg_yz_if(s1_y, s1_z, yz + n1, !have1 && n1 >= r0);
      s2_row = n2 >= r0 ? n2 : -1;
      ld_cg_yz_if(s2_y, s2_z, yz + n2, n2 >= r0);
    }
    // candidates of this step's search: their bin ranges were loaded during the last step; touch them now
    const uint32_t* bs = bin_start + (size_t)(sec_base + trow) * g.nb_stride;
    if (mode == M_SEARCH && (pk_z >> 24) == (uint32_t)trow) {
      if (pq.b0 > pq.a0) prefetch_l1(srt + pq.a0);
      if (pq.b1 > pq.a1) prefetch_l1(srt + pq.a1);
    }
    // bin ranges of the NEXT step's search window, at the position extrapolated from the state before this step
    // (issued here so that this step's transport and update hide the latency; ptxas waits for loads that are in
    // flight at the loop's back edge, so nothing may be issued at the end of the body)
    {
      int nrow = -1;
      if (((ph == PH_A && rc.up < 0) || ph == PH_B) && trow + 1 < nr) nrow = trow + 1;
      if ((ph == PH_CS || ph == PH_CD) && trow - 1 < r0 && trow >= 1) nrow = trow - 1;
      const bool pred = nrow >= 0;
      const int srow = pred ? nrow : row;
      const float ndx = (float)(s_row_x[srow] - s_row_x[row]);
      const float ps = p.s;
      const float ic = rsqrtf(fmaxf(1.f - ps * ps, 0.05f)) * g.units;
      const float py = p.y + ndx * ps * ic, pz = p.z + ndx * p.t * ic;
      const Window w = search_window(g, py, pz, C.var_y() + g.sy2, C.var_z() + g.sz2, p.oy, p.oz, org_z);
      BinRanges nq = pq;
      load_ranges_if(g, bin_start + (size_t)(sec_base + srow) * g.nb_stride, w, nq, pred);
      nk_y = pred ? w.key_y() : pk_y;
      nk_z = pred ? w.key_z(nrow) : pk_z;
      npq = nq;
    }

    bool ok = ph != PH_IDLE && ph != PH_DONE;
    if (ok && tr) ok = transport<true>(g, dx, p, C);
    if (ok) {
      row = trow;
      float ym = resid_y(g, p, hy), zm = resid_z(g, p, hz);   // residuals of the hit, cm
      if (mode == M_SEARCH) {
        const float vy = C.var_y() + g.sy2, vz = C.var_z() + g.sz2;
        const Window w = search_window(g, p.y, p.z, vy, vz, p.oy, p.oz, org_z);
        Found f;
        f.id = -1;
        f.ry = f.rz = 0.f;
        f.hy = f.hz = 0;
        float bestd = __int_as_float(0x7f800000);
        const float wy = 1.f / vy, wz = 1.f / vz;
        if (w.iz_hi <= w.iz_lo + 1) {   // always so on the coarse grid (bins >= 2 gate_z wide)
          BinRanges q = pq;
          load_ranges_if(g, bs, w, q, w.key_y() != pk_y || w.key_z(row) != pk_z);
          search_ranges(g, q, p, wy, wz, srt, f, bestd);
        } else {   // refined grid (dense call) and a wide gate: two z-bin rows at a time
          for (int iz = w.iz_lo; iz <= w.iz_hi; iz += 2) {
            Window w2 = w;
            w2.iz_lo = iz;
            w2.iz_hi = min(iz + 1, w.iz_hi);
            BinRanges q2 = {0, 0, 0, 0};
            load_ranges_if(g, bs, w2, q2, true);
            search_ranges(g, q2, p, wy, wz, srt, f, bestd);
          }
        }
        if (!(bestd < g.gate_d)) f.id = -1;   // P21
        hid = f.id;
        ym = f.ry;
        zm = f.rz;
        tab[row] = hid;
        if (ph == PH_B) yz[row] = make_int2(hid >= 0 ? f.hy : YZ_NONE, f.hz);
        rmin = min(rmin, row);
        rmax = max(rmax, row);
        if (hid >= 0) {
          ++nh;
          miss = 0;
          if (ph == PH_CD) lowest = row;
        } else {
          ++miss;
        }
      } else if (mode == M_LINK) {
        tab[row] = hid;
        yz[row] = make_int2(hy, hz);
        rmax = row;
        ++nh;
        more = rc.up >= 0;
      }
      if (mode != M_NONE && hid >= 0) chi2 += update(g, p, C, ym, zm);
      if (ph == PH_INIT) phase = PH_A;
      if (ph == PH_CS) phase = PH_CD;
      if (ph == PH_FIN) phase = PH_DONE;
    } else {
      // transport failed (P18): the state stays where it is
      if (ph == PH_A || ph == PH_B) phase = PH_CS;
      if (ph == PH_CD) { fail_dn = true; phase = PH_FIN; }
      if (ph == PH_FIN) phase = PH_DONE;
    }

    pk_y = nk_y;
    pk_z = nk_z;
    pq = npq;

    // ---- tracklets that ended: record, visited span and ownership votes ----
    const unsigned done = __ballot_sync(FULL, phase == PH_DONE);
    if (done) {
      if (phase == PH_DONE) {
        float4* o = tl_rec + (size_t)i * TL_REC_V4;
        o[0] = make_float4((float)s_row_x[row], (float)(((double)p.y + (double)p.oy) * g.inv_units_d),
                           (float)(((double)p.z + (double)p.oz) * g.inv_units_d), (float)p.s);
        o[1] = make_float4((float)p.t, (float)p.q, chi2, __int_as_float(nh));
        float cv[15];
        C.lower(cv);
        o[2] = make_float4(cv[0], cv[1], cv[2], cv[3]);
        o[3] = make_float4(cv[4], cv[5], cv[6], cv[7]);
        o[4] = make_float4(cv[8], cv[9], cv[10], cv[11]);
        o[5] = make_float4(cv[12], cv[13], cv[14], __int_as_float(sec_base + r0));
        tl_span[i] = (uint32_t)rmin | ((uint32_t)rmax << 8);   // the rows outside hold nothing: a5 masks by the span
      }
      __syncwarp();   // the table entries of the ending lanes are visible to the whole warp
      unsigned dm = done;
      while (dm) {
        const int src = __ffs(dm) - 1;
        dm &= dm - 1;
        const int si = __shfl_sync(FULL, i, src), snh = __shfl_sync(FULL, nh, src);
        const int smin = __shfl_sync(FULL, rmin, src), smax = __shfl_sync(FULL, rmax, src);
        // P24, P26: owner(h) = surviving tracklet with the most hits, ties -> smallest rank
        const uint32_t word = snh >= g.n_min_tracklet ? (((uint32_t)snh << 24) | (0xFFFFFFu - (uint32_t)si)) : 0u;
        int32_t* out = tl_hits + (size_t)si * nr;
        int v[8];   // n_rows <= 255: all loads of the table first, then the votes
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int r = k * 32 + lane;
          v[k] = -1;
          ld_cg_s32_if(v[k], out + r, r >= smin && r <= smax);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int r = k * 32 + lane;
          if (word && v[k] >= 0) atomicMax(&owner[v[k]], word);
        }
      }
      if (phase == PH_DONE) phase = PH_IDLE;
    }
  }
}

}  // namespace

static size_t a4_smem_bytes(const DevGeom& g) { return (size_t)g.n_rows * (8 + 4); }

cudaError_t setup_a4_attributes(tpc_tracker* t) {
  int sms = 0;
  cudaError_t e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, t->device);
  if (e != cudaSuccess) return e;
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, a4_follow_kernel, A4_THREADS, a4_smem_bytes(t->g));
  if (e != cudaSuccess) return e;
  t->a4_sms = sms;
  t->a4_blocks = per_sm * sms;   // persistent grid: every resident warp slot of the device
  return t->a4_blocks > 0 ? cudaSuccess : cudaErrorInvalidConfiguration;
}

cudaError_t launch_a4_follow(const tpc_tracker* t, int64_t n, cudaStream_t st) {
  if (n == 0 || t->s_cap == 0) return cudaSuccess;
  a4_follow_kernel<<<t->a4_blocks, A4_THREADS, a4_smem_bytes(t->g), st>>>(
      t->g, t->s.ctl, t->s.srt, t->s.clean_up, t->s.sec_key, t->s.bin_start, t->s.seed_pos, t->s.seed_sr, t->s.tl_rec, t->s.tl_hits,
      t->s.tl_yz, t->s.tl_span, t->s.owner);
  return cudaGetLastError();
}
