// a4_phases.cu -- stage a4 as four phase-specialised persistent kernels (same arithmetic, same results as
// a4_follow.cu).  In the single uniform kernel every warp pays for the row search in every
// step although only ~7 of its 32 lanes search; here the tracklets of one phase run together:
//   A  P19 state + fit up the seed chain          (no search: transport + update, next chain record a step ahead)
//   B  extend up with the gated search            (every live lane searches)
//   C  covariance reset + refit down to the seed's first row over the recorded hits (no search)
//   D  extend down with the search, final transport, tracklet record, table padding and ownership votes
// Between two phases a tracklet's filter state is parked in HBM (128 bytes) and its seed rank is pushed into the next
// phase's queue; a kernel boundary separates producers and consumers, so the queues need no flags or fences.
#include "tpc_internal.cuh"
#include "a4_search.cuh"

namespace {

constexpr int AP_THREADS = 128;
constexpr int A4_REFILL_MIN = 8;   // free lanes a warp collects before it refills (4: +2 % a4 time, 16: equal)
enum : int { Q_B = 0, Q_C = 1, Q_D = 2 };

struct Env {   // everything a warp needs that does not change during a kernel
  DevGeom g;
  DevCtl* ctl;
  const int4* srt;
  const int32_t* clean_up;   // a3: cleaned up link of every sorted position
  const uint32_t* sec_key;
  const uint32_t* bin_start;
  const int4* seed_rec;
  float4* tl_rec;
  int32_t* tl_hits;
  int2* tl_yz;
  int4* tl_state;
  uint32_t* q_items;
  uint32_t* tl_span;
  const double* s_row_x;   // shared-memory copies
  const float* s_row_dx;
  int2* s_yz;              // this lane's staging column for the (y, z) stream: slot k at s_yz[k * AP_THREADS]
  int* s_tab;              // likewise for the hit table: eight rows = one 32-byte group
  uint32_t* q_buf;         // this warp's collected queue items [2 slots][A4_Q_BUCKETS][A4_Q_BATCH] and their counts
  int* q_cnt;
  bool tab_groups;         // n_rows is a multiple of 8: every aligned group of eight rows lies inside the tracklet's table
  float bucket_scale;      // A4_Q_BUCKETS / n_rows
  int yz_stride;           // entries per tracklet in tl_yz: n_rows rounded up to a multiple of 4 (32-byte groups)
  uint32_t n_seeds, s_cap;
  int lane, lanes_used;
};

struct Trk {   // per-tracklet constants, recomputed from the seed rank when a lane picks the tracklet up
  int i, id0, y0, z0, up0, sec_base, r0, org_z;   // (y0, z0, id0, up0): the seed's first cluster (its srt record)
  int y1, z1;     // the seed's second cluster (P19 initial direction); valid in phase A only
  int32_t* tab;   // its row -> hit id table = its final hit list
  int2* yz;       // its row -> (y, z) of the recorded hit: what the downward refit streams
};

__device__ __forceinline__ Trk trk_of(const Env& e, int i) {
  Trk t;
  t.i = i;
  const int4 q0 = e.seed_rec[2 * i], q1 = e.seed_rec[2 * i + 1];   // one 32-byte sector (a3_rank_kernel)
  const int sr = q0.x;
  const int sec = sr / e.g.n_rows;
  t.sec_base = sec * e.g.n_rows;
  t.r0 = sr - t.sec_base;
  t.org_z = zmin_from_key(e.sec_key[sec]);
  t.tab = e.tl_hits + (size_t)i * e.g.n_rows;
  t.yz = e.tl_yz + (size_t)i * e.yz_stride;
  t.y0 = q0.y;
  t.z0 = q0.z;
  t.id0 = q0.w;
  t.up0 = q1.x;
  t.y1 = q1.y;
  t.z1 = q1.z;
  return t;
}

struct Book {   // bookkeeping that travels with the filter state
  int row, nh, miss, lowest, rmin, rmax;
  bool fail_dn;
  float chi2;
};

__device__ __forceinline__ void state_save(const Env& e, const Trk& t, const State& p, const Cov& C, const Book& b) {
  float4* f = (float4*)(e.tl_state + (size_t)t.i * A4_STATE_V4);
  f[0] = make_float4(C.d0, C.d1, C.d2, C.d3);
  f[1] = make_float4(C.d4, C.u01, C.u02, C.u03);
  f[2] = make_float4(C.u04, C.u12, C.u13, C.u14);
  f[3] = make_float4(C.u23, C.u24, C.u34, p.y);
  f[4] = make_float4(p.z, p.s, p.t, p.q);
  f[5] = make_float4(b.chi2, __int_as_float(b.row), __int_as_float(b.nh), __int_as_float(b.miss));
  f[6] = make_float4(__int_as_float(b.lowest), __int_as_float(b.rmin | (b.rmax << 8) | (b.fail_dn ? 1 << 16 : 0)),
                     0.f, 0.f);
  ((int4*)f)[7] = make_int4(p.oy, p.oz, t.sec_base + t.r0, t.org_z);   // so that the next phase needs one gather level
}

__device__ __forceinline__ void state_load(const Env& e, int i, Trk& t, State& p, Cov& C, Book& b) {
  const float4* f = (const float4*)(e.tl_state + (size_t)i * A4_STATE_V4);
  const float4 f0 = f[0], f1 = f[1], f2 = f[2], f3 = f[3], f4 = f[4], f5 = f[5], f6 = f[6];
  const int4 o = ((const int4*)f)[7];
  t.i = i;
  t.y0 = p.oy = o.x;
  t.z0 = p.oz = o.y;
  t.sec_base = (o.z / e.g.n_rows) * e.g.n_rows;
  t.r0 = o.z - t.sec_base;
  t.org_z = o.w;
  t.tab = e.tl_hits + (size_t)i * e.g.n_rows;
  t.yz = e.tl_yz + (size_t)i * e.yz_stride;
  t.id0 = t.up0 = -1;
  t.y1 = t.z1 = 0;
  C.d0 = f0.x; C.d1 = f0.y; C.d2 = f0.z; C.d3 = f0.w; C.d4 = f1.x; C.u01 = f1.y; C.u02 = f1.z; C.u03 = f1.w;
  C.u04 = f2.x; C.u12 = f2.y; C.u13 = f2.z; C.u14 = f2.w; C.u23 = f3.x; C.u24 = f3.y; C.u34 = f3.z;
  p.y = f3.w; p.z = f4.x; p.s = f4.y; p.t = f4.z; p.q = f4.w;
  b.chi2 = f5.x;
  b.row = __float_as_int(f5.y);
  b.nh = __float_as_int(f5.z);
  b.miss = __float_as_int(f5.w);
  b.lowest = __float_as_int(f6.x);
  const int pk = __float_as_int(f6.y);
  b.rmin = pk & 0xff;
  b.rmax = (pk >> 8) & 0xff;
  b.fail_dn = (pk >> 16) & 1;
}

// Length bucket of a tracklet entering a phase: the rows it has left to cover.  Longest first (bucket 0), so that
// the tail of each phase kernel consists of short tracklets.
__device__ __forceinline__ int len_bucket(const Env& e, int rows_left) {
  // evaluated by every lane in every step: a multiplication, not an integer division (the bucket only orders the work)
  const int b = (A4_Q_BUCKETS - 1) - __float2int_rz((float)min(max(rows_left, 0), e.g.n_rows - 1) * e.bucket_scale);
  return b < 0 ? 0 : b;
}

// Producer side (lanes with pred, after state_save).  A warp collects the items it produces per (queue, bucket) in
// shared memory and hands them over A4_Q_BATCH at a time: the fetch-add that claims their place in the queue -- a
// round trip the warp waits for -- is paid once per batch instead of in every step in which a lane leaves.
constexpr int A4_Q_BATCH = 16;

__device__ __forceinline__ void queue_flush(const Env& e, int q, int slot, int bk) {
  const int n = e.q_cnt[slot * A4_Q_BUCKETS + bk];
  if (n == 0) return;   // warp-uniform
  const int qq = q * A4_Q_BUCKETS + bk;
  uint32_t base = 0;
  if (e.lane == 0) base = atomicAdd(&e.ctl->q_alloc[qq].v, (uint32_t)n);
  base = __shfl_sync(0xffffffffu, base, 0);
  if (e.lane < n)
    e.q_items[(size_t)qq * e.s_cap + base + e.lane] = e.q_buf[(slot * A4_Q_BUCKETS + bk) * A4_Q_BATCH + e.lane];
  __syncwarp();
  if (e.lane == 0) e.q_cnt[slot * A4_Q_BUCKETS + bk] = 0;
  __syncwarp();
}

// slot: which of the phase's destination queues (0, or 1 for phase A's second one)
__device__ __forceinline__ void queue_push(const Env& e, int q, int slot, int bucket, int i, bool pred) {
  unsigned todo = __ballot_sync(0xffffffffu, pred);
  while (todo) {   // one round per distinct bucket among the leaving lanes (usually one or two)
    const int bk = __shfl_sync(0xffffffffu, bucket, __ffs(todo) - 1);
    const bool mine = pred && bucket == bk;
    const unsigned m = __ballot_sync(0xffffffffu, mine);
    const int cell = slot * A4_Q_BUCKETS + bk;
    int done = 0;   // items of this round already stored
    const int total = __popc(m), rank = __popc(m & ((1u << e.lane) - 1u));
    while (done < total) {   // at most three rounds (32 lanes, batches of 16)
      const int have = e.q_cnt[cell];
      const int take = min(total - done, A4_Q_BATCH - have);
      if (mine && rank >= done && rank < done + take) e.q_buf[cell * A4_Q_BATCH + have + rank - done] = (uint32_t)i;
      __syncwarp();
      if (e.lane == 0) e.q_cnt[cell] = have + take;
      __syncwarp();
      done += take;
      if (have + take == A4_Q_BATCH) queue_flush(e, q, slot, bk);
    }
    todo &= ~m;
  }
}

// before a warp leaves a phase kernel: everything it still holds
__device__ __forceinline__ void queue_flush_all(const Env& e, int q0, int q1) {
  for (int bk = 0; bk < A4_Q_BUCKETS; ++bk) {
    queue_flush(e, q0, 0, bk);
    if (q1 >= 0) queue_flush(e, q1, 1, bk);
  }
}

// Consumer side: the queues are complete (their producers ran in earlier launches); a claim is one fetch-add.
// `bk` is the bucket the warp currently drains (warp-uniform); `dry` is set once the last bucket ran out.
__device__ __forceinline__ int queue_pop(const Env& e, int q, unsigned want, bool mine, int* bk, bool* dry) {
  int i = -1;
  unsigned w = want;
  while (w && *bk < A4_Q_BUCKETS) {   // warp-uniform loop
    const int qq = q * A4_Q_BUCKETS + *bk;
    const uint32_t total = e.ctl->q_alloc[qq].v;
    uint32_t base = 0;
    if (e.lane == 0) base = atomicAdd(&e.ctl->q_head[qq].v, (uint32_t)__popc(w));
    base = __shfl_sync(0xffffffffu, base, 0);
    const uint32_t k = base + (uint32_t)__popc(w & ((1u << e.lane) - 1u));
    const bool got = mine && i < 0 && ((w >> e.lane) & 1u) && k < total;
    if (got) i = (int)e.q_items[(size_t)qq * e.s_cap + k];
    const uint32_t claimed = (uint32_t)__popc(w);
    w &= ~__ballot_sync(0xffffffffu, got);
    if (base + claimed >= total) ++*bk;   // this bucket is empty now: move on to the next
  }
  *dry = *bk >= A4_Q_BUCKETS;
  return i;
}

// The (y, z) stream of a tracklet (tl_yz) is written through a four-row staging column in shared memory, one
// aligned 32-byte group per store: single 8-byte stores made the two upward phases ~25 % slower, because every
// partially written sector is first filled from DRAM (measured: +9 B of DRAM reads per step).  A group may carry
// stale slots for rows the phase did not visit: rows below the seed's first row and above the last visited row
// are never read (phase C runs from the last visited row down to the seed's first row).
__device__ __forceinline__ void yz_stage(const Env& e, int row, int y, int z) {
  e.s_yz[(row & 3) * AP_THREADS] = make_int2(y, z);
}
// rows [first, row] of the group of `row` are staged; rows below `first` belong to an earlier phase and must stay
__device__ __forceinline__ void yz_flush(const Env& e, const Trk& t, int row, int first) {
  const int base = row & ~3;
  if (base >= first) {
    const int2 v0 = e.s_yz[0], v1 = e.s_yz[AP_THREADS], v2 = e.s_yz[2 * AP_THREADS], v3 = e.s_yz[3 * AP_THREADS];
    int4* dst = (int4*)(t.yz + base);
    dst[0] = make_int4(v0.x, v0.y, v1.x, v1.y);
    dst[1] = make_int4(v2.x, v2.y, v3.x, v3.y);
  } else {
    for (int r = first; r <= row; ++r) t.yz[r] = e.s_yz[(r & 3) * AP_THREADS];
  }
}

// The hit table (4-byte entries) goes through an eight-row staging column in the same way, for the same reason.
// Stale slots of a group land in rows the phase did not visit: a later phase that visits them rewrites them (it
// stores row by row inside a group it shares with an earlier phase), and rows no phase visits lie outside
// [rmin, rmax] and are padded with -1 by the votes kernel.
__device__ __forceinline__ void tab_stage(const Env& e, int row, int id) { e.s_tab[(row & 7) * AP_THREADS] = id; }
__device__ __forceinline__ void tab_store_group(const Env& e, const Trk& t, int base) {
  const int* c = e.s_tab;
  int4* dst = (int4*)(t.tab + base);
  dst[0] = make_int4(c[0], c[AP_THREADS], c[2 * AP_THREADS], c[3 * AP_THREADS]);
  dst[1] = make_int4(c[4 * AP_THREADS], c[5 * AP_THREADS], c[6 * AP_THREADS], c[7 * AP_THREADS]);
}
// upward phases: rows [first, row] of the group of `row` are staged; rows below `first` are an earlier phase's
__device__ __forceinline__ void tab_flush_up(const Env& e, const Trk& t, int row, int first) {
  const int base = row & ~7;
  if (e.tab_groups && base >= first) {
    tab_store_group(e, t, base);
  } else {
    for (int r = max(first, base); r <= row; ++r) t.tab[r] = e.s_tab[(r & 7) * AP_THREADS];
  }
}
// downward phase: rows [row, last] of the group of `row` are staged; rows above `last` are an earlier phase's
__device__ __forceinline__ void tab_flush_down(const Env& e, const Trk& t, int row, int last) {
  const int base = row & ~7;
  if (e.tab_groups && base + 7 <= last) {
    tab_store_group(e, t, base);
  } else {
    for (int r = row; r <= min(last, base + 7); ++r) t.tab[r] = e.s_tab[(r & 7) * AP_THREADS];
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Phase A: P19 initial state + fit up the seed chain, no gate.  Items = seed ranks from ctl->next_seed.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void phase_a(const Env& e) {
  const unsigned FULL = 0xffffffffu;
  const DevGeom& g = e.g;
  bool live = false, first = false, exhausted = false;
  Trk t = {};
  Book b = {};
  State p;
  Cov C;
  p.y = p.z = p.s = p.t = p.q = 0; p.oy = p.oz = 0;
  cov_reset(g, C);
  Rec rcn = {0, 0, -1, -1};   // the chain hit of the next step (requested one step ahead: its record and its link)
  bool more = false;          // rcn holds a chain hit
  bool dirty = false;         // the staging column holds rows that are not in tl_yz yet
  bool dirty_t = false;       // likewise for the hit table
  while (true) {
    const bool want = !live && e.lane < e.lanes_used && !exhausted;
    const unsigned idle = __ballot_sync(FULL, want);
    // refill in batches: a refill stalls the warp for its gathers, so wait until several lanes are free
    if (idle && (__popc(idle) >= A4_REFILL_MIN || !__any_sync(FULL, live))) {
      uint32_t base = 0;
      if (e.lane == 0) base = atomicAdd(&e.ctl->next_seed, (uint32_t)__popc(idle));
      base = __shfl_sync(FULL, base, 0);
      if (base + (uint32_t)__popc(idle) >= e.n_seeds) exhausted = true;
      const uint32_t k = base + (uint32_t)__popc(idle & ((1u << e.lane) - 1u));
      if (want && k < e.n_seeds) {
        t = trk_of(e, (int)k);
        rcn.y = t.y0; rcn.z = t.z0; rcn.id = t.id0; rcn.up = t.up0;
        more = true;
        const float dxr = e.s_row_dx[t.r0];
        const float dy = (float)(t.y1 - t.y0) * g.inv_units, dz = (float)(t.z1 - t.z0) * g.inv_units;
        const float ichord = rsqrtf(fmaf(dxr, dxr, dy * dy));
        p.y = 0; p.z = 0; p.s = dy * ichord; p.t = dz * ichord; p.q = 0;
        p.oy = t.y0; p.oz = t.z0;
        b.row = b.rmin = b.rmax = b.lowest = t.r0;
        b.nh = 0; b.miss = 0; b.chi2 = 0.f; b.fail_dn = false;
        first = true;
        live = true;
      }
    }
    if (!__any_sync(FULL, live)) {
      queue_flush_all(e, Q_B, Q_C);
      return;
    }

    if (live && first) cov_reset(g, C);   // P19
    const bool tr = live && !first;
    const int trow = b.row + (tr ? 1 : 0);
    const float dx = e.s_row_dx[b.row];
    const Rec rc = rcn;
    ld_rec_if(rcn, e.srt + rc.up, e.clean_up + rc.up, live && rc.up >= 0);   // the next chain hit, one step ahead
    bool ok = live;
    if (tr) ok = transport<true>(g, dx, p, C);
    if (ok) {
      b.row = trow;
      update(g, p, C, resid_y(g, p, rc.y), resid_z(g, p, rc.z));
      tab_stage(e, trow, rc.id);
      yz_stage(e, trow, rc.y, rc.z);
      dirty = true;
      dirty_t = true;
      b.rmax = trow;
      ++b.nh;
      more = rc.up >= 0;
      first = false;
    }
    // the chain ended, or the transport failed (P18; then phase B is skipped)
    const bool leave = live && (!ok || !more);
    if (dirty && ((b.row & 3) == 3 || leave)) {
      yz_flush(e, t, b.row, 0);   // rows of the group below the seed's first row are never read: whole groups
      dirty = false;
    }
    if (dirty_t && ((b.row & 7) == 7 || leave)) {
      tab_flush_up(e, t, b.row, 0);
      dirty_t = false;
    }
    if (leave) state_save(e, t, p, C, b);
    const bool to_b = leave && ok && b.row + 1 < g.n_rows;
    queue_push(e, Q_B, 0, len_bucket(e, g.n_rows - 1 - b.row), t.i, to_b);
    queue_push(e, Q_C, 1, len_bucket(e, b.row - t.r0), t.i, leave && !to_b);
    if (leave) live = false;
  }
}

// Search step shared by phases B and D (P17, P21): exact window after the transport, bin ranges from the prediction
// when it matches, candidates.
__device__ __forceinline__ Found search_step(const Env& e, const Trk& t, const State& p, const Cov& C, int row,
                                             uint32_t pk_y, uint32_t pk_z, const BinRanges& pq) {
  const DevGeom& g = e.g;
  const float vy = C.var_y() + g.sy2, vz = C.var_z() + g.sz2;
  const Window w = search_window(g, p.y, p.z, vy, vz, p.oy, p.oz, t.org_z);
  const uint32_t* bs = e.bin_start + (size_t)(t.sec_base + row) * g.nb_stride;
  Found f;
  f.id = -1;
  f.ry = f.rz = 0.f;
  f.hy = f.hz = 0;
  float bestd = __int_as_float(0x7f800000);
  const float wy = 1.f / vy, wz = 1.f / vz;
  if (w.iz_hi <= w.iz_lo + 1) {   // always so on the coarse grid
    BinRanges q = pq;
    load_ranges_if(g, bs, w, q, w.key_y() != pk_y || w.key_z(row) != pk_z);
    search_ranges(g, q, p, wy, wz, e.srt, f, bestd);
  } else {   // refined grid and a wide gate: two z-bin rows at a time
    for (int iz = w.iz_lo; iz <= w.iz_hi; iz += 2) {
      Window w2 = w;
      w2.iz_lo = iz;
      w2.iz_hi = min(iz + 1, w.iz_hi);
      BinRanges q2 = {0, 0, 0, 0};
      load_ranges_if(g, bs, w2, q2, true);
      search_ranges(g, q2, p, wy, wz, e.srt, f, bestd);
    }
  }
  if (!(bestd < g.gate_d)) f.id = -1;   // P21
  return f;
}

// Bin ranges of the search window of row `nrow` at the position extrapolated from the state at row `row`
// (requested before the current step's transport so that the step hides the latency).
__device__ __forceinline__ void predict_ranges(const Env& e, const Trk& t, const State& p, const Cov& C, int row,
                                               int nrow, bool pred, uint32_t& nk_y, uint32_t& nk_z, BinRanges& nq) {
  const DevGeom& g = e.g;
  const int srow = pred ? nrow : row;
  const float ndx = (float)(e.s_row_x[srow] - e.s_row_x[row]);
  const float ps = p.s;
  const float ic = rsqrtf(fmaxf(1.f - ps * ps, 0.05f)) * g.units;
  const float py = p.y + ndx * ps * ic, pz = p.z + ndx * p.t * ic;
  const Window w = search_window(g, py, pz, C.var_y() + g.sy2, C.var_z() + g.sz2, p.oy, p.oz, t.org_z);
  load_ranges_if(g, e.bin_start + (size_t)(t.sec_base + srow) * g.nb_stride, w, nq, pred);
  if (pred) {
    nk_y = w.key_y();
    nk_z = w.key_z(nrow);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Phase B: extend up with the gated nearest-hit search (P17, P20, P21).  Every live lane searches in every step.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void phase_b(const Env& e) {
  const unsigned FULL = 0xffffffffu;
  const DevGeom& g = e.g;
  int bk = 0;
  bool live = false, dry = false;
  Trk t = {};
  Book b = {};
  State p;
  Cov C;
  p.y = p.z = p.s = p.t = p.q = 0; p.oy = p.oz = 0;
  cov_reset(g, C);
  uint32_t pk_y = 0xFFFFFFFFu, pk_z = 0xFFFFFFFFu;
  BinRanges pq = {0, 0, 0, 0};
  int fr = 0;           // first row this phase visits for the tracklet (the rows below are phase A's)
  bool dirty = false;   // the staging column holds rows that are not in tl_yz yet
  bool dirty_t = false; // likewise for the hit table
  while (true) {
    const bool want = !live && e.lane < e.lanes_used && !dry;
    const unsigned idle = __ballot_sync(FULL, want);
    // refill in batches: a refill stalls the warp for its gathers, so wait until several lanes are free
    if (idle && (__popc(idle) >= A4_REFILL_MIN || !__any_sync(FULL, live))) {
      const int i = queue_pop(e, Q_B, idle, want, &bk, &dry);
      if (i >= 0) {
        state_load(e, i, t, p, C, b);
        pk_y = pk_z = 0xFFFFFFFFu;
        fr = b.row + 1;
        live = true;
      }
    }
    if (!__any_sync(FULL, live)) {
      queue_flush_all(e, Q_C, -1);
      return;
    }

    const int trow = b.row + 1;   // a live lane always has a row above and fewer than max_miss misses
    const float dx = e.s_row_dx[b.row];
    if (live && (pk_z >> 24) == (uint32_t)trow) {   // this step's first candidates into L1 during the transport
      if (pq.b0 > pq.a0) prefetch_l1(e.srt + pq.a0);
      if (pq.b1 > pq.a1) prefetch_l1(e.srt + pq.a1);
    }
    uint32_t nk_y = pk_y, nk_z = pk_z;
    BinRanges nq = pq;
    predict_ranges(e, t, p, C, b.row, trow + 1, live && trow + 1 < g.n_rows, nk_y, nk_z, nq);
    bool ok = live;
    if (ok) ok = transport<true>(g, dx, p, C);
    if (ok) {
      b.row = trow;
      const Found f = search_step(e, t, p, C, trow, pk_y, pk_z, pq);
      tab_stage(e, trow, f.id);
      yz_stage(e, trow, f.id >= 0 ? f.hy : YZ_NONE, f.hz);
      dirty = true;
      dirty_t = true;
      b.rmax = trow;
      if (f.id >= 0) {
        update(g, p, C, f.ry, f.rz);
        ++b.nh;
        b.miss = 0;
      } else {
        ++b.miss;
      }
    }
    pk_y = nk_y;
    pk_z = nk_z;
    pq = nq;
    const bool leave = live && (!ok || !(b.row + 1 < g.n_rows && b.miss < g.max_miss));   // P18, P20
    if (dirty && ((b.row & 3) == 3 || leave)) {
      yz_flush(e, t, b.row, fr);
      dirty = false;
    }
    if (dirty_t && ((b.row & 7) == 7 || leave)) {
      tab_flush_up(e, t, b.row, fr);
      dirty_t = false;
    }
    if (leave) state_save(e, t, p, C, b);
    queue_push(e, Q_C, 0, len_bucket(e, b.row - t.r0), t.i, leave);
    if (leave) live = false;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Phase C: covariance reset (P22), then refit down over the recorded hits to the seed's first row.  The first step
// of a tracklet (reset + update with the top row's hit) has no transport.  The hits come from the tracklet's own
// (y, z) stream, written row by row on the way up: one sequential 8-byte load per step, requested two rows ahead --
// no gather by cluster id, no table look-up.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void phase_c(const Env& e) {
  const unsigned FULL = 0xffffffffu;
  const DevGeom& g = e.g;
  int bk = 0;
  bool live = false, first = false, dry = false;
  Trk t = {};
  Book b = {};
  State p;
  Cov C;
  p.y = p.z = p.s = p.t = p.q = 0; p.oy = p.oz = 0;
  cov_reset(g, C);
  int s1_row = -1, s1_y = YZ_NONE, s1_z = 0;   // stream entries of this step's row and of the one below
  int s2_row = -1, s2_y = YZ_NONE, s2_z = 0;
  while (true) {
    const bool want = !live && e.lane < e.lanes_used && !dry;
    const unsigned idle = __ballot_sync(FULL, want);
    // refill in batches: a refill stalls the warp for its gathers, so wait until several lanes are free
    if (idle && (__popc(idle) >= A4_REFILL_MIN || !__any_sync(FULL, live))) {
      const int i = queue_pop(e, Q_C, idle, want, &bk, &dry);
      if (i >= 0) {
        state_load(e, i, t, p, C, b);
        s1_row = s2_row = -1;
        first = true;
        live = true;
      }
    }
    if (!__any_sync(FULL, live)) {
      queue_flush_all(e, Q_D, -1);
      return;
    }

    if (live && first) {   // P22
      cov_reset(g, C);
      b.chi2 = 0.f;
      b.miss = 0;
      b.lowest = t.r0;
    }
    const bool tr = live && !first;
    const int trow = b.row - (tr ? 1 : 0);
    const float dx = -e.s_row_dx[max(b.row - 1, 0)];
    int hy = YZ_NONE, hz = 0;
    if (live) {   // rolling two-deep pipeline over the stream on the way down
      ld_ca_yz_if(s1_y, s1_z, t.yz + trow, s1_row != trow);
      hy = s1_y;
      hz = s1_z;
      const int n1 = trow - 1, n2 = trow - 2;
      const bool have1 = s2_row == n1;
      s1_y = s2_y;
      s1_z = s2_z;
      s1_row = n1 >= t.r0 ? n1 : -1;
      ld_ca_yz_if(s1_y, s1_z, t.yz + n1, !have1 && n1 >= t.r0);
      s2_row = n2 >= t.r0 ? n2 : -1;
      ld_ca_yz_if(s2_y, s2_z, t.yz + n2, n2 >= t.r0);
    }
    bool ok = live;
    if (tr) ok = transport<true>(g, dx, p, C);
    if (ok) {
      b.row = trow;
      if (hy != YZ_NONE) b.chi2 += update(g, p, C, resid_y(g, p, hy), resid_z(g, p, hz));
      first = false;
    } else if (live) {
      b.fail_dn = true;   // P18: the state stays at the row where it stopped
    }
    const bool leave = live && (!ok || b.row <= t.r0);   // below the seed's first row phase D searches
    if (leave) state_save(e, t, p, C, b);
    queue_push(e, Q_D, 0, len_bucket(e, b.row), t.i, leave);
    if (leave) live = false;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Phase D: extend down below the seed's first row with the search (P20), then the final transport to the
// lowest-row hit (P23) and the tracklet record.  The padding of the hit tables and the ownership votes (P24, P26)
// are a flat kernel of their own (a4_votes_kernel): a warp per tracklet, 32 rows per instruction.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void phase_d(const Env& e) {
  const unsigned FULL = 0xffffffffu;
  const DevGeom& g = e.g;
  const int nr = g.n_rows;
  int bk = 0;
  bool live = false, dry = false;
  Trk t = {};
  Book b = {};
  State p;
  Cov C;
  p.y = p.z = p.s = p.t = p.q = 0; p.oy = p.oz = 0;
  cov_reset(g, C);
  uint32_t pk_y = 0xFFFFFFFFu, pk_z = 0xFFFFFFFFu;
  BinRanges pq = {0, 0, 0, 0};
  int d_last = 0;         // first (= highest) row this phase visits for the tracklet; the rows above are earlier phases'
  bool dirty_t = false;   // the staging column holds hit-table rows that are not in tl_hits yet
  while (true) {
    const bool want = !live && e.lane < e.lanes_used && !dry;
    const unsigned idle = __ballot_sync(FULL, want);
    // refill in batches: a refill stalls the warp for its gathers, so wait until several lanes are free
    if (idle && (__popc(idle) >= A4_REFILL_MIN || !__any_sync(FULL, live))) {
      const int i = queue_pop(e, Q_D, idle, want, &bk, &dry);
      if (i >= 0) {
        state_load(e, i, t, p, C, b);
        pk_y = pk_z = 0xFFFFFFFFu;
        d_last = b.row - 1;
        live = true;
      }
    }
    if (!__any_sync(FULL, live)) return;

    // search step down, or the final transport once the extension is over
    const bool srch = live && !b.fail_dn && b.row > 0 && b.miss < g.max_miss;
    const bool fin = live && !srch;
    bool tr = srch;
    int trow = b.row - (srch ? 1 : 0);
    float dx = -e.s_row_dx[max(b.row - 1, 0)];
    if (fin && !b.fail_dn && b.lowest != b.row) {   // P23
      tr = true;
      trow = b.lowest;
      dx = (float)(e.s_row_x[b.lowest] - e.s_row_x[b.row]);
    }
    if (srch && (pk_z >> 24) == (uint32_t)trow) {
      if (pq.b0 > pq.a0) prefetch_l1(e.srt + pq.a0);
      if (pq.b1 > pq.a1) prefetch_l1(e.srt + pq.a1);
    }
    uint32_t nk_y = pk_y, nk_z = pk_z;
    BinRanges nq = pq;
    predict_ranges(e, t, p, C, b.row, trow - 1, srch && trow >= 1, nk_y, nk_z, nq);
    bool ok = live;
    if (tr) ok = transport<true>(g, dx, p, C);
    if (ok) b.row = trow;
    if (srch) {
      if (ok) {
        const Found f = search_step(e, t, p, C, trow, pk_y, pk_z, pq);
        tab_stage(e, trow, f.id);
        dirty_t = true;
        if ((trow & 7) == 0) {
          tab_flush_down(e, t, trow, d_last);
          dirty_t = false;
        }
        b.rmin = min(b.rmin, trow);
        if (f.id >= 0) {
          b.chi2 += update(g, p, C, f.ry, f.rz);
          ++b.nh;
          b.miss = 0;
          b.lowest = trow;
        } else {
          ++b.miss;
        }
      } else {
        b.fail_dn = true;
      }
    }
    pk_y = nk_y;
    pk_z = nk_z;
    pq = nq;

    // ---- tracklets that ended: record, padding of the hit table and ownership votes ----
    const unsigned done = __ballot_sync(FULL, fin);
    if (done) {
      if (fin && dirty_t) {   // b.rmin is the lowest row this phase wrote
        tab_flush_down(e, t, b.rmin, d_last);
        dirty_t = false;
      }
      if (fin) {
        float4* o = e.tl_rec + (size_t)t.i * TL_REC_V4;
        o[0] = make_float4((float)e.s_row_x[b.row], (float)(((double)p.y + (double)p.oy) * g.inv_units_d),
                           (float)(((double)p.z + (double)p.oz) * g.inv_units_d), (float)p.s);
        o[1] = make_float4((float)p.t, (float)p.q, b.chi2, __int_as_float(b.nh));
        float cv[15];
        C.lower(cv);
        o[2] = make_float4(cv[0], cv[1], cv[2], cv[3]);
        o[3] = make_float4(cv[4], cv[5], cv[6], cv[7]);
        o[4] = make_float4(cv[8], cv[9], cv[10], cv[11]);
        o[5] = make_float4(cv[12], cv[13], cv[14], __int_as_float(t.sec_base + t.r0));
        e.tl_span[t.i] = (uint32_t)b.rmin | ((uint32_t)b.rmax << 8);
      }
      if (fin) live = false;
    }
  }
}

// P24, P26: owner(h) = surviving tracklet with the most hits, ties -> smallest rank.  Only the rows the tracklet
// visited (tl_span) hold entries; the rest of its table is never written and never read (a5 masks by the span too).
// One warp per tracklet, grid-stride.
__global__ void __launch_bounds__(256)
a4_votes_kernel(const DevGeom g, const DevCtl* __restrict__ ctl, const float4* __restrict__ tl_rec,
                const uint32_t* __restrict__ tl_span, const int32_t* __restrict__ tl_hits,
                uint32_t* __restrict__ owner) {
  const int nr = g.n_rows, lane = threadIdx.x & 31;
  const uint32_t n_seeds = ctl->n_seeds;
  const uint32_t warps = gridDim.x * (blockDim.x >> 5);
  for (uint32_t i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < n_seeds; i += warps) {
    const int nh = __float_as_int(tl_rec[(size_t)i * TL_REC_V4 + 1].w);
    const uint32_t span = tl_span[i];
    const int smin = span & 0xff, smax = (span >> 8) & 0xff;
    const uint32_t word = nh >= g.n_min_tracklet ? (((uint32_t)nh << 24) | (0xFFFFFFu - i)) : 0u;
    if (!word) continue;   // P24: a discarded tracklet casts no vote
    const int32_t* out = tl_hits + (size_t)i * nr;
    for (int r = (smin & ~7) + lane; r <= smax; r += 32) {   // from the 32-byte group that holds the first row
      if (r >= smin) {
        const int v = out[r];
        if (v >= 0) atomicMax(&owner[v], word);
      }
    }
  }
}

// Resident CTAs per SM (measured per phase, profiles/r02_summary.md): the two phases that search run best at 16 warps
// per SM (5 CTAs: B +0.06, D +0.03 ms; 3: slower too), the refit phase, which streams its measurements, at 28 (6 or
// 8 CTAs: +0.01 / +0.03 ms).  The chain fit alone on the GPU is 0.01 ms faster at 20 warps than at 16 (24: +0.03),
// but with a second call on a second stream the step is 0.7 % slower then: 16.
constexpr int ap_min_blocks(int ph) { return ph == 2 ? 7 : 4; }
// CTAs per SM actually launched.  A call that shares the GPU with other calls (K handles on K streams) leaves CTA
// slots to them: with three streams 3 / 4 (C) per SM give 6.42 G clusters/s against 6.21 at 4 / 7, alone 5.32 against
// 5.64 (profiles/r02_summary.md).
constexpr int ap_grid_blocks(int ph, bool shared) { return shared ? (ph == 2 ? 4 : 3) : ap_min_blocks(ph); }

template <int PH>
__global__ void __launch_bounds__(AP_THREADS, ap_min_blocks(PH))
a4_phase_kernel(const DevGeom g, uint32_t s_cap, DevCtl* __restrict__ ctl, const int4* __restrict__ srt,
                const int32_t* __restrict__ clean_up,
                const uint32_t* __restrict__ sec_key, const uint32_t* __restrict__ bin_start,
                const int4* __restrict__ seed_rec, float4* __restrict__ tl_rec, int32_t* __restrict__ tl_hits, int2* __restrict__ tl_yz,
                int4* __restrict__ tl_state, uint32_t* __restrict__ q_items, uint32_t* __restrict__ tl_span) {
  extern __shared__ double smem_ap[];
  __shared__ int2 s_yz[4][AP_THREADS];
  __shared__ int s_tab[8][AP_THREADS];
  __shared__ uint32_t s_qbuf[AP_THREADS / 32][2 * A4_Q_BUCKETS * A4_Q_BATCH];
  __shared__ int s_qcnt[AP_THREADS / 32][2 * A4_Q_BUCKETS];
  const int nr = g.n_rows;
  const uint32_t n_seeds = ctl->n_seeds;
  if (n_seeds == 0) return;
  double* const s_row_x = smem_ap;
  float* const s_row_dx = (float*)(s_row_x + nr);
  for (int r = threadIdx.x; r < nr; r += blockDim.x) {
    s_row_x[r] = g.row_x[r];
    s_row_dx[r] = g.row_dx[r];
  }
  __syncthreads();
  Env e;
  e.g = g;
  e.ctl = ctl; e.srt = srt; e.clean_up = clean_up; e.sec_key = sec_key; e.bin_start = bin_start;
  e.seed_rec = seed_rec; e.tl_rec = tl_rec; e.tl_hits = tl_hits; e.tl_yz = tl_yz;
  e.tl_state = tl_state;
  e.q_items = q_items; e.tl_span = tl_span; e.s_row_x = s_row_x; e.s_row_dx = s_row_dx;
  e.n_seeds = n_seeds; e.s_cap = s_cap;
  e.s_yz = &s_yz[0][threadIdx.x];
  e.s_tab = &s_tab[0][threadIdx.x];
  e.q_buf = &s_qbuf[threadIdx.x >> 5][0];
  e.q_cnt = &s_qcnt[threadIdx.x >> 5][0];
  if ((threadIdx.x & 31) < 2 * A4_Q_BUCKETS) s_qcnt[threadIdx.x >> 5][threadIdx.x & 31] = 0;
  __syncwarp();
  e.tab_groups = (nr & 7) == 0;
  e.yz_stride = (nr + 3) & ~3;
  e.bucket_scale = (float)A4_Q_BUCKETS / (float)nr;
  e.lane = threadIdx.x & 31;
  // few seeds (one small event): spread them over all warps instead of filling the first warps' 32 lanes
  const uint32_t n_warps = gridDim.x * (blockDim.x >> 5);
  e.lanes_used = (int)min(32u, (n_seeds + n_warps - 1) / n_warps);
  if (PH == 0) phase_a(e);
  if (PH == 1) phase_b(e);
  if (PH == 2) phase_c(e);
  if (PH == 3) phase_d(e);
}

}  // namespace

cudaError_t launch_a4_phases(const tpc_tracker* t, int64_t n, cudaStream_t st) {
  if (n == 0 || t->s_cap == 0) return cudaSuccess;
  const size_t smem = (size_t)t->g.n_rows * (8 + 4);
  const bool shared = t->concurrency >= 2;   // tpc_set_concurrency: other calls run next to this one
#define AP_LAUNCH(PH)                                                                                         \
  a4_phase_kernel<PH><<<t->a4_sms * ap_grid_blocks(PH, shared), AP_THREADS, smem, st>>>(                                                \
      t->g, (uint32_t)t->s_cap, t->s.ctl, t->s.srt, t->s.clean_up, t->s.sec_key, t->s.bin_start, t->s.seed_rec, \
      t->s.tl_rec, t->s.tl_hits, t->s.tl_yz, t->s.tl_state, t->s.q_items, t->s.tl_span)
  AP_LAUNCH(0);
  AP_LAUNCH(1);
  AP_LAUNCH(2);
  AP_LAUNCH(3);
#undef AP_LAUNCH
  a4_votes_kernel<<<t->a4_sms * 64, 256, 0, st>>>(t->g, t->s.ctl, t->s.tl_rec, t->s.tl_span, t->s.tl_hits, t->s.owner);
  return cudaGetLastError();
}
