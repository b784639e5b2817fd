// a2_neighbours.cu -- stage a2: neighbour finding (SURVEY 8(c) "Stage 1-2", P5, P7-P10; north_star
// "each cluster links to the best pair of clusters in the adjacent rows").  Integer only -> bit-exact.
//
// For cluster h in row r (1 <= r <= n_rows-2): U = clusters of row r+1 with |dy| <= w_y and |dz| <= w_z,
// D likewise in row r-1; pick the pair minimising (cost, id_u, id_d), cost = cost_wy*(yu+yd-2yh)^2 +
// cost_wz*(zu+zd-2zh)^2; accept iff cost <= c_max.  Ties are broken by cluster id (P9); the links are written in
// SORTED space (the position of the linked cluster in srt), at the sorted position of h: coalesced stores, and a3 / a4
// follow them through the same bin-ordered array the searches read.
// The a1 grid prunes the candidates: bins are at least 2*w wide, so a window touches at most 2 x 2 bins, and
// with y-fastest bin order each z-bin contributes one contiguous range of sorted clusters.
#include "tpc_internal.cuh"

namespace {

constexpr int A2_THREADS = 128;
constexpr int A2_MASK_UNROLL = 2;   // independent loads per trip of the window test

struct Ranges {
  uint32_t a0, b0, a1, b1;   // up to two contiguous sorted ranges (second empty if the window is in one z-bin)
};

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

struct Window {
  int iy_lo, iy_hi, iz_lo, iz_hi;   // inclusive bin ranges
};

// Rows of one sector share the grid shape and origin, so one window serves both neighbour rows.
__device__ __forceinline__ Window window_bins(const DevGeom& g, int yh, int zh, int org_z) {
  Window w;
  w.iy_lo = clampi((yh - g.w_y - g.org_y) >> g.shift_y, 0, g.ny - 1);
  w.iy_hi = clampi((yh + g.w_y - g.org_y) >> g.shift_y, 0, g.ny - 1);
  w.iz_lo = clampi((zh - g.w_z - org_z) >> g.shift_z, 0, g.nz - 1);
  w.iz_hi = clampi((zh + g.w_z - org_z) >> g.shift_z, 0, g.nz - 1);
  return w;
}

// Coarse grid (bins >= 2*w_z wide): the window touches at most two z-bins, both ranges are loaded up front.
__device__ __forceinline__ Ranges load_ranges(const DevGeom& g, const Window& w, const uint32_t* __restrict__ bs) {
  Ranges q;
  q.a0 = bs[w.iz_lo * g.ny + w.iy_lo];
  q.b0 = bs[w.iz_lo * g.ny + w.iy_hi + 1];
  q.a1 = q.b1 = 0;
  if (w.iz_hi != w.iz_lo) {
    q.a1 = bs[w.iz_hi * g.ny + w.iy_lo];
    q.b1 = bs[w.iz_hi * g.ny + w.iy_hi + 1];
  }
  return q;
}

struct Best {   // running best pair: cost and sorted positions (what is stored).  The ids that break cost ties
  int cost, pu, pd;   // (P9) are read back from srt only when a tie happens: one pair in ~1e4
};

// P9 on a cost tie: does the pair (idu, idd) come before the running best in (id_u, id_d) order?
__device__ __forceinline__ bool tie_wins(const int4* __restrict__ srt, const Best& b, int idu, int idd) {
  const int bu = srt[b.pu].z;
  return idu < bu || (idu == bu && idd < srt[b.pd].z);
}

// One candidate pair against the running best (P8, P9).
__device__ __forceinline__ void try_pair(const DevGeom& g, const int4* __restrict__ srt, int dyu, int dzu, int idu,
                                         uint32_t pu, const int4& cd, uint32_t pd, int yh, int zh, Best& b) {
  const int dyd = cd.x - yh, dzd = cd.y - zh;
  if (abs(dyd) > g.w_y || abs(dzd) > g.w_z) return;
  const int ddy = dyu + dyd, ddz = dzu + dzd;
  const int cost = g.cost_wy * ddy * ddy + g.cost_wz * ddz * ddz;
  if (cost > b.cost) return;
  if (cost < b.cost || tie_wins(srt, b, idu, cd.z)) {
    b.cost = cost;
    b.pu = (int)pu;
    b.pd = (int)pd;
  }
}

// The definition's nested scan over the up and down candidates of the window.  FINE: the call refined the grid
// (api.cu: choose_grid), a window may span any number of z-bins and the ranges are read bin row by bin row.
template <bool FINE>
__device__ __forceinline__ void pair_search_nested(const DevGeom& g, const int4* __restrict__ srt, const Window& w,
                                                   const uint32_t* __restrict__ bs_u,
                                                   const uint32_t* __restrict__ bs_d, int yh, int zh, Best& b) {
  if (!FINE) {
    const Ranges qu = load_ranges(g, w, bs_u), qd = load_ranges(g, w, bs_d);
#pragma unroll 1
    for (int pu = 0; pu < 2; ++pu) {
      const uint32_t ua = pu ? qu.a1 : qu.a0, ub = pu ? qu.b1 : qu.b0;
      for (uint32_t u = ua; u < ub; ++u) {
        const int4 cu = srt[u];
        const int dyu = cu.x - yh, dzu = cu.y - zh;
        if (abs(dyu) > g.w_y || abs(dzu) > g.w_z) continue;
#pragma unroll 1
        for (int pd = 0; pd < 2; ++pd) {
          const uint32_t da = pd ? qd.a1 : qd.a0, db = pd ? qd.b1 : qd.b0;
          for (uint32_t d = da; d < db; ++d) try_pair(g, srt, dyu, dzu, cu.z, u, srt[d], d, yh, zh, b);
        }
      }
    }
  } else {
    for (int izu = w.iz_lo; izu <= w.iz_hi; ++izu) {
      const uint32_t ua = bs_u[izu * g.ny + w.iy_lo], ub = bs_u[izu * g.ny + w.iy_hi + 1];
      for (uint32_t u = ua; u < ub; ++u) {
        const int4 cu = srt[u];
        const int dyu = cu.x - yh, dzu = cu.y - zh;
        if (abs(dyu) > g.w_y || abs(dzu) > g.w_z) continue;
        for (int izd = w.iz_lo; izd <= w.iz_hi; ++izd) {
          const uint32_t da = bs_d[izd * g.ny + w.iy_lo], db = bs_d[izd * g.ny + w.iy_hi + 1];
          for (uint32_t d = da; d < db; ++d) try_pair(g, srt, dyu, dzu, cu.z, u, srt[d], d, yh, zh, b);
        }
      }
    }
  }
}

template <bool FINE>
__global__ void __launch_bounds__(A2_THREADS)
a2_neighbours_kernel(const DevGeom g, const DevCtl* __restrict__ ctl, const uint32_t* __restrict__ ro, const int4* __restrict__ srt,
                     const uint32_t* __restrict__ sec_key, const uint32_t* __restrict__ bin_start,
                     int32_t* __restrict__ link_up, int32_t* __restrict__ link_dn) {
  if (ctl->bad_offsets) return;
  const int sr = blockIdx.x;
  const int r = sr % g.n_rows;
  const uint32_t a = ro[sr], b = ro[sr + 1];
  const bool inner = r >= 1 && r <= g.n_rows - 2;   // P5
  const int org_z = zmin_from_key(sec_key[sr / g.n_rows]);
  const uint32_t *bs_u = nullptr, *bs_d = nullptr;
  if (inner) {
    bs_u = bin_start + (size_t)(sr + 1) * g.nb_stride;
    bs_d = bin_start + (size_t)(sr - 1) * g.nb_stride;
  }
  for (uint32_t j = a + threadIdx.x; j < b; j += A2_THREADS) {
    const int4 ch = srt[j];
    const int yh = ch.x, zh = ch.y;
    Best b = {INT32_MAX, -1, -1};
    if (inner) {
      const Window w = window_bins(g, yh, zh, org_z);
      pair_search_nested<FINE>(g, srt, w, bs_u, bs_d, yh, zh, b);
      if (b.pu < 0 || b.cost > g.c_max) b.pu = b.pd = -1;   // P10
    }
    link_up[j] = b.pu;
    link_dn[j] = b.pd;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Sparse and medium rows on the coarse grid (the common case).  In the nested scan a warp pays, per up candidate of
// any lane, the longest down range of any lane, although a lane's own window holds one or two clusters per side.
// Here each side's ranges are tested once, the clusters inside the window become bits of a 32-bit mask (bit t = the
// t-th cluster of the concatenated ranges), and the pair loop visits set bits only.  More than 32 range clusters on
// a side: the nested scan.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t range_at(const Ranges& q, uint32_t n0, uint32_t t) {
  return t < n0 ? q.a0 + t : q.a1 + (t - n0);
}

__device__ __forceinline__ uint32_t side_mask(const DevGeom& g, const int4* __restrict__ srt, const Ranges& q,
                                              uint32_t n0, uint32_t n, int yh, int zh) {
  uint32_t m = 0;
  const uint32_t span_y = 2u * (uint32_t)g.w_y, span_z = 2u * (uint32_t)g.w_z;
  // A2_MASK_UNROLL independent loads per trip (the tail re-reads the last cluster; its bits are masked off)
  for (uint32_t t = 0; t < n; t += A2_MASK_UNROLL) {
    int2 c[A2_MASK_UNROLL];
#pragma unroll
    for (int i = 0; i < A2_MASK_UNROLL; ++i)
      c[i] = *reinterpret_cast<const int2*>(srt + range_at(q, n0, min(t + (uint32_t)i, n - 1u)));
#pragma unroll
    for (int i = 0; i < A2_MASK_UNROLL; ++i) {
      // P7, inclusive: |dy| <= w_y and |dz| <= w_z
      const bool in = (uint32_t)(c[i].x - yh + g.w_y) <= span_y && (uint32_t)(c[i].y - zh + g.w_z) <= span_z &&
                      t + (uint32_t)i < n;
      m |= (uint32_t)in << ((t + (uint32_t)i) & 31u);
    }
  }
  return m;
}

// Best pair of one cluster through the window masks.  su / sd: where the up / down row's records are read from,
// indexed by GLOBAL sorted position (the direct kernel passes srt for both; the staged kernel passes shared-memory
// copies of the two rows, biased by the rows' first positions); srt: the global array (rare paths: ids on cost ties,
// more than 32 range clusters on a side).
__device__ __forceinline__ Best mask_best_pair(const DevGeom& g, const int4* __restrict__ srt, const int4* su,
                                               const int4* sd, const uint32_t* bs_u, const uint32_t* bs_d, int yh,
                                               int zh, int org_z) {
  Best b = {INT32_MAX, -1, -1};
  const Window w = window_bins(g, yh, zh, org_z);
  const Ranges qu = load_ranges(g, w, bs_u), qd = load_ranges(g, w, bs_d);
  const uint32_t nu0 = qu.b0 - qu.a0, nu = nu0 + (qu.b1 - qu.a1);
  const uint32_t nd0 = qd.b0 - qd.a0, nd = nd0 + (qd.b1 - qd.a1);
  if (nu > 32u || nd > 32u) {
    pair_search_nested<false>(g, srt, w, bs_u, bs_d, yh, zh, b);
  } else if (nu && nd) {
    const uint32_t mu = side_mask(g, su, qu, nu0, nu, yh, zh);
    const uint32_t md = mu ? side_mask(g, sd, qd, nd0, nd, yh, zh) : 0u;
    if (md) {
      for (uint32_t bu = mu; bu; bu &= bu - 1u) {
        const uint32_t pu = range_at(qu, nu0, (uint32_t)__ffs((int)bu) - 1u);
        const int4 cu = su[pu];
        const int dyu = cu.x - yh, dzu = cu.y - zh, idu = cu.z;
        for (uint32_t bd = md; bd; bd &= bd - 1u) {
          const uint32_t pd = range_at(qd, nd0, (uint32_t)__ffs((int)bd) - 1u);
          const int4 cd = sd[pd];
          const int ddy = dyu + (cd.x - yh), ddz = dzu + (cd.y - zh);
          const int cost = g.cost_wy * ddy * ddy + g.cost_wz * ddz * ddz;   // P8
          if (cost < b.cost || (cost == b.cost && tie_wins(srt, b, idu, cd.z))) {   // P9
            b.cost = cost;
            b.pu = (int)pu;
            b.pd = (int)pd;
          }
        }
      }
    }
  }
  if (b.pu < 0 || b.cost > g.c_max) b.pu = b.pd = -1;   // P10
  return b;
}

// 16 CTAs of 128 threads per SM (32 registers): the kernel hides its gathers with resident warps
__global__ void __launch_bounds__(A2_THREADS, 16)
a2_neighbours_mask_kernel(const DevGeom g, const DevCtl* __restrict__ ctl, const uint32_t* __restrict__ ro, const int4* __restrict__ srt,
                          const uint32_t* __restrict__ sec_key, const uint32_t* __restrict__ bin_start,
                          int32_t* __restrict__ link_up, int32_t* __restrict__ link_dn) {
  if (ctl->bad_offsets) return;
  const int sr = blockIdx.x;
  const int r = sr % g.n_rows;
  const uint32_t a = ro[sr], b = ro[sr + 1];
  const bool inner = r >= 1 && r <= g.n_rows - 2;   // P5
  const int org_z = zmin_from_key(sec_key[sr / g.n_rows]);
  const uint32_t *bs_u = nullptr, *bs_d = nullptr;
  if (inner) {
    bs_u = bin_start + (size_t)(sr + 1) * g.nb_stride;
    bs_d = bin_start + (size_t)(sr - 1) * g.nb_stride;
  }
  for (uint32_t j = a + threadIdx.x; j < b; j += A2_THREADS) {
    const int4 ch = srt[j];
    Best bp = {INT32_MAX, -1, -1};
    if (inner) bp = mask_best_pair(g, srt, srt, srt, bs_u, bs_d, ch.x, ch.y, org_z);
    link_up[j] = bp.pu;
    link_dn[j] = bp.pd;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// north_star's a2: "stages the r-1 / r+1 row grids in shared memory via TMA".  A CTA owns A2S_ROWS consecutive rows of
// one sector and slides a three-row window over them: every row's cluster records and bin starts are copied into a
// four-slot shared-memory ring ONCE, by 1-D bulk copies (cp.async.bulk, completion on an mbarrier), two rows ahead
// of their use, and serve as down row, own row and up row in turn.  Rows that do not fit a slot are read from global
// memory through the same pointers.  Same arithmetic (mask_best_pair), same links; which of the two kernels a call
// runs is decided in launch_a2_neighbours from the measurement in profiles/r02_a2_staged.md.
// ---------------------------------------------------------------------------------------------------------------
constexpr int A2S_ROWS = 19;       // rows per CTA (152 = 8 x 19); two extra rows are staged per CTA
constexpr int A2S_RING = 4;
constexpr int A2S_ROWCAP = 320;    // records per slot (5 KB); longer rows stay in global memory
constexpr int A2S_BINCAP = 1024;   // bin starts per slot (4 KB)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t phase) {
  asm volatile(
      "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @p bra DONE_%=;\n"
      " bra WAIT_%=;\n DONE_%=:\n}" ::"r"(smem_u32(bar)), "r"(phase) : "memory");
}
// 1-D bulk copy global -> shared (TMA without a tensor map): 16-byte aligned addresses, size a multiple of 16
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__global__ void __launch_bounds__(A2_THREADS)
a2_neighbours_staged_kernel(const DevGeom g, const DevCtl* __restrict__ ctl, const uint32_t* __restrict__ ro,
                            const int4* __restrict__ srt, const uint32_t* __restrict__ sec_key,
                            const uint32_t* __restrict__ bin_start, int32_t* __restrict__ link_up,
                            int32_t* __restrict__ link_dn) {
  __shared__ __align__(128) int4 s_rec[A2S_RING][A2S_ROWCAP];
  __shared__ __align__(128) uint32_t s_bin[A2S_RING][A2S_BINCAP];
  __shared__ __align__(8) uint64_t s_bar[A2S_RING];
  __shared__ uint32_t s_a[A2S_RING], s_b[A2S_RING];      // position range of the row in each slot
  __shared__ int s_staged[A2S_RING];                      // the slot holds a copy (else: read global memory)
  __shared__ uint32_t s_uses[A2S_RING], s_phase[A2S_RING];   // copies issued into the slot so far; parity to wait for
  if (ctl->bad_offsets) return;
  const int nr = g.n_rows;
  const int chunks = (nr + A2S_ROWS - 1) / A2S_ROWS;
  const int sec = blockIdx.x / chunks, chunk = blockIdx.x % chunks;
  const int r_lo = chunk * A2S_ROWS, r_hi = min(r_lo + A2S_ROWS, nr);   // rows [r_lo, r_hi)
  const int org_z = zmin_from_key(sec_key[sec]);
  const int64_t sr0 = (int64_t)sec * nr;
  const bool bins_fit = g.nb_stride <= A2S_BINCAP;
  if (threadIdx.x == 0) {
    for (int k = 0; k < A2S_RING; ++k) {
      mbar_init(&s_bar[k], 1);
      s_uses[k] = 0;
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // thread 0 stages row `row` (any row of the sector, or nothing outside it) into slot row & 3
  auto stage = [&](int row) {
    const int slot = row & (A2S_RING - 1);
    if (row < 0 || row >= nr) {
      s_staged[slot] = 0;
      s_a[slot] = s_b[slot] = 0;
      return;
    }
    const uint32_t a = ro[sr0 + row], b = ro[sr0 + row + 1];
    s_a[slot] = a;
    s_b[slot] = b;
    const bool fit = bins_fit && b - a <= (uint32_t)A2S_ROWCAP;
    s_staged[slot] = fit ? 1 : 0;
    if (fit) {
      const uint32_t bytes_rec = (b - a) * 16u, bytes_bin = (uint32_t)g.nb_stride * 4u;
      s_phase[slot] = s_uses[slot] & 1u;   // the mbarrier's phase flips once per completed copy into this slot
      ++s_uses[slot];
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // earlier reads of the slot precede the copy
      mbar_expect_tx(&s_bar[slot], bytes_rec + bytes_bin);
      if (bytes_rec) bulk_g2s(&s_rec[slot][0], srt + a, bytes_rec, &s_bar[slot]);
      bulk_g2s(&s_bin[slot][0], bin_start + (size_t)(sr0 + row) * g.nb_stride, bytes_bin, &s_bar[slot]);
    }
  };
  if (threadIdx.x == 0) {
    stage(r_lo - 1);
    stage(r_lo);
    stage(r_lo + 1);
  }
  __syncthreads();
  for (int r = r_lo; r < r_hi; ++r) {
    if (threadIdx.x == 0 && r + 2 <= r_hi) stage(r + 2);   // two rows ahead; its slot was the down row of row r - 1
    __syncthreads();                                        // s_a / s_b / s_staged of the new slot are visible
    const int sc = r & 3, su_ = (r + 1) & 3, sd_ = (r - 1) & 3;
    const bool inner = r >= 1 && r <= nr - 2;               // P5
    const uint32_t a = s_a[sc], b = s_b[sc];
    auto wait_slot = [&](int row) {
      const int slot = row & 3;
      if (row >= 0 && row < nr && s_staged[slot]) mbar_wait(&s_bar[slot], s_phase[slot]);
    };
    wait_slot(r - 1);
    wait_slot(r);
    wait_slot(r + 1);
    // pointers indexed by global sorted position: the shared copy biased by the row's first position, or srt itself
    const int4* pc = s_staged[sc] ? &s_rec[sc][0] - a : srt;
    const int4* pu = srt;
    const int4* pd = srt;
    const uint32_t *bs_u = nullptr, *bs_d = nullptr;
    if (inner) {
      pu = s_staged[su_] ? &s_rec[su_][0] - s_a[su_] : srt;
      pd = s_staged[sd_] ? &s_rec[sd_][0] - s_a[sd_] : srt;
      bs_u = s_staged[su_] ? &s_bin[su_][0] : bin_start + (size_t)(sr0 + r + 1) * g.nb_stride;
      bs_d = s_staged[sd_] ? &s_bin[sd_][0] : bin_start + (size_t)(sr0 + r - 1) * g.nb_stride;
    }
    for (uint32_t j = a + threadIdx.x; j < b; j += A2_THREADS) {
      const int4 ch = pc[j];
      Best bp = {INT32_MAX, -1, -1};
      if (inner) bp = mask_best_pair(g, srt, pu, pd, bs_u, bs_d, ch.x, ch.y, org_z);
      link_up[j] = bp.pu;
      link_dn[j] = bp.pd;
    }
    __syncthreads();   // everybody is done with the down row's slot before it is staged again
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Dense rows (several clusters per grid bin: pile-up at high density).  The nested scan above tests every cluster
// of the down ranges once per up candidate; here each side's ranges are filtered once into a short list in shared
// memory and the pair loop runs over |U| x |D| window candidates only (a few, against hundreds of range pairs).
// A cluster with more than A2_KEEP candidates on a side falls back to the nested scan.
// ---------------------------------------------------------------------------------------------------------------
constexpr int A2_KEEP = 20;   // in-window candidates kept per side (60 KB of lists per CTA); configs[3] literal: 12 -> 13.1 ms,
                              // 20 -> 8.2 ms, 32 -> 10.9 ms, 48 -> 21.0 ms (fewer fallbacks against fewer resident CTAs)

__device__ __forceinline__ int filter_side(const DevGeom& g, const int4* __restrict__ srt, const Window& w,
                                           const uint32_t* __restrict__ bs, int yh, int zh,
                                           int* __restrict__ col /* [A2_KEEP][3][A2_THREADS] column: dy, dz, sorted position */) {
  int cnt = 0;
  for (int iz = w.iz_lo; iz <= w.iz_hi; ++iz) {   // one contiguous sorted range per z-bin row of the window
    const uint32_t ra = bs[iz * g.ny + w.iy_lo], rb = bs[iz * g.ny + w.iy_hi + 1];
    if (ra >= rb) continue;
    int4 nx = srt[ra];
    for (uint32_t t = ra; t < rb; ++t) {
      const int4 c = nx;
      nx = srt[min(t + 1, rb - 1)];   // next one in flight (the last iteration re-reads itself)
      const int dy = c.x - yh, dz = c.y - zh;
      if (abs(dy) <= g.w_y && abs(dz) <= g.w_z) {   // P7, inclusive
        if (cnt < A2_KEEP) {
          int* e = col + cnt * 3 * A2_THREADS;
          e[0] = dy;
          e[A2_THREADS] = dz;
          e[2 * A2_THREADS] = (int)t;   // sorted position; ids are only needed on cost ties (P9)
        }
        ++cnt;
      }
    }
  }
  return cnt;
}

template <bool FINE>
__global__ void __launch_bounds__(A2_THREADS)
a2_neighbours_dense_kernel(const DevGeom g, const DevCtl* __restrict__ ctl, const uint32_t* __restrict__ ro, const int4* __restrict__ srt,
                           const uint32_t* __restrict__ sec_key, const uint32_t* __restrict__ bin_start,
                           int32_t* __restrict__ link_up, int32_t* __restrict__ link_dn) {
  extern __shared__ int cand[];   // [side][slot][dy, dz, position][thread]: a thread reads only its column
  if (ctl->bad_offsets) return;
  const int sr = blockIdx.x;
  const int r = sr % g.n_rows;
  const uint32_t a = ro[sr], b = ro[sr + 1];
  const bool inner = r >= 1 && r <= g.n_rows - 2;   // P5
  const int org_z = zmin_from_key(sec_key[sr / g.n_rows]);
  const uint32_t *bs_u = nullptr, *bs_d = nullptr;
  if (inner) {
    bs_u = bin_start + (size_t)(sr + 1) * g.nb_stride;
    bs_d = bin_start + (size_t)(sr - 1) * g.nb_stride;
  }
  int* const col_u = cand + threadIdx.x;
  int* const col_d = cand + A2_KEEP * 3 * A2_THREADS + threadIdx.x;
  // gridDim.y CTAs share a row (dense rows hold thousands of clusters)
  for (uint32_t j = a + blockIdx.y * A2_THREADS + threadIdx.x; j < b; j += gridDim.y * A2_THREADS) {
    const int4 ch = srt[j];
    const int yh = ch.x, zh = ch.y;
    Best b = {INT32_MAX, -1, -1};
    if (inner) {
      const Window w = window_bins(g, yh, zh, org_z);
      const int nu = filter_side(g, srt, w, bs_u, yh, zh, col_u);
      const int nd = nu > 0 ? filter_side(g, srt, w, bs_d, yh, zh, col_d) : 0;
      if (nu > A2_KEEP || nd > A2_KEEP) {
        pair_search_nested<FINE>(g, srt, w, bs_u, bs_d, yh, zh, b);
      } else {
        const int np = nu * nd;   // one flat loop over the pairs
        int iu = 0, id = 0;
        for (int t = 0; t < np; ++t) {
          const int* eu = col_u + iu * 3 * A2_THREADS;
          const int* ed = col_d + id * 3 * A2_THREADS;
          const int ddy = eu[0] + ed[0], ddz = eu[A2_THREADS] + ed[A2_THREADS];
          const int cost = g.cost_wy * ddy * ddy + g.cost_wz * ddz * ddz;   // P8
          const int pu = eu[2 * A2_THREADS], pd = ed[2 * A2_THREADS];
          if (cost < b.cost || (cost == b.cost && tie_wins(srt, b, srt[pu].z, srt[pd].z))) {   // P9
            b.cost = cost;
            b.pu = pu;
            b.pd = pd;
          }
          if (++id == nd) { id = 0; ++iu; }
        }
      }
      if (b.pu < 0 || b.cost > g.c_max) b.pu = b.pd = -1;   // P10
    }
    link_up[j] = b.pu;
    link_dn[j] = b.pd;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// P48 (NEXT-4): rows that are not equidistant.  The straightness of (d, h, u) is the pitch-weighted second difference
// wa c_u + wb c_d - (wa + wb) c_h with the integer weights of the gaps below (wa) and above (wb) the row of h; its
// square needs 64 bits, and the acceptance is 4 cost <= c_max (wa + wb)^2.  One plain kernel for every grid shape
// (the definition's nested scan over the window's bin rows); geometries with equal pitches never come here, their
// cost is the same up to the common factor wa^2 and stays in the 32-bit kernels above.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(A2_THREADS)
a2_neighbours_weighted_kernel(const DevGeom g, const DevCtl* __restrict__ ctl, const uint32_t* __restrict__ ro,
                              const int4* __restrict__ srt, const uint32_t* __restrict__ sec_key,
                              const uint32_t* __restrict__ bin_start, int32_t* __restrict__ link_up,
                              int32_t* __restrict__ link_dn) {
  if (ctl->bad_offsets) return;
  const int sr = blockIdx.x;
  const int r = sr % g.n_rows;
  const uint32_t a = ro[sr], b = ro[sr + 1];
  const bool inner = r >= 1 && r <= g.n_rows - 2;   // P5
  const int org_z = zmin_from_key(sec_key[sr / g.n_rows]);
  const uint32_t *bs_u = nullptr, *bs_d = nullptr;
  long long wa = 1, wb = 1;
  if (inner) {
    bs_u = bin_start + (size_t)(sr + 1) * g.nb_stride;
    bs_d = bin_start + (size_t)(sr - 1) * g.nb_stride;
    wa = g.gap_w[r - 1];
    wb = g.gap_w[r];
  }
  const long long wab = wa + wb;
  for (uint32_t j = a + blockIdx.y * A2_THREADS + threadIdx.x; j < b; j += gridDim.y * A2_THREADS) {
    const int4 ch = srt[j];
    const int yh = ch.x, zh = ch.y;
    long long best_cost = LLONG_MAX;
    int best_u = -1, best_d = -1, pu_best = -1, pd_best = -1;
    if (inner) {
      const Window w = window_bins(g, yh, zh, org_z);
      for (int izu = w.iz_lo; izu <= w.iz_hi; ++izu) {
        const uint32_t ua = bs_u[izu * g.ny + w.iy_lo], ub = bs_u[izu * g.ny + w.iy_hi + 1];
        for (uint32_t u = ua; u < ub; ++u) {
          const int4 cu = srt[u];
          if (abs(cu.x - yh) > g.w_y || abs(cu.y - zh) > g.w_z) continue;   // P7
          for (int izd = w.iz_lo; izd <= w.iz_hi; ++izd) {
            const uint32_t da = bs_d[izd * g.ny + w.iy_lo], db = bs_d[izd * g.ny + w.iy_hi + 1];
            for (uint32_t d = da; d < db; ++d) {
              const int4 cd = srt[d];
              if (abs(cd.x - yh) > g.w_y || abs(cd.y - zh) > g.w_z) continue;
              const long long ddy = wa * cu.x + wb * cd.x - wab * yh, ddz = wa * cu.y + wb * cd.y - wab * zh;
              const long long cost = (long long)g.cost_wy * ddy * ddy + (long long)g.cost_wz * ddz * ddz;
              if (cost < best_cost || (cost == best_cost && (cu.z < best_u || (cu.z == best_u && cd.z < best_d)))) {   // P9
                best_cost = cost;
                best_u = cu.z;
                best_d = cd.z;
                pu_best = (int)u;
                pd_best = (int)d;
              }
            }
          }
        }
      }
      if (pu_best < 0 || 4 * best_cost > (long long)g.c_max * wab * wab) pu_best = pd_best = -1;   // P10 (P48)
    }
    link_up[j] = pu_best;
    link_dn[j] = pd_best;
  }
}

}  // namespace

cudaError_t setup_a2_attributes() {
  const int bytes = 2 * A2_KEEP * 3 * A2_THREADS * (int)sizeof(int);
  cudaError_t e = cudaFuncSetAttribute(a2_neighbours_dense_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(a2_neighbours_dense_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

cudaError_t launch_a2_neighbours(const tpc_tracker* t, const uint32_t* ro, int64_t n, cudaStream_t st) {
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  if (R == 0) return cudaSuccess;
  // clusters per grid bin decide the variant (both compute the same links); a refined grid (choose_grid) may have
  // z-bins narrower than the window
  const bool dense = (double)n > 0.75 * (double)R * (double)(t->g.ny * t->g.nz);
  const bool fine = t->g.shift_z < t->base_shift_z;
#define A2_ARGS t->g, t->s.ctl, ro, t->s.srt, t->s.sec_key, t->s.bin_start, t->s.link_up, t->s.link_dn
  // dense rows: CTAs per row from the average row length (a longer row just loops)
  int64_t per_row = (n / R + A2_THREADS - 1) / A2_THREADS;
  per_row = per_row < 1 ? 1 : (per_row > 64 ? 64 : per_row);
  const dim3 grid2((unsigned)R, (unsigned)per_row);
  const size_t dense_smem = (size_t)2 * A2_KEEP * 3 * A2_THREADS * sizeof(int);
  if (t->g.gap_w) a2_neighbours_weighted_kernel<<<grid2, A2_THREADS, 0, st>>>(A2_ARGS);
  else if (dense && fine) a2_neighbours_dense_kernel<true><<<grid2, A2_THREADS, dense_smem, st>>>(A2_ARGS);
  else if (dense) a2_neighbours_dense_kernel<false><<<grid2, A2_THREADS, dense_smem, st>>>(A2_ARGS);
  else if (fine) a2_neighbours_kernel<true><<<(unsigned)R, A2_THREADS, 0, st>>>(A2_ARGS);
  else if (t->a2_variant == 1) {
    const int chunks = (t->g.n_rows + A2S_ROWS - 1) / A2S_ROWS;
    a2_neighbours_staged_kernel<<<(unsigned)(t->g.n_sectors * chunks), A2_THREADS, 0, st>>>(A2_ARGS);
  } else a2_neighbours_mask_kernel<<<(unsigned)R, A2_THREADS, 0, st>>>(A2_ARGS);
#undef A2_ARGS
  return cudaGetLastError();
}
