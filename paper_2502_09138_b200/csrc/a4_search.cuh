// a4_search.cuh -- the row search of the tracklet follower (P17/P21) and the predicated loads its gathers use.
// Shared by the a4 kernels; included after kalman.cuh.
#pragma once
#include "kalman.cuh"

namespace {


__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

struct Found {
  int id;
  int hy, hz;     // its fixed-point coordinates
  float ry, rz;   // residuals (hit - state) of the accepted hit, cm
};

// The search window of P17/P21 in grid bins.  A cluster can only be accepted if dy^2/(Cyy+sy2) < gate_d, so the
// bins that are read cover |dy| <= min(gate_y, sqrt(gate_d (Cyy+sy2))) (widened by 0.2 % + 2 units against
// rounding), likewise in z: the grid only prunes, every accept/compare in search_row is the definition's.
struct Window {
  int iy_lo, iy_hi, iz_lo, iz_hi;
  __device__ __forceinline__ uint32_t key_y() const { return ((uint32_t)iy_lo << 16) | (uint32_t)iy_hi; }
  __device__ __forceinline__ uint32_t key_z(int row) const {
    return ((uint32_t)row << 24) | ((uint32_t)iz_lo << 8) | (uint32_t)min(iz_hi - iz_lo, 255);   // nz < 2^16
  }
};

// (py, pz) = fraction of the position in units relative to the integer origin (oy, oz) (kalman.cuh: State).
__device__ __forceinline__ Window search_window(const DevGeom& g, float py, float pz, float vy, float vz, int oy, int oz,
                                                int org_z) {
  // half widths in units: gate_d*v*rsqrt(gate_d*v) = sqrt(gate_d*v) to 2 ulp, inside the 0.2 % margin.
  // float -> int conversions saturate; a state so far off that oy + (...) wraps has no cluster within the gate
  // (coordinates stay within +-2^24 units of the extents), and the clamps keep every index in range regardless.
  const float ay = g.gate_d * vy, az = g.gate_d * vz;
  const float hy = fminf(g.gate_y, ay * rsqrtf(ay) * 1.002f) * g.units + 2.f;
  const float hz = fminf(g.gate_z, az * rsqrtf(az) * 1.002f) * g.units + 2.f;
  const int by = oy - g.org_y, bz = oz - org_z;
  Window w;
  w.iy_lo = min(max((__float2int_rd(py - hy) + by) >> g.shift_y, 0), g.ny - 1);
  w.iy_hi = min(max((__float2int_ru(py + hy) + by) >> g.shift_y, 0), g.ny - 1);
  w.iz_lo = min(max((__float2int_rd(pz - hz) + bz) >> g.shift_z, 0), g.nz - 1);
  w.iz_hi = min(max((__float2int_ru(pz + hz) + bz) >> g.shift_z, 0), g.nz - 1);   // bins >= 2 gate_z: iz_hi <= iz_lo + 1
  return w;
}

// Bin starts of a window: (a0,b0) = sorted range of the low z-bin, (a1,b1) of the high one (empty if the same).
struct BinRanges {
  uint32_t a0, b0, a1, b1;
};

__device__ __forceinline__ BinRanges load_ranges(const DevGeom& g, const uint32_t* __restrict__ bs, const Window& w) {
  BinRanges q;
  q.a0 = bs[w.iz_lo * g.ny + w.iy_lo];
  q.b0 = bs[w.iz_lo * g.ny + w.iy_hi + 1];
  q.a1 = q.b1 = 0;
  if (w.iz_hi != w.iz_lo) {
    q.a1 = bs[w.iz_hi * g.ny + w.iy_lo];
    q.b1 = bs[w.iz_hi * g.ny + w.iy_hi + 1];
  }
  return q;
}

__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

// Predicated loads that write straight into their destination registers (the old value stays when `pred` is
// false).  Written as PTX because `if (c) v = *p;` compiles to load-into-temporary + select, and the select waits
// for the load right there -- which would turn every gather that is issued one step ahead into a blocking one.
// (y, z, up link) of a cluster record as three scalar loads: a predicated 128-bit load needs an aligned register
// quad, which ptxas then copies out of right behind the load (and so waits for it); scalars land in place.
struct Rec {   // a chain hit: its srt record (y, z, cluster id) and its cleaned up link (a sorted position, a3's table)
  int y, z, id, up;
};
__device__ __forceinline__ void ld_rec_if(Rec& v, const int4* p, const int32_t* link, bool pred) {
  asm volatile("{ .reg .pred q; setp.ne.s32 q, %4, 0; @q ld.global.nc.s32 %0, [%5]; @q ld.global.nc.s32 %1, [%5+4];"
               " @q ld.global.nc.s32 %2, [%5+8]; @q ld.global.nc.s32 %3, [%6]; }"
               : "+r"(v.y), "+r"(v.z), "+r"(v.id), "+r"(v.up) : "r"((int)pred), "l"(p), "l"(link));
}
// (y, z) of a recorded hit out of the tracklet's own stream (written by this call's upward pass: read through L2)
__device__ __forceinline__ void ld_cg_yz_if(int& y, int& z, const int2* p, bool pred) {
  asm volatile("{ .reg .pred q; setp.ne.s32 q, %2, 0; @q ld.global.cg.v2.s32 {%0, %1}, [%3]; }"
               : "+r"(y), "+r"(z) : "r"((int)pred), "l"(p) : "memory");
}
// the same in a kernel that only reads the stream (phase C: written by earlier launches): through L1, where the other
// three entries of the 32-byte group are found when their rows come up
__device__ __forceinline__ void ld_ca_yz_if(int& y, int& z, const int2* p, bool pred) {
  asm volatile("{ .reg .pred q; setp.ne.s32 q, %2, 0; @q ld.global.ca.v2.s32 {%0, %1}, [%3]; }"
               : "+r"(y), "+r"(z) : "r"((int)pred), "l"(p) : "memory");
}
__device__ __forceinline__ void ld_u32_if(uint32_t& v, const uint32_t* p, bool pred) {
  asm volatile("{ .reg .pred q; setp.ne.s32 q, %1, 0; @q ld.global.nc.u32 %0, [%2]; }" : "+r"(v) : "r"((int)pred), "l"(p));
}
// .cg: the hit table is written by this kernel, so it is read from L2, never from a stale L1 line
__device__ __forceinline__ void ld_cg_s32_if(int& v, const int32_t* p, bool pred) {
  asm volatile("{ .reg .pred q; setp.ne.s32 q, %1, 0; @q ld.global.cg.s32 %0, [%2]; }" : "+r"(v) : "r"((int)pred), "l"(p) : "memory");
}

// Bin starts of window w of the row whose bin_start segment is bs, loaded into q iff pred.
__device__ __forceinline__ void load_ranges_if(const DevGeom& g, const uint32_t* __restrict__ bs, const Window& w,
                                               BinRanges& q, bool pred) {
  const bool two = pred && w.iz_hi != w.iz_lo;
  if (pred && !two) q.a1 = q.b1 = 0;
  ld_u32_if(q.a0, bs + w.iz_lo * g.ny + w.iy_lo, pred);
  ld_u32_if(q.b0, bs + w.iz_lo * g.ny + w.iy_hi + 1, pred);
  ld_u32_if(q.a1, bs + w.iz_hi * g.ny + w.iy_lo, two);
  ld_u32_if(q.b1, bs + w.iz_hi * g.ny + w.iy_hi + 1, two);
}

// P17/P21: among the candidates minimise (d, id), d = dy^2/(Cyy + sy2) + dz^2/(Czz + sz2), restricted to
// |dy| <= gate_y and |dz| <= gate_z (cm).  Accumulates into (f, bestd); the caller applies the gate d < gate_d.
__device__ __forceinline__ void search_take(const DevGeom& g, const int4& c, const State& p, float wy, float wz,
                                            Found& f, float& bestd) {
  const float dy = resid_y(g, p, c.x), dz = resid_z(g, p, c.y);
  if (fabsf(dy) > g.gate_y || fabsf(dz) > g.gate_z) return;
  const float d = dy * dy * wy + dz * dz * wz;
  if (d < bestd || (d == bestd && c.z < f.id)) {
    bestd = d;
    f.id = c.z;
    f.hy = c.x;
    f.hz = c.y;
    f.ry = dy;
    f.rz = dz;
  }
}

__device__ __forceinline__ void search_ranges(const DevGeom& g, const BinRanges& q, const State& p, float wy, float wz,
                                              const int4* __restrict__ srt, Found& f, float& bestd) {
  const uint32_t n0 = q.b0 - q.a0, total = n0 + (q.b1 - q.a1);
  if (total) {
    // a search has 1.8 candidates on average: the first two are requested together and tested in line, the flat loop
    // over both z-bins takes over from the third (an index beyond the last re-reads the last: never tested)
    auto at = [&](uint32_t t) { t = min(t, total - 1); return t < n0 ? q.a0 + t : q.a1 + (t - n0); };
    const int4 c0 = srt[at(0)], c1 = srt[at(1)], c2 = srt[at(2)], c3 = srt[at(3)];
    int4 nx = srt[at(4)];
    search_take(g, c0, p, wy, wz, f, bestd);
    if (total > 1) search_take(g, c1, p, wy, wz, f, bestd);
    if (total > 2) search_take(g, c2, p, wy, wz, f, bestd);
    if (total > 3) search_take(g, c3, p, wy, wz, f, bestd);
    for (uint32_t t = 4; t < total; ++t) {
      const int4 c = nx;
      nx = srt[at(t + 1)];   // next one in flight
      search_take(g, c, p, wy, wz, f, bestd);
    }
  }
}

}  // namespace
