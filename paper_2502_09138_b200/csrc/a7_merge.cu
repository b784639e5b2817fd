// a7_merge.cu -- NEXT-1: merging of sector tracks across sector edges, across the central membrane and
// inside a sector (readings P42..P46).  tpc_merge in include/tpc_track.h.
//
// For an ordered pair a -> b ("b continues a"): the rows must leave a gap of 1..gap_max between a's last and b's first
// owned hit and the sectors must be the same, azimuthal neighbours on one side, or face each other across the central
// membrane (P43).  a's record is rotated into b's frame (P42), transported along its helix to b's reference plane,
// and chi2 = D^T (C_a' + C_b)^-1 D over the five parameters decides (P44).  succ(a) and pred(b) are the candidates
// of smallest (chi2, index) below chi2_max; a link stands iff both agree (P45).
//
// One thread per track; the lanes of a warp are consecutive tracks, i.e. mostly one sector, so the loop over a
// candidate sector's tracks is uniform and the partner's record is a broadcast load.  Everything that decides is in
// fp64: the step is outside the hot path (a few hundred chi2 evaluations per track), and with fp64 the decisions are
// the oracle's.  Tracks arrive ordered by seed cluster id, hence by sector (P29): the per-sector track ranges come
// from one binary search per sector.
#include "tpc_internal.cuh"

namespace {

struct MState {
  double x, y, z, s, t, q;
  double C[15];   // packed lower triangle 00 10 11 20 21 22 30 31 32 33 40 41 42 43 44
};

__device__ __forceinline__ int tri(int i, int j) { return i >= j ? i * (i + 1) / 2 + j : j * (j + 1) / 2 + i; }

__device__ __forceinline__ void load_state(const tpc_track_rec_t* __restrict__ r, MState& m) {
  m.x = r->x; m.y = r->y; m.z = r->z; m.s = r->sinphi; m.t = r->tanl; m.q = r->qpt;
#pragma unroll
  for (int k = 0; k < 15; ++k) m.C[k] = r->cov[k];
}

// C <- J C J^T for a 5x5 J given as full matrix (row-major), C packed.
__device__ __forceinline__ void congruence(const double J[25], double C[15]) {
  double M[25];   // M = J C
#pragma unroll
  for (int i = 0; i < 5; ++i)
#pragma unroll
    for (int j = 0; j < 5; ++j) {
      double a = 0.0;
#pragma unroll
      for (int l = 0; l < 5; ++l) a += J[i * 5 + l] * C[tri(l, j)];
      M[i * 5 + j] = a;
    }
#pragma unroll
  for (int i = 0; i < 5; ++i)
#pragma unroll
    for (int j = 0; j <= i; ++j) {
      double a = 0.0;
#pragma unroll
      for (int l = 0; l < 5; ++l) a += M[i * 5 + l] * J[j * 5 + l];
      C[tri(i, j)] = a;
    }
}

// P42: the same point and direction in the frame turned by alpha (sa = sin alpha, ca = cos alpha).
__device__ __forceinline__ bool rotate_frame(double cq, double smax, double sa, double ca, MState& m) {
  if (!(fabs(m.s) < 1.0)) return false;
  const double c = sqrt(1.0 - m.s * m.s);
  const double s1 = m.s * ca - c * sa, c1 = c * ca + m.s * sa;
  if (!(c1 > 0.0) || !(fabs(s1) < smax)) return false;
  double J[25];
#pragma unroll
  for (int k = 0; k < 25; ++k) J[k] = (k % 6 == 0) ? 1.0 : 0.0;
  J[0] = c / c1;                     // dy'/dy
  J[5] = -sa * m.t / c1;             // dz'/dy
  J[10] = -sa * cq * m.q;            // dsin phi'/dy
  J[12] = c1 / c;                    // dsin phi'/dsin phi
  congruence(J, m.C);
  const double x0 = m.x, y0 = m.y;
  m.x = x0 * ca + y0 * sa;
  m.y = -x0 * sa + y0 * ca;
  m.s = s1;
  return true;
}

// Appendix C in fp64: one helix step of dx with covariance.
__device__ __forceinline__ bool transport64(double cq, double smax, double dx, MState& m) {
  const double k = cq * m.q, s0 = m.s, s1 = s0 + k * dx;
  if (!(fabs(s0) < smax) || !(fabs(s1) < smax)) return false;
  const double c0 = sqrt(1.0 - s0 * s0), c1 = sqrt(1.0 - s1 * s1);
  const double tau = (s0 + s1) / (c0 + c1);
  const double dy = dx * tau;
  const double chord = copysign(sqrt(dx * dx + dy * dy), dx);
  const double u = 0.5 * k * chord;
  const double dS = fabs(u) < 1e-6 ? chord * (1.0 + u * u / 6.0) : chord * asin(u) / u;
  const double d = 0.5 * k * dS;
  const double sinc = fabs(d) < 1e-6 ? 1.0 - d * d / 6.0 : sin(d) / d;
  const double gg = fabs(d) < 1e-2 ? 1.0 / 3.0 - d * d / 30.0 + d * d * d * d / 840.0 : (sin(d) - d * cos(d)) / (d * d * d);
  const double cm = 1.0 / sqrt(1.0 + tau * tau), sm = tau * cm;
  const double mm = c0 + s0 * tau;
  const double dSdk = (0.5 * dS * dS * sm * sinc + 0.25 * k * dS * dS * dS * cm * gg) / c1;
  double J[25];
#pragma unroll
  for (int i = 0; i < 25; ++i) J[i] = (i % 6 == 0) ? 1.0 : 0.0;
  J[2] = dx * mm / (c0 * c1);
  J[4] = cq * dx * dx * mm / (c1 * (c0 + c1));
  J[7] = m.t * dy / (c0 * c1);
  J[8] = dS;
  J[9] = m.t * cq * dSdk;
  J[14] = cq * dx;
  congruence(J, m.C);
  m.x += dx;
  m.y += dy;
  m.z += m.t * dS;
  m.s = s1;
  return true;
}

// P44.  Negative: no match possible (rotation / transport failed, or S not positive definite).
__device__ __forceinline__ double match_chi2(double cq, double smax, int rot, double sa, double ca, const MState& a0,
                                             const MState& b) {
  MState a = a0;
  if (rot != 0 && !rotate_frame(cq, smax, rot > 0 ? sa : -sa, ca, a)) return -1.0;
  if (!transport64(cq, smax, b.x - a.x, a)) return -1.0;
  double L[15];
#pragma unroll
  for (int k = 0; k < 15; ++k) L[k] = a.C[k] + b.C[k];
  const double D[5] = {b.y - a.y, b.z - a.z, b.s - a.s, b.t - a.t, b.q - a.q};
  // in-place Cholesky of the packed lower triangle, then forward substitution
#pragma unroll
  for (int i = 0; i < 5; ++i)
#pragma unroll
    for (int j = 0; j <= i; ++j) {
      double v = L[tri(i, j)];
#pragma unroll
      for (int l = 0; l < j; ++l) v -= L[tri(i, l)] * L[tri(j, l)];
      if (i == j) {
        if (!(v > 0.0)) return -1.0;
        L[tri(i, i)] = sqrt(v);
      } else {
        L[tri(i, j)] = v / L[tri(j, j)];
      }
    }
  double chi2 = 0.0, w[5];
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    double v = D[i];
#pragma unroll
    for (int l = 0; l < i; ++l) v -= L[tri(i, l)] * w[l];
    w[i] = v / L[tri(i, i)];
    chi2 += w[i] * w[i];
  }
  return chi2;
}

struct MergeCfg {
  double cq, smax, sa, ca, chi2_max;
  int gap_max, nps, n_sectors;
};

__global__ void a7_sector_ranges_kernel(const tpc_track_rec_t* __restrict__ tracks, const int32_t* __restrict__ counts,
                                        int32_t cap, int n_sectors, int32_t* __restrict__ sec_start) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s > n_sectors) return;
  const int nt = min(counts[0], cap);
  int lo = 0, hi = nt;   // first track with sector >= s
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (tracks[mid].sector < s) lo = mid + 1; else hi = mid;
  }
  sec_start[s] = lo;
}

// The up to four sectors whose tracks can be joined with a track of sector s, with the rotation from a's frame to
// b's frame when a is in `s` and b in the listed sector (rot = +1: b's frame is a's turned by +sector_angle).
__device__ __forceinline__ int partner_sectors(const MergeCfg& c, int s, int sec[4], int rot[4]) {
  const int side_base = (s / c.nps) * c.nps, i = s - side_base;
  int n = 0;
  sec[n] = s; rot[n++] = 0;
  if (c.nps > 1) {
    const int up = side_base + (i + 1) % c.nps, dn = side_base + (i + c.nps - 1) % c.nps;
    sec[n] = up; rot[n++] = 1;
    if (dn != up) { sec[n] = dn; rot[n++] = -1; }
  }
  const int grp = s / (2 * c.nps);
  const int other = (s / c.nps) % 2 == 0 ? s + c.nps : s - c.nps;
  if (other >= 0 && other < c.n_sectors && other / (2 * c.nps) == grp) { sec[n] = other; rot[n++] = 0; }
  return n;
}

// FORWARD: thread per a, best successor.  !FORWARD: thread per b, best predecessor.
template <bool FORWARD>
__global__ void __launch_bounds__(128)
a7_best_kernel(const MergeCfg c, const tpc_track_rec_t* __restrict__ tracks, const int32_t* __restrict__ counts,
               int32_t cap, const int32_t* __restrict__ sec_start, int32_t* __restrict__ best,
               double* __restrict__ best_chi2) {
  const int nt = min(counts[0], cap);
  const int me = blockIdx.x * blockDim.x + threadIdx.x;
  if (me >= nt) return;
  MState m;
  load_state(tracks + me, m);
  const int my_sec = tracks[me].sector, my_first = tracks[me].first_row, my_last = tracks[me].last_row;
  int sec[4], rot[4];
  const int np = partner_sectors(c, my_sec, sec, rot);
  int bi = -1;
  double bc = c.chi2_max;
  for (int k = 0; k < np; ++k) {
    const int t0 = sec_start[sec[k]], t1 = sec_start[sec[k] + 1];
    for (int o = t0; o < t1; ++o) {
      if (o == me) continue;
      const tpc_track_rec_t* r = tracks + o;
      const int gap = FORWARD ? r->first_row - my_last : my_first - r->last_row;
      if (gap < 1 || gap > c.gap_max) continue;
      // exact prefilter: tan lambda and q/pT (and their variances) change neither in the rotation nor along the
      // helix, and D^T S^-1 D >= D_i^2 / S_ii for a positive definite S, so a pair that fails on one of them alone
      // cannot pass the full chi2
      {
        const double dt = (double)r->tanl - m.t, dq = (double)r->qpt - m.q;
        if (dt * dt >= c.chi2_max * ((double)r->cov[9] + m.C[9]) || dq * dq >= c.chi2_max * ((double)r->cov[14] + m.C[14]))
          continue;
      }
      MState other;
      load_state(r, other);
      // rotation goes from the inner segment's frame to the outer one's
      const double chi2 = FORWARD ? match_chi2(c.cq, c.smax, rot[k], c.sa, c.ca, m, other)
                                  : match_chi2(c.cq, c.smax, -rot[k], c.sa, c.ca, other, m);
      if (chi2 < 0.0) continue;
      if (chi2 < bc || (chi2 == bc && bi >= 0 && o < bi)) {   // (chi2, index) lexicographic, chi2 < chi2_max
        bc = chi2;
        bi = o;
      }
    }
  }
  best[me] = bi;
  best_chi2[me] = bc;
}

__global__ void a7_link_kernel(const int32_t* __restrict__ counts, int32_t cap, const int32_t* __restrict__ best_s,
                               const int32_t* __restrict__ best_p, const double* __restrict__ chi_s,
                               int32_t* __restrict__ succ, int32_t* __restrict__ pred, float* __restrict__ link_chi2,
                               int32_t* __restrict__ merge_counts) {
  const int nt = min(counts[0], cap);
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a == 0) merge_counts[2] = nt;
  if (a >= nt) return;
  const int b = best_s[a];
  const bool link = b >= 0 && best_p[b] == a;   // P45: mutual best
  succ[a] = link ? b : -1;
  link_chi2[a] = link ? (float)chi_s[a] : -1.f;
  if (link) {
    pred[b] = a;
    atomicAdd(&merge_counts[0], 1);
  }
}

__global__ void a7_init_kernel(const int32_t* __restrict__ counts, int32_t cap, int32_t* __restrict__ pred,
                               int32_t* __restrict__ merge_counts) {
  const int nt = min(counts[0], cap);
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a < 4) merge_counts[a] = 0;
  if (a < nt) pred[a] = -1;
}

__global__ void a7_finish_kernel(int32_t* __restrict__ merge_counts) {
  merge_counts[1] = merge_counts[2] - merge_counts[0];   // merged tracks = tracks - links
}

}  // namespace

cudaError_t launch_a7_merge(const tpc_tracker* t, const tpc_merge_params_t* mp, const tpc_track_rec_t* tracks,
                            const int32_t* counts, int32_t cap, int32_t* succ, int32_t* pred, float* link_chi2,
                            int32_t* merge_counts, cudaStream_t st) {
  if (cap <= 0) return cudaSuccess;
  MergeCfg c;
  c.cq = t->params.cq_per_tesla * t->bz;
  c.smax = t->params.sinphi_max;
  c.sa = sin(mp->sector_angle);
  c.ca = cos(mp->sector_angle);
  c.chi2_max = mp->chi2_max;
  c.gap_max = mp->gap_max;
  c.nps = mp->n_per_side;
  c.n_sectors = t->g.n_sectors;
  const unsigned blocks = (unsigned)((cap + 127) / 128);
  a7_init_kernel<<<blocks, 128, 0, st>>>(counts, cap, pred, merge_counts);
  a7_sector_ranges_kernel<<<(unsigned)(t->g.n_sectors / 128 + 1), 128, 0, st>>>(tracks, counts, cap, t->g.n_sectors,
                                                                                t->merge_sec);
  a7_best_kernel<true><<<blocks, 128, 0, st>>>(c, tracks, counts, cap, t->merge_sec, t->merge_best, t->merge_chi2);
  a7_best_kernel<false><<<blocks, 128, 0, st>>>(c, tracks, counts, cap, t->merge_sec, t->merge_best + cap,
                                               t->merge_chi2 + cap);
  a7_link_kernel<<<blocks, 128, 0, st>>>(counts, cap, t->merge_best, t->merge_best + cap, t->merge_chi2, succ, pred,
                                         link_chi2, merge_counts);
  a7_finish_kernel<<<1, 1, 0, st>>>(merge_counts);
  return cudaGetLastError();
}
