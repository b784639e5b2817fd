// tpc_oracle.cpp -- CPU oracle (fp64) for TPC sector track finding.  TEST INFRASTRUCTURE, NOT PRODUCT.
// See tpc_oracle.h for the contract.  Follows SURVEY.md section 8(c) / Appendix C step by step
// (PAPER.md:29, :40 name the task only; BASELINE.json north_star names the five stages).
// Independent of the CUDA path: no shared code, headers, tables or constants.
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"; the table is in DESIGN.md section 3): grid == brute force; mutual
// links; chain partition invariants; transport == closed-form circle/helix and reversibility; Jacobian == central finite
// differences and == long-double closed form; update == information form and, for Bz -> 0, weighted least squares
// (numpy lstsq); the follower's rules (row search and gate, miss/stop logic, initial state, final transport) and the
// selection filters on hand-made straight tracks with closed-form line-fit variances (test_oracle_follower_rules.py);
// exact helices reconstructed to 1e-4; <= 1 owner per hit; refit == generator truth; rotation == plane geometry, the
// generator's helix in the next sector and finite differences; merge rules on hand-made records; pitch-weighted cost on
// hand-made unequal gaps; residual transform values, exactness on lines / parabolas and the lossless round trip;
// clusterizer centroids, plateau and threshold rules worked out by hand and resolution against the digit generator;
// rANS stage: frequency tables and chunk bytes worked out by hand (with and without an emission, x = f 2^16), a
// certain symbol costs 0 bits, a symbol of probability 1/16 exactly 4, size against the Shannon bound, round trip.
// No function is left "parity unpinned".  Unpinned by the paper: the free constants of orc_params_t (and of the merge,
// compression and clusterizer readings) and the efficiency / fake-rate values themselves beyond the 100 % zero-
// smearing case -- they are whatever this written algorithm yields.
#include "tpc_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" void orc_default_params(orc_params_t* p) {
  p->w_y = 1280;  // P7: 2.0 cm
  p->w_z = 1600;  // P7: 2.5 cm
  p->cost_wy = 9; // P8
  p->cost_wz = 4;
  p->c_max = 3538944;  // P10 = 16 * 221184
  p->l_min = 5;        // P13
  p->units_per_cm = 640.0;  // P3
  p->sigma_y = 0.1;         // P15
  p->sigma_z = 0.15;
  p->sinphi_max = 0.95;  // P18
  p->max_miss = 5;       // P20
  p->n_min_tracklet = 10;  // P24
  p->gate_d = 15.0;        // P21
  p->gate_y_cm = 2.0;
  p->gate_z_cm = 2.5;
  p->c_reset[0] = 0.25;  // P22
  p->c_reset[1] = 0.25;
  p->c_reset[2] = 0.05;
  p->c_reset[3] = 0.05;
  p->c_reset[4] = 25.0;
  p->cq_per_tesla = -0.00299792458;  // P4
  p->n_min_owned = 10;               // P27
}

extern "C" int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ------------------------------------------------------------------------------------------------
// Stage 1-2: neighbours.  SURVEY 8(c): for cluster h in row r (1 <= r <= n_rows-2, P5), candidates
// U in row r+1 and D in row r-1 of the same sector inside the inclusive window (P7); choose the pair
// minimising (cost, id_u, id_d) lexicographically (P8, P9); accept iff cost <= c_max (P10).
// ------------------------------------------------------------------------------------------------
static inline bool in_window(const orc_params_t* p, int32_t yh, int32_t zh, int32_t yc, int32_t zc) {
  int64_t dy = (int64_t)yc - yh, dz = (int64_t)zc - zh;
  return std::llabs(dy) <= p->w_y && std::llabs(dz) <= p->w_z;
}

// P8 for any row pitches (P48): the straight line through d and u, evaluated at the row of h, misses h by
// (wa y_u + wb y_d - (wa + wb) y_h) / (wa + wb) with wa, wb the integer pitch weights of the gaps below and above h.
// The cost is that numerator squared and weighted; for equal pitches (wa == wb == 1) it is the plain second difference.
static inline int64_t pair_cost(const orc_params_t* p, int64_t wa, int64_t wb, int32_t yh, int32_t zh, int32_t yu,
                                int32_t zu, int32_t yd, int32_t zd) {
  int64_t ddy = wa * yu + wb * yd - (wa + wb) * (int64_t)yh;
  int64_t ddz = wa * zu + wb * zd - (wa + wb) * (int64_t)zh;
  return p->cost_wy * ddy * ddy + p->cost_wz * ddz * ddz;
}

static void best_pair(const orc_params_t* p, int64_t wa, int64_t wb, const int32_t* y, const int32_t* z, int32_t h,
                      const std::vector<int32_t>& U, const std::vector<int32_t>& D, int32_t* up, int32_t* dn) {
  int64_t best_cost = std::numeric_limits<int64_t>::max();
  int32_t bu = -1, bd = -1;
  for (int32_t u : U)
    for (int32_t d : D) {
      int64_t c = pair_cost(p, wa, wb, y[h], z[h], y[u], z[u], y[d], z[d]);
      bool better = c < best_cost || (c == best_cost && (u < bu || (u == bu && d < bd)));
      if (better) {
        best_cost = c;
        bu = u;
        bd = d;
      }
    }
  // P10 with the pitch weights: cost / ((wa + wb) / 2)^2 <= c_max
  if (bu >= 0 && 4 * best_cost <= (int64_t)p->c_max * (wa + wb) * (wa + wb)) {
    *up = bu;
    *dn = bd;
  } else {
    *up = -1;
    *dn = -1;
  }
}

extern "C" void orc_neighbours_brute_w(const orc_params_t* p, int32_t n_sectors, int32_t n_rows, const int32_t* gap_w,
                                       const int32_t* y, const int32_t* z, const uint32_t* ro, int32_t* link_up,
                                       int32_t* link_dn) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t s = 0; s < n_sectors; ++s) {
    std::vector<int32_t> U, D;
    for (int32_t r = 0; r < n_rows; ++r) {
      const uint32_t* o = ro + (int64_t)s * n_rows + r;
      for (uint32_t h = o[0]; h < o[1]; ++h) {
        link_up[h] = -1;
        link_dn[h] = -1;
        if (r < 1 || r > n_rows - 2) continue;
        U.clear();
        D.clear();
        for (uint32_t c = o[1]; c < o[2]; ++c)
          if (in_window(p, y[h], z[h], y[c], z[c])) U.push_back((int32_t)c);
        for (uint32_t c = o[-1]; c < o[0]; ++c)
          if (in_window(p, y[h], z[h], y[c], z[c])) D.push_back((int32_t)c);
        best_pair(p, gap_w ? gap_w[r - 1] : 1, gap_w ? gap_w[r] : 1, y, z, (int32_t)h, U, D, &link_up[h], &link_dn[h]);
      }
    }
  }
}

extern "C" void orc_neighbours_brute(const orc_params_t* p, int32_t n_sectors, int32_t n_rows, const int32_t* y,
                                     const int32_t* z, const uint32_t* ro, int32_t* link_up, int32_t* link_dn) {
  orc_neighbours_brute_w(p, n_sectors, n_rows, nullptr, y, z, ro, link_up, link_dn);
}

// z-sorted index per row: the oracle's own pruning structure (not the GPU's (y,z) bin grid).
template <typename T>
static void build_zorder(int64_t n_sr, const uint32_t* ro, const T* z, std::vector<int32_t>& idx) {
  idx.resize(ro[n_sr]);
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t sr = 0; sr < n_sr; ++sr) {
    for (uint32_t h = ro[sr]; h < ro[sr + 1]; ++h) idx[h] = (int32_t)h;
    std::sort(idx.begin() + ro[sr], idx.begin() + ro[sr + 1],
              [&](int32_t a, int32_t b) { return z[a] < z[b] || (z[a] == z[b] && a < b); });
  }
}

extern "C" void orc_neighbours_pruned_w(const orc_params_t* p, int32_t n_sectors, int32_t n_rows, const int32_t* gap_w,
                                        const int32_t* y, const int32_t* z, const uint32_t* ro, int32_t* link_up,
                                        int32_t* link_dn) {
  std::vector<int32_t> zo;
  build_zorder<int32_t>((int64_t)n_sectors * n_rows, ro, z, zo);
  auto collect = [&](uint32_t a, uint32_t b, int32_t yh, int32_t zh, std::vector<int32_t>& out) {
    out.clear();
    int64_t zlo = (int64_t)zh - p->w_z;
    auto first = std::lower_bound(zo.begin() + a, zo.begin() + b, zlo,
                                  [&](int32_t c, int64_t v) { return (int64_t)z[c] < v; });
    for (auto it = first; it != zo.begin() + b; ++it) {
      if ((int64_t)z[*it] > (int64_t)zh + p->w_z) break;
      if (in_window(p, yh, zh, y[*it], z[*it])) out.push_back(*it);
    }
  };
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t s = 0; s < n_sectors; ++s) {
    std::vector<int32_t> U, D;
    for (int32_t r = 0; r < n_rows; ++r) {
      const uint32_t* o = ro + (int64_t)s * n_rows + r;
      for (uint32_t h = o[0]; h < o[1]; ++h) {
        link_up[h] = -1;
        link_dn[h] = -1;
        if (r < 1 || r > n_rows - 2) continue;
        collect(o[1], o[2], y[h], z[h], U);
        collect(o[-1], o[0], y[h], z[h], D);
        best_pair(p, gap_w ? gap_w[r - 1] : 1, gap_w ? gap_w[r] : 1, y, z, (int32_t)h, U, D, &link_up[h], &link_dn[h]);
      }
    }
  }
}

extern "C" void orc_neighbours_pruned(const orc_params_t* p, int32_t n_sectors, int32_t n_rows, const int32_t* y,
                                      const int32_t* z, const uint32_t* ro, int32_t* link_up, int32_t* link_dn) {
  orc_neighbours_pruned_w(p, n_sectors, n_rows, nullptr, y, z, ro, link_up, link_dn);
}

// ------------------------------------------------------------------------------------------------
// Stage 3.  SURVEY 8(c): one synchronous step from the raw tables (P11); chain start = no down link,
// has up link (P12); length counts clusters; seed iff L >= l_min (P13); seeds ascend by start id (P14).
// ------------------------------------------------------------------------------------------------
extern "C" void orc_clean_links(int64_t n, const int32_t* up, const int32_t* dn, int32_t* up_c, int32_t* dn_c) {
  for (int64_t h = 0; h < n; ++h) {
    up_c[h] = (up[h] >= 0 && dn[up[h]] == (int32_t)h) ? up[h] : -1;
    dn_c[h] = (dn[h] >= 0 && up[dn[h]] == (int32_t)h) ? dn[h] : -1;
  }
}

extern "C" int64_t orc_find_seeds(const orc_params_t* p, int64_t n, const int32_t* up_c, const int32_t* dn_c,
                                  int32_t* seed_start, int32_t* seed_len) {
  int64_t ns = 0;
  for (int64_t h = 0; h < n; ++h) {
    if (dn_c[h] >= 0 || up_c[h] < 0) continue;
    int32_t len = 1;
    for (int32_t c = up_c[h]; c >= 0; c = up_c[c]) ++len;
    if (len >= p->l_min) {
      seed_start[ns] = (int32_t)h;
      seed_len[ns] = len;
      ++ns;
    }
  }
  return ns;
}

// ------------------------------------------------------------------------------------------------
// Stage 4 building blocks.  SURVEY Appendix C (textbook circle/helix geometry in the sector frame).
// State (y, z, s = sin phi, t = tan lambda = dz/ds_xy, q = q/pT) at x; k = cq * q is the signed curvature:
// s(x + dx) = s + k dx exactly on a circle.
// ------------------------------------------------------------------------------------------------
struct Step {
  double s1, c0, c1, tau, dy, dS, m, dSdk;
};

// Geometry of one step.  dy = dx (s+s1)/(c0+c1) [= (c0-c1)/k]; chord = sign(dx) sqrt(dx^2+dy^2);
// u = k chord / 2; dS = chord asin(u)/u [= (asin s1 - asin s)/k].
// d(dS)/dk = (dx/c1 - dS)/k, evaluated without the 0/0 at k -> 0: with phi_m = (phi0+phi1)/2 (tan phi_m = tau)
// and delta = k dS / 2 = (phi1-phi0)/2,
//   dx/c1 - dS = (2/(k c1)) [cos phi_m (sin d - d cos d) + d sin phi_m sin d]
//   => d(dS)/dk = [ (dS^2/2) sin phi_m sinc(d) + (k dS^3/4) cos phi_m g(d) ] / c1,  g(d) = (sin d - d cos d)/d^3.
static bool step_geometry(double k, double s, double dx, double smax, Step* g) {
  double s1 = s + k * dx;
  if (std::fabs(s) >= smax || std::fabs(s1) >= smax) return false;
  double c0 = std::sqrt(1.0 - s * s), c1 = std::sqrt(1.0 - s1 * s1);
  double tau = (s + s1) / (c0 + c1);
  double dy = dx * tau;
  double chord = std::copysign(std::sqrt(dx * dx + dy * dy), dx);
  double u = 0.5 * k * chord;
  double dS = (std::fabs(u) < 1e-6) ? chord * (1.0 + u * u / 6.0) : chord * std::asin(u) / u;
  double d = 0.5 * k * dS;
  double sinc = (std::fabs(d) < 1e-6) ? 1.0 - d * d / 6.0 : std::sin(d) / d;
  double gg = (std::fabs(d) < 1e-2) ? 1.0 / 3.0 - d * d / 30.0 + d * d * d * d / 840.0
                                   : (std::sin(d) - d * std::cos(d)) / (d * d * d);
  double cm = 1.0 / std::sqrt(1.0 + tau * tau), sm = tau * cm;
  g->s1 = s1;
  g->c0 = c0;
  g->c1 = c1;
  g->tau = tau;
  g->dy = dy;
  g->dS = dS;
  g->m = c0 + s * tau;  // = sin(phi1-phi0)/(k dx)
  g->dSdk = (0.5 * dS * dS * sm * sinc + 0.25 * k * dS * dS * dS * cm * gg) / c1;
  return true;
}

static void jacobian_from(const Step& g, double cq, double dx, double t, double F[25]) {
  for (int i = 0; i < 25; ++i) F[i] = 0.0;
  for (int i = 0; i < 5; ++i) F[i * 5 + i] = 1.0;
  F[0 * 5 + 2] = dx * g.m / (g.c0 * g.c1);                      // dy1/ds
  F[0 * 5 + 4] = cq * dx * dx * g.m / (g.c1 * (g.c0 + g.c1));   // dy1/dq
  F[1 * 5 + 2] = t * g.dy / (g.c0 * g.c1);                      // dz1/ds
  F[1 * 5 + 3] = g.dS;                                          // dz1/dt
  F[1 * 5 + 4] = t * cq * g.dSdk;                               // dz1/dq
  F[2 * 5 + 4] = cq * dx;                                       // ds1/dq
}

extern "C" void orc_jacobian(double cq, double dx, const double* st, double* F) {
  Step g;
  if (!step_geometry(cq * st[4], st[2], dx, 1.0, &g)) {
    for (int i = 0; i < 25; ++i) F[i] = std::numeric_limits<double>::quiet_NaN();
    return;
  }
  jacobian_from(g, cq, dx, st[3], F);
}

extern "C" int orc_transport(double cq, double smax, double dx, double* st, double* C) {
  Step g;
  if (!step_geometry(cq * st[4], st[2], dx, smax, &g)) return 0;
  if (C) {
    double F[25], FC[25];
    jacobian_from(g, cq, dx, st[3], F);
    for (int i = 0; i < 5; ++i)
      for (int j = 0; j < 5; ++j) {
        double a = 0.0;
        for (int l = 0; l < 5; ++l) a += F[i * 5 + l] * C[l * 5 + j];
        FC[i * 5 + j] = a;
      }
    for (int i = 0; i < 5; ++i)
      for (int j = 0; j < 5; ++j) {
        double a = 0.0;
        for (int l = 0; l < 5; ++l) a += FC[i * 5 + l] * F[j * 5 + l];
        C[i * 5 + j] = a;
      }
  }
  st[0] += g.dy;
  st[1] += st[3] * g.dS;
  st[2] = g.s1;
  return 1;
}

// Standard Kalman update with H = [I2 | 0], V = diag(sy2, sz2) (Appendix C):
// S = C[0:2,0:2] + V; K = C[:,0:2] S^-1; p += K r; C -= K C[0:2,:]; symmetrise; chi2 = r^T S^-1 r.
extern "C" double orc_update(double* st, double* C, double ym, double zm, double sy2, double sz2) {
  double S00 = C[0] + sy2, S01 = C[1], S10 = C[5], S11 = C[6] + sz2;
  double det = S00 * S11 - S01 * S10;
  double I00 = S11 / det, I01 = -S01 / det, I10 = -S10 / det, I11 = S00 / det;
  double r0 = ym - st[0], r1 = zm - st[1];
  double K[5][2];
  for (int i = 0; i < 5; ++i) {
    K[i][0] = C[i * 5 + 0] * I00 + C[i * 5 + 1] * I10;
    K[i][1] = C[i * 5 + 0] * I01 + C[i * 5 + 1] * I11;
  }
  double HC[2][5];
  for (int j = 0; j < 5; ++j) {
    HC[0][j] = C[0 * 5 + j];
    HC[1][j] = C[1 * 5 + j];
  }
  for (int i = 0; i < 5; ++i) st[i] += K[i][0] * r0 + K[i][1] * r1;
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < 5; ++j) C[i * 5 + j] -= K[i][0] * HC[0][j] + K[i][1] * HC[1][j];
  for (int i = 0; i < 5; ++i)
    for (int j = i + 1; j < 5; ++j) {
      double a = 0.5 * (C[i * 5 + j] + C[j * 5 + i]);
      C[i * 5 + j] = a;
      C[j * 5 + i] = a;
    }
  return r0 * (I00 * r0 + I01 * r1) + r1 * (I10 * r0 + I11 * r1);
}

// ------------------------------------------------------------------------------------------------
// Stage 4: follower.  SURVEY 8(c) "Stage 4" (P15..P24).
// ------------------------------------------------------------------------------------------------
struct FollowCtx {
  const orc_params_t* p;
  double cq;  // cq_per_tesla * Bz
  int32_t n_rows;
  int64_t n_sr;  // n_sectors * n_rows
  const double* row_x;
  const double* y;
  const double* z;
  const uint32_t* ro;
  const int32_t* zorder;  // NULL in search_mode 0
  double sy2, sz2;
};

// P17/P21: among all clusters of the sector-row inside |dy| <= gate_y, |dz| <= gate_z, minimise (d, id),
// d = dy^2/(Cyy + sy2) + dz^2/(Czz + sz2); accept iff d < gate_d.
static int32_t search_row(const FollowCtx& c, int64_t sr, const double* st, const double* C) {
  const orc_params_t* p = c.p;
  double wy = 1.0 / (C[0] + c.sy2), wz = 1.0 / (C[6] + c.sz2);
  double bestd = std::numeric_limits<double>::infinity();
  int32_t best = -1;
  auto consider = [&](int32_t id) {
    double dy = c.y[id] - st[0], dz = c.z[id] - st[1];
    if (std::fabs(dy) > p->gate_y_cm || std::fabs(dz) > p->gate_z_cm) return;
    double d = dy * dy * wy + dz * dz * wz;
    if (d < bestd || (d == bestd && id < best)) {
      bestd = d;
      best = id;
    }
  };
  uint32_t a = c.ro[sr], b = c.ro[sr + 1];
  if (!c.zorder) {
    for (uint32_t h = a; h < b; ++h) consider((int32_t)h);
  } else {
    double zlo = st[1] - p->gate_z_cm - 1e-9, zhi = st[1] + p->gate_z_cm + 1e-9;  // pruning only, superset
    const int32_t* first = std::lower_bound(c.zorder + a, c.zorder + b, zlo,
                                            [&](int32_t id, double v) { return c.z[id] < v; });
    for (const int32_t* it = first; it != c.zorder + b && c.z[*it] <= zhi; ++it) consider(*it);
  }
  return (best >= 0 && bestd < p->gate_d) ? best : -1;
}

static void reset_cov(const orc_params_t* p, double* C) {
  for (int i = 0; i < 25; ++i) C[i] = 0.0;
  for (int i = 0; i < 5; ++i) C[i * 5 + i] = p->c_reset[i];
}

static void follow_one(const FollowCtx& c, int32_t h0, int32_t L, const int32_t* up_c, double* par, double* cov,
                       double* chi2_out, int32_t* n_hits_out, int32_t* hits) {
  const orc_params_t* p = c.p;
  const int32_t nr = c.n_rows;
  // locate (sector,row) of h0 by binary search over the CSR offsets: ro[lo] <= h0 < ro[lo+1]
  int64_t lo = 0, hi = c.n_sr;
  while (hi - lo > 1) {
    int64_t mid = (lo + hi) / 2;
    if (c.ro[mid] <= (uint32_t)h0) lo = mid; else hi = mid;
  }
  const int64_t sec_base = (lo / nr) * nr;
  const int32_t r0 = (int32_t)(lo % nr);
  for (int32_t r = 0; r < nr; ++r) hits[r] = -1;

  // P19 init from the first two chain hits
  int32_t c0 = h0, c1 = up_c[h0];
  double x = c.row_x[r0];
  double dxr = c.row_x[r0 + 1] - c.row_x[r0];
  double dy = c.y[c1] - c.y[c0], dz = c.z[c1] - c.z[c0];
  double chord = std::sqrt(dxr * dxr + dy * dy);
  double st[5] = {c.y[c0], c.z[c0], dy / chord, dz / chord, 0.0};
  double C[25];
  reset_cov(p, C);
  orc_update(st, C, c.y[c0], c.z[c0], c.sy2, c.sz2);
  hits[r0] = c0;
  int32_t row = r0;
  bool fail_up = false;

  // Phase A: fit up the chain, no gate
  int32_t h = c0;
  for (int32_t i = 1; i < L; ++i) {
    h = up_c[h];
    if (!orc_transport(c.cq, p->sinphi_max, c.row_x[r0 + i] - x, st, C)) {
      fail_up = true;
      break;
    }
    row = r0 + i;
    x = c.row_x[row];
    orc_update(st, C, c.y[h], c.z[h], c.sy2, c.sz2);
    hits[row] = h;
  }
  // Phase B: extend up with gated nearest-hit search (P20: stop after max_miss consecutive empty rows)
  if (!fail_up) {
    int32_t miss = 0;
    while (row + 1 <= nr - 1 && miss < p->max_miss) {
      if (!orc_transport(c.cq, p->sinphi_max, c.row_x[row + 1] - x, st, C)) break;
      ++row;
      x = c.row_x[row];
      int32_t f = search_row(c, sec_base + row, st, C);
      if (f >= 0) {
        orc_update(st, C, c.y[f], c.z[f], c.sy2, c.sz2);
        hits[row] = f;
        miss = 0;
      } else {
        ++miss;
      }
    }
  }
  // Phase C: keep the state, reset the covariance (P22), refit downwards over the recorded hits;
  // Phase D: below the seed's first row, search as in B.
  reset_cov(p, C);
  double chi2 = 0.0;
  if (hits[row] >= 0) chi2 += orc_update(st, C, c.y[hits[row]], c.z[hits[row]], c.sy2, c.sz2);
  bool fail_dn = false;
  int32_t miss = 0;
  while (row > 0) {
    if (row - 1 < r0 && miss >= p->max_miss) break;
    if (!orc_transport(c.cq, p->sinphi_max, c.row_x[row - 1] - x, st, C)) {
      fail_dn = true;
      break;
    }
    --row;
    x = c.row_x[row];
    if (row >= r0) {
      if (hits[row] >= 0) chi2 += orc_update(st, C, c.y[hits[row]], c.z[hits[row]], c.sy2, c.sz2);
    } else {
      int32_t f = search_row(c, sec_base + row, st, C);
      if (f >= 0) {
        chi2 += orc_update(st, C, c.y[f], c.z[f], c.sy2, c.sz2);
        hits[row] = f;
        miss = 0;
      } else {
        ++miss;
      }
    }
  }
  // P23: transport (no update) back to the lowest-row hit
  int32_t lowest = 0, nh = 0;
  for (int32_t r = nr - 1; r >= 0; --r)
    if (hits[r] >= 0) {
      lowest = r;
      ++nh;
    }
  if (!fail_dn && lowest != row) {
    if (orc_transport(c.cq, p->sinphi_max, c.row_x[lowest] - x, st, C)) x = c.row_x[lowest];
  }
  par[0] = x;
  for (int i = 0; i < 5; ++i) par[1 + i] = st[i];
  int q = 0;
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j) cov[q++] = C[i * 5 + j];
  *chi2_out = chi2;
  *n_hits_out = nh;
}

extern "C" void orc_follow(const orc_params_t* p, double bz, int32_t n_sectors, int32_t n_rows, const double* row_x,
                           const double* y_cm, const double* z_cm, const uint32_t* ro, const int32_t* up_c,
                           int64_t n_seeds, const int32_t* seed_start, const int32_t* seed_len, int search_mode,
                           double* par, double* cov, double* chi2, int32_t* n_hits, int32_t* hits) {
  std::vector<int32_t> zo;
  if (search_mode == 1) build_zorder<double>((int64_t)n_sectors * n_rows, ro, z_cm, zo);
  FollowCtx c;
  c.p = p;
  c.cq = p->cq_per_tesla * bz;
  c.n_rows = n_rows;
  c.n_sr = (int64_t)n_sectors * n_rows;
  c.row_x = row_x;
  c.y = y_cm;
  c.z = z_cm;
  c.ro = ro;
  c.zorder = search_mode == 1 ? zo.data() : nullptr;
  c.sy2 = p->sigma_y * p->sigma_y;
  c.sz2 = p->sigma_z * p->sigma_z;
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t i = 0; i < n_seeds; ++i) {
    follow_one(c, seed_start[i], seed_len[i], up_c, par + i * 6, cov + i * 15, chi2 + i, n_hits + i,
               hits + i * (int64_t)n_rows);
  }
}

// ------------------------------------------------------------------------------------------------
// Stage 5.  SURVEY 8(c): surviving tracklets have n_hits >= n_min_tracklet (P24); owner(h) = surviving
// tracklet containing h with the largest n_hits, ties -> smallest seed start id (P26); output iff owned
// >= n_min_owned (P27); hit list = owned hits ascending row; output order = ascending seed start id (P29).
// ------------------------------------------------------------------------------------------------
extern "C" int64_t orc_select(const orc_params_t* p, int64_t n, int32_t n_rows, int64_t n_seeds,
                              const int32_t* seed_start, const int32_t* n_hits, const int32_t* hits, int32_t* owner,
                              int32_t* trk_seed, int32_t* trk_n_owned, int32_t* trk_hit_offset, int32_t* hit_ids,
                              int64_t* n_out_hits) {
  for (int64_t h = 0; h < n; ++h) owner[h] = -1;
  for (int64_t i = 0; i < n_seeds; ++i) {
    if (n_hits[i] < p->n_min_tracklet) continue;
    for (int32_t r = 0; r < n_rows; ++r) {
      int32_t h = hits[i * n_rows + r];
      if (h < 0) continue;
      int32_t o = owner[h];
      // seeds ascend by start id, so "smaller start id" == "smaller rank"
      if (o < 0 || n_hits[i] > n_hits[o] || (n_hits[i] == n_hits[o] && seed_start[i] < seed_start[o]))
        owner[h] = (int32_t)i;
    }
  }
  int64_t nt = 0, nh = 0;
  for (int64_t i = 0; i < n_seeds; ++i) {
    if (n_hits[i] < p->n_min_tracklet) continue;
    int32_t owned = 0;
    for (int32_t r = 0; r < n_rows; ++r) {
      int32_t h = hits[i * n_rows + r];
      if (h >= 0 && owner[h] == (int32_t)i) ++owned;
    }
    if (owned < p->n_min_owned) continue;
    trk_seed[nt] = (int32_t)i;
    trk_n_owned[nt] = owned;
    trk_hit_offset[nt] = (int32_t)nh;
    for (int32_t r = 0; r < n_rows; ++r) {
      int32_t h = hits[i * n_rows + r];
      if (h >= 0 && owner[h] == (int32_t)i) hit_ids[nh++] = h;
    }
    ++nt;
  }
  *n_out_hits = nh;
  return nt;
}

// ------------------------------------------------------------------------------------------------
// NEXT-1: refit of an output track over its owned hits only.  Reading P41.
// ------------------------------------------------------------------------------------------------
extern "C" void orc_refit(const orc_params_t* p, double bz, int32_t n_sectors, int32_t n_rows, const double* row_x,
                          const double* y, const double* z, const uint32_t* ro, int64_t n_tracks,
                          const int32_t* trk_hit_offset, const int32_t* trk_n_owned, const int32_t* hit_ids,
                          double* par, double* cov, double* chi2_out, int32_t* n_used) {
  const double cq = p->cq_per_tesla * bz;
  const double sy2 = p->sigma_y * p->sigma_y, sz2 = p->sigma_z * p->sigma_z;
  const int64_t n_sr = (int64_t)n_sectors * n_rows;
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t t = 0; t < n_tracks; ++t) {
    const int32_t* h = hit_ids + trk_hit_offset[t];
    const int32_t m = trk_n_owned[t];
    std::vector<double> xs(m);
    for (int32_t j = 0; j < m; ++j) {   // row of hit j: ro[lo] <= h_j < ro[lo+1]
      int64_t lo = 0, hi = n_sr;
      while (hi - lo > 1) {
        int64_t mid = (lo + hi) / 2;
        if (ro[mid] <= (uint32_t)h[j]) lo = mid; else hi = mid;
      }
      xs[j] = row_x[lo % n_rows];
    }
    double st[5] = {m > 0 ? y[h[0]] : 0.0, m > 0 ? z[h[0]] : 0.0, 0.0, 0.0, 0.0};
    double C[25];
    reset_cov(p, C);
    double x = m > 0 ? xs[0] : 0.0, chi2 = 0.0;
    int32_t used = 0;
    if (m >= 2) {
      const double dx01 = xs[1] - xs[0], dy = y[h[1]] - y[h[0]], dz = z[h[1]] - z[h[0]];
      const double chord = std::sqrt(dx01 * dx01 + dy * dy);
      st[2] = dy / chord;
      st[3] = dz / chord;
    }
    if (m > 0) {
      orc_update(st, C, y[h[0]], z[h[0]], sy2, sz2);
      int32_t last = 0;
      for (int32_t j = 1; j < m; ++j) {   // up
        if (!orc_transport(cq, p->sinphi_max, xs[j] - x, st, C)) break;
        x = xs[j];
        orc_update(st, C, y[h[j]], z[h[j]], sy2, sz2);
        last = j;
      }
      reset_cov(p, C);
      chi2 += orc_update(st, C, y[h[last]], z[h[last]], sy2, sz2);
      used = 1;
      for (int32_t j = last - 1; j >= 0; --j) {   // down
        if (!orc_transport(cq, p->sinphi_max, xs[j] - x, st, C)) break;
        x = xs[j];
        chi2 += orc_update(st, C, y[h[j]], z[h[j]], sy2, sz2);
        ++used;
      }
    }
    par[t * 6] = x;
    for (int i = 0; i < 5; ++i) par[t * 6 + 1 + i] = st[i];
    int q = 0;
    for (int i = 0; i < 5; ++i)
      for (int j = 0; j <= i; ++j) cov[t * 15 + q++] = C[i * 5 + j];
    chi2_out[t] = chi2;
    n_used[t] = used;
  }
}

// ------------------------------------------------------------------------------------------------
// NEXT-1: merging of sector tracks across sector edges, the central membrane and inside a sector.
// Readings P42..P46.  Geometry: the frame of sector s' = s + 1 is the frame of s turned by +20 degrees.
// ------------------------------------------------------------------------------------------------
// P42.  Point (x, y) and direction phi in the old frame; in the frame turned by alpha:
//   x' = x cos a + y sin a,  y' = -x sin a + y cos a,  phi' = phi - a,  z, tan lambda, q/pT unchanged.
// The state is "at the plane x = const", so a variation of y moves the point off the new plane x'; bringing it back
// along the track (dy'/dx' = tan phi', dz/dx' = tan lambda / cos phi', d sin phi'/dx' = k) gives the Jacobian
//   dy'/dy = cos phi / cos phi',  dz'/dy = -sin a tan lambda / cos phi',  dsin phi'/dy = -k sin a,
//   dsin phi'/dsin phi = cos phi' / cos phi,  all other entries as the identity.
extern "C" int orc_rotate(double cq, double smax, double alpha, double* x, double* st, double* C) {
  const double ca = std::cos(alpha), sa = std::sin(alpha);
  const double s = st[2];
  if (!(std::fabs(s) < 1.0)) return 0;
  const double c = std::sqrt(1.0 - s * s);
  const double s1 = s * ca - c * sa, c1 = c * ca + s * sa;
  if (!(c1 > 0.0) || !(std::fabs(s1) < smax)) return 0;
  if (C) {
    double R[25];
    for (int i = 0; i < 25; ++i) R[i] = 0.0;
    for (int i = 0; i < 5; ++i) R[i * 5 + i] = 1.0;
    R[0 * 5 + 0] = c / c1;
    R[1 * 5 + 0] = -sa * st[3] / c1;
    R[2 * 5 + 0] = -sa * cq * st[4];
    R[2 * 5 + 2] = c1 / c;
    double RC[25];
    for (int i = 0; i < 5; ++i)
      for (int j = 0; j < 5; ++j) {
        double a = 0.0;
        for (int l = 0; l < 5; ++l) a += R[i * 5 + l] * C[l * 5 + j];
        RC[i * 5 + j] = a;
      }
    for (int i = 0; i < 5; ++i)
      for (int j = 0; j < 5; ++j) {
        double a = 0.0;
        for (int l = 0; l < 5; ++l) a += RC[i * 5 + l] * R[j * 5 + l];
        C[i * 5 + j] = a;
      }
  }
  const double x0 = *x, y0 = st[0];
  *x = x0 * ca + y0 * sa;
  st[0] = -x0 * sa + y0 * ca;
  st[2] = s1;
  return 1;
}

static void unpack_cov(const double* c15, double* C) {
  int q = 0;
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j) {
      C[i * 5 + j] = c15[q];
      C[j * 5 + i] = c15[q];
      ++q;
    }
}

// P44.  chi2 = D^T S^-1 D by Cholesky S = L L^T (S is the sum of two covariances).
extern "C" double orc_match_chi2(double cq, double smax, double alpha, const double* pa, const double* ca15,
                                 const double* pb, const double* cb15) {
  double x = pa[0], st[5], Ca[25], Cb[25];
  for (int i = 0; i < 5; ++i) st[i] = pa[1 + i];
  unpack_cov(ca15, Ca);
  unpack_cov(cb15, Cb);
  if (alpha != 0.0 && !orc_rotate(cq, smax, alpha, &x, st, Ca)) return -1.0;
  if (!orc_transport(cq, smax, pb[0] - x, st, Ca)) return -1.0;
  double S[25], D[5], L[25];
  for (int i = 0; i < 25; ++i) S[i] = Ca[i] + Cb[i];
  for (int i = 0; i < 5; ++i) D[i] = pb[1 + i] - st[i];
  for (int i = 0; i < 25; ++i) L[i] = 0.0;
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j) {
      double a = S[i * 5 + j];
      for (int l = 0; l < j; ++l) a -= L[i * 5 + l] * L[j * 5 + l];
      if (i == j) {
        if (!(a > 0.0)) return -1.0;
        L[i * 5 + i] = std::sqrt(a);
      } else {
        L[i * 5 + j] = a / L[j * 5 + j];
      }
    }
  double chi2 = 0.0, w[5];
  for (int i = 0; i < 5; ++i) {   // forward substitution L w = D; chi2 = |w|^2
    double a = D[i];
    for (int l = 0; l < i; ++l) a -= L[i * 5 + l] * w[l];
    w[i] = a / L[i * 5 + i];
    chi2 += w[i] * w[i];
  }
  return chi2;
}

// P43: is a -> b a candidate, and by which rotation?
static bool merge_candidate(int32_t n_per_side, double sector_angle, int32_t gap_max, int32_t sa, int32_t sb,
                            int32_t last_a, int32_t first_b, double* alpha) {
  const int32_t g = first_b - last_a;
  if (g < 1 || g > gap_max) return false;
  if (sa == sb) {
    *alpha = 0.0;
    return true;
  }
  const int32_t side_a = sa / n_per_side, side_b = sb / n_per_side;
  const int32_t ia = sa % n_per_side, ib = sb % n_per_side;
  if (side_a == side_b) {
    const int32_t d = ((ib - ia) % n_per_side + n_per_side) % n_per_side;
    if (d == 1) { *alpha = sector_angle; return true; }
    if (d == n_per_side - 1) { *alpha = -sector_angle; return true; }
    return false;
  }
  // across the central membrane: same azimuth, other side of the same event (a batch of events is laid out as
  // groups of 2 n_per_side sectors)
  if (ia == ib && sa / (2 * n_per_side) == sb / (2 * n_per_side)) {
    *alpha = 0.0;
    return true;
  }
  return false;
}

extern "C" int64_t orc_merge(double cq, double smax, int32_t n_per_side, double sector_angle, int32_t gap_max,
                             double chi2_max, int64_t nt, const double* par, const double* cov, const int32_t* sector,
                             const int32_t* first_row, const int32_t* last_row, int32_t* succ, int32_t* pred,
                             double* link_chi2) {
  std::vector<int32_t> best_s(nt, -1), best_p(nt, -1);
  std::vector<double> chi_s(nt, std::numeric_limits<double>::infinity()), chi_p(nt, std::numeric_limits<double>::infinity());
  // plain all-pairs scan; ascending b (a) with a strict "<" keeps the smaller index on ties (P45)
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t a = 0; a < nt; ++a)
    for (int64_t b = 0; b < nt; ++b) {
      double alpha;
      if (a == b || !merge_candidate(n_per_side, sector_angle, gap_max, sector[a], sector[b], last_row[a], first_row[b], &alpha)) continue;
      const double c = orc_match_chi2(cq, smax, alpha, par + a * 6, cov + a * 15, par + b * 6, cov + b * 15);
      if (c < 0.0 || !(c < chi2_max)) continue;
      if (c < chi_s[a]) { chi_s[a] = c; best_s[a] = (int32_t)b; }
    }
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t b = 0; b < nt; ++b)
    for (int64_t a = 0; a < nt; ++a) {
      double alpha;
      if (a == b || !merge_candidate(n_per_side, sector_angle, gap_max, sector[a], sector[b], last_row[a], first_row[b], &alpha)) continue;
      const double c = orc_match_chi2(cq, smax, alpha, par + a * 6, cov + a * 15, par + b * 6, cov + b * 15);
      if (c < 0.0 || !(c < chi2_max)) continue;
      if (c < chi_p[b]) { chi_p[b] = c; best_p[b] = (int32_t)a; }
    }
  int64_t links = 0;
  for (int64_t t = 0; t < nt; ++t) { succ[t] = -1; pred[t] = -1; link_chi2[t] = -1.0; }
  for (int64_t a = 0; a < nt; ++a) {
    const int32_t b = best_s[a];
    if (b >= 0 && best_p[b] == (int32_t)a) {
      succ[a] = b;
      pred[b] = (int32_t)a;
      link_chi2[a] = chi_s[a];
      ++links;
    }
  }
  return links;
}

// ------------------------------------------------------------------------------------------------
// P47: refit over a chain of linked tracks (the "global refit" of SURVEY 8(f) NEXT-1).
// ------------------------------------------------------------------------------------------------
// angle by which the frame of sector sb is turned against the frame of sa (P42); the pair must be related (P43)
static double frame_angle(int32_t n_per_side, double sector_angle, int32_t sa, int32_t sb) {
  if (sa == sb) return 0.0;
  if (sa / n_per_side != sb / n_per_side) return 0.0;   // across the membrane: same frame
  const int32_t d = ((sb % n_per_side - sa % n_per_side) % n_per_side + n_per_side) % n_per_side;
  return d == 1 ? sector_angle : -sector_angle;
}

extern "C" void orc_refit_merged(const orc_params_t* p, double bz, int32_t n_sectors, int32_t n_rows,
                                 const double* row_x, const double* y, const double* z, const uint32_t* ro,
                                 int32_t n_per_side, double sector_angle, int64_t n_tracks,
                                 const int32_t* trk_hit_offset, const int32_t* trk_n_owned, const int32_t* hit_ids,
                                 const int32_t* succ, const int32_t* pred, double* par, double* cov, double* chi2_out,
                                 int32_t* n_used, int32_t* out_sector) {
  const double cq = p->cq_per_tesla * bz;
  const double sy2 = p->sigma_y * p->sigma_y, sz2 = p->sigma_z * p->sigma_z;
  const int64_t n_sr = (int64_t)n_sectors * n_rows;
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t t = 0; t < n_tracks; ++t) {
    n_used[t] = 0;
    if (pred[t] >= 0) continue;
    // the chain's hits with their row x and sector
    std::vector<int32_t> h;
    for (int64_t c = t; c >= 0; c = succ[c])
      for (int32_t j = 0; j < trk_n_owned[c]; ++j) h.push_back(hit_ids[trk_hit_offset[c] + j]);
    const int32_t m = (int32_t)h.size();
    std::vector<double> xs(m);
    std::vector<int32_t> sec(m);
    for (int32_t j = 0; j < m; ++j) {
      int64_t lo = 0, hi = n_sr;
      while (hi - lo > 1) {
        int64_t mid = (lo + hi) / 2;
        if (ro[mid] <= (uint32_t)h[j]) lo = mid; else hi = mid;
      }
      xs[j] = row_x[lo % n_rows];
      sec[j] = (int32_t)(lo / n_rows);
    }
    if (m == 0) continue;
    double st[5] = {y[h[0]], z[h[0]], 0.0, 0.0, 0.0};
    double C[25];
    reset_cov(p, C);
    double x = xs[0], chi2 = 0.0;
    int32_t cur = sec[0], used = 0;
    if (m >= 2 && sec[1] == sec[0]) {   // a chain's first track owns >= n_min_owned hits of one sector
      const double dx01 = xs[1] - xs[0], dy = y[h[1]] - y[h[0]], dz = z[h[1]] - z[h[0]];
      const double chord = std::sqrt(dx01 * dx01 + dy * dy);
      st[2] = dy / chord;
      st[3] = dz / chord;
    }
    // move the state to hit j: rotate into its sector's frame if needed, then transport to its row
    // (all or nothing: if the rotation works but the transport fails, the state stays in the old frame)
    auto move_to = [&](int32_t j) -> bool {
      if (sec[j] != cur) {
        double x2 = x, st2[5], C2[25];
        for (int i = 0; i < 5; ++i) st2[i] = st[i];
        for (int i = 0; i < 25; ++i) C2[i] = C[i];
        const double a = frame_angle(n_per_side, sector_angle, cur, sec[j]);
        if (a != 0.0 && !orc_rotate(cq, p->sinphi_max, a, &x2, st2, C2)) return false;
        if (!orc_transport(cq, p->sinphi_max, xs[j] - x2, st2, C2)) return false;
        for (int i = 0; i < 5; ++i) st[i] = st2[i];
        for (int i = 0; i < 25; ++i) C[i] = C2[i];
        cur = sec[j];
        x = xs[j];
        return true;
      }
      if (!orc_transport(cq, p->sinphi_max, xs[j] - x, st, C)) return false;
      x = xs[j];
      return true;
    };
    orc_update(st, C, y[h[0]], z[h[0]], sy2, sz2);
    int32_t last = 0;
    for (int32_t j = 1; j < m; ++j) {   // up
      if (!move_to(j)) break;
      orc_update(st, C, y[h[j]], z[h[j]], sy2, sz2);
      last = j;
    }
    reset_cov(p, C);
    chi2 += orc_update(st, C, y[h[last]], z[h[last]], sy2, sz2);
    used = 1;
    for (int32_t j = last - 1; j >= 0; --j) {   // down
      if (!move_to(j)) break;
      chi2 += orc_update(st, C, y[h[j]], z[h[j]], sy2, sz2);
      ++used;
    }
    par[t * 6] = x;
    for (int i = 0; i < 5; ++i) par[t * 6 + 1 + i] = st[i];
    int q = 0;
    for (int i = 0; i < 5; ++i)
      for (int j = 0; j <= i; ++j) cov[t * 15 + q++] = C[i * 5 + j];
    chi2_out[t] = chi2;
    n_used[t] = used;
    out_sector[t] = cur;
  }
}

// ------------------------------------------------------------------------------------------------
// NEXT-3: track-model residual transform.  Readings P50..P52.
// ------------------------------------------------------------------------------------------------
static inline int64_t floor_div(int64_t a, int64_t b) {   // b > 0
  int64_t q = a / b;
  if ((a % b != 0) && (a < 0)) --q;
  return q;
}

// P50 predictor for hit j >= 2 from the previous hits' rows r[] and coordinates c[] (j indexes the current hit)
static inline int64_t predict(const int32_t* r, const int32_t* c, int32_t j) {
  const bool four = j >= 4 && r[j] - r[j - 1] == 1 && r[j - 1] - r[j - 2] == 1 && r[j - 2] - r[j - 3] == 1 &&
                    r[j - 3] - r[j - 4] == 1;
  if (four) return floor_div(2 * (int64_t)c[j - 1] + c[j - 2] - c[j - 4], 2);
  const int64_t g1 = r[j - 1] - r[j - 2], g2 = r[j] - r[j - 1];
  return (int64_t)c[j - 1] + floor_div(((int64_t)c[j - 1] - c[j - 2]) * g2, g1);
}

extern "C" void orc_compress(int32_t n_rows, const int32_t* y, const int32_t* z, const uint32_t* ro, int64_t n_sr,
                             int64_t n_tracks, const int32_t* off, const int32_t* cnt, const int32_t* hit_ids,
                             uint8_t* drow, int32_t* ry, int32_t* rz) {
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t t = 0; t < n_tracks; ++t) {
    const int32_t m = cnt[t];
    std::vector<int32_t> r(m), cy(m), cz(m);
    for (int32_t j = 0; j < m; ++j) {
      const int32_t h = hit_ids[off[t] + j];
      int64_t lo = 0, hi = n_sr;
      while (hi - lo > 1) {
        int64_t mid = (lo + hi) / 2;
        if (ro[mid] <= (uint32_t)h) lo = mid; else hi = mid;
      }
      r[j] = (int32_t)(lo % n_rows);
      cy[j] = y[h];
      cz[j] = z[h];
    }
    for (int32_t j = 0; j < m; ++j) {
      const int64_t k = off[t] + j;
      if (j == 0) {
        drow[k] = (uint8_t)r[0];
        ry[k] = cy[0];
        rz[k] = cz[0];
      } else if (j == 1) {
        drow[k] = (uint8_t)(r[1] - r[0]);
        ry[k] = cy[1] - cy[0];
        rz[k] = cz[1] - cz[0];
      } else {
        drow[k] = (uint8_t)(r[j] - r[j - 1]);
        ry[k] = (int32_t)(cy[j] - predict(r.data(), cy.data(), j));
        rz[k] = (int32_t)(cz[j] - predict(r.data(), cz.data(), j));
      }
    }
  }
}

extern "C" void orc_decompress(int64_t n_tracks, const int32_t* off, const int32_t* cnt, const uint8_t* drow,
                               const int32_t* ry, const int32_t* rz, int32_t* row, int32_t* y, int32_t* z) {
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t t = 0; t < n_tracks; ++t) {
    const int32_t m = cnt[t];
    int32_t* r = row + off[t];
    int32_t* cy = y + off[t];
    int32_t* cz = z + off[t];
    for (int32_t j = 0; j < m; ++j) {
      const int64_t k = off[t] + j;
      if (j == 0) {
        r[0] = drow[k];
        cy[0] = ry[k];
        cz[0] = rz[k];
      } else if (j == 1) {
        r[1] = r[0] + drow[k];
        cy[1] = cy[0] + ry[k];
        cz[1] = cz[0] + rz[k];
      } else {
        r[j] = r[j - 1] + drow[k];
        cy[j] = (int32_t)(predict(r, cy, j) + ry[k]);
        cz[j] = (int32_t)(predict(r, cz, j) + rz[k]);
      }
    }
  }
}

extern "C" void orc_residual_histogram(int64_t n_tracks, const int32_t* off, const int32_t* cnt, const int32_t* res,
                                       int32_t j_min, int64_t* hist) {
  for (int i = 0; i < 65536; ++i) hist[i] = 0;
  for (int64_t t = 0; t < n_tracks; ++t)
    for (int32_t j = j_min; j < cnt[t]; ++j) {
      int64_t v = (int64_t)res[off[t] + j] + 32768;
      if (v < 0) v = 0;
      if (v > 65535) v = 65535;
      ++hist[v];
    }
}

// ------------------------------------------------------------------------------------------------
// NEXT-3, entropy stage: static rANS over chunks.  Readings P57..P60 (tpc_oracle.h).
// ------------------------------------------------------------------------------------------------
static const uint64_t RANS_M = 65536;   // probabilities in units of 1/M; also the lower bound of the state

extern "C" int32_t orc_rans_symbol(int32_t v, int32_t alphabet_bits) {   // P57
  const int64_t half = (int64_t)1 << (alphabet_bits - 1);
  return ((int64_t)v > -half && (int64_t)v < half) ? (int32_t)(v + half) : 0;
}

extern "C" void orc_rans_normalise(int32_t alphabet, const int64_t* counts, uint32_t* freq) {   // P58
  int64_t N = 0, K = 0;
  for (int32_t s = 0; s < alphabet; ++s) {
    N += counts[s];
    if (counts[s] > 0) ++K;
    freq[s] = 0;
  }
  if (N == 0) return;
  int64_t sum = 0;
  int32_t top = 0;
  for (int32_t s = 0; s < alphabet; ++s) {
    if (counts[s] == 0) continue;
    freq[s] = (uint32_t)(1 + (counts[s] * ((int64_t)RANS_M - K)) / N);
    sum += freq[s];
    if (counts[s] > counts[top]) top = s;   // the first of the most frequent
  }
  freq[top] += (uint32_t)((int64_t)RANS_M - sum);
}

extern "C" int64_t orc_rans_encode(const int32_t* values, int64_t n, int32_t alphabet_bits, int32_t chunk,
                                   uint32_t* freq, uint32_t* chunk_off, uint32_t* esc_off, uint8_t* payload,
                                   int32_t* escapes) {
  const int32_t A = 1 << alphabet_bits;
  std::vector<int64_t> counts((size_t)A, 0);
  for (int64_t i = 0; i < n; ++i) ++counts[orc_rans_symbol(values[i], alphabet_bits)];
  orc_rans_normalise(A, counts.data(), freq);
  std::vector<uint64_t> cum((size_t)A + 1, 0);
  for (int32_t s = 0; s < A; ++s) cum[s + 1] = cum[s] + freq[s];
  const int64_t n_chunks = (n + chunk - 1) / chunk;
  int64_t bytes = 0, n_esc = 0;
  chunk_off[0] = 0;
  esc_off[0] = 0;
  for (int64_t c = 0; c < n_chunks; ++c) {
    const int64_t i0 = c * chunk, i1 = std::min<int64_t>(n, i0 + chunk);
    for (int64_t i = i0; i < i1; ++i)   // escapes in stream order
      if (orc_rans_symbol(values[i], alphabet_bits) == 0) escapes[n_esc++] = values[i];
    std::vector<uint16_t> words;   // in emission order
    uint64_t x = RANS_M;
    for (int64_t i = i1 - 1; i >= i0; --i) {
      const int32_t s = orc_rans_symbol(values[i], alphabet_bits);
      const uint64_t f = freq[s];
      if (x >= f * 65536) {
        words.push_back((uint16_t)(x & 0xFFFF));
        x >>= 16;
      }
      x = (x / f) * RANS_M + (x % f) + cum[s];
    }
    for (int b = 0; b < 4; ++b) payload[bytes++] = (uint8_t)((x >> (8 * b)) & 0xFF);
    for (size_t k = words.size(); k-- > 0;) {   // the decoder reads the last emitted word first
      payload[bytes++] = (uint8_t)(words[k] & 0xFF);
      payload[bytes++] = (uint8_t)(words[k] >> 8);
    }
    chunk_off[c + 1] = (uint32_t)bytes;
    esc_off[c + 1] = (uint32_t)n_esc;
  }
  return bytes;
}

extern "C" void orc_rans_decode(int64_t n, int32_t alphabet_bits, int32_t chunk, const uint32_t* freq,
                                const uint32_t* chunk_off, const uint32_t* esc_off, const uint8_t* payload,
                                const int32_t* escapes, int32_t* values) {
  const int32_t A = 1 << alphabet_bits;
  const int64_t half = (int64_t)A / 2;
  std::vector<uint64_t> cum((size_t)A + 1, 0);
  for (int32_t s = 0; s < A; ++s) cum[s + 1] = cum[s] + freq[s];
  const int64_t n_chunks = (n + chunk - 1) / chunk;
  for (int64_t c = 0; c < n_chunks; ++c) {
    const int64_t i0 = c * chunk, i1 = std::min<int64_t>(n, i0 + chunk);
    const uint8_t* in = payload + chunk_off[c];
    uint64_t x = 0;
    for (int b = 0; b < 4; ++b) x |= (uint64_t)(*in++) << (8 * b);
    int64_t e = esc_off[c];
    for (int64_t i = i0; i < i1; ++i) {
      const uint64_t slot = x % RANS_M;
      // the symbol whose interval [c_s, c_s + f_s) holds the slot (binary search over the cumulative table)
      const int32_t s = (int32_t)(std::upper_bound(cum.begin(), cum.end(), slot) - cum.begin()) - 1;
      x = (uint64_t)freq[s] * (x / RANS_M) + slot - cum[s];
      if (x < RANS_M) {
        const uint64_t w = (uint64_t)in[0] | ((uint64_t)in[1] << 8);
        in += 2;
        x = x * 65536 + w;
      }
      values[i] = s == 0 ? escapes[e++] : (int32_t)(s - half);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// NEXT-2: clusterizer.  Readings P53..P56.  A dense (time x pad) image per row.
// ------------------------------------------------------------------------------------------------
static inline int64_t rdiv(int64_t a, int64_t b) {   // floor((2a + b) / (2b)), b > 0: round to nearest, halves up
  const int64_t n = 2 * a + b, d = 2 * b;
  int64_t q = n / d;
  if ((n % d != 0) && (n < 0)) --q;
  return q;
}

extern "C" int64_t orc_clusterize(int32_t n_sectors, int32_t n_rows, int32_t n_per_side, int32_t n_pads,
                                  int32_t n_time, int32_t pad_units, int32_t time_units, int32_t q_peak_min,
                                  const uint16_t* pad, const uint16_t* time, const uint16_t* adc,
                                  const uint32_t* doff, int32_t* y, int32_t* z, int32_t* qtot, int32_t* qmax,
                                  uint32_t* row_offsets) {
  const int64_t n_sr = (int64_t)n_sectors * n_rows;
  const int64_t W = n_pads + 2, H = n_time + 2;   // one empty cell of margin all around
  std::vector<int32_t> img((size_t)(W * H), 0);
  const int64_t y_off = ((int64_t)(n_pads - 1) * pad_units) / 2;   // non-negative: floor
  int64_t nc = 0;
  row_offsets[0] = 0;
  for (int64_t sr = 0; sr < n_sr; ++sr) {
    const int32_t side = (int32_t)((sr / n_rows) / n_per_side) % 2;
    for (uint32_t i = doff[sr]; i < doff[sr + 1]; ++i) img[(size_t)((time[i] + 1) * W + pad[i] + 1)] = adc[i];
    for (uint32_t i = doff[sr]; i < doff[sr + 1]; ++i) {   // digits ascend by (time, pad): so do the peaks (P55)
      const int32_t a = adc[i];
      if (a < q_peak_min) continue;
      const int64_t c = (int64_t)(time[i] + 1) * W + pad[i] + 1;
      bool peak = true;
      int64_t Q = 0, Sy = 0, St = 0;
      for (int dt = -1; dt <= 1; ++dt)
        for (int dp = -1; dp <= 1; ++dp) {
          const int32_t v = img[(size_t)(c + dt * W + dp)];
          Q += v;
          Sy += (int64_t)v * dp;
          St += (int64_t)v * dt;
          if (dt == 0 && dp == 0) continue;
          const bool before = dt < 0 || (dt == 0 && dp < 0);   // precedes (t, p) in (time, pad) order
          if (before ? !(a > v) : !(a >= v)) peak = false;
        }
      if (!peak) continue;
      const int64_t yy = (int64_t)pad[i] * pad_units - y_off + rdiv((int64_t)pad_units * Sy, Q);
      const int64_t zz = (int64_t)time[i] * time_units + rdiv((int64_t)time_units * St, Q);
      y[nc] = (int32_t)yy;
      z[nc] = (int32_t)(side ? -zz : zz);
      qtot[nc] = (int32_t)Q;
      qmax[nc] = a;
      ++nc;
    }
    for (uint32_t i = doff[sr]; i < doff[sr + 1]; ++i) img[(size_t)((time[i] + 1) * W + pad[i] + 1)] = 0;
    row_offsets[sr + 1] = (uint32_t)nc;
  }
  return nc;
}
