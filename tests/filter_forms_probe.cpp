// filter_forms_probe.cpp -- TEST INFRASTRUCTURE (tests/test_filter_forms.py), neither product nor oracle.
// Replays the a4 filter schedule (SURVEY 8(c) Stage 4: fit up, reset, refit down, final transport) over GIVEN hit
// tables in a chosen arithmetic, to measure which fp32 form of the filter keeps the 1e-4 bar against the fp64 oracle:
//   replay:   positions as plain floats relative to the first cluster; variants fp64 covariance (0), fp32 covariance
//             (1), fp32 Joseph form (2), fp32 U-D factors with Bierman updates (3), fp64 U-D (4)
//   replay_s: positions split into an integer origin + fp32 fraction (what kalman.cuh does); variants 1, 2, 3 as above
// It shares no code with csrc/ or oracle/: the arithmetic is restated here so that the forms can be compared.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <vector>

template <typename R>
struct St { R y, z, s, t, q; };

template <typename R>
struct Geo { R dy, dS, s1, a, b, c, d, e, f; };

template <typename R>
static bool geom(R cq, R smax, R dx, const St<R>& p, Geo<R>& g) {
  R k = cq * p.q, s0 = p.s, s1 = s0 + k * dx;
  if (!(std::fabs(s0) < smax) || !(std::fabs(s1) < smax)) return false;
  R c0 = std::sqrt(1 - s0 * s0), c1 = std::sqrt(1 - s1 * s1);
  R tau = (s0 + s1) / (c0 + c1);
  R dy = dx * tau;
  R chord = std::copysign(std::sqrt(dx * dx + dy * dy), dx);
  R u = R(0.5) * k * chord;
  R dS = (std::fabs(u) < R(1e-3)) ? chord * (1 + u * u / 6 + 3 * u * u * u * u / 40) : chord * std::asin(u) / u;
  R dd = R(0.5) * k * dS;
  R sinc = (std::fabs(dd) < R(1e-2)) ? 1 - dd * dd / 6 + dd*dd*dd*dd/120 : std::sin(dd) / dd;
  R gg = (std::fabs(dd) < R(1e-1)) ? R(1.0 / 3) - dd * dd / 30 + dd * dd * dd * dd / 840 : (std::sin(dd) - dd * std::cos(dd)) / (dd * dd * dd);
  R cm = 1 / std::sqrt(1 + tau * tau), sm = tau * cm;
  R m = c0 + s0 * tau;
  R dSdk = (R(0.5) * dS * dS * sm * sinc + R(0.25) * k * dS * dS * dS * cm * gg) / c1;
  g.dy = dy; g.dS = dS; g.s1 = s1;
  g.a = dx * m / (c0 * c1);
  g.b = cq * dx * dx * m / (c1 * (c0 + c1));
  g.c = p.t * dy / (c0 * c1);
  g.d = dS;
  g.e = p.t * cq * dSdk;
  g.f = cq * dx;
  return true;
}

// ---- standard covariance form (full 5x5) ----
template <typename R, int JOSEPH>
struct FilterCov {
  R C[5][5];
  void reset(const double* cr) { for (int i = 0; i < 5; ++i) for (int j = 0; j < 5; ++j) C[i][j] = i == j ? (R)cr[i] : 0; }
  void transport(const Geo<R>& g) {
    R F[5][5] = {};
    for (int i = 0; i < 5; ++i) F[i][i] = 1;
    F[0][2] = g.a; F[0][4] = g.b; F[1][2] = g.c; F[1][3] = g.d; F[1][4] = g.e; F[2][4] = g.f;
    R M[5][5];
    for (int i = 0; i < 5; ++i) for (int j = 0; j < 5; ++j) { R a = 0; for (int l = 0; l < 5; ++l) a += F[i][l] * C[l][j]; M[i][j] = a; }
    for (int i = 0; i < 5; ++i) for (int j = 0; j < 5; ++j) { R a = 0; for (int l = 0; l < 5; ++l) a += M[i][l] * F[j][l]; C[i][j] = a; }
  }
  R update(St<R>& p, R ym, R zm, R sy2, R sz2) {
    R S00 = C[0][0] + sy2, S01 = C[0][1], S11 = C[1][1] + sz2;
    R det = S00 * S11 - S01 * S01;
    R I00 = S11 / det, I01 = -S01 / det, I11 = S00 / det;
    R r0 = ym - p.y, r1 = zm - p.z;
    R K[5][2];
    for (int i = 0; i < 5; ++i) { K[i][0] = C[i][0] * I00 + C[i][1] * I01; K[i][1] = C[i][0] * I01 + C[i][1] * I11; }
    R* ps = &p.y;
    for (int i = 0; i < 5; ++i) ps[i] += K[i][0] * r0 + K[i][1] * r1;
    R N[5][5];
    if (!JOSEPH) {
      for (int i = 0; i < 5; ++i) for (int j = 0; j < 5; ++j) N[i][j] = C[i][j] - (K[i][0] * C[0][j] + K[i][1] * C[1][j]);
    } else {   // (I-KH) C (I-KH)^T + K V K^T
      R A[5][5];
      for (int i = 0; i < 5; ++i) for (int j = 0; j < 5; ++j) A[i][j] = (i == j ? 1 : 0) - (j < 2 ? K[i][j] : 0);
      R M[5][5];
      for (int i = 0; i < 5; ++i) for (int j = 0; j < 5; ++j) { R a = 0; for (int l = 0; l < 5; ++l) a += A[i][l] * C[l][j]; M[i][j] = a; }
      for (int i = 0; i < 5; ++i) for (int j = 0; j < 5; ++j) { R a = 0; for (int l = 0; l < 5; ++l) a += M[i][l] * A[j][l]; N[i][j] = a + K[i][0] * sy2 * K[j][0] + K[i][1] * sz2 * K[j][1]; }
    }
    for (int i = 0; i < 5; ++i) for (int j = 0; j < 5; ++j) C[i][j] = R(0.5) * (N[i][j] + N[j][i]);
    return r0 * (I00 * r0 + I01 * r1) + r1 * (I01 * r0 + I11 * r1);
  }
  void cov_out(double* o) { int q = 0; for (int i = 0; i < 5; ++i) for (int j = 0; j <= i; ++j) o[q++] = C[i][j]; }
};

// ---- UD form: C = U D U^T, U unit upper triangular.  F is unit upper triangular too, so U <- F U, D unchanged. ----
template <typename R>
struct FilterUD {
  R U[5][5], D[5];
  void reset(const double* cr) { for (int i = 0; i < 5; ++i) { D[i] = (R)cr[i]; for (int j = 0; j < 5; ++j) U[i][j] = i == j ? 1 : 0; } }
  void transport(const Geo<R>& g) {
    // row 0 += a row2 + b row4 ; row 1 += c row2 + d row3 + e row4 ; row 2 += f row4
    U[0][2] += g.a; U[0][3] += g.a * U[2][3]; U[0][4] += g.a * U[2][4] + g.b;
    U[1][2] += g.c; U[1][3] += g.c * U[2][3] + g.d; U[1][4] += g.c * U[2][4] + g.d * U[3][4] + g.e;
    U[2][4] += g.f;
  }
  // Bierman scalar update, measurement of component m with variance Rv.  Returns chi2 increment.
  R scalar(St<R>& p, int m, R meas, R Rv) {
    R* ps = &p.y;
    R b[5] = {0, 0, 0, 0, 0};
    R alpha = Rv;
    for (int j = m; j < 5; ++j) {
      R fj = j == m ? R(1) : U[m][j];
      R vj = D[j] * fj;
      R an = alpha + fj * vj;
      R lam = -fj / alpha;
      D[j] = D[j] * alpha / an;
      for (int i = 0; i < j; ++i) {
        R uij = U[i][j];
        U[i][j] = uij + lam * b[i];
        b[i] += uij * vj;
      }
      b[j] = vj;
      alpha = an;
    }
    R r = meas - ps[m];
    R ia = 1 / alpha;
    for (int i = 0; i < 5; ++i) ps[i] += b[i] * (r * ia);
    return r * r * ia;
  }
  R update(St<R>& p, R ym, R zm, R sy2, R sz2) {
    R c = scalar(p, 0, ym, sy2);
    c += scalar(p, 1, zm, sz2);
    return c;
  }
  void cov_out(double* o) {
    int q = 0;
    for (int i = 0; i < 5; ++i) for (int j = 0; j <= i; ++j) {
      double a = 0;
      for (int l = 0; l < 5; ++l) a += (double)U[i][l] * (double)D[l] * (double)U[j][l];
      o[q++] = a;
    }
  }
};

template <typename R, typename FL>
static void replay_one(const double* prm, int nr, const double* row_x, const double* y, const double* z, int r0, int L,
                       const int32_t* hits, double* par, double* cov, double* chi2o) {
  const R cq = (R)prm[0], smax = (R)prm[1], sy2 = (R)prm[2], sz2 = (R)prm[3];
  const int max_miss = (int)prm[4];
  const double* cr = prm + 5;
  const int h0 = hits[r0], h1 = hits[r0 + 1];
  const double y0 = y[h0], z0 = z[h0];   // coordinates relative to the first cluster, as the device does
  auto Y = [&](int h) { return (R)(y[h] - y0); };
  auto Z = [&](int h) { return (R)(z[h] - z0); };
  R dxr = (R)(row_x[r0 + 1] - row_x[r0]);
  R dy = Y(h1), dz = Z(h1);
  R chord = std::sqrt(dxr * dxr + dy * dy);
  St<R> p = {0, 0, dy / chord, dz / chord, 0};
  FL f;
  f.reset(cr);
  f.update(p, Y(h0), Z(h0), sy2, sz2);
  int row = r0;
  bool fail_up = false;
  Geo<R> g;
  for (int i = 1; i < L; ++i) {
    if (!geom<R>(cq, smax, (R)(row_x[row + 1] - row_x[row]), p, g)) { fail_up = true; break; }
    f.transport(g); p.y += g.dy; p.z += p.t * g.dS; p.s = g.s1;
    ++row;
    f.update(p, Y(hits[row]), Z(hits[row]), sy2, sz2);
  }
  if (!fail_up) {
    int miss = 0;
    while (row + 1 <= nr - 1 && miss < max_miss) {
      if (!geom<R>(cq, smax, (R)(row_x[row + 1] - row_x[row]), p, g)) break;
      f.transport(g); p.y += g.dy; p.z += p.t * g.dS; p.s = g.s1;
      ++row;
      if (hits[row] >= 0) { f.update(p, Y(hits[row]), Z(hits[row]), sy2, sz2); miss = 0; } else ++miss;
    }
  }
  f.reset(cr);
  R chi2 = 0;
  if (hits[row] >= 0) chi2 += f.update(p, Y(hits[row]), Z(hits[row]), sy2, sz2);
  bool fail_dn = false;
  int miss = 0;
  while (row > 0) {
    if (row - 1 < r0 && miss >= max_miss) break;
    if (!geom<R>(cq, smax, (R)(row_x[row - 1] - row_x[row]), p, g)) { fail_dn = true; break; }
    f.transport(g); p.y += g.dy; p.z += p.t * g.dS; p.s = g.s1;
    --row;
    if (row >= r0) {
      if (hits[row] >= 0) chi2 += f.update(p, Y(hits[row]), Z(hits[row]), sy2, sz2);
    } else {
      if (hits[row] >= 0) { chi2 += f.update(p, Y(hits[row]), Z(hits[row]), sy2, sz2); miss = 0; } else ++miss;
    }
  }
  int lowest = 0;
  for (int r = nr - 1; r >= 0; --r) if (hits[r] >= 0) lowest = r;
  if (!fail_dn && lowest != row) {
    if (geom<R>(cq, smax, (R)(row_x[lowest] - row_x[row]), p, g)) { f.transport(g); p.y += g.dy; p.z += p.t * g.dS; p.s = g.s1; row = lowest; }
  }
  par[0] = row_x[row]; par[1] = (double)p.y + y0; par[2] = (double)p.z + z0; par[3] = p.s; par[4] = p.t; par[5] = p.q;
  f.cov_out(cov);
  *chi2o = chi2;
}


// Split positions: y, z = integer origin (units) + fp32 fraction (units); everything else fp32 in cm.
template <typename FL>
static void replay_split(const double* prm, int nr, const double* row_x, const int32_t* yi, const int32_t* zi, int r0, int L,
                         const int32_t* hits, double* par, double* cov, double* chi2o) {
  typedef float R;
  const R cq = (R)prm[0], smax = (R)prm[1], sy2 = (R)prm[2], sz2 = (R)prm[3];
  const int max_miss = (int)prm[4];
  const double* cr = prm + 5;
  const R U = 640.f, IU = 1.f / 640.f;
  const int h0 = hits[r0], h1 = hits[r0 + 1];
  int64_t oy = yi[h0], oz = zi[h0];
  R dxr = (R)(row_x[r0 + 1] - row_x[r0]);
  R dy = (R)(yi[h1] - yi[h0]) * IU, dz = (R)(zi[h1] - zi[h0]) * IU;
  R chord = std::sqrt(dxr * dxr + dy * dy);
  St<R> p = {0, 0, dy / chord, dz / chord, 0};   // p.y, p.z: fraction in units
  FL f;
  f.reset(cr);
  auto upd = [&](int h) {
    St<R> q = {0, 0, p.s, p.t, p.q};
    R ry = ((R)(yi[h] - oy) - p.y) * IU, rz = ((R)(zi[h] - oz) - p.z) * IU;
    R c = f.update(q, ry, rz, sy2, sz2);
    p.y += q.y * U; p.z += q.z * U; p.s = q.s; p.t = q.t; p.q = q.q;
    return c;
  };
  auto recentre = [&]() {
    R ry = std::nearbyint(p.y), rz = std::nearbyint(p.z);
    oy += (int64_t)ry; oz += (int64_t)rz; p.y -= ry; p.z -= rz;
  };
  auto step = [&](R dx) {
    Geo<R> g;
    if (!geom<R>(cq, smax, dx, p, g)) return false;
    f.transport(g); p.y += g.dy * U; p.z += p.t * g.dS * U; p.s = g.s1;
    recentre();
    return true;
  };
  upd(h0);
  int row = r0;
  bool fail_up = false;
  for (int i = 1; i < L; ++i) {
    if (!step((R)(row_x[row + 1] - row_x[row]))) { fail_up = true; break; }
    ++row;
    upd(hits[row]);
  }
  if (!fail_up) {
    int miss = 0;
    while (row + 1 <= nr - 1 && miss < max_miss) {
      if (!step((R)(row_x[row + 1] - row_x[row]))) break;
      ++row;
      if (hits[row] >= 0) { upd(hits[row]); miss = 0; } else ++miss;
    }
  }
  f.reset(cr);
  R chi2 = 0;
  if (hits[row] >= 0) chi2 += upd(hits[row]);
  bool fail_dn = false;
  int miss = 0;
  while (row > 0) {
    if (row - 1 < r0 && miss >= max_miss) break;
    if (!step((R)(row_x[row - 1] - row_x[row]))) { fail_dn = true; break; }
    --row;
    if (row >= r0) {
      if (hits[row] >= 0) chi2 += upd(hits[row]);
    } else {
      if (hits[row] >= 0) { chi2 += upd(hits[row]); miss = 0; } else ++miss;
    }
  }
  int lowest = 0;
  for (int r = nr - 1; r >= 0; --r) if (hits[r] >= 0) lowest = r;
  if (!fail_dn && lowest != row) {
    if (step((R)(row_x[lowest] - row_x[row]))) row = lowest;
  }
  par[0] = row_x[row]; par[1] = ((double)oy + (double)p.y) / 640.0; par[2] = ((double)oz + (double)p.z) / 640.0;
  par[3] = p.s; par[4] = p.t; par[5] = p.q;
  f.cov_out(cov);
  *chi2o = chi2;
}

extern "C" void replay_s(int variant, const double* prm, int nr, const double* row_x, const int32_t* yi, const int32_t* zi,
                       int64_t ns, const int32_t* r0, const int32_t* L, const int32_t* hits, double* par, double* cov,
                       double* chi2) {
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < ns; ++i) {
    const int32_t* h = hits + i * nr;
    if (variant == 3) replay_split<FilterUD<float>>(prm, nr, row_x, yi, zi, r0[i], L[i], h, par + i * 6, cov + i * 15, chi2 + i);
    else if (variant == 2) replay_split<FilterCov<float, 1>>(prm, nr, row_x, yi, zi, r0[i], L[i], h, par + i * 6, cov + i * 15, chi2 + i);
    else replay_split<FilterCov<float, 0>>(prm, nr, row_x, yi, zi, r0[i], L[i], h, par + i * 6, cov + i * 15, chi2 + i);
  }
}

extern "C" void replay(int variant, const double* prm, int nr, const double* row_x, const double* y, const double* z,
                       int64_t ns, const int32_t* r0, const int32_t* L, const int32_t* hits, double* par, double* cov,
                       double* chi2) {
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < ns; ++i) {
    const int32_t* h = hits + i * nr;
    double* pp = par + i * 6; double* cc = cov + i * 15; double* xx = chi2 + i;
    switch (variant) {
      case 0: replay_one<double, FilterCov<double, 0>>(prm, nr, row_x, y, z, r0[i], L[i], h, pp, cc, xx); break;
      case 1: replay_one<float, FilterCov<float, 0>>(prm, nr, row_x, y, z, r0[i], L[i], h, pp, cc, xx); break;
      case 2: replay_one<float, FilterCov<float, 1>>(prm, nr, row_x, y, z, r0[i], L[i], h, pp, cc, xx); break;
      case 3: replay_one<float, FilterUD<float>>(prm, nr, row_x, y, z, r0[i], L[i], h, pp, cc, xx); break;
      case 4: replay_one<double, FilterUD<double>>(prm, nr, row_x, y, z, r0[i], L[i], h, pp, cc, xx); break;
    }
  }
}
