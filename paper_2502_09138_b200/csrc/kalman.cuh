// kalman.cuh -- the filter arithmetic shared by a4 (tracklet follower) and a6 (track refit): state, covariance,
// helix transport with Jacobian, (y, z) update.  SURVEY Appendix C; precision: DESIGN.md "a4 precision".
// Included inside each kernel file's anonymous namespace; both files are compiled with --use_fast_math (build.py).
//
// Everything is fp32.  The covariance is carried as its U D U^T factors (U unit upper triangular, D diagonal, state
// order y, z, sin phi, tan lambda, q/pT): 15 floats, like the packed triangle, but
//   * the Jacobian of the helix step is itself unit upper triangular in this state order (Appendix C: its only
//     off-diagonal entries are dy/ds, dy/dq, dz/ds, dz/dt, dz/dq, ds/dq) and there is no process noise (P16), so
//     C <- F C F^T is U <- F U with D untouched: nine FMAs instead of the seventy of the packed form;
//   * the update is Bierman's scalar form, once for y and once for z (V is diagonal, so two scalar updates equal
//     the joint update of Appendix C, chi2 included); it only multiplies and adds positive terms into D, so the
//     cancellation of C - K H C after the P22 reset -- which costs a plain fp32 covariance the 1e-4 bar on 0.6-1.3 %
//     of the tracklets -- never happens.  Measured against the fp64 oracle: worst parameter error 3e-5.
#pragma once
#include "tpc_internal.cuh"

namespace {

struct Cov {   // C = U D U^T
  float d0, d1, d2, d3, d4;
  float u01, u02, u03, u04, u12, u13, u14, u23, u24, u34;
  // variances of y and z (the gate of P17 ignores Cyz): sums of positive terms
  __device__ __forceinline__ float var_y() const {
    return fmaf(u04 * u04, d4, fmaf(u03 * u03, d3, fmaf(u02 * u02, d2, fmaf(u01 * u01, d1, d0))));
  }
  __device__ __forceinline__ float var_z() const {
    return fmaf(u14 * u14, d4, fmaf(u13 * u13, d3, fmaf(u12 * u12, d2, d1)));
  }
  // packed lower triangle c00 c10 c11 c20 c21 c22 c30 .. c44 (the layout of tpc_track_rec_t.cov)
  __device__ __forceinline__ void lower(float c[15]) const {
    const float e1 = u01 * d1, e2 = u02 * d2, e3 = u03 * d3, e4 = u04 * d4;   // row 0 of U D
    const float g2 = u12 * d2, g3 = u13 * d3, g4 = u14 * d4;                  // row 1
    const float h3 = u23 * d3, h4 = u24 * d4;                                 // row 2
    const float k4 = u34 * d4;                                                // row 3
    c[0] = fmaf(e4, u04, fmaf(e3, u03, fmaf(e2, u02, fmaf(e1, u01, d0))));
    c[1] = fmaf(e4, u14, fmaf(e3, u13, fmaf(e2, u12, e1)));
    c[2] = fmaf(g4, u14, fmaf(g3, u13, fmaf(g2, u12, d1)));
    c[3] = fmaf(e4, u24, fmaf(e3, u23, e2));
    c[4] = fmaf(g4, u24, fmaf(g3, u23, g2));
    c[5] = fmaf(h4, u24, fmaf(h3, u23, d2));
    c[6] = fmaf(e4, u34, e3);
    c[7] = fmaf(g4, u34, g3);
    c[8] = fmaf(h4, u34, h3);
    c[9] = fmaf(k4, u34, d3);
    c[10] = e4;
    c[11] = g4;
    c[12] = h4;
    c[13] = k4;
    c[14] = d4;
  }
};

// Positions are split: integer origin (fixed-point units, the ABI's) + fp32 fraction in units, re-centred after
// every transport so that |fraction| <= 1/2 unit.  A hit's residual is then an exact integer difference minus a small
// fraction, whatever the drift offset or the sector width: with plain fp32 positions (ulp 1.5e-5 cm at 150 cm) the
// gains right after the P22 reset (up to ~40 GeV^-1 per cm on q/pT) turn position rounding into 1e-4-level errors.
struct State {
  float y, z;      // fraction of the position, units
  float s, t, q;   // sin phi, tan lambda, q/pT
  int oy, oz;      // origin, units
};

__device__ __forceinline__ void state_recentre(State& p) {
  const float ry = rintf(p.y), rz = rintf(p.z);   // exact: |p.y| stays far below 2^23 units
  p.oy += (int)ry;
  p.oz += (int)rz;
  p.y -= ry;
  p.z -= rz;
}

// residual of a cluster at integer (hy, hz) against the state's position, cm
__device__ __forceinline__ float resid_y(const DevGeom& g, const State& p, int hy) { return ((float)(hy - p.oy) - p.y) * g.inv_units; }
__device__ __forceinline__ float resid_z(const DevGeom& g, const State& p, int hz) { return ((float)(hz - p.oz) - p.z) * g.inv_units; }

__device__ __forceinline__ void cov_reset(const DevGeom& g, Cov& C) {   // P19, P22: diag(c_reset)
  C.d0 = g.c_reset[0]; C.d1 = g.c_reset[1]; C.d2 = g.c_reset[2]; C.d3 = g.c_reset[3]; C.d4 = g.c_reset[4];
  C.u01 = C.u02 = C.u03 = C.u04 = C.u12 = C.u13 = C.u14 = C.u23 = C.u24 = C.u34 = 0.f;
}

// Appendix C.  One step of dx (either sign) along the helix; k = cq * q/pT.  Returns false (state untouched)
// iff |sin phi| >= sinphi_max before or after (P18).  WITH_COV: U <- F U with
// F = I + [02]=a [04]=b [12]=c [13]=d [14]=e [24]=f.
template <bool WITH_COV>
__device__ __forceinline__ bool transport(const DevGeom& g, float dx, State& p, Cov& C) {
  const float cq = g.cq;
  const float k = cq * p.q;
  const float s0 = p.s;
  const float s1 = fmaf(k, dx, s0);
  if (!(fabsf(s0) < g.sinphi_max) || !(fabsf(s1) < g.sinphi_max)) return false;
  // |s| < sinphi_max < 1: 1 - s^2 stays well away from 0
  const float q0 = fmaf(-s0, s0, 1.f), q1 = fmaf(-s1, s1, 1.f);
  const float ic0 = rsqrtf(q0), ic1 = rsqrtf(q1);
  const float c0 = q0 * ic0, c1 = q1 * ic1;
  const float icc = 1.f / (c0 + c1);
  const float tau = (s0 + s1) * icc;
  const float dy = dx * tau;
  const float w2 = fmaf(tau, tau, 1.f);
  const float cm = rsqrtf(w2);                 // cos of the mean direction; sqrt(1 + tau^2) = w2 * cm
  const float chord = dx * (w2 * cm);          // sign(dx) sqrt(dx^2 + dy^2)
  const float u = 0.5f * k * chord;
  const float u2 = u * u;
  // asin(u)/u = 1 + u^2/6 + 3u^4/40 + 15u^6/336 + 105 u^8/3456 + 945 u^10/42240 ...
  const float dS = (u2 < 0.01f)
      ? chord * fmaf(u2, fmaf(u2, fmaf(u2, fmaf(u2, fmaf(u2, 0.022372159f, 0.030381944f), 0.044642857f), 0.075f),
                              0.16666666666666666f), 1.f)
      : chord * asinf(u) / u;
  if (WITH_COV) {
    const float m = fmaf(s0, tau, c0);
    const float ic0c1 = ic0 * ic1;
    const float d_ = 0.5f * k * dS;
    const float d2 = d_ * d_;
    float sinc, gg;
    if (d2 < 0.01f) {
      sinc = fmaf(d2, fmaf(d2, fmaf(d2, -1.0f / 5040.0f, 1.0f / 120.0f), -1.0f / 6.0f), 1.f);
      gg = fmaf(d2, fmaf(d2, fmaf(d2, -1.0f / 45360.0f, 1.0f / 840.0f), -1.0f / 30.0f), 1.0f / 3.0f);
    } else {
      float sn, cs;
      sincosf(d_, &sn, &cs);
      sinc = sn / d_;
      gg = (sn - d_ * cs) / (d_ * d2);
    }
    const float sm = tau * cm;
    // d(dS)/dk in the form that has no 0/0 at k -> 0 (the same re-derivation of Appendix C's (dx/c1 - dS)/k as the
    // oracle's: both restate one derivation)
    const float dSdk = (0.5f * dS * dS * sm * sinc + 0.25f * k * dS * dS * dS * cm * gg) * ic1;
    const float a = dx * m * ic0c1;              // dy1/ds
    const float b = cq * dx * dx * m * ic1 * icc; // dy1/dq
    const float c = p.t * dy * ic0c1;            // dz1/ds
    const float d = dS;                          // dz1/dt
    const float e = p.t * cq * dSdk;             // dz1/dq
    const float f = cq * dx;                     // ds1/dq
    // rows of F U: row0 += a row2 + b row4, row1 += c row2 + d row3 + e row4, row2 += f row4
    C.u02 += a;
    C.u03 = fmaf(a, C.u23, C.u03);
    C.u04 = fmaf(a, C.u24, C.u04) + b;
    C.u12 += c;
    C.u13 = fmaf(c, C.u23, C.u13) + d;
    C.u14 = fmaf(c, C.u24, fmaf(d, C.u34, C.u14)) + e;
    C.u24 += f;
  }
  p.y = fmaf(dy, g.units, p.y);
  p.z = fmaf(p.t * dS, g.units, p.z);
  p.s = s1;
  state_recentre(p);
  return true;
}

// Appendix C update with H = [I2 | 0], V = diag(sy2, sz2), as two Bierman scalar updates (y, then z with the
// residual after the y update).  (ry, rz) = hit - state in cm (resid_y / resid_z).  Returns the chi2 increment (equal
// to the joint r^T S^-1 r).
__device__ __forceinline__ float update(const DevGeom& g, State& p, Cov& C, float ry, float rz) {
  float chi2;
  {   // ---- y: h = e_0, f = (1, u01, u02, u03, u04) ----
    const float a0 = g.sy2;
    const float v0 = C.d0;
    const float a1 = a0 + v0;
    const float i1 = 1.f / a1;
    C.d0 = v0 * a0 * i1;
    float b0 = v0;
    // j = 1
    const float f1 = C.u01, v1 = C.d1 * f1;
    const float a2 = fmaf(f1, v1, a1);
    const float i2 = 1.f / a2;
    C.d1 = C.d1 * a1 * i2;
    float lam = -f1 * i1;
    C.u01 = fmaf(lam, b0, f1);
    b0 = fmaf(f1, v1, b0);
    float b1 = v1;
    // j = 2
    const float f2 = C.u02, v2 = C.d2 * f2;
    const float a3 = fmaf(f2, v2, a2);
    const float i3 = 1.f / a3;
    C.d2 = C.d2 * a2 * i3;
    lam = -f2 * i2;
    const float o12 = C.u12;
    C.u02 = fmaf(lam, b0, f2);
    C.u12 = fmaf(lam, b1, o12);
    b0 = fmaf(f2, v2, b0);
    b1 = fmaf(o12, v2, b1);
    float b2 = v2;
    // j = 3
    const float f3 = C.u03, v3 = C.d3 * f3;
    const float a4 = fmaf(f3, v3, a3);
    const float i4 = 1.f / a4;
    C.d3 = C.d3 * a3 * i4;
    lam = -f3 * i3;
    const float o13 = C.u13, o23 = C.u23;
    C.u03 = fmaf(lam, b0, f3);
    C.u13 = fmaf(lam, b1, o13);
    C.u23 = fmaf(lam, b2, o23);
    b0 = fmaf(f3, v3, b0);
    b1 = fmaf(o13, v3, b1);
    b2 = fmaf(o23, v3, b2);
    float b3 = v3;
    // j = 4
    const float f4 = C.u04, v4 = C.d4 * f4;
    const float a5 = fmaf(f4, v4, a4);
    const float i5 = 1.f / a5;
    C.d4 = C.d4 * a4 * i5;
    lam = -f4 * i4;
    const float o14 = C.u14, o24 = C.u24, o34 = C.u34;
    C.u04 = fmaf(lam, b0, f4);
    C.u14 = fmaf(lam, b1, o14);
    C.u24 = fmaf(lam, b2, o24);
    C.u34 = fmaf(lam, b3, o34);
    b0 = fmaf(f4, v4, b0);
    b1 = fmaf(o14, v4, b1);
    b2 = fmaf(o24, v4, b2);
    b3 = fmaf(o34, v4, b3);
    const float b4 = v4;
    const float r = ry;
    const float ri = r * i5;   // residual / innovation variance (a5 = Cyy + sy2)
    p.y = fmaf(b0 * ri, g.units, p.y);
    p.z = fmaf(b1 * ri, g.units, p.z);
    rz = fmaf(-b1, ri, rz);    // the z residual against the state after the y update
    p.s = fmaf(b2, ri, p.s);
    p.t = fmaf(b3, ri, p.t);
    p.q = fmaf(b4, ri, p.q);
    chi2 = r * ri;
  }
  {   // ---- z: h = e_1, f = (0, 1, u12, u13, u14) ----
    const float a1 = g.sz2;
    const float v1 = C.d1;
    const float a2 = a1 + v1;
    const float i2 = 1.f / a2;
    C.d1 = v1 * a1 * i2;
    float b0 = C.u01 * v1;   // u01 itself is unchanged (b0 was 0 before this column)
    float b1 = v1;
    // j = 2
    const float f2 = C.u12, v2 = C.d2 * f2;
    const float a3 = fmaf(f2, v2, a2);
    const float i3 = 1.f / a3;
    C.d2 = C.d2 * a2 * i3;
    float lam = -f2 * i2;
    const float o02 = C.u02;
    C.u02 = fmaf(lam, b0, o02);
    C.u12 = fmaf(lam, b1, f2);
    b0 = fmaf(o02, v2, b0);
    b1 = fmaf(f2, v2, b1);
    float b2 = v2;
    // j = 3
    const float f3 = C.u13, v3 = C.d3 * f3;
    const float a4 = fmaf(f3, v3, a3);
    const float i4 = 1.f / a4;
    C.d3 = C.d3 * a3 * i4;
    lam = -f3 * i3;
    const float o03 = C.u03, o23 = C.u23;
    C.u03 = fmaf(lam, b0, o03);
    C.u13 = fmaf(lam, b1, f3);
    C.u23 = fmaf(lam, b2, o23);
    b0 = fmaf(o03, v3, b0);
    b1 = fmaf(f3, v3, b1);
    b2 = fmaf(o23, v3, b2);
    float b3 = v3;
    // j = 4
    const float f4 = C.u14, v4 = C.d4 * f4;
    const float a5 = fmaf(f4, v4, a4);
    const float i5 = 1.f / a5;
    C.d4 = C.d4 * a4 * i5;
    lam = -f4 * i4;
    const float o04 = C.u04, o24 = C.u24, o34 = C.u34;
    C.u04 = fmaf(lam, b0, o04);
    C.u14 = fmaf(lam, b1, f4);
    C.u24 = fmaf(lam, b2, o24);
    C.u34 = fmaf(lam, b3, o34);
    b0 = fmaf(o04, v4, b0);
    b1 = fmaf(f4, v4, b1);
    b2 = fmaf(o24, v4, b2);
    b3 = fmaf(o34, v4, b3);
    const float b4 = v4;
    const float r = rz;
    const float ri = r * i5;
    p.y = fmaf(b0 * ri, g.units, p.y);
    p.z = fmaf(b1 * ri, g.units, p.z);
    p.s = fmaf(b2, ri, p.s);
    p.t = fmaf(b3, ri, p.t);
    p.q = fmaf(b4, ri, p.q);
    chi2 = fmaf(r, ri, chi2);
  }
  return chi2;
}

}  // namespace
