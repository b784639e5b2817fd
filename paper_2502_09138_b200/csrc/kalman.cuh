// kalman.cuh -- the filter arithmetic shared by a4 (tracklet follower) and a6 (track refit): state, covariance,
// helix transport with Jacobian, joint (y, z) update.  SURVEY Appendix C; precision: DESIGN.md "a4 precision".
// Included inside each kernel file's anonymous namespace; both files are compiled with --use_fast_math (build.py).
#pragma once
#include "tpc_internal.cuh"

namespace {

// Precision: state in fp32, covariance and gain in fp64.  With an fp32 covariance
// 0.6 % (config 1) to 1.3 % (config 4) of the tracklets miss the 1e-4 bar on q/pT (cancellation in C - K H C
// after the P22 reset); with the covariance in fp64 none does.
#ifdef TPC_A4_COV32
typedef float creal;
#else
typedef double creal;
#endif
#ifdef TPC_A4_STATE64
typedef double sreal;
#else
typedef float sreal;
#endif

struct Cov {   // symmetric 5x5, lower triangle
  creal c00, c10, c11, c20, c21, c22, c30, c31, c32, c33, c40, c41, c42, c43, c44;
};

struct State {
  sreal y, z, s, t, q;   // relative y, relative z, sin phi, tan lambda, q/pT
};

__device__ __forceinline__ void cov_reset(const DevGeom& g, Cov& C) {
  C.c00 = g.c_reset[0]; C.c11 = g.c_reset[1]; C.c22 = g.c_reset[2]; C.c33 = g.c_reset[3]; C.c44 = g.c_reset[4];
  C.c10 = C.c20 = C.c21 = C.c30 = C.c31 = C.c32 = C.c40 = C.c41 = C.c42 = C.c43 = 0.f;
}

// Appendix C.  One step of dx (either sign) along the helix; k = cq * q/pT.  Returns false (state untouched)
// iff |sin phi| >= sinphi_max before or after (P18).  WITH_COV: C <- F C F^T with
// F = I + [02]=a [04]=b [12]=c [13]=d [14]=e [24]=f.
template <bool WITH_COV>
__device__ __forceinline__ bool transport(const DevGeom& g, float dxf, State& p, Cov& C) {
  const sreal dx = dxf;
  const sreal cq = g.cq;
  const sreal k = cq * p.q;
  const sreal s0 = p.s;
  const sreal s1 = fma(k, dx, s0);
  if (!(fabs(s0) < (sreal)g.sinphi_max) || !(fabs(s1) < (sreal)g.sinphi_max)) return false;
  const sreal c0 = sqrt(fma(-s0, s0, (sreal)1)), c1 = sqrt(fma(-s1, s1, (sreal)1));
  const sreal tau = (s0 + s1) / (c0 + c1);
  const sreal dy = dx * tau;
  const sreal chord = copysign(sqrt(fma(dx, dx, dy * dy)), dx);
  const sreal u = (sreal)0.5 * k * chord;
  const sreal u2 = u * u;
  // asin(u)/u = 1 + u^2/6 + 3u^4/40 + 15u^6/336 + 105 u^8/3456 + 945 u^10/42240 ...
  const sreal dS = (u2 < (sreal)0.01)
      ? chord * fma(u2, fma(u2, fma(u2, fma(u2, fma(u2, (sreal)0.022372159, (sreal)0.030381944), (sreal)0.044642857),
                                   (sreal)0.075), (sreal)0.16666666666666666), (sreal)1)
      : chord * asin(u) / u;
  if (WITH_COV) {
    const sreal m = fma(s0, tau, c0);
    const sreal ic0c1 = (sreal)1 / (c0 * c1);
    const sreal d_ = (sreal)0.5 * k * dS;
    const sreal d2 = d_ * d_;
    sreal sinc, gg;
    if (d2 < (sreal)0.01) {
      sinc = fma(d2, fma(d2, fma(d2, (sreal)(-1.0 / 5040.0), (sreal)(1.0 / 120.0)), (sreal)(-1.0 / 6.0)), (sreal)1);
      gg = fma(d2, fma(d2, fma(d2, (sreal)(-1.0 / 45360.0), (sreal)(1.0 / 840.0)), (sreal)(-1.0 / 30.0)), (sreal)(1.0 / 3.0));
    } else {
      sreal sn, cs;
      sincos(d_, &sn, &cs);
      sinc = sn / d_;
      gg = (sn - d_ * cs) / (d_ * d2);
    }
    const sreal cm = rsqrt(fma(tau, tau, (sreal)1)), sm = tau * cm;
    const sreal dSdk = ((sreal)0.5 * dS * dS * sm * sinc + (sreal)0.25 * k * dS * dS * dS * cm * gg) / c1;
    const creal a = dx * m * ic0c1;                     // dy1/ds
    const creal b = cq * dx * dx * m / (c1 * (c0 + c1)); // dy1/dq
    const creal c = p.t * dy * ic0c1;                   // dz1/ds
    const creal d = dS;                                 // dz1/dt
    const creal e = p.t * cq * dSdk;                    // dz1/dq
    const creal f = cq * dx;                            // ds1/dq
    // M = F C (rows 0..2 change), then C' = M F^T
    const creal m00 = C.c00 + a * C.c20 + b * C.c40;
    const creal m02 = C.c20 + a * C.c22 + b * C.c42;
    const creal m04 = C.c40 + a * C.c42 + b * C.c44;
    const creal m10 = C.c10 + c * C.c20 + d * C.c30 + e * C.c40;
    const creal m11 = C.c11 + c * C.c21 + d * C.c31 + e * C.c41;
    const creal m12 = C.c21 + c * C.c22 + d * C.c32 + e * C.c42;
    const creal m13 = C.c31 + c * C.c32 + d * C.c33 + e * C.c43;
    const creal m14 = C.c41 + c * C.c42 + d * C.c43 + e * C.c44;
    const creal m20 = C.c20 + f * C.c40;
    const creal m21 = C.c21 + f * C.c41;
    const creal m22 = C.c22 + f * C.c42;
    const creal m23 = C.c32 + f * C.c43;
    const creal m24 = C.c42 + f * C.c44;
    Cov N;
    N.c00 = m00 + a * m02 + b * m04;
    N.c10 = m10 + a * m12 + b * m14;
    N.c11 = m11 + c * m12 + d * m13 + e * m14;
    N.c20 = m20 + a * m22 + b * m24;
    N.c21 = m21 + c * m22 + d * m23 + e * m24;
    N.c22 = m22 + f * m24;
    N.c30 = C.c30 + a * C.c32 + b * C.c43;
    N.c31 = C.c31 + c * C.c32 + d * C.c33 + e * C.c43;
    N.c32 = C.c32 + f * C.c43;
    N.c33 = C.c33;
    N.c40 = C.c40 + a * C.c42 + b * C.c44;
    N.c41 = C.c41 + c * C.c42 + d * C.c43 + e * C.c44;
    N.c42 = C.c42 + f * C.c44;
    N.c43 = C.c43;
    N.c44 = C.c44;
    C = N;
  }
  p.y += dy;
  p.z = fma(p.t, dS, p.z);
  p.s = s1;
  return true;
}

// Appendix C update with H = [I2 | 0], V = diag(sy2, sz2).  Returns the chi2 increment.
__device__ __forceinline__ float update(const DevGeom& g, State& p, Cov& C, float ym, float zm) {
  const creal S00 = C.c00 + (creal)g.sy2, S01 = C.c10, S11 = C.c11 + (creal)g.sz2;
#ifdef TPC_A4_COV32
  const creal idet = (creal)1 / (S00 * S11 - S01 * S01);
#else
  // 1/det: fp32 reciprocal + two Newton steps in fp64 (relative error ~1e-15) instead of the IEEE fp64 division
  // sequence; det = (Cyy + sy2)(Czz + sz2) - Cyz^2 >= sy2 sz2 stays far inside the fp32 range.
  const double det = S00 * S11 - S01 * S01;
  double idet = (double)(1.0f / (float)det);
  idet = idet * (2.0 - det * idet);
  idet = idet * (2.0 - det * idet);
#endif
  const creal I00 = S11 * idet, I01 = -S01 * idet, I11 = S00 * idet;
  const creal r0 = (sreal)ym - p.y, r1 = (sreal)zm - p.z;
  // K = C[:,0:2] S^-1
  const creal k00 = C.c00 * I00 + C.c10 * I01, k01 = C.c00 * I01 + C.c10 * I11;
  const creal k10 = C.c10 * I00 + C.c11 * I01, k11 = C.c10 * I01 + C.c11 * I11;
  const creal k20 = C.c20 * I00 + C.c21 * I01, k21 = C.c20 * I01 + C.c21 * I11;
  const creal k30 = C.c30 * I00 + C.c31 * I01, k31 = C.c30 * I01 + C.c31 * I11;
  const creal k40 = C.c40 * I00 + C.c41 * I01, k41 = C.c40 * I01 + C.c41 * I11;
  p.y += (sreal)(k00 * r0 + k01 * r1);
  p.z += (sreal)(k10 * r0 + k11 * r1);
  p.s += (sreal)(k20 * r0 + k21 * r1);
  p.t += (sreal)(k30 * r0 + k31 * r1);
  p.q += (sreal)(k40 * r0 + k41 * r1);
  // C <- C - K (H C), lower triangle: C_ij -= K_i0 C_0j + K_i1 C_1j
  Cov N;
  N.c00 = C.c00 - (k00 * C.c00 + k01 * C.c10);
  N.c10 = C.c10 - (k10 * C.c00 + k11 * C.c10);
  N.c11 = C.c11 - (k10 * C.c10 + k11 * C.c11);
  N.c20 = C.c20 - (k20 * C.c00 + k21 * C.c10);
  N.c21 = C.c21 - (k20 * C.c10 + k21 * C.c11);
  N.c22 = C.c22 - (k20 * C.c20 + k21 * C.c21);
  N.c30 = C.c30 - (k30 * C.c00 + k31 * C.c10);
  N.c31 = C.c31 - (k30 * C.c10 + k31 * C.c11);
  N.c32 = C.c32 - (k30 * C.c20 + k31 * C.c21);
  N.c33 = C.c33 - (k30 * C.c30 + k31 * C.c31);
  N.c40 = C.c40 - (k40 * C.c00 + k41 * C.c10);
  N.c41 = C.c41 - (k40 * C.c10 + k41 * C.c11);
  N.c42 = C.c42 - (k40 * C.c20 + k41 * C.c21);
  N.c43 = C.c43 - (k40 * C.c30 + k41 * C.c31);
  N.c44 = C.c44 - (k40 * C.c40 + k41 * C.c41);
  C = N;
  return (float)(r0 * (I00 * r0 + I01 * r1) + r1 * (I01 * r0 + I11 * r1));
}


}  // namespace
