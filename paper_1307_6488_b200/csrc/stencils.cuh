// stencils.cuh -- finite-difference operators of the CUDA path (4th order; 8th for the wave system).
// Reading S2/S6: centred 1st (1,-8,0,8,-1)/12h, 2nd (-1,16,-30,16,-1)/12h^2, mixed = 1st(a) o 1st(b),
// upwind (-3,-10,18,-6,1)/12h on offsets -1..+3 (mirrored for beta<0), KO5 (1,-6,15,-20,15,-6,1) eps/64h.
// All in difference form (reading R-H1): only differences of neighbouring values are ever scaled and summed,
// so flat data differentiates to exactly 0 and near-flat data keeps full relative accuracy.
#pragma once
#include "bssn_point.cuh"

namespace chm {

// Reads a field through global memory (L1/L2 cached, read-only path).  `p` points at the evaluation point of
// variable 0 in the padded layout; sy, sz, sv are the y, z and variable strides in doubles.
struct GlobalPoint {
  const double* __restrict__ p;
  long sy, sz, sv;
  __device__ __forceinline__ double at(int v, int di, int dj, int dk) const {
    return __ldg(p + v * sv + dk * sz + dj * sy + di);
  }
  // offset `m` along axis a (0=x,1=y,2=z)
  __device__ __forceinline__ double ax(int v, int a, int m) const {
    return a == 0 ? at(v, m, 0, 0) : (a == 1 ? at(v, 0, m, 0) : at(v, 0, 0, m));
  }
  // offsets m along a and n along b, a != b
  __device__ __forceinline__ double ax2(int v, int a, int m, int b, int n) const {
    int d[3] = {0, 0, 0};
    d[a] = m; d[b] = n;
    return at(v, d[0], d[1], d[2]);
  }
};

// ---- 4th order ---------------------------------------------------------------------------------------
template <class P>
CHM_HD double d1_o4(const P& f, int v, int a, double inv_h) {
  double e1 = f.ax(v, a, 1) - f.ax(v, a, -1);
  double e2 = f.ax(v, a, 2) - f.ax(v, a, -2);
  return (8.0 * e1 - e2) * (inv_h * (1.0 / 12.0));
}

template <class P>
CHM_HD double d2_o4(const P& f, int v, int a, double inv_h2) {
  double f0 = f.at(v, 0, 0, 0);
  double s1 = (f.ax(v, a, 1) - f0) + (f.ax(v, a, -1) - f0);
  double s2 = (f.ax(v, a, 2) - f0) + (f.ax(v, a, -2) - f0);
  return (16.0 * s1 - s2) * (inv_h2 * (1.0 / 12.0));
}

// row(m) = undivided first difference along b at offset m along a
template <class P>
CHM_HD double dmix_o4(const P& f, int v, int a, int b, double inv_h2) {
  double r[4];
  const int off[4] = {1, -1, 2, -2};
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    int m = off[t];
    double e1 = f.ax2(v, a, m, b, 1) - f.ax2(v, a, m, b, -1);
    double e2 = f.ax2(v, a, m, b, 2) - f.ax2(v, a, m, b, -2);
    r[t] = 8.0 * e1 - e2;
  }
  return (8.0 * (r[0] - r[1]) - (r[2] - r[3])) * (inv_h2 * (1.0 / 144.0));
}

// beta^a * upwinded d_a f, side by the sign of beta (beta == 0 gives exactly 0)
template <class P>
CHM_HD double adv_o4(const P& f, int v, int a, double beta, double inv_h) {
  double f0 = f.at(v, 0, 0, 0);
  int s = beta > 0.0 ? 1 : -1;
  double m1 = f.ax(v, a, -s) - f0;
  double p1 = f.ax(v, a, s) - f0;
  double p2 = f.ax(v, a, 2 * s) - f0;
  double p3 = f.ax(v, a, 3 * s) - f0;
  double r = (18.0 * p1 - 3.0 * m1) + (p3 - 6.0 * p2);
  double sb = beta > 0.0 ? beta : -beta;   // beta * side = |beta|
  return sb * r * (inv_h * (1.0 / 12.0));
}

// Kreiss-Oliger dissipation along one axis, undivided: s3 - 6 s2 + 15 s1
template <class P>
CHM_HD double ko5_axis(const P& f, int v, int a) {
  double f0 = f.at(v, 0, 0, 0);
  double s1 = (f.ax(v, a, 1) - f0) + (f.ax(v, a, -1) - f0);
  double s2 = (f.ax(v, a, 2) - f0) + (f.ax(v, a, -2) - f0);
  double s3 = (f.ax(v, a, 3) - f0) + (f.ax(v, a, -3) - f0);
  return (s3 - 6.0 * s2) + 15.0 * s1;
}

template <class P>
CHM_HD double ko5(const P& f, int v, double ko) {
  return ko * ((ko5_axis(f, v, 0) + ko5_axis(f, v, 1)) + ko5_axis(f, v, 2));
}
// dissipation with the five weights of Coef::kq (order 5 or 9; needs 5 ghost zones): 8th-order BSSN kernels
template <class P>
CHM_HD double ko_kq(const P& f, int v, const double* kq) {
  const double f0 = f.at(v, 0, 0, 0);
  double r = 0.0;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double s[6];
#pragma unroll
    for (int k = 1; k <= 5; ++k) s[k] = (f.ax(v, a, k) - f0) + (f.ax(v, a, -k) - f0);
    const double q = ((kq[4] * s[5] + kq[3] * s[4]) + (kq[2] * s[3] + kq[1] * s[2])) + kq[0] * s[1];
    r = a == 0 ? q : r + q;
  }
  return r;
}

// ---- 8th order (wave systems) ------------------------------------------------------------------------
// 1st derivative (3,-32,168,-672,0,672,-168,32,-3)/840h
template <class P>
CHM_HD double d1_o8(const P& f, int v, int a, double inv_h) {
  double e1 = f.ax(v, a, 1) - f.ax(v, a, -1);
  double e2 = f.ax(v, a, 2) - f.ax(v, a, -2);
  double e3 = f.ax(v, a, 3) - f.ax(v, a, -3);
  double e4 = f.ax(v, a, 4) - f.ax(v, a, -4);
  return ((672.0 * e1 - 168.0 * e2) + (32.0 * e3 - 3.0 * e4)) * (inv_h * (1.0 / 840.0));
}

// mixed derivative: the 1-D first-derivative stencil along a applied to the one along b (64 points)
template <class P>
CHM_HD double dmix_o8(const P& f, int v, int a, int b, double inv_h2) {
  double r[8];
  const int off[8] = {1, -1, 2, -2, 3, -3, 4, -4};
#pragma unroll
  for (int t = 0; t < 8; ++t) {
    const int m = off[t];
    const double e1 = f.ax2(v, a, m, b, 1) - f.ax2(v, a, m, b, -1);
    const double e2 = f.ax2(v, a, m, b, 2) - f.ax2(v, a, m, b, -2);
    const double e3 = f.ax2(v, a, m, b, 3) - f.ax2(v, a, m, b, -3);
    const double e4 = f.ax2(v, a, m, b, 4) - f.ax2(v, a, m, b, -4);
    r[t] = (672.0 * e1 - 168.0 * e2) + (32.0 * e3 - 3.0 * e4);
  }
  return ((672.0 * (r[0] - r[1]) - 168.0 * (r[2] - r[3])) + (32.0 * (r[4] - r[5]) - 3.0 * (r[6] - r[7]))) *
         (inv_h2 * (1.0 / (840.0 * 840.0)));
}

// beta^a * upwinded d_a f at 8th order: offsets -3..+5 on the side of beta,
// (-5, 60, -420, -378, 1050, -420, 140, -30, 3)/840h, in differences from the centre value (5 ghosts)
template <class P>
CHM_HD double adv_o8(const P& f, int v, int a, double beta, double inv_h) {
  const double f0 = f.at(v, 0, 0, 0);
  const int s = beta > 0.0 ? 1 : -1;
  const double m3 = f.ax(v, a, -3 * s) - f0, m2 = f.ax(v, a, -2 * s) - f0, m1 = f.ax(v, a, -s) - f0;
  const double p1 = f.ax(v, a, s) - f0, p2 = f.ax(v, a, 2 * s) - f0, p3 = f.ax(v, a, 3 * s) - f0;
  const double p4 = f.ax(v, a, 4 * s) - f0, p5 = f.ax(v, a, 5 * s) - f0;
  const double r = ((1050.0 * p1 - 420.0 * m1) + (60.0 * m2 - 420.0 * p2)) + ((140.0 * p3 - 5.0 * m3) + (3.0 * p5 - 30.0 * p4));
  const double sb = beta > 0.0 ? beta : -beta;   // beta * side = |beta|
  return sb * r * (inv_h * (1.0 / 840.0));
}

// 2nd derivative (-9,128,-1008,8064,-14350,8064,-1008,128,-9)/5040h^2
template <class P>
CHM_HD double d2_o8(const P& f, int v, int a, double inv_h2) {
  double f0 = f.at(v, 0, 0, 0);
  double s1 = (f.ax(v, a, 1) - f0) + (f.ax(v, a, -1) - f0);
  double s2 = (f.ax(v, a, 2) - f0) + (f.ax(v, a, -2) - f0);
  double s3 = (f.ax(v, a, 3) - f0) + (f.ax(v, a, -3) - f0);
  double s4 = (f.ax(v, a, 4) - f0) + (f.ax(v, a, -4) - f0);
  return ((8064.0 * s1 - 1008.0 * s2) + (128.0 * s3 - 9.0 * s4)) * (inv_h2 * (1.0 / 5040.0));
}

// differentiates on the fly from a point accessor P
template <class P, int ORDER = 4>
struct OnTheFly {
  P pt;
  Coef C;
  double beta[3];
  CHM_HD double f(int v) const { return pt.at(v, 0, 0, 0); }
  CHM_HD double d1(int v, int a) const {
    return ORDER == 4 ? d1_o4(pt, v, a, C.inv_h) : d1_o8(pt, v, a, C.inv_h);
  }
  CHM_HD double d2(int v, int a, int b) const {
    if (ORDER == 4) return a == b ? d2_o4(pt, v, a, C.inv_h2) : dmix_o4(pt, v, a, b, C.inv_h2);
    return a == b ? d2_o8(pt, v, a, C.inv_h2) : dmix_o8(pt, v, a, b, C.inv_h2);
  }
  CHM_HD double adv(int v, int a) const {
    return ORDER == 4 ? adv_o4(pt, v, a, beta[a], C.inv_h) : adv_o8(pt, v, a, beta[a], C.inv_h);
  }
  CHM_HD double ad(int v) const {
    double r = ORDER == 4 ? ko5(pt, v, C.ko) : ko_kq(pt, v, C.kq);
    if (v != V_A) r += (adv(v, 0) + adv(v, 1)) + adv(v, 2);
    return r;
  }
};

}  // namespace chm
