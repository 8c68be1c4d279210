// bssn_point.cuh -- pointwise BSSN right-hand side of the CUDA path (readings S3-S6, S10 in DESIGN.md):
// vacuum, chi variant, 1+log lapse, Gamma-driver shift.  Written against a "derivative provider" D so the
// same expression serves the fused kernel (D differentiates on the fly) and the split kernel (D reads the
// precomputed derivative arrays).  D supplies
//     D.f(v)          field value            D.d1(v,a)   centred d_a
//     D.d2(v,a,b)     centred d_a d_b, a<=b  D.ad(v)     beta^k d^up_k v + KO dissipation of v
// and the results leave through emit(v, rhs) as soon as they are complete (short live ranges; the stage
// update and store happen inside emit).  Symmetric tensors are packed (11,12,13,22,23,33) -> 0..5.
#pragma once
#include "common.cuh"

namespace chm {

enum { V_CHI = 0, V_GT = 1, V_K = 7, V_AT = 8, V_GAM = 14, V_ALPHA = 17, V_BETA = 18, V_B = 21, V_A = 24 };

CHM_HD constexpr int sym(int i, int j) {
  return i <= j ? (i == 0 ? j : i + j + 1) : (j == 0 ? i : i + j + 1);   // (0,0)0 (0,1)1 (0,2)2 (1,1)3 (1,2)4 (2,2)5
}

// contraction of a packed symmetric tensor with another: A^{ij} B_{ij}
CHM_HD double sdot(const double* A, const double* B) {
  return (A[0] * B[0] + A[3] * B[3] + A[5] * B[5]) + 2.0 * (A[1] * B[1] + A[2] * B[2] + A[4] * B[4]);
}

template <class D, class Emit>
CHM_HD void bssn_point(const D& d, const Coef& C, Emit&& emit) {
  const double third = 1.0 / 3.0, two_thirds = 2.0 / 3.0;

  // ---- metric, inverse metric ----------------------------------------------------------------------
  double g[6], gu[6];
#pragma unroll
  for (int s = 0; s < 6; ++s) g[s] = d.f(V_GT + s);
  {
    double c00 = g[3] * g[5] - g[4] * g[4];
    double c01 = g[2] * g[4] - g[1] * g[5];
    double c02 = g[1] * g[4] - g[2] * g[3];
    double det = g[0] * c00 + g[1] * c01 + g[2] * c02;
    double idet = 1.0 / det;
    gu[0] = c00 * idet;
    gu[1] = c01 * idet;
    gu[2] = c02 * idet;
    gu[3] = (g[0] * g[5] - g[2] * g[2]) * idet;
    gu[4] = (g[1] * g[2] - g[0] * g[4]) * idet;
    gu[5] = (g[0] * g[3] - g[1] * g[1]) * idet;
  }
  const double chi = d.f(V_CHI), alpha = d.f(V_ALPHA), trK = d.f(V_K);
  const double ichi = 1.0 / chi;

  // ---- shift derivatives; db[j][i] = d_j beta^i ------------------------------------------------------
  double db[3][3];
#pragma unroll
  for (int j = 0; j < 3; ++j)
#pragma unroll
    for (int i = 0; i < 3; ++i) db[j][i] = d.d1(V_BETA + i, j);
  const double divb = (db[0][0] + db[1][1]) + db[2][2];

  // ---- d_t chi, d_t gt_ij, d_t alpha, d_t beta^i -----------------------------------------------------
  emit(V_CHI, two_thirds * chi * (alpha * trK - divb) + d.ad(V_CHI));
  double At[6];
#pragma unroll
  for (int s = 0; s < 6; ++s) At[s] = d.f(V_AT + s);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) {
      double lie = 0.0;   // gt_ik d_j beta^k + gt_jk d_i beta^k
#pragma unroll
      for (int k = 0; k < 3; ++k) lie += g[sym(i, k)] * db[j][k] + g[sym(j, k)] * db[i][k];
      int s = sym(i, j);
      emit(V_GT + s, (lie - two_thirds * g[s] * divb) - 2.0 * alpha * At[s] + d.ad(V_GT + s));
    }
  emit(V_ALPHA, -2.0 * alpha * trK + d.ad(V_ALPHA));
  double Bv[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    Bv[i] = d.f(V_B + i);
    emit(V_BETA + i, C.sgc * Bv[i] + d.ad(V_BETA + i));
  }

  // ---- Christoffel symbols of gt ---------------------------------------------------------------------
  // Cl[k][s(i,j)] = Gamma~_kij = 1/2 (d_i gt_kj + d_j gt_ki - d_k gt_ij);  Cu[k][s] = gtu^{kl} Cl[l][s]
  double Cl[3][6], Cu[3][6], Gn[3];
  {
    double dg[3][6];   // dg[c][s] = d_c gt_s
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int s = 0; s < 6; ++s) dg[c][s] = d.d1(V_GT + s, c);
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = i; j < 3; ++j)
          Cl[k][sym(i, j)] = 0.5 * ((dg[i][sym(k, j)] + dg[j][sym(k, i)]) - dg[k][sym(i, j)]);
  }
#pragma unroll
  for (int k = 0; k < 3; ++k) {
#pragma unroll
    for (int s = 0; s < 6; ++s)
      Cu[k][s] = gu[sym(k, 0)] * Cl[0][s] + gu[sym(k, 1)] * Cl[1][s] + gu[sym(k, 2)] * Cl[2][s];
    Gn[k] = sdot(gu, Cu[k]);
  }

  // ---- conformal Ricci tensor R~_ij --------------------------------------------------------------------
  double Rt[6];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) {
      // 1/2 Gamma~^k_n (Gamma~_ijk + Gamma~_jik)
      double acc = 0.0;
#pragma unroll
      for (int k = 0; k < 3; ++k) acc += Gn[k] * (Cl[i][sym(j, k)] + Cl[j][sym(i, k)]);
      acc *= 0.5;
      // gtu^{lm} (Gamma~^k_li Gamma~_jkm + Gamma~^k_lj Gamma~_ikm + Gamma~^k_im Gamma~_klj)
#pragma unroll
      for (int l = 0; l < 3; ++l)
#pragma unroll
        for (int m = 0; m < 3; ++m) {
          double q = 0.0;
#pragma unroll
          for (int k = 0; k < 3; ++k)
            q += Cu[k][sym(l, i)] * Cl[j][sym(k, m)] + Cu[k][sym(l, j)] * Cl[i][sym(k, m)] +
                 Cu[k][sym(i, m)] * Cl[k][sym(l, j)];
          acc += gu[sym(l, m)] * q;
        }
      Rt[sym(i, j)] = acc;
    }
  // -1/2 gtu^{lm} d_l d_m gt_ij
#pragma unroll
  for (int s = 0; s < 6; ++s) {
    double dd[6];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b) dd[sym(a, b)] = d.d2(V_GT + s, a, b);
    Rt[s] -= 0.5 * sdot(gu, dd);
  }
  // 1/2 (gt_ki d_j Gt^k + gt_kj d_i Gt^k)
  {
    double dG[3][3];   // dG[j][k] = d_j Gt^k
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
      for (int k = 0; k < 3; ++k) dG[j][k] = d.d1(V_GAM + k, j);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j) {
        double q = 0.0;
#pragma unroll
        for (int k = 0; k < 3; ++k) q += g[sym(k, i)] * dG[j][k] + g[sym(k, j)] * dG[i][k];
        Rt[sym(i, j)] += 0.5 * q;
      }
  }

  // ---- chi and lapse second covariant derivatives ----------------------------------------------------------
  double dchi[3], dal[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) { dchi[a] = d.d1(V_CHI, a); dal[a] = d.d1(V_ALPHA, a); }
  double X[6];         // X_ij = -D_i D_j alpha + alpha (R~_ij + R^chi_ij)
  double lap_alpha;    // D^2 alpha
  {
    double cdchi[6], cdal[6];   // conformal Hessians  d_i d_j u - Gamma~^k_ij d_k u
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b) {
        int s = sym(a, b);
        cdchi[s] = d.d2(V_CHI, a, b) - (Cu[0][s] * dchi[0] + Cu[1][s] * dchi[1] + Cu[2][s] * dchi[2]);
        cdal[s] = d.d2(V_ALPHA, a, b) - (Cu[0][s] * dal[0] + Cu[1][s] * dal[1] + Cu[2][s] * dal[2]);
      }
    double chichi[6], chial[6];  // d_i chi d_j chi ; d_i chi d_j alpha + d_j chi d_i alpha
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b) {
        chichi[sym(a, b)] = dchi[a] * dchi[b];
        chial[sym(a, b)] = dchi[a] * dal[b] + dchi[b] * dal[a];
      }
    const double tr_cdchi = sdot(gu, cdchi), tr_cdal = sdot(gu, cdal);
    const double tr_chichi = sdot(gu, chichi), tr_chial = 0.5 * sdot(gu, chial);  // gtu^{kl} d_k chi d_l alpha
    lap_alpha = chi * tr_cdal - 0.5 * tr_chial;
    const double h2 = 0.5 * ichi, h4 = 0.25 * ichi * ichi;
#pragma unroll
    for (int s = 0; s < 6; ++s) {
      double DDa = cdal[s] + h2 * (chial[s] - g[s] * tr_chial);
      double Rchi = h2 * (cdchi[s] + g[s] * tr_cdchi) - h4 * (chichi[s] + 3.0 * g[s] * tr_chichi);
      X[s] = alpha * (Rt[s] + Rchi) - DDa;
    }
  }

  // ---- extrinsic curvature ------------------------------------------------------------------------------
  // Am[i][j] = At^i_j = gtu^{ik} At_kj ; Au = At^{ij} packed
  double Am[3][3], Au[6];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      Am[i][j] = gu[sym(i, 0)] * At[sym(0, j)] + gu[sym(i, 1)] * At[sym(1, j)] + gu[sym(i, 2)] * At[sym(2, j)];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j)
      Au[sym(i, j)] = Am[i][0] * gu[sym(0, j)] + Am[i][1] * gu[sym(1, j)] + Am[i][2] * gu[sym(2, j)];

  emit(V_K, (alpha * (sdot(Au, At) + third * trK * trK) - lap_alpha) + d.ad(V_K));

  {
    const double trX = sdot(gu, X);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j) {
        int s = sym(i, j);
        double AA = 0.0, lie = 0.0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          AA += At[sym(i, k)] * Am[k][j];
          lie += At[sym(i, k)] * db[j][k] + At[sym(j, k)] * db[i][k];
        }
        double r = chi * (X[s] - third * g[s] * trX) + alpha * (trK * At[s] - 2.0 * AA) +
                   (lie - two_thirds * At[s] * divb);
        emit(V_AT + s, r + d.ad(V_AT + s));
      }
  }

  // ---- Gamma~^i and B^i ---------------------------------------------------------------------------------------
  double dK[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) dK[a] = d.d1(V_K, a);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double ddb[6];   // d_j d_k beta^i
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a; b < 3; ++b) ddb[sym(a, b)] = d.d2(V_BETA + i, a, b);
    double r = sdot(gu, ddb);
    // 1/3 gtu^{ij} d_j (d_k beta^k)
    double graddiv = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      double dj_div = (d.d2(V_BETA + 0, j < 0 ? j : 0, j > 0 ? j : 0) + d.d2(V_BETA + 1, j < 1 ? j : 1, j > 1 ? j : 1)) +
                      d.d2(V_BETA + 2, j < 2 ? j : 2, j > 2 ? j : 2);
      graddiv += gu[sym(i, j)] * dj_div;
    }
    r += third * graddiv;
    double t = sdot(Cu[i], Au);   // Gamma~^i_jk At^{jk}
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      t -= two_thirds * gu[sym(i, j)] * dK[j] + 1.5 * ichi * Au[sym(i, j)] * dchi[j];
      r -= 2.0 * Au[sym(i, j)] * dal[j] + Gn[j] * db[j][i];
    }
    r += 2.0 * alpha * t + two_thirds * Gn[i] * divb;
    emit(V_GAM + i, r + d.ad(V_GAM + i));
    emit(V_B + i, (r - C.eta * Bv[i]) + d.ad(V_B + i));
  }

  // ---- slot 25 (S3): inert, dissipation only ----------------------------------------------------------------
  emit(V_A, d.ad(V_A));
}

}  // namespace chm
