// oracle/oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU restatement (fp64) of the hot path of the codes Chemora
// generates (arXiv:1307.6488): "a calculation is applied to all grid points" (PAPER.md:133,
// :187, :218-220) with high-order finite differences, ghost-zone
// synchronisation and a method-of-lines time integrator (PAPER.md:338,
// :408).  The paper prints no equations, stencil coefficients or integrator formula; the
// readings used here are SURVEY.md section 8(c) S1-S14, restated in DESIGN.md "Readings".
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
// build, load or call this file.  It shares no code with paper_1307_6488_b200/ (the CUDA
// path): no headers, no tables, no helpers.
//
// Data layout of the ORACLE (its own; the CUDA library uses a padded one): a "state" is
// V arrays, each (nz+2g) x (ny+2g) x (nx+2g) doubles, x fastest, no row padding.
//
// Every stencil is evaluated in *difference form* (pairs f[+k]-f[-k] for antisymmetric
// stencils, (f[+k]-f0)+(f[-k]-f0) for symmetric ones, (f[m]-f0) for one-sided ones; valid
// because the coefficients sum to zero).  DESIGN.md reading R-H1 says why.
//
// Pins (tests/test_oracle_*.py): polynomial exactness of every stencil (O1), the exact
// discrete Fourier solution of the wave system (O2), convergence order (O3), flat stays
// flat bitwise (O4), Kasner (O5), linearised BSSN (O6), Schwarzschild in isotropic (O7) and
// Kerr-Schild (O8) coordinates; for system 2 (the paper's Sample 1) the exact
// discrete Fourier solution, the discrete energy identity and the energy of the Gaussian pulse
// (W1-W3, tests/test_oracle_wave1.py).  "Parity unpinned" (conventions of this build that the
// paper does not fix, so nothing external can pin them): eta, eps_diss, dx, the inert 25th
// slot A, KO order 5 on BSSN.
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC oracle.cpp -o liboracle.so
#include <cmath>
#include <cstddef>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct Grid {
  int nx, ny, nz, g;   // interior sizes and ghost width
  long tx, ty, tz;     // totals including ghosts
  int order;           // 4 or 8 (centred FD order)
  double h;            // grid spacing, same in x,y,z
  long npts() const { return tx * ty * tz; }
};

Grid make_grid(int nx, int ny, int nz, int g, int order, double h) {
  Grid G;
  G.nx = nx; G.ny = ny; G.nz = nz; G.g = g;
  G.tx = nx + 2L * g; G.ty = ny + 2L * g; G.tz = nz + 2L * g;
  G.order = order; G.h = h;
  return G;
}

// linear index of interior coordinate (i,j,k); i in [-g, nx+g)
inline long idx(const Grid& G, int i, int j, int k) {
  return ((long)(k + G.g) * G.ty + (j + G.g)) * G.tx + (i + G.g);
}

// value of f at point p=(i,j,k) shifted by `off` cells along `axis` (0=x,1=y,2=z)
inline double at(const double* f, const Grid& G, int i, int j, int k, int axis, int off) {
  if (axis == 0) return f[idx(G, i + off, j, k)];
  if (axis == 1) return f[idx(G, i, j + off, k)];
  return f[idx(G, i, j, k + off)];
}

// ---------------------------------------------------------------------------------------
// Finite-difference operators (reading S2).  Coefficients as exact integers over a common
// denominator:
//   1st, O4: ( 1, -8, 0, 8, -1)/12h
//   1st, O8: ( 3, -32, 168, -672, 0, 672, -168, 32, -3)/840h
//   2nd, O4: (-1, 16, -30, 16, -1)/12h^2
//   2nd, O8: (-9, 128, -1008, 8064, -14350, 8064, -1008, 128, -9)/5040h^2
// ---------------------------------------------------------------------------------------

// centred first derivative d/dx_axis, undivided by h: sum_m c_m (f[+m] - f[-m])
double d1_undivided(const double* f, const Grid& G, int i, int j, int k, int axis) {
  if (G.order == 4) {
    double a1 = at(f, G, i, j, k, axis, +1) - at(f, G, i, j, k, axis, -1);
    double a2 = at(f, G, i, j, k, axis, +2) - at(f, G, i, j, k, axis, -2);
    return (8.0 * a1 - a2) / 12.0;
  } else {
    double a1 = at(f, G, i, j, k, axis, +1) - at(f, G, i, j, k, axis, -1);
    double a2 = at(f, G, i, j, k, axis, +2) - at(f, G, i, j, k, axis, -2);
    double a3 = at(f, G, i, j, k, axis, +3) - at(f, G, i, j, k, axis, -3);
    double a4 = at(f, G, i, j, k, axis, +4) - at(f, G, i, j, k, axis, -4);
    return (672.0 * a1 - 168.0 * a2 + 32.0 * a3 - 3.0 * a4) / 840.0;
  }
}

double d1(const double* f, const Grid& G, int i, int j, int k, int axis) {
  return d1_undivided(f, G, i, j, k, axis) / G.h;
}

// centred second derivative d^2/dx_axis^2:  sum_m c_m ((f[+m]-f0) + (f[-m]-f0)) / h^2
double d2(const double* f, const Grid& G, int i, int j, int k, int axis) {
  double f0 = f[idx(G, i, j, k)];
  double s[5];
  int half = G.order / 2;
  for (int m = 1; m <= half; ++m)
    s[m] = (at(f, G, i, j, k, axis, +m) - f0) + (at(f, G, i, j, k, axis, -m) - f0);
  if (G.order == 4) return (16.0 * s[1] - s[2]) / (12.0 * G.h * G.h);
  return (8064.0 * s[1] - 1008.0 * s[2] + 128.0 * s[3] - 9.0 * s[4]) / (5040.0 * G.h * G.h);
}

// mixed derivative d^2/(dx_a dx_b), a != b: the 1-D first-derivative stencil along a applied
// to the 1-D first-derivative stencil along b (16 points at O4, 64 at O8).
double dmixed(const double* f, const Grid& G, int i, int j, int k, int a, int b) {
  int half = G.order / 2;
  double e[5];
  for (int m = 1; m <= half; ++m) {
    int ip = i, jp = j, kp = k, im = i, jm = j, km = k;
    if (a == 0) { ip += m; im -= m; } else if (a == 1) { jp += m; jm -= m; } else { kp += m; km -= m; }
    e[m] = d1_undivided(f, G, ip, jp, kp, b) - d1_undivided(f, G, im, jm, km, b);
  }
  double r;
  if (G.order == 4) r = (8.0 * e[1] - e[2]) / 12.0;
  else r = (672.0 * e[1] - 168.0 * e[2] + 32.0 * e[3] - 3.0 * e[4]) / 840.0;
  return r / (G.h * G.h);
}

// generic second derivative d_a d_b
double dd(const double* f, const Grid& G, int i, int j, int k, int a, int b) {
  return a == b ? d2(f, G, i, j, k, a) : dmixed(f, G, i, j, k, a, b);
}

// one-sided ("partially upwinded") first derivative, one point off centre.
// side = +1 (used when beta^axis > 0):  O4 offsets -1..+3  (-3,-10,18,-6,1)/12h
//                                       O8 offsets -3..+5  (-5,60,-420,-378,1050,-420,140,-30,3)/840h
// side = -1 (beta^axis < 0): the mirror image, i.e. offsets negated and coefficients negated.
double dupw(const double* f, const Grid& G, int i, int j, int k, int axis, int side) {
  double f0 = f[idx(G, i, j, k)];
  double r;
  if (G.order == 4) {
    double m1 = at(f, G, i, j, k, axis, -1 * side) - f0;
    double p1 = at(f, G, i, j, k, axis, +1 * side) - f0;
    double p2 = at(f, G, i, j, k, axis, +2 * side) - f0;
    double p3 = at(f, G, i, j, k, axis, +3 * side) - f0;
    r = (-3.0 * m1 + 18.0 * p1 - 6.0 * p2 + p3) / 12.0;
  } else {
    double m3 = at(f, G, i, j, k, axis, -3 * side) - f0;
    double m2 = at(f, G, i, j, k, axis, -2 * side) - f0;
    double m1 = at(f, G, i, j, k, axis, -1 * side) - f0;
    double p1 = at(f, G, i, j, k, axis, +1 * side) - f0;
    double p2 = at(f, G, i, j, k, axis, +2 * side) - f0;
    double p3 = at(f, G, i, j, k, axis, +3 * side) - f0;
    double p4 = at(f, G, i, j, k, axis, +4 * side) - f0;
    double p5 = at(f, G, i, j, k, axis, +5 * side) - f0;
    r = (-5.0 * m3 + 60.0 * m2 - 420.0 * m1 + 1050.0 * p1 - 420.0 * p2 + 140.0 * p3 - 30.0 * p4 +
         3.0 * p5) / 840.0;
  }
  return (double)side * r / G.h;
}

// Kreiss-Oliger dissipation of order p=5 (reading S6), summed over the three axes:
//   + (eps/64h) sum_axes (u[-3] - 6u[-2] + 15u[-1] - 20u0 + 15u[+1] - 6u[+2] + u[+3])
double ko5(const double* f, const Grid& G, int i, int j, int k, double eps) {
  double f0 = f[idx(G, i, j, k)];
  double total = 0.0;
  for (int axis = 0; axis < 3; ++axis) {
    double s1 = (at(f, G, i, j, k, axis, +1) - f0) + (at(f, G, i, j, k, axis, -1) - f0);
    double s2 = (at(f, G, i, j, k, axis, +2) - f0) + (at(f, G, i, j, k, axis, -2) - f0);
    double s3 = (at(f, G, i, j, k, axis, +3) - f0) + (at(f, G, i, j, k, axis, -3) - f0);
    total += s3 - 6.0 * s2 + 15.0 * s1;
  }
  return eps * total / (64.0 * G.h);
}

// Kreiss-Oliger dissipation of order p=9 (reading S6b; SURVEY 8(f)-1 "9th-order KO (11-point)", the operator
// that goes with 8th-order differencing and 5 ghost zones), summed over the three axes:
//   + (eps/1024h) sum_axes (u[-5] - 10u[-4] + 45u[-3] - 120u[-2] + 210u[-1] - 252u0 + 210u[+1] - ... + u[+5])
// = + (eps/1024h) h^10 (D+ D-)^5 u, written in difference form like ko5 (the coefficients sum to zero).
double ko9(const double* f, const Grid& G, int i, int j, int k, double eps) {
  double f0 = f[idx(G, i, j, k)];
  double total = 0.0;
  for (int axis = 0; axis < 3; ++axis) {
    double s1 = (at(f, G, i, j, k, axis, +1) - f0) + (at(f, G, i, j, k, axis, -1) - f0);
    double s2 = (at(f, G, i, j, k, axis, +2) - f0) + (at(f, G, i, j, k, axis, -2) - f0);
    double s3 = (at(f, G, i, j, k, axis, +3) - f0) + (at(f, G, i, j, k, axis, -3) - f0);
    double s4 = (at(f, G, i, j, k, axis, +4) - f0) + (at(f, G, i, j, k, axis, -4) - f0);
    double s5 = (at(f, G, i, j, k, axis, +5) - f0) + (at(f, G, i, j, k, axis, -5) - f0);
    total += s5 - 10.0 * s4 + 45.0 * s3 - 120.0 * s2 + 210.0 * s1;
  }
  return eps * total / (1024.0 * G.h);
}

// advective term beta^k d^{up}_k u, side chosen by the sign of beta^k at the point (S2);
// beta^k == 0 contributes exactly 0.
double advect(const double* u, const double* const beta[3], const Grid& G, int i, int j, int k) {
  double total = 0.0;
  for (int axis = 0; axis < 3; ++axis) {
    double b = beta[axis][idx(G, i, j, k)];
    if (b > 0.0) total += b * dupw(u, G, i, j, k, axis, +1);
    else if (b < 0.0) total += b * dupw(u, G, i, j, k, axis, -1);
  }
  return total;
}

// ---------------------------------------------------------------------------------------
// Ghost-zone fill, periodic in all three axes (reading S8; PAPER.md:105 is the exchange this
// stands in for on one process): ghost (i,j,k) <- interior ((i mod nx),(j mod ny),(k mod nz)).
// ---------------------------------------------------------------------------------------
inline int wrap(int i, int n) { int r = i % n; return r < 0 ? r + n : r; }

void fill_ghosts(double* f, const Grid& G) {
  for (int k = -G.g; k < G.nz + G.g; ++k)
    for (int j = -G.g; j < G.ny + G.g; ++j)
      for (int i = -G.g; i < G.nx + G.g; ++i) {
        bool interior = (i >= 0 && i < G.nx && j >= 0 && j < G.ny && k >= 0 && k < G.nz);
        if (!interior) f[idx(G, i, j, k)] = f[idx(G, wrap(i, G.nx), wrap(j, G.ny), wrap(k, G.nz))];
      }
}

// ---------------------------------------------------------------------------------------
// System 0 (reading S1): scalar wave equation, first order in time, V = 2: (phi, pi)
//   d_t phi = pi (+ KO),   d_t pi = delta^{ij} d_i d_j phi (+ KO)
// ---------------------------------------------------------------------------------------
enum { SYS_WAVE = 0, SYS_BSSN = 1, SYS_WAVE1 = 2 };
int nvars_of(int system) { return system == SYS_WAVE ? 2 : system == SYS_BSSN ? 25 : 5; }

struct Params {
  double eps_diss;  // KO strength; 0 switches the KO term off (and its +-3 reads)
  double eta;       // Gamma-driver damping (S5)
  double shift_gamma_coeff;  // 3/4 (S5)
  int ko_order;     // 5 (S6, the default) or 9 (S6b: needs 5 ghost zones)
};
// the dissipation operator the parameters select
inline double ko(const double* f, const Grid& G, int i, int j, int k, const Params& P) {
  return P.ko_order == 9 ? ko9(f, G, i, j, k, P.eps_diss) : ko5(f, G, i, j, k, P.eps_diss);
}

void wave_rhs(const double* state, double* rhs, const Grid& G, const Params& P) {
  const long n = G.npts();
  const double* phi = state;
  const double* pi = state + n;
#pragma omp parallel for schedule(static)
  for (int k = 0; k < G.nz; ++k)
    for (int j = 0; j < G.ny; ++j)
      for (int i = 0; i < G.nx; ++i) {
        long p = idx(G, i, j, k);
        double rphi = pi[p];
        double rpi = (d2(phi, G, i, j, k, 0) + d2(phi, G, i, j, k, 1)) + d2(phi, G, i, j, k, 2);
        if (P.eps_diss != 0.0) {
          rphi += ko(phi, G, i, j, k, P);
          rpi += ko(pi, G, i, j, k, P);
        }
        rhs[p] = rphi;
        rhs[n + p] = rpi;
      }
}

// ---------------------------------------------------------------------------------------
// System 2 ("Sample 1"): the scalar wave equation in fully first-order form,
// V = 5: (u, rho, v_1, v_2, v_3), propagation speed 1:
//   D_t u = rho ;  D_t rho = delta^{ij} D_i v_j ;  D_t v_i = D_i rho      (+ KO on every variable)
// D_i = centred first derivative of the chosen order (reading S2).
// ---------------------------------------------------------------------------------------
void wave1_rhs(const double* state, double* rhs, const Grid& G, const Params& P) {
  const long n = G.npts();
  const double* u = state;
  const double* rho = state + n;
  const double* v[3] = {state + 2 * n, state + 3 * n, state + 4 * n};
#pragma omp parallel for schedule(static)
  for (int k = 0; k < G.nz; ++k)
    for (int j = 0; j < G.ny; ++j)
      for (int i = 0; i < G.nx; ++i) {
        long p = idx(G, i, j, k);
        double r[5];
        r[0] = rho[p];
        r[1] = (d1(v[0], G, i, j, k, 0) + d1(v[1], G, i, j, k, 1)) + d1(v[2], G, i, j, k, 2);
        for (int a = 0; a < 3; ++a) r[2 + a] = d1(rho, G, i, j, k, a);
        if (P.eps_diss != 0.0) {
          r[0] += ko(u, G, i, j, k, P);
          r[1] += ko(rho, G, i, j, k, P);
          for (int a = 0; a < 3; ++a) r[2 + a] += ko(v[a], G, i, j, k, P);
        }
        for (int c = 0; c < 5; ++c) rhs[c * n + p] = r[c];
      }
}

// ---------------------------------------------------------------------------------------
// System 1 (readings S3-S6, S10): vacuum BSSN, chi variant, 1+log lapse, Gamma-driver shift.
// Slots: 0 chi | 1..6 gt11 gt12 gt13 gt22 gt23 gt33 | 7 trK | 8..13 At11..At33 | 14..16 Gt^i
//        | 17 alpha | 18..20 beta^i | 21..23 B^i | 24 A (inert: d_t A = KO only)
// ---------------------------------------------------------------------------------------
const int SYM[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};  // (i,j) -> packed symmetric slot

void bssn_rhs_point(const double* const u[25], double* const r[25], const Grid& G, const Params& P,
                    int i, int j, int k) {
  const long p = idx(G, i, j, k);
  const double* chi_f = u[0];
  const double* K_f = u[7];
  const double* alpha_f = u[17];
  const double* const beta_f[3] = {u[18], u[19], u[20]};

  // fields at the point
  double chi = chi_f[p], K = K_f[p], alpha = alpha_f[p];
  double gt[3][3], At[3][3], Gt[3], beta[3], B[3];
  for (int a = 0; a < 3; ++a) {
    for (int b = 0; b < 3; ++b) {
      gt[a][b] = u[1 + SYM[a][b]][p];
      At[a][b] = u[8 + SYM[a][b]][p];
    }
    Gt[a] = u[14 + a][p];
    beta[a] = u[18 + a][p];
    B[a] = u[21 + a][p];
  }
  (void)Gt;  // undifferentiated Gamma-tilde is taken from the metric (reading S10)

  // centred first derivatives; first index = direction of differentiation
  double dchi[3], dK[3], dalpha[3], dgt[3][3][3], dGt[3][3], dbeta[3][3];
  for (int c = 0; c < 3; ++c) {
    dchi[c] = d1(chi_f, G, i, j, k, c);
    dK[c] = d1(K_f, G, i, j, k, c);
    dalpha[c] = d1(alpha_f, G, i, j, k, c);
    for (int a = 0; a < 3; ++a) {
      dGt[c][a] = d1(u[14 + a], G, i, j, k, c);      // d_c Gt^a
      dbeta[c][a] = d1(u[18 + a], G, i, j, k, c);    // d_c beta^a
      for (int b = 0; b < 3; ++b) dgt[c][a][b] = d1(u[1 + SYM[a][b]], G, i, j, k, c);  // d_c gt_ab
    }
  }
  // centred second derivatives
  double ddchi[3][3], ddalpha[3][3], ddgt[3][3][3][3], ddbeta[3][3][3];
  for (int c = 0; c < 3; ++c)
    for (int d = 0; d < 3; ++d) {
      ddchi[c][d] = dd(chi_f, G, i, j, k, c, d);
      ddalpha[c][d] = dd(alpha_f, G, i, j, k, c, d);
      for (int a = 0; a < 3; ++a) {
        ddbeta[c][d][a] = dd(u[18 + a], G, i, j, k, c, d);  // d_c d_d beta^a
        for (int b = 0; b < 3; ++b) ddgt[c][d][a][b] = dd(u[1 + SYM[a][b]], G, i, j, k, c, d);
      }
    }

  // inverse conformal metric gtu = gt^{-1} (cofactors / determinant)
  double det = gt[0][0] * (gt[1][1] * gt[2][2] - gt[1][2] * gt[2][1]) -
               gt[0][1] * (gt[1][0] * gt[2][2] - gt[1][2] * gt[2][0]) +
               gt[0][2] * (gt[1][0] * gt[2][1] - gt[1][1] * gt[2][0]);
  double gtu[3][3];
  gtu[0][0] = (gt[1][1] * gt[2][2] - gt[1][2] * gt[2][1]) / det;
  gtu[0][1] = (gt[0][2] * gt[2][1] - gt[0][1] * gt[2][2]) / det;
  gtu[0][2] = (gt[0][1] * gt[1][2] - gt[0][2] * gt[1][1]) / det;
  gtu[1][1] = (gt[0][0] * gt[2][2] - gt[0][2] * gt[2][0]) / det;
  gtu[1][2] = (gt[0][2] * gt[1][0] - gt[0][0] * gt[1][2]) / det;
  gtu[2][2] = (gt[0][0] * gt[1][1] - gt[0][1] * gt[1][0]) / det;
  gtu[1][0] = gtu[0][1]; gtu[2][0] = gtu[0][2]; gtu[2][1] = gtu[1][2];

  // Christoffel symbols of gt:  Gl[k][i][j] = Gamma~_{kij} = 1/2 (d_i gt_kj + d_j gt_ki - d_k gt_ij)
  double Gl[3][3][3], Gu[3][3][3], Gn[3];
  for (int c = 0; c < 3; ++c)
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) Gl[c][a][b] = 0.5 * (dgt[a][c][b] + dgt[b][c][a] - dgt[c][a][b]);
  // Gu[k][i][j] = Gamma~^k_{ij} = gtu^{kl} Gamma~_{lij};   Gn[k] = gtu^{ij} Gamma~^k_{ij}
  for (int c = 0; c < 3; ++c) {
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) {
        double s = 0.0;
        for (int l = 0; l < 3; ++l) s += gtu[c][l] * Gl[l][a][b];
        Gu[c][a][b] = s;
      }
    double s = 0.0;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) s += gtu[a][b] * Gu[c][a][b];
    Gn[c] = s;
  }

  // At with indices raised: Atm[i][j] = At^i_j = gtu^{ik} At_kj ; Atu[i][j] = At^{ij}
  double Atm[3][3], Atu[3][3];
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) {
      double s = 0.0;
      for (int c = 0; c < 3; ++c) s += gtu[a][c] * At[c][b];
      Atm[a][b] = s;
    }
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) {
      double s = 0.0;
      for (int c = 0; c < 3; ++c) s += Atm[a][c] * gtu[c][b];
      Atu[a][b] = s;
    }

  double divbeta = (dbeta[0][0] + dbeta[1][1]) + dbeta[2][2];

  // dissipation + advection of variable v
  auto diss = [&](int v) { return P.eps_diss != 0.0 ? ko(u[v], G, i, j, k, P) : 0.0; };
  auto adv = [&](int v) { return advect(u[v], beta_f, G, i, j, k); };

  // d_t chi = 2/3 chi (alpha K - d_k beta^k) + adv
  r[0][p] = (2.0 / 3.0) * chi * (alpha * K - divbeta) + adv(0) + diss(0);

  // d_t gt_ij = -2 alpha At_ij + gt_ik d_j beta^k + gt_jk d_i beta^k - 2/3 gt_ij d_k beta^k + adv
  for (int a = 0; a < 3; ++a)
    for (int b = a; b < 3; ++b) {
      double s = -2.0 * alpha * At[a][b];
      for (int c = 0; c < 3; ++c) s += gt[a][c] * dbeta[b][c] + gt[b][c] * dbeta[a][c];
      s -= (2.0 / 3.0) * gt[a][b] * divbeta;
      int v = 1 + SYM[a][b];
      r[v][p] = s + adv(v) + diss(v);
    }

  // D^2 alpha = chi gtu^{ij} (d_i d_j alpha - Gamma~^k_ij d_k alpha) - 1/2 gtu^{ij} d_i chi d_j alpha
  double DDalpha_trace = 0.0, dchi_dalpha = 0.0, dchi_dchi = 0.0;
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) {
      double cd = ddalpha[a][b];
      for (int c = 0; c < 3; ++c) cd -= Gu[c][a][b] * dalpha[c];
      DDalpha_trace += gtu[a][b] * cd;
      dchi_dalpha += gtu[a][b] * dchi[a] * dalpha[b];
      dchi_dchi += gtu[a][b] * dchi[a] * dchi[b];
    }
  double lap_alpha = chi * DDalpha_trace - 0.5 * dchi_dalpha;

  // d_t K = -D^2 alpha + alpha (At_ij At^ij + K^2/3) + adv
  double AtAt = 0.0;
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) AtAt += At[a][b] * Atu[a][b];
  r[7][p] = -lap_alpha + alpha * (AtAt + K * K / 3.0) + adv(7) + diss(7);

  // conformal covariant Hessian of chi and its trace
  double DDchi[3][3], DDchi_trace = 0.0;
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) {
      double s = ddchi[a][b];
      for (int c = 0; c < 3; ++c) s -= Gu[c][a][b] * dchi[c];
      DDchi[a][b] = s;
      DDchi_trace += gtu[a][b] * s;
    }

  // X_ij = -D_i D_j alpha + alpha (R~_ij + R^chi_ij)
  double X[3][3];
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) {
      // D_i D_j alpha = d_i d_j alpha - Gamma~^k_ij d_k alpha
      //               + (1/2chi)(d_i chi d_j alpha + d_j chi d_i alpha - gt_ij gtu^{kl} d_k chi d_l alpha)
      double DDa = ddalpha[a][b];
      for (int c = 0; c < 3; ++c) DDa -= Gu[c][a][b] * dalpha[c];
      DDa += (dchi[a] * dalpha[b] + dchi[b] * dalpha[a] - gt[a][b] * dchi_dalpha) / (2.0 * chi);

      // R~_ij = -1/2 gtu^{lm} d_l d_m gt_ij + 1/2 (gt_ki d_j Gt^k + gt_kj d_i Gt^k)
      //         + 1/2 Gamma~^k_n (Gamma~_ijk + Gamma~_jik)
      //         + gtu^{lm} (Gamma~^k_li Gamma~_jkm + Gamma~^k_lj Gamma~_ikm + Gamma~^k_im Gamma~_klj)
      double Rt = 0.0;
      for (int l = 0; l < 3; ++l)
        for (int m = 0; m < 3; ++m) Rt -= 0.5 * gtu[l][m] * ddgt[l][m][a][b];
      for (int c = 0; c < 3; ++c) {
        Rt += 0.5 * (gt[c][a] * dGt[b][c] + gt[c][b] * dGt[a][c]);
        Rt += 0.5 * Gn[c] * (Gl[a][b][c] + Gl[b][a][c]);
      }
      for (int l = 0; l < 3; ++l)
        for (int m = 0; m < 3; ++m) {
          double s = 0.0;
          for (int c = 0; c < 3; ++c)
            s += Gu[c][l][a] * Gl[b][c][m] + Gu[c][l][b] * Gl[a][c][m] + Gu[c][a][m] * Gl[c][l][b];
          Rt += gtu[l][m] * s;
        }

      // R^chi_ij = (1/2chi)(D~_i D~_j chi + gt_ij gtu^{kl} D~_k D~_l chi)
      //            - (1/4chi^2) d_i chi d_j chi - (3/4chi^2) gt_ij gtu^{kl} d_k chi d_l chi
      double Rchi = (DDchi[a][b] + gt[a][b] * DDchi_trace) / (2.0 * chi) -
                    dchi[a] * dchi[b] / (4.0 * chi * chi) -
                    3.0 * gt[a][b] * dchi_dchi / (4.0 * chi * chi);

      X[a][b] = -DDa + alpha * (Rt + Rchi);
    }
  double Xtrace = 0.0;
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) Xtrace += gtu[a][b] * X[a][b];

  // d_t At_ij = chi X^TF_ij + alpha (K At_ij - 2 At_ik At^k_j)
  //             + At_ik d_j beta^k + At_jk d_i beta^k - 2/3 At_ij d_k beta^k + adv
  for (int a = 0; a < 3; ++a)
    for (int b = a; b < 3; ++b) {
      double XTF = X[a][b] - gt[a][b] * Xtrace / 3.0;
      double AA = 0.0;
      for (int c = 0; c < 3; ++c) AA += At[a][c] * Atm[c][b];
      double s = chi * XTF + alpha * (K * At[a][b] - 2.0 * AA);
      for (int c = 0; c < 3; ++c) s += At[a][c] * dbeta[b][c] + At[b][c] * dbeta[a][c];
      s -= (2.0 / 3.0) * At[a][b] * divbeta;
      int v = 8 + SYM[a][b];
      r[v][p] = s + adv(v) + diss(v);
    }

  // d_t Gt^i |_0 = -2 At^{ij} d_j alpha
  //               + 2 alpha (Gamma~^i_jk At^{jk} - 2/3 gtu^{ij} d_j K - (3/2chi) At^{ij} d_j chi)
  //               + gtu^{jk} d_j d_k beta^i + 1/3 gtu^{ij} d_j d_k beta^k
  //               - Gamma~^j_n d_j beta^i + 2/3 Gamma~^i_n d_j beta^j
  double dtGt0[3];
  for (int a = 0; a < 3; ++a) {
    double s = 0.0;
    for (int b = 0; b < 3; ++b) s -= 2.0 * Atu[a][b] * dalpha[b];
    double t = 0.0;
    for (int b = 0; b < 3; ++b) {
      for (int c = 0; c < 3; ++c) t += Gu[a][b][c] * Atu[b][c];
      t -= (2.0 / 3.0) * gtu[a][b] * dK[b];
      t -= 1.5 * Atu[a][b] * dchi[b] / chi;
    }
    s += 2.0 * alpha * t;
    for (int b = 0; b < 3; ++b)
      for (int c = 0; c < 3; ++c) {
        s += gtu[b][c] * ddbeta[b][c][a];
        s += gtu[a][b] * ddbeta[b][c][c] / 3.0;
      }
    for (int b = 0; b < 3; ++b) s -= Gn[b] * dbeta[b][a];
    s += (2.0 / 3.0) * Gn[a] * divbeta;
    dtGt0[a] = s;
    r[14 + a][p] = s + adv(14 + a) + diss(14 + a);
  }

  // gauge (S5): d_t alpha = -2 alpha K + adv ; d_t beta^i = 3/4 B^i + adv ;
  //             d_t B^i = d_t Gt^i|_0 - eta B^i + adv
  r[17][p] = -2.0 * alpha * K + adv(17) + diss(17);
  for (int a = 0; a < 3; ++a) {
    r[18 + a][p] = P.shift_gamma_coeff * B[a] + adv(18 + a) + diss(18 + a);
    r[21 + a][p] = dtGt0[a] - P.eta * B[a] + adv(21 + a) + diss(21 + a);
  }
  // slot 25 (S3): inert, dissipation only
  r[24][p] = diss(24);
}

void bssn_rhs(const double* state, double* rhs, const Grid& G, const Params& P) {
  const long n = G.npts();
  const double* u[25];
  double* r[25];
  for (int v = 0; v < 25; ++v) { u[v] = state + v * n; r[v] = rhs + v * n; }
#pragma omp parallel for schedule(static)
  for (int k = 0; k < G.nz; ++k)
    for (int j = 0; j < G.ny; ++j)
      for (int i = 0; i < G.nx; ++i) bssn_rhs_point(u, r, G, P, i, j, k);
}

void rhs_any(int system, const double* state, double* rhs, const Grid& G, const Params& P) {
  if (system == SYS_WAVE) wave_rhs(state, rhs, G, P);
  else if (system == SYS_WAVE1) wave1_rhs(state, rhs, G, P);
  else bssn_rhs(state, rhs, G, P);
}

// ---------------------------------------------------------------------------------------
// Classical RK4 with the association fixed by reading S9 (4 buffers U, Y, S, k):
//   S = k1 ; Y2 = U + (dt/2) k1 ; S += 2 k2 ; Y3 = U + (dt/2) k2 ; S += 2 k3 ; Y4 = U + dt k3 ;
//   U+ = U + (dt/6) (S + k4).      Ghost fill before every RHS evaluation.
// ---------------------------------------------------------------------------------------
void rk4_step(int system, double* U, const Grid& G, const Params& P, double dt) {
  const int V = nvars_of(system);
  const long n = G.npts(), tot = V * n;
  std::vector<double> Y(tot, 0.0), S(tot, 0.0), kk(tot, 0.0);
  auto fill_all = [&](double* st) { for (int v = 0; v < V; ++v) fill_ghosts(st + v * n, G); };
  auto interior_loop = [&](auto body) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < G.nz; ++k)
      for (int v = 0; v < V; ++v)
        for (int j = 0; j < G.ny; ++j)
          for (int i = 0; i < G.nx; ++i) body(v * n + idx(G, i, j, k));
  };
  // stage 1
  fill_all(U);
  rhs_any(system, U, kk.data(), G, P);
  interior_loop([&](long q) { S[q] = kk[q]; Y[q] = U[q] + (dt / 2.0) * kk[q]; });
  // stage 2
  fill_all(Y.data());
  rhs_any(system, Y.data(), kk.data(), G, P);
  interior_loop([&](long q) { S[q] = S[q] + 2.0 * kk[q]; Y[q] = U[q] + (dt / 2.0) * kk[q]; });
  // stage 3
  fill_all(Y.data());
  rhs_any(system, Y.data(), kk.data(), G, P);
  interior_loop([&](long q) { S[q] = S[q] + 2.0 * kk[q]; Y[q] = U[q] + dt * kk[q]; });
  // stage 4
  fill_all(Y.data());
  rhs_any(system, Y.data(), kk.data(), G, P);
  interior_loop([&](long q) { U[q] = U[q] + (dt / 6.0) * (S[q] + kk[q]); });
}

// ---------------------------------------------------------------------------------------
// Second boundary kind (the paper's blocks have outer faces as well as inter-block
// faces; it prints no boundary condition): radiative (Sommerfeld) outer
// boundary, reading S16 of DESIGN.md.  Every point of the padded block outside the interior (the g
// ghost layers: faces, edges, corners) is a BOUNDARY POINT that is evolved, not filled:
//     d_t u = - v [ n^i D_i u + (u - u_inf) / r ],   n^i = x^i / r,   v = 1,
// with the block centred on the origin, x^i = (i - (N_i - 1)/2) h for i in [-g, N_i + g), r = |x|,
// u_inf = 1 for chi, gt11, gt22, gt33, alpha of the BSSN system and 0 for every other variable, and
// D_i the second-order first derivative: centred (u[+1] - u[-1]) / 2h where both neighbours exist in
// the padded array, else the one-sided three-point formula pointing into the block,
//     lowest index:  (-3 u[0] + 4 u[+1] - u[+2]) / 2h ;   highest:  (3 u[0] - 4 u[-1] + u[-2]) / 2h ,
// both evaluated in difference form (reading R-H1).
// No dissipation at boundary points.  The interior right-hand side is unchanged (it reads the
// boundary points as its stencil neighbours); there is no ghost fill.
// ---------------------------------------------------------------------------------------
double u_infinity(int system, int v) {
  if (system != SYS_BSSN) return 0.0;
  return (v == 0 || v == 1 || v == 4 || v == 6 || v == 17) ? 1.0 : 0.0;
}

inline bool is_interior(const Grid& G, int i, int j, int k) {
  return i >= 0 && i < G.nx && j >= 0 && j < G.ny && k >= 0 && k < G.nz;
}

// second-order first derivative along `axis` at a point of the padded array (centred, or one-sided at its two ends)
double d1_boundary(const double* f, const Grid& G, int i, int j, int k, int axis) {
  const int c = axis == 0 ? i : axis == 1 ? j : k;
  const int n = axis == 0 ? G.nx : axis == 1 ? G.ny : G.nz;
  // difference form (reading R-H1): -3 u0 + 4 u1 - u2 = 4 (u1 - u0) - (u2 - u0), every subtraction of near-equal
  // values exact, so near-flat data keeps its relative accuracy and flat data gives exactly 0
  const double u0 = at(f, G, i, j, k, axis, 0);
  if (c == -G.g) return (4.0 * (at(f, G, i, j, k, axis, 1) - u0) - (at(f, G, i, j, k, axis, 2) - u0)) / (2.0 * G.h);
  if (c == n + G.g - 1) return -(4.0 * (at(f, G, i, j, k, axis, -1) - u0) - (at(f, G, i, j, k, axis, -2) - u0)) / (2.0 * G.h);
  return (at(f, G, i, j, k, axis, 1) - at(f, G, i, j, k, axis, -1)) / (2.0 * G.h);
}

double radiative_rhs_point(const double* f, const Grid& G, int i, int j, int k, double uinf) {
  const double x = (i - 0.5 * (G.nx - 1)) * G.h, y = (j - 0.5 * (G.ny - 1)) * G.h, z = (k - 0.5 * (G.nz - 1)) * G.h;
  const double r = std::sqrt(x * x + y * y + z * z);
  const double nd = (x * d1_boundary(f, G, i, j, k, 0) + y * d1_boundary(f, G, i, j, k, 1) +
                     z * d1_boundary(f, G, i, j, k, 2)) / r;
  return -(nd + (f[idx(G, i, j, k)] - uinf) / r);
}

// rhs at every boundary point of every variable (interior entries untouched)
void radiative_rhs(int system, const double* state, double* rhs, const Grid& G) {
  const int V = nvars_of(system);
  const long n = G.npts();
  for (int v = 0; v < V; ++v)
    for (int k = -G.g; k < G.nz + G.g; ++k)
      for (int j = -G.g; j < G.ny + G.g; ++j)
        for (int i = -G.g; i < G.nx + G.g; ++i)
          if (!is_interior(G, i, j, k))
            rhs[v * n + idx(G, i, j, k)] = radiative_rhs_point(state + v * n, G, i, j, k, u_infinity(system, v));
}

// RK4 (reading S9, same association) on a block with radiative outer boundaries: the stage updates run over ALL
// points of the padded array, the right-hand side is the system's in the interior and the radiative one outside.
void rk4_step_radiative(int system, double* U, const Grid& G, const Params& P, double dt) {
  const int V = nvars_of(system);
  const long tot = V * G.npts();
  std::vector<double> Y(tot, 0.0), S(tot, 0.0), kk(tot, 0.0);
  auto rhs_all = [&](const double* st) { rhs_any(system, st, kk.data(), G, P); radiative_rhs(system, st, kk.data(), G); };
  rhs_all(U);
  for (long q = 0; q < tot; ++q) { S[q] = kk[q]; Y[q] = U[q] + (dt / 2.0) * kk[q]; }
  rhs_all(Y.data());
  for (long q = 0; q < tot; ++q) { S[q] = S[q] + 2.0 * kk[q]; Y[q] = U[q] + (dt / 2.0) * kk[q]; }
  rhs_all(Y.data());
  for (long q = 0; q < tot; ++q) { S[q] = S[q] + 2.0 * kk[q]; Y[q] = U[q] + dt * kk[q]; }
  rhs_all(Y.data());
  for (long q = 0; q < tot; ++q) U[q] = U[q] + (dt / 6.0) * (S[q] + kk[q]);
}

}  // namespace

// ---------------------------------------------------------------------------------------
// C entry points for the ctypes harness (oracle/oracle.py).  All arrays are host memory in
// the oracle layout described at the top.  params = {eps_diss, eta, shift_gamma_coeff, ko_order}.
// ---------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------
// RK3 (reading S9b; the paper's runs use "RK3", without a formula): the third-order
// strong-stability-preserving scheme of Shu and Osher,
//   U1 = U + dt f(U) ;  U2 = 3/4 U + 1/4 (U1 + dt f(U1)) ;  U+ = 1/3 U + 2/3 (U2 + dt f(U2)),
// every stage written as  a*U + b*(Y + dt*k)  with each product and sum rounded once.
// Ghost fill before every RHS evaluation.
// ---------------------------------------------------------------------------------------
static void rk3_step(int system, double* U, const Grid& G, const Params& P, double dt) {
  const int V = nvars_of(system);
  const long n = G.npts(), tot = V * n;
  std::vector<double> Ya(tot, 0.0), Yb(tot, 0.0), kk(tot, 0.0);
  auto fill_all = [&](double* st) { for (int v = 0; v < V; ++v) fill_ghosts(st + v * n, G); };
  auto stage = [&](const double* Y, double* out, double a, double b) {
    rhs_any(system, Y, kk.data(), G, P);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < G.nz; ++k)
      for (int v = 0; v < V; ++v)
        for (int j = 0; j < G.ny; ++j)
          for (int i = 0; i < G.nx; ++i) {
            long q = v * n + idx(G, i, j, k);
            out[q] = a * U[q] + b * (Y[q] + dt * kk[q]);
          }
  };
  fill_all(U);
  stage(U, Ya.data(), 0.0, 1.0);
  fill_all(Ya.data());
  stage(Ya.data(), Yb.data(), 3.0 / 4.0, 1.0 / 4.0);
  fill_all(Yb.data());
  stage(Yb.data(), U, 1.0 / 3.0, 2.0 / 3.0);
}

// ---------------------------------------------------------------------------------------
// Algebraic constraint enforcement of the BSSN variables (reading S10b; not in the paper, the
// standard companion of the evolution in its production runs): at every interior point
//   gt_ij <- gt_ij + gt_ij (det(gt)^(-1/3) - 1)   (det gt = 1)
//   At_ij <- At_ij - 1/3 gt_ij gtu^{kl} At_kl (tr At = 0), with the new gt and its inverse.
// ---------------------------------------------------------------------------------------
static void enforce_constraints(double* state, const Grid& G) {
  const long n = G.npts();
#pragma omp parallel for schedule(static)
  for (int k = 0; k < G.nz; ++k)
    for (int j = 0; j < G.ny; ++j)
      for (int i = 0; i < G.nx; ++i) {
        long p = idx(G, i, j, k);
        double g[6], A[6];
        for (int s = 0; s < 6; ++s) { g[s] = state[(1 + s) * n + p]; A[s] = state[(8 + s) * n + p]; }
        // packed order 11 12 13 22 23 33
        double det = g[0] * (g[3] * g[5] - g[4] * g[4]) - g[1] * (g[1] * g[5] - g[4] * g[2]) +
                     g[2] * (g[1] * g[4] - g[3] * g[2]);
        // rounding-aware form (reading R-H1): the correction factor minus one, det^(-1/3) - 1, is a small number
        // known to full relative accuracy, and gt_ij is rounded once at its own magnitude when it is added
        double f1 = std::expm1(-std::log(det) / 3.0);
        for (int s = 0; s < 6; ++s) g[s] = g[s] + g[s] * f1;
        // inverse of the rescaled metric (its determinant is 1 up to rounding; divide by it anyway)
        double c00 = g[3] * g[5] - g[4] * g[4], c01 = g[2] * g[4] - g[1] * g[5], c02 = g[1] * g[4] - g[2] * g[3];
        double d = g[0] * c00 + g[1] * c01 + g[2] * c02;
        double u[6] = {c00 / d, c01 / d, c02 / d, (g[0] * g[5] - g[2] * g[2]) / d, (g[1] * g[2] - g[0] * g[4]) / d,
                       (g[0] * g[3] - g[1] * g[1]) / d};
        double tr = (u[0] * A[0] + u[3] * A[3] + u[5] * A[5]) + 2.0 * (u[1] * A[1] + u[2] * A[2] + u[4] * A[4]);
        for (int s = 0; s < 6; ++s) {
          state[(1 + s) * n + p] = g[s];
          state[(8 + s) * n + p] = A[s] - (tr / 3.0) * g[s];
        }
      }
}

extern "C" {

void oracle_set_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n > 0 ? n : 1);
#else
  (void)n;
#endif
}

int oracle_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// op: 0 d1(axis a) | 1 dd(a,b) | 2 dupw(axis a, side b=+-1) | 3 ko5(eps) | 4 ko9(eps) ; `f` has ghosts,
// `out` is interior-packed nz*ny*nx.
void oracle_apply_op(int op, const double* f, double* out, int nx, int ny, int nz, int g, int order,
                     double h, int a, int b, double eps) {
  Grid G = make_grid(nx, ny, nz, g, order, h);
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        double v = 0.0;
        if (op == 0) v = d1(f, G, i, j, k, a);
        else if (op == 1) v = dd(f, G, i, j, k, a, b);
        else if (op == 2) v = dupw(f, G, i, j, k, a, b);
        else if (op == 3) v = ko5(f, G, i, j, k, eps);
        else if (op == 4) v = ko9(f, G, i, j, k, eps);
        out[((long)k * ny + j) * nx + i] = v;
      }
}

void oracle_fill_ghosts(double* state, int nvars, int nx, int ny, int nz, int g) {
  Grid G = make_grid(nx, ny, nz, g, 4, 1.0);
  for (int v = 0; v < nvars; ++v) fill_ghosts(state + v * G.npts(), G);
}

// rhs has the same ghosted shape as state; only interior entries are written.
void oracle_rhs(int system, const double* state, double* rhs, int nx, int ny, int nz, int g, int order,
                double h, const double* params) {
  Grid G = make_grid(nx, ny, nz, g, order, h);
  Params P = {params[0], params[1], params[2], (int)params[3]};
  rhs_any(system, state, rhs, G, P);
}

// U (ghosted) is advanced in place by `nsteps` RK4 steps; ghosts of the result are NOT refilled.
void oracle_rk4(int system, double* U, int nx, int ny, int nz, int g, int order, double h, double dt,
                const double* params, int nsteps) {
  Grid G = make_grid(nx, ny, nz, g, order, h);
  Params P = {params[0], params[1], params[2], (int)params[3]};
  for (int s = 0; s < nsteps; ++s) rk4_step(system, U, G, P, dt);
}

// U (ghosted) is advanced in place by `nsteps` RK3 steps (reading S9b); with enforce != 0 (BSSN only) the algebraic
// constraints are enforced after every step.
void oracle_rk3(int system, double* U, int nx, int ny, int nz, int g, int order, double h, double dt,
                const double* params, int nsteps, int enforce) {
  Grid G = make_grid(nx, ny, nz, g, order, h);
  Params P = {params[0], params[1], params[2], (int)params[3]};
  for (int s = 0; s < nsteps; ++s) {
    rk3_step(system, U, G, P, dt);
    if (enforce && system == SYS_BSSN) enforce_constraints(U, G);
  }
}

// The "Energy" calculation of the paper's Sample 1: eps = 1/2 (rho^2 + delta^ij v_i v_j) at every
// interior point of a ghosted system-2 state, written to a packed nz x ny x nx array.
void oracle_energy(const double* U, int nx, int ny, int nz, int g, double* eps) {
  Grid G = make_grid(nx, ny, nz, g, 4, 1.0);
  const long n = G.npts();
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        long p = idx(G, i, j, k);
        double rho = U[n + p], v1 = U[2 * n + p], v2 = U[3 * n + p], v3 = U[4 * n + p];
        eps[((long)k * ny + j) * nx + i] = 0.5 * (rho * rho + ((v1 * v1 + v2 * v2) + v3 * v3));
      }
}

void oracle_enforce(double* U, int nx, int ny, int nz, int g) {
  Grid G = make_grid(nx, ny, nz, g, 4, 1.0);
  enforce_constraints(U, G);
}

// Radiative outer boundary (reading S16): rhs at the boundary points of a ghosted state (interior entries of `rhs`
// are left as they are), and RK4 steps of a block whose ghost layers are evolved boundary points.
void oracle_radiative_rhs(int system, const double* state, double* rhs, int nx, int ny, int nz, int g, double h) {
  Grid G = make_grid(nx, ny, nz, g, 4, h);
  radiative_rhs(system, state, rhs, G);
}

void oracle_rk4_radiative(int system, double* U, int nx, int ny, int nz, int g, int order, double h, double dt,
                          const double* params, int nsteps) {
  Grid G = make_grid(nx, ny, nz, g, order, h);
  Params P = {params[0], params[1], params[2], (int)params[3]};
  for (int s = 0; s < nsteps; ++s) rk4_step_radiative(system, U, G, P, dt);
}

}  // extern "C"
