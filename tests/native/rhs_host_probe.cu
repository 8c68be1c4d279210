// Host-side probe of the CUDA path's own right-hand-side arithmetic (no device needed): the finite-difference
// templates of csrc/stencils.cuh, the derivative provider OnTheFly and the pointwise BSSN expression of
// csrc/bssn_point.cuh -- the code the derivative-split kernels and the L1-path wave kernels instantiate on the
// device -- compiled for the host and run over a periodic block read from a file.
//   rhs_host_probe <system 0|1|2> <order> <nx> <ny> <nz> <g> <h> <eps> <eta> <sgc> <ko_order> <in.bin> <out.bin>
// in.bin: ghosted state [V][nz+2g][ny+2g][nx+2g] doubles (ghosts filled); out.bin: rhs [V][nz][ny][nx].
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "../../paper_1307_6488_b200/csrc/stencils.cuh"

using namespace chm;

struct HostPoint {   // same interface as GlobalPoint
  const double* p;
  long sy, sz, sv;
  __host__ __device__ double at(int v, int di, int dj, int dk) const { return p[v * sv + dk * sz + dj * sy + di]; }
  __host__ __device__ double ax(int v, int a, int m) const { return a == 0 ? at(v, m, 0, 0) : (a == 1 ? at(v, 0, m, 0) : at(v, 0, 0, m)); }
  __host__ __device__ double ax2(int v, int a, int m, int b, int n) const {
    int d[3] = {0, 0, 0};
    d[a] = m; d[b] = n;
    return at(v, d[0], d[1], d[2]);
  }
};

int main(int argc, char** argv) {
  if (argc != 14) return 2;
  const int system = atoi(argv[1]), order = atoi(argv[2]), nx = atoi(argv[3]), ny = atoi(argv[4]), nz = atoi(argv[5]),
            g = atoi(argv[6]), ko_order = atoi(argv[11]);
  const double h = atof(argv[7]), eps = atof(argv[8]), eta = atof(argv[9]), sgc = atof(argv[10]);
  const int V = system == 0 ? 2 : system == 1 ? 25 : 5;
  const long tx = nx + 2 * g, ty = ny + 2 * g, tz = nz + 2 * g, n = tx * ty * tz;
  std::vector<double> st((size_t)V * n), out((size_t)V * nx * ny * nz);
  FILE* f = fopen(argv[12], "rb");
  if (!f || fread(st.data(), 8, st.size(), f) != st.size()) return 3;
  fclose(f);
  Coef C;   // as chemora.cu's make_coef
  C.inv_h = 1.0 / h; C.inv_h2 = 1.0 / (h * h); C.ko = eps / (64.0 * h); C.eta = eta; C.sgc = sgc;
  const double w5[5] = {15.0, -6.0, 1.0, 0.0, 0.0}, w9[5] = {210.0, -120.0, 45.0, -10.0, 1.0};
  for (int k = 0; k < 5; ++k) C.kq[k] = ko_order == 9 ? eps / (1024.0 * h) * w9[k] : C.ko * w5[k];
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        HostPoint P{st.data() + ((long)(k + g) * ty + (j + g)) * tx + (i + g), tx, tx * ty, n};
        auto put = [&](int v, double r) { out[(((size_t)v * nz + k) * ny + j) * nx + i] = r; };
        if (system == 1) {
          if (order == 4) {
            OnTheFly<HostPoint, 4> d{P, C, {P.at(V_BETA, 0, 0, 0), P.at(V_BETA + 1, 0, 0, 0), P.at(V_BETA + 2, 0, 0, 0)}};
            bssn_point(d, C, put);
          } else {
            OnTheFly<HostPoint, 8> d{P, C, {P.at(V_BETA, 0, 0, 0), P.at(V_BETA + 1, 0, 0, 0), P.at(V_BETA + 2, 0, 0, 0)}};
            bssn_point(d, C, put);
          }
        } else if (system == 0) {   // as wave_kernel: d_t phi = pi, d_t pi = laplacian(phi), KO on both
          double lap = order == 4 ? (d2_o4(P, 0, 0, C.inv_h2) + d2_o4(P, 0, 1, C.inv_h2)) + d2_o4(P, 0, 2, C.inv_h2)
                                  : (d2_o8(P, 0, 0, C.inv_h2) + d2_o8(P, 0, 1, C.inv_h2)) + d2_o8(P, 0, 2, C.inv_h2);
          double r0 = P.at(1, 0, 0, 0), r1 = lap;
          if (eps != 0.0) { r0 += ko5(P, 0, C.ko); r1 += ko5(P, 1, C.ko); }
          put(0, r0); put(1, r1);
        } else {                    // Sample 1: d_t u = rho, d_t rho = d_i v_i, d_t v_i = d_i rho
          auto d1 = [&](int v, int a) { return order == 4 ? d1_o4(P, v, a, C.inv_h) : d1_o8(P, v, a, C.inv_h); };
          double r[5] = {P.at(1, 0, 0, 0), (d1(2, 0) + d1(3, 1)) + d1(4, 2), d1(1, 0), d1(1, 1), d1(1, 2)};
          for (int v = 0; v < 5; ++v) put(v, eps != 0.0 ? r[v] + ko5(P, v, C.ko) : r[v]);
        }
      }
  f = fopen(argv[13], "wb");
  if (!f || fwrite(out.data(), 8, out.size(), f) != out.size()) return 4;
  fclose(f);
  return 0;
}
