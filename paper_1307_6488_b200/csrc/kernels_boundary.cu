// kernels_boundary.cu -- the radiative (Sommerfeld) face kernel (reading S16) and the runtime sweep's
// agreement norm.  Plain loads and stores, no TMA.  Like the TMA kernels this file also compiles for the host
// (-DCHM_EMULATE on top of tests/native/cta_emu.hpp), where its launchers are left out.
#include "common.cuh"

namespace chm {

// ---------------------------------------------------------------------------------------------------
// Radiative (Sommerfeld) outer boundary, reading S16 (the second boundary kind; block faces:
// PAPER.md:105, :117-123).  The g ghost layers are evolved BOUNDARY POINTS: at each of them
//   k = -[ n^i D_i u + (u - u_inf) / r ],  n^i = x^i / r,  x^i = (i - (N_i - 1)/2) h  (block centred on the origin),
// D_i second order: centred where both neighbours exist in the padded array, one-sided three-point at its two ends;
// then the same Runge-Kutta stage epilogue as the interior kernels.  Same warp-per-row task decomposition as the
// ghost fill (regions A, B: whole padded rows; C: the 2g ghost columns of the interior rows).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) radiative_kernel(Layout L, Stage st, double h, unsigned uinf_mask, int rowsA,
                                                        int rowsAB, int lpr_shift) {
  const int g = L.g, tx = L.nx + 2 * g, lane = threadIdx.x & 31;
  const int task = blockIdx.x * 8 + (threadIdx.x >> 5);
  const int v = blockIdx.y;
  const double uinf = ((uinf_mask >> v) & 1u) ? 1.0 : 0.0;
  const double* u = st.in + (long)v * L.vstride + (L.xo - g);   // column 0 = first ghost column of a padded row
  const double ih2 = 1.0 / (2.0 * h);
  // second-order first derivative along a direction with element stride s, at padded coordinate c of n
  auto d1 = [&](const double* c0, long s, int c, int n) {
    // difference form (reading R-H1): -3 u0 + 4 u1 - u2 = 4 (u1 - u0) - (u2 - u0)
    if (c == 0) return (4.0 * (c0[s] - c0[0]) - (c0[2 * s] - c0[0])) * ih2;
    if (c == n - 1) return -(4.0 * (c0[-s] - c0[0]) - (c0[-2 * s] - c0[0])) * ih2;
    return (c0[s] - c0[-s]) * ih2;
  };
  auto point = [&](int i, int j, int k) {   // padded coordinates
    const long off = (long)k * L.plane + (long)j * L.pitch + i;
    const double* c0 = u + off;
    const double x = ((i - g) - 0.5 * (L.nx - 1)) * h, y = ((j - g) - 0.5 * (L.ny - 1)) * h,
                 z = ((k - g) - 0.5 * (L.nz - 1)) * h;
    const double r = sqrt(x * x + y * y + z * z);
    const double nd = (x * d1(c0, 1, i, tx) + y * d1(c0, L.pitch, j, L.tot_y) + z * d1(c0, L.plane, k, L.tot_z)) / r;
    const double kk = -(nd + (c0[0] - uinf) / r);
    stage_emit(st, (long)v * L.vstride + (L.xo - g) + off, kk);
  };
  if (task < rowsAB) {
    int j, k;
    if (task < rowsA) {
      const int kk = task / L.tot_y;
      j = task - kk * L.tot_y;
      k = kk < g ? kk : kk + L.nz;
    } else {
      const int r = task - rowsA, kk = r / (2 * g), jj = r - kk * 2 * g;
      k = kk + g;
      j = jj < g ? jj : jj + L.ny;
    }
    for (int i = lane; i < tx; i += 32) point(i, j, k);
  } else {
    const int lpr = 1 << lpr_shift;
    const int row = (task - rowsAB) * (32 >> lpr_shift) + (lane >> lpr_shift);
    if (row < L.nz * L.ny) {
      const int kk = row / L.ny, jj = row - kk * L.ny;
      for (int ii = lane & (lpr - 1); ii < 2 * g; ii += lpr) point(ii < g ? ii : ii + L.nx, jj + g, kk + g);
    }
  }
}

// launch geometry: one warp per task, 8 tasks per 256-thread block, grid.y = variables
struct RadGeom { long rowsA, rowsAB, tasks; int lpr_shift; };
inline RadGeom rad_geom(const Layout& L) {
  const int g = L.g;
  RadGeom G;
  G.rowsA = 2L * g * L.tot_y;
  G.rowsAB = G.rowsA + 2L * g * L.nz;
  const long rowsC = (long)L.nz * L.ny;
  G.lpr_shift = 0;
  while ((1 << G.lpr_shift) < 2 * g && G.lpr_shift < 5) ++G.lpr_shift;
  G.tasks = G.rowsAB + (rowsC + (32 >> G.lpr_shift) - 1) / (32 >> G.lpr_shift);
  return G;
}

#ifndef CHM_EMULATE
cudaError_t launch_radiative(const Layout& L, const Stage& st, double h, unsigned uinf_mask, cudaStream_t s) {
  if (L.g < 2) return cudaErrorInvalidValue;   // the one-sided formula reads two points inward
  const RadGeom G = rad_geom(L);
  if (G.tasks > 0x7fffffffL - 8 || (long)L.nz * L.ny > 0x7fffffffL) return cudaErrorInvalidValue;
  dim3 grid((unsigned)((G.tasks + 7) / 8), L.nvars);
  radiative_kernel<<<grid, 256, 0, s>>>(L, st, h, uinf_mask, (int)G.rowsA, (int)G.rowsAB, G.lpr_shift);
  return cudaGetLastError();
}
#endif   // CHM_EMULATE

// Per variable v: out[2 v] = max |a - b|, out[2 v + 1] = max |b| over the variable's whole padded array, as the bit
// patterns of non-negative doubles (which order like unsigned integers, so atomicMax works); a NaN on either side
// counts as an infinite difference.  The runtime sweep's guard: a candidate variant must reproduce the reference
// variant's result in the norm of reading S11.
__global__ void __launch_bounds__(256) maxdiff_kernel(const double* __restrict__ a, const double* __restrict__ b,
                                                      long vstride, unsigned long long* out) {
  const long base = (long)blockIdx.y * vstride;
  double d = 0.0, m = 0.0;
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < vstride; i += (long)gridDim.x * blockDim.x) {
    const double x = a[base + i], y = b[base + i];
    double e = fabs(x - y);
    if (!(e == e)) e = __longlong_as_double(0x7ff0000000000000LL);
    d = fmax(d, e);
    m = fmax(m, fabs(y));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    d = fmax(d, __shfl_xor_sync(0xffffffffu, d, o));
    m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  }
  if ((threadIdx.x & 31) == 0) {
    atomicMax(out + 2 * blockIdx.y, (unsigned long long)__double_as_longlong(d));
    atomicMax(out + 2 * blockIdx.y + 1, (unsigned long long)__double_as_longlong(m));
  }
}

#ifndef CHM_EMULATE
cudaError_t launch_maxdiff(const double* a, const double* b, long vstride, int nvars, unsigned long long* out,
                           cudaStream_t s) {
  long blocks = (vstride + 256L * 8 - 1) / (256L * 8);
  if (blocks > 1024) blocks = 1024;
  if (blocks < 1) blocks = 1;
  maxdiff_kernel<<<dim3((unsigned)blocks, nvars), 256, 0, s>>>(a, b, vstride, out);
  return cudaGetLastError();
}
#endif   // CHM_EMULATE

}  // namespace chm
