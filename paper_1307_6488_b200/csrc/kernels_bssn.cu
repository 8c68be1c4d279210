// kernels_bssn.cu -- BSSN right-hand side, split variant: one kernel writes the derivative
// arrays to global memory, a second evaluates the RHS from them (+ RK4 stage update).  The fused kernel is in
// kernels_bssn_tma.cu.
#include "bssn_point.cuh"
#include "stencils.cuh"

namespace chm {

// derivative-array slots of the split variant: 45 first, 66 second, 25 advection+dissipation
__device__ __forceinline__ constexpr int slot_d1(int v, int a) {
  int base = v == V_CHI ? 0 : v < V_K ? 3 + 3 * (v - V_GT) : v == V_K ? 21 : v < V_ALPHA ? 24 + 3 * (v - V_GAM)
             : v == V_ALPHA ? 33 : 36 + 3 * (v - V_BETA);
  return base + a;
}
__device__ __forceinline__ constexpr int slot_d2(int v, int a, int b) {
  int base = v == V_CHI ? 0 : v < V_K ? 6 + 6 * (v - V_GT) : v == V_ALPHA ? 42 : 48 + 6 * (v - V_BETA);
  return 45 + base + sym(a, b);
}
__device__ __forceinline__ constexpr int slot_ad(int v) { return 111 + v; }

// reads the precomputed derivative arrays (packed interior layout, stride n per array)
struct FromArrays {
  const double* __restrict__ fields;   // at the point, padded layout
  long sv;
  const double* __restrict__ dv;       // at the point, packed layout
  long n;
  __device__ __forceinline__ double f(int v) const { return __ldg(fields + v * sv); }
  __device__ __forceinline__ double d1(int v, int a) const { return __ldg(dv + slot_d1(v, a) * n); }
  __device__ __forceinline__ double d2(int v, int a, int b) const { return __ldg(dv + slot_d2(v, a, b) * n); }
  __device__ __forceinline__ double ad(int v) const { return __ldg(dv + slot_ad(v) * n); }
};

__host__ __device__ inline long packed_stride(const Layout& L) {
  long n = (long)L.nx * L.ny * L.nz;
  return (n + 15) / 16 * 16;
}

template <int TX, int TY, int TZ, int ORDER>
__global__ void __launch_bounds__(TX* TY) bssn_derivs_kernel(Layout L, Coef C, const double* __restrict__ in,
                                                            double* __restrict__ derivs) {
  const int i = blockIdx.x * TX + threadIdx.x, j = blockIdx.y * TY + threadIdx.y;
  if (i >= L.nx || j >= L.ny) return;
  const int k0 = blockIdx.z * TZ;
  const long n = packed_stride(L);
#pragma unroll 1
  for (int kk = 0; kk < TZ; ++kk) {
    const int k = k0 + kk;
    if (k >= L.nz) break;
    const long q = (long)(k + L.g) * L.plane + (long)(j + L.g) * L.pitch + (i + L.xo);
    double* o = derivs + ((long)k * L.ny + j) * L.nx + i;
    OnTheFly<GlobalPoint, ORDER> D{{in + q, L.pitch, L.plane, L.vstride}, C, {0, 0, 0}};
    D.beta[0] = D.f(V_BETA); D.beta[1] = D.f(V_BETA + 1); D.beta[2] = D.f(V_BETA + 2);
#pragma unroll
    for (int v = 0; v < 25; ++v) {
      const bool has_d1 = v <= V_K || (v >= V_GAM && v < V_B);
      const bool has_d2 = v <= V_GT + 5 || (v >= V_ALPHA && v < V_B);
      if (has_d1) {
#pragma unroll
        for (int a = 0; a < 3; ++a) o[slot_d1(v, a) * n] = D.d1(v, a);
      }
      if (has_d2) {
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
          for (int b = a; b < 3; ++b) o[slot_d2(v, a, b) * n] = D.d2(v, a, b);
      }
      o[slot_ad(v) * n] = D.ad(v);
    }
  }
}

template <int TX, int TY, int TZ>
__global__ void __launch_bounds__(TX* TY) bssn_from_derivs_kernel(Layout L, Coef C, const double* __restrict__ derivs,
                                                                 Stage st) {
  const int i = blockIdx.x * TX + threadIdx.x, j = blockIdx.y * TY + threadIdx.y;
  if (i >= L.nx || j >= L.ny) return;
  const int k0 = blockIdx.z * TZ;
  const long n = packed_stride(L);
#pragma unroll 1
  for (int kk = 0; kk < TZ; ++kk) {
    const int k = k0 + kk;
    if (k >= L.nz) break;
    const long q = (long)(k + L.g) * L.plane + (long)(j + L.g) * L.pitch + (i + L.xo);
    FromArrays D{st.in + q, L.vstride, derivs + ((long)k * L.ny + j) * L.nx + i, n};
    bssn_point(D, C, [&](int v, double r) { stage_emit(st, q + v * L.vstride, r); });
  }
}

// which: 1 derivs, 2 from_derivs
#ifndef CHM_EMULATE
template <int TX, int TY, int TZ>
static cudaError_t bssn_go(int which, const Layout& L, const Coef& C, const Stage* st, const double* in,
                           double* derivs, cudaStream_t s, cudaFuncAttributes* a) {
  dim3 grid((L.nx + TX - 1) / TX, (L.ny + TY - 1) / TY, (L.nz + TZ - 1) / TZ), block(TX, TY);
  if (which == 1) {
    auto kern = bssn_derivs_kernel<TX, TY, TZ, 4>;
    if (a) return cudaFuncGetAttributes(a, kern);
    kern<<<grid, block, 0, s>>>(L, C, in, derivs);
  } else if (which == 3) {   // 8th-order derivatives (the paper's configuration; split variant only)
    auto kern = bssn_derivs_kernel<TX, TY, TZ, 8>;
    if (a) return cudaFuncGetAttributes(a, kern);
    kern<<<grid, block, 0, s>>>(L, C, in, derivs);
  } else {
    auto kern = bssn_from_derivs_kernel<TX, TY, TZ>;
    if (a) return cudaFuncGetAttributes(a, kern);
    kern<<<grid, block, 0, s>>>(L, C, derivs, *st);
  }
  return cudaGetLastError();
}
#endif   // CHM_EMULATE

#ifndef CHM_EMULATE
static cudaError_t bssn_dispatch(int which, int tile, const Layout& L, const Coef& C, const Stage* st,
                                 const double* in, double* derivs, cudaStream_t s, cudaFuncAttributes* a) {
  switch (tile) {
    case 0: return bssn_go<32, 4, 8>(which, L, C, st, in, derivs, s, a);
    case 1: return bssn_go<32, 8, 8>(which, L, C, st, in, derivs, s, a);
    case 2: return bssn_go<64, 2, 8>(which, L, C, st, in, derivs, s, a);
    case 3: return bssn_go<64, 4, 8>(which, L, C, st, in, derivs, s, a);
    case 4: return bssn_go<128, 2, 8>(which, L, C, st, in, derivs, s, a);
    case 5: return bssn_go<16, 16, 8>(which, L, C, st, in, derivs, s, a);
  }
  return cudaErrorInvalidValue;
}
#endif   // CHM_EMULATE

#ifndef CHM_EMULATE
cudaError_t launch_bssn_derivs(const Layout& L, const Coef& C, int order, int tile, const double* in, double* derivs,
                               cudaStream_t s) {
  return bssn_dispatch(order == 8 ? 3 : 1, tile, L, C, nullptr, in, derivs, s, nullptr);
}
#endif   // CHM_EMULATE
#ifndef CHM_EMULATE
cudaError_t launch_bssn_from_derivs(const Layout& L, const Coef& C, int tile, const double* derivs, const Stage& st,
                                    cudaStream_t s) {
  return bssn_dispatch(2, tile, L, C, &st, nullptr, const_cast<double*>(derivs), s, nullptr);
}
#endif   // CHM_EMULATE
#ifndef CHM_EMULATE
cudaError_t kernel_info_bssn_split(int which, int tile, cudaFuncAttributes* a) {
  Layout L{}; Coef C{};
  return bssn_dispatch(which, tile, L, C, nullptr, nullptr, nullptr, 0, a);
}
#endif   // CHM_EMULATE

}  // namespace chm
