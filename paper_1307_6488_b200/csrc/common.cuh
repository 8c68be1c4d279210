// common.cuh -- shared declarations of libchemora's translation units (host + device).
// Part of the CUDA product path; shares nothing with oracle/.
#pragma once
#ifndef CHM_EMULATE   // tests/native/cta_emu.hpp stands in for the CUDA headers when the kernel source is compiled for the host
#include <cuda_runtime.h>
#endif
#include <stdint.h>

// inline helper usable from device code and from host-side probes of the same arithmetic (tests/native/)
#define CHM_HD __host__ __device__ __forceinline__

namespace chm {

#define CHM_ST(p, v) __stcs(p, v)   // streaming store: written once, re-read only by a later launch
// Device-side view of the padded SoA layout (include/chemora.h "Conventions").
struct Layout {
  int nx, ny, nz, g;     // interior dims, ghost width
  int xo;                // x index of interior point 0 inside a row: g, or g+1 when that makes (xo - 3) even,
                         // so that the fused BSSN kernel's TMA halo boxes start on a 16-byte boundary
  int nvars;
  long pitch;            // doubles per row, multiple of 16 (128-byte rows)
  long plane;            // pitch * tot_y
  long vstride;          // plane * tot_z
  int tot_y, tot_z;
  int col_rows;          // fused BSSN kernel: y-extent (grid rows) of a tile-traversal column (L2 reuse of halos)
  unsigned* err;         // the handle's device error word (0 = fine): bounded mbarrier waits record a code here
};

// Stencil scale factors and model parameters, precomputed on the host once per launch.
struct Coef {
  double inv_h;          // 1/h
  double inv_h2;         // 1/h^2
  double ko;             // eps_diss / (64 h); 0 => dissipation off (no +-3 reads)
  double kq[5];          // 8th-order BSSN kernels: dissipation = sum_k kq[k-1] s_k, s_k = (u[+k]-u0) + (u[-k]-u0);
                         // KO order 5: ko * (15, -6, 1, 0, 0); order 9 (reading S6b): eps/(1024 h) * (210, -120, 45, -10, 1)
  double eta;            // Gamma-driver damping
  double sgc;            // shift_gamma_coeff (3/4)
};

// Runge-Kutta epilogue fused into the RHS kernels (reading S9).
//   MODE_RHS   : out = k
//   MODE_FIRST : S = k          ; Y = U + a k        (U == the input state)
//   MODE_MID   : S = S + 2 k    ; Y = U + a k
//   MODE_LAST  : U = U + a (S + k)                   (a = dt/6)
// and of the Shu-Osher RK3 (reading S9b):
//   MODE_SSP   : out = ca U + cb (in + a k)          (a = dt; out may be U itself: each point is read, then written)
enum { MODE_RHS = 0, MODE_FIRST = 1, MODE_MID = 2, MODE_LAST = 3, MODE_SSP = 4 };

struct Stage {
  const double* in;      // state the RHS is evaluated on (ghosts filled)
  double* U;             // MODE_LAST: read+written.  MODE_FIRST/MID: read only.  MODE_RHS: unused
  double* S;             // accumulator
  double* out;           // MODE_RHS: rhs ; MODE_FIRST/MID: next stage state Y
  double a;              // dt/2, dt/2, dt, dt/6
  int mode;
  double ca, cb;         // MODE_SSP only
};

// a U + b (Y + dt k), every product and sum rounded once
__device__ __forceinline__ double ssp_combine(const Stage& st, double u, double y, double k) {
  return __dadd_rn(__dmul_rn(st.ca, u), __dmul_rn(st.cb, __dadd_rn(y, __dmul_rn(st.a, k))));
}

// The stage combination, one rounding per operation and no FMA contraction, so that it is
// bit-identical to the association written in reading S9 for a given k.
__device__ __forceinline__ void stage_emit(const Stage& st, long q, double k) {
  if (st.mode == MODE_RHS) {
    st.out[q] = k;
  } else if (st.mode == MODE_FIRST) {
    st.S[q] = k;
    st.out[q] = __dadd_rn(st.in[q], __dmul_rn(st.a, k));
  } else if (st.mode == MODE_MID) {
    st.S[q] = __dadd_rn(st.S[q], __dmul_rn(2.0, k));
    st.out[q] = __dadd_rn(st.U[q], __dmul_rn(st.a, k));
  } else if (st.mode == MODE_LAST) {
    st.U[q] = __dadd_rn(st.U[q], __dmul_rn(st.a, __dadd_rn(st.S[q], k)));
  } else {
    st.out[q] = ssp_combine(st, st.U[q], st.in[q], k);
  }
}

// Split form of stage_emit: fetch the operands early (stage_prefetch), combine and store later.
struct StagePre { double u, s; };
__device__ __forceinline__ void stage_prefetch(const Stage& st, long q, StagePre& r) {
  if (st.mode == MODE_FIRST) r.u = st.in[q];
  else if (st.mode == MODE_SSP) { r.u = st.U[q]; r.s = st.in[q]; }
  else if (st.mode != MODE_RHS) { r.u = st.U[q]; r.s = st.S[q]; }
}
__device__ __forceinline__ void stage_emit(const Stage& st, long q, double k, const StagePre& pr) {
  if (st.mode == MODE_RHS) {
    CHM_ST(&st.out[q], k);
  } else if (st.mode == MODE_FIRST) {
    CHM_ST(&st.S[q], k);
    CHM_ST(&st.out[q], __dadd_rn(pr.u, __dmul_rn(st.a, k)));
  } else if (st.mode == MODE_MID) {
    CHM_ST(&st.S[q], __dadd_rn(pr.s, __dmul_rn(2.0, k)));
    CHM_ST(&st.out[q], __dadd_rn(pr.u, __dmul_rn(st.a, k)));
  } else if (st.mode == MODE_LAST) {
    CHM_ST(&st.U[q], __dadd_rn(pr.u, __dmul_rn(st.a, __dadd_rn(pr.s, k))));
  } else {
    CHM_ST(&st.out[q], ssp_combine(st, pr.u, pr.s, k));
  }
}

// Same with the mode as a compile-time constant (no branches in the epilogue of the fused BSSN kernel):
// values first, stores under one predicate (no divergent region around the arithmetic)
template <int MODE>
__device__ __forceinline__ void stage_emit_t(const Stage& st, long q, double k, const StagePre& pr, bool valid) {
  if (MODE == MODE_RHS) {
    if (valid) CHM_ST(&st.out[q], k);
  } else if (MODE == MODE_FIRST) {
    const double y = __dadd_rn(pr.u, __dmul_rn(st.a, k));
    if (valid) { CHM_ST(&st.S[q], k); CHM_ST(&st.out[q], y); }
  } else if (MODE == MODE_MID) {
    const double s2 = __dadd_rn(pr.s, __dmul_rn(2.0, k)), y = __dadd_rn(pr.u, __dmul_rn(st.a, k));
    if (valid) { CHM_ST(&st.S[q], s2); CHM_ST(&st.out[q], y); }
  } else if (MODE == MODE_LAST) {
    const double u = __dadd_rn(pr.u, __dmul_rn(st.a, __dadd_rn(pr.s, k)));
    if (valid) CHM_ST(&st.U[q], u);
  } else {
    const double y = ssp_combine(st, pr.u, pr.s, k);   // pr.u = U, pr.s = the evaluated state at the point
    if (valid) CHM_ST(&st.out[q], y);
  }
}

// Tile shapes of the variant sweep.  Fused kernel: 3-D tile, one point per thread.  Split kernels and the wave
// kernel: x,y = thread block, z = planes marched per block.
struct TileShape { int tx, ty, tz; };
// fused BSSN tile ids 0..6 (8th order: id 0 only); id 5: 16x4x4 with the interleaved section layout; id 6: the same
// with a full variable's own right-hand side emitted before the plane barrier of its mixed derivatives; id 7: id 6
// with a six-slot box ring
constexpr int kNumFused = 8;
static const TileShape kTilesFused[kNumFused] = {{16, 4, 4}, {16, 8, 2}, {8, 4, 8}, {16, 2, 8}, {16, 4, 2}, {16, 4, 4}, {16, 4, 4}, {16, 4, 4}};
// wave system ids 6..8: the TMA plane-ring kernel (x, y = thread block, z = planes per work item)
static const TileShape kTilesWaveTma[3] = {{32, 16, 32}, {32, 16, 64}, {64, 8, 32}};
// Sample-1 system ids 6..8: the same plane-ring kernel with five variables (smaller tiles: the ring holds 5 boxes a plane)
static const TileShape kTilesWave1Tma[3] = {{16, 8, 64}, {16, 16, 64}, {32, 8, 64}};
static const TileShape kTilesMarch[6] = {{32, 4, 8}, {32, 8, 8}, {64, 2, 8}, {64, 4, 8}, {128, 2, 8}, {16, 16, 8}};

// launchers implemented in the kernel translation units; each returns the cudaError_t of the launch
// Source of the ghost z-planes when the block is linked to z-neighbours (multi-block interface): the same state
// buffer of the lower / upper neighbour block (same nx, ny, ghost width and row layout; its own nz).
struct FillLink {
  const double* lo;  long lo_vstride;  int lo_nz;    // lower neighbour: its top g interior planes
  const double* hi;  long hi_vstride;                // upper neighbour: its bottom g interior planes
};
// link: where the ghost z-planes come from (nullptr: the block's own periodic images)
cudaError_t launch_fill_ghosts(const Layout& L, double* state, cudaStream_t s, const FillLink* link = nullptr);
// radiative outer boundary (reading S16): RHS + stage epilogue at the boundary points (the g ghost layers)
cudaError_t launch_radiative(const Layout& L, const Stage& st, double h, unsigned uinf_mask, cudaStream_t s);
cudaError_t launch_maxdiff(const double* a, const double* b, long vstride, int nvars, unsigned long long* out, cudaStream_t s);
cudaError_t launch_energy(const Layout& L, const double* state, double* eps_out, double* sum, cudaStream_t s);
cudaError_t launch_enforce(const Layout& L, double* state, cudaStream_t s);
cudaError_t launch_pack(const Layout& L, const double* packed, double* state, bool to_state, cudaStream_t s);
cudaError_t launch_wave(const Layout& L, const Coef& C, int order, int tile, const Stage& st, cudaStream_t s);
cudaError_t launch_wave_tma(const Layout& L, const Coef& C, int order, int which, const Stage& st, cudaStream_t s);
cudaError_t kernel_info_wave_tma(int order, int which, cudaFuncAttributes* a);
bool wave_tma_ok(const Layout& L, int order, bool ko);
cudaError_t launch_wave1_tma(const Layout& L, const Coef& C, int order, int which, const Stage& st, cudaStream_t s);
cudaError_t kernel_info_wave1_tma(int order, int which, cudaFuncAttributes* a);
bool wave1_tma_ok(const Layout& L, int order, bool ko, int which);
cudaError_t launch_wave1(const Layout& L, const Coef& C, int order, int tile, const Stage& st, cudaStream_t s);
cudaError_t kernel_info_wave1(int order, int tile, cudaFuncAttributes* a);
cudaError_t launch_bssn_fused(const Layout& L, const Coef& C, int order, int tile, const Stage& st, cudaStream_t s);
cudaError_t launch_bssn_fill(const Layout& L, const Coef& C, int tile, const Stage& st, cudaStream_t s);   // fill-only mode
cudaError_t launch_bssn_derivs(const Layout& L, const Coef& C, int order, int tile, const double* in, double* derivs,
                               cudaStream_t s);
cudaError_t launch_bssn_from_derivs(const Layout& L, const Coef& C, int tile, const double* derivs,
                                    const Stage& st, cudaStream_t s);
cudaError_t kernel_info_wave(int order, int tile, cudaFuncAttributes* a);
cudaError_t kernel_info_bssn_fused(int order, int tile, cudaFuncAttributes* a);
cudaError_t kernel_info_bssn_split(int which, int tile, cudaFuncAttributes* a);
cudaError_t launch_dfma_peak(int blocks, int threads, int iters, double* sink, cudaStream_t s);

// number of derivative arrays of the split variant: 45 first + 66 second + 25 advection+dissipation
constexpr int kNumDerivArrays = 136;

}  // namespace chm
