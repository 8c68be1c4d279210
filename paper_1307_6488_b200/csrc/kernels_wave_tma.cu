// kernels_wave_tma.cu -- the (phi, pi) wave-system RHS + RK stage (reading S1) as a z-marching kernel, sm_100a.
// HBM-bound work (2 variables, 68 B per point and launch): persistent CTAs; each work item is an (x, y) tile of
// TX x TY points and a chunk of ZC planes.  The (TX + 2R) x (TY + 2R) box of one z-plane of BOTH variables is one
// TMA load (cp.async.bulk.tensor.4d, box 4th extent 2) into a ring of NP plane slots, issued PF planes ahead, so no
// thread ever waits for global-memory latency; all 44 stencil reads of a point come from shared memory with
// compile-time x/y offsets and a per-step table of the 2R+1 plane bases.  The RK operands (U, S) of the next plane
// are prefetched into registers while the current plane is evaluated.  Slots are released warp by warp (mbarrier
// whose returned state tells the last arriver, see bssn_tma.cuh); the last warp out issues the slot's next load.
#include "bssn_tma.cuh"
#include <cstdio>

#include "stencils.cuh"
#include "tma_check.cuh"

namespace chm {

namespace wv {

// NV = 2: the (phi, pi) system; NV = 5: the paper's Sample-1 system (u, rho, v_i), reading S1b
template <int ORDER, bool KO, int TX, int TY, int NV = 2>
struct Cfg {
  static constexpr int R0 = ORDER / 2, R = (KO && R0 < 3) ? 3 : R0;
  static constexpr int ROW = TX + 2 * R, COLS = TY + 2 * R;
  static constexpr int PB = ROW * COLS;                       // doubles per variable in one plane box
  static constexpr int SLOT = (NV * PB + 15) / 16 * 16;       // all variables, 128-byte multiple
  static constexpr uint32_t BYTES = (uint32_t)NV * PB * 8u;
  static constexpr size_t smem_of(int pf) { return (size_t)(2 * R + 1 + pf) * SLOT * 8 + 2 * (2 * R + 1 + pf) * 8 + 128; }
  // planes in flight ahead of the one being evaluated: as many as fit (five variables leave room for fewer)
  static constexpr int PF0 = TX * TY == 512 && TX == 32 ? 5 : 3;
  static constexpr int PF = NV == 2 ? PF0 : (smem_of(3) <= 227 * 1024 ? 3 : (smem_of(2) <= 227 * 1024 ? 2 : 1));
  static constexpr int NP = 2 * R + 1 + PF;                   // ring slots
  static constexpr int THREADS = TX * TY, NW = THREADS / 32;
  static constexpr size_t SMEM = smem_of(PF);
  static constexpr bool FITS = SMEM <= 227 * 1024;
  static_assert(TX % 2 == 0, "TMA rows start on 16-byte boundaries");
};

// stencil accessor: x/y offsets inside the centre plane, z offsets through the table of plane bases
template <int R>
struct RingPoint {
  const double* const* zp;   // zp[R + dk]: this thread's point in the phi box of plane k + dk (pi box at + pb)
  int row, pb;
  __device__ __forceinline__ double at(int v, int di, int dj, int dk) const { return zp[R + dk][v * pb + dj * row + di]; }
  __device__ __forceinline__ double ax(int v, int a, int m) const {
    return a == 0 ? at(v, m, 0, 0) : (a == 1 ? at(v, 0, m, 0) : at(v, 0, 0, m));
  }
};

}  // namespace wv

template <int ORDER, bool KO, int TX, int TY, int ZC, int NV>
__global__ void __launch_bounds__(TX* TY, 1)
wave_tma_kernel(const __grid_constant__ CUtensorMap tm, Layout L, Coef C, Stage st, int ntx, int nty, int ntz) {
  using K = wv::Cfg<ORDER, KO, TX, TY, NV>;
  constexpr int R = K::R, ROW = K::ROW, PB = K::PB, SLOT = K::SLOT, NP = K::NP, PF = K::PF;
  CHM_DYNAMIC_SMEM(smem_raw);
  double* sm = reinterpret_cast<double*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(sm + NP * SLOT);   // [NP] plane arrived
  uint64_t* empty = full + NP;                                     // [NP] plane released by all warps
  const int tid = threadIdx.y * TX + threadIdx.x, lane = tid & 31;
  const int poff = (threadIdx.y + R) * ROW + threadIdx.x + R;     // this thread's point inside a plane box
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NP; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], K::NW); }
    fence_mbar_init();
  }
  __syncthreads();

  const int nitems = ntx * nty * ntz;
  int n = 0;    // planes this CTA has loaded so far = load sequence number (slot n % NP, parity (n / NP) & 1)
  for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
    const int bz = item / (ntx * nty), r2 = item - bz * ntx * nty, by = r2 / ntx, bx = r2 - by * ntx;
    const int i0 = bx * TX, j0 = by * TY, k0 = bz * ZC, k1 = min(k0 + ZC, L.nz);
    const int x0 = i0 + L.xo - R, y0 = j0 + L.g - R;               // box origin, padded coordinates
    const int nplanes = (k1 - k0) + 2 * R;                          // planes k0-R .. k1-1+R
    const int nbase = n;
    // plane number p (0-based inside the item) is padded z = k0 + g - R + p; load sequence number nbase + p
    auto issue = [&](int p) {
      const int m = nbase + p;
      const int slot = m % NP;
      mbar_expect_tx(&full[slot], K::BYTES);
      tma_load_4d(sm + slot * SLOT, &tm, &full[slot], x0, y0, k0 + L.g - R + p, 0);
    };
    // The ring is empty at an item boundary only logically: the previous item's last planes may still be read by
    // slower warps, so a slot is refilled by the last warp that releases it (below); the first NP loads of an item
    // are issued by thread 0 once every slot it needs has been released (it waits on `empty` for slots used before).
    if (tid == 0) {
      const int first = nplanes < NP ? nplanes : NP;               // fill the whole ring
      for (int p = 0; p < first; ++p) {
        const int m = nbase + p;
        if (m >= NP) mbar_wait(&empty[m % NP], (uint32_t)(((m / NP) - 1) & 1), L.err, 0x20001u);
        issue(p);
      }
    }
    const int i = i0 + threadIdx.x, j = j0 + threadIdx.y;
    const bool inxy = i < L.nx && j < L.ny;
    long q = (long)(k0 + L.g) * L.plane + (long)((inxy ? j : 0) + L.g) * L.pitch + ((inxy ? i : 0) + L.xo);
    // RK operands (U, S) of planes k, k+1, k+2 travel in registers: loaded two planes before they are used
    StagePre pr[NV], n1[NV], n2[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) stage_prefetch(st, q + v * L.vstride, pr[v]);
    if (k0 + 1 < k1) {
#pragma unroll
      for (int v = 0; v < NV; ++v) stage_prefetch(st, q + L.plane + v * L.vstride, n1[v]);
    }
    for (int k = k0; k < k1; ++k) {
      const int pc = (k - k0) + R;                                  // centre plane number inside the item
      // wait for the newest plane this step needs (older ones were waited for in earlier steps / below)
      if (k == k0) {
        for (int p = 0; p <= pc + R; ++p) { const int m = nbase + p; mbar_wait(&full[m % NP], (uint32_t)((m / NP) & 1), L.err, 0x20002u); }
      } else {
        const int m = nbase + pc + R;
        mbar_wait(&full[m % NP], (uint32_t)((m / NP) & 1), L.err, 0x20003u);
      }
      const double* zp[2 * R + 1];
#pragma unroll
      for (int d = 0; d <= 2 * R; ++d) zp[d] = sm + ((nbase + pc - R + d) % NP) * SLOT + poff;
      if (k + 2 < k1) {
#pragma unroll
        for (int v = 0; v < NV; ++v) stage_prefetch(st, q + 2 * L.plane + v * L.vstride, n2[v]);
      }
      wv::RingPoint<R> P{zp, ROW, PB};
      double r[NV];
      if constexpr (NV == 2) {
        double lap;
        if (ORDER == 4) lap = (d2_o4(P, 0, 0, C.inv_h2) + d2_o4(P, 0, 1, C.inv_h2)) + d2_o4(P, 0, 2, C.inv_h2);
        else lap = (d2_o8(P, 0, 0, C.inv_h2) + d2_o8(P, 0, 1, C.inv_h2)) + d2_o8(P, 0, 2, C.inv_h2);
        r[0] = P.at(1, 0, 0, 0);
        r[1] = lap;
      } else {   // D_t u = rho ; D_t rho = d_i v_i ; D_t v_i = d_i rho
        auto d1 = [&](int v, int a) { return ORDER == 4 ? d1_o4(P, v, a, C.inv_h) : d1_o8(P, v, a, C.inv_h); };
        r[0] = P.at(1, 0, 0, 0);
        r[1] = (d1(2, 0) + d1(3, 1)) + d1(4, 2);
#pragma unroll
        for (int a = 0; a < 3; ++a) r[2 + a] = d1(1, a);
      }
      if (KO) {
#pragma unroll
        for (int v = 0; v < NV; ++v) r[v] += ko5(P, v, C.ko);
      }
      // the oldest plane (k - R) is not needed after this step: release it; the last warp out refills its slot
      __syncwarp();
      if (lane == 0) {
        const int mo = nbase + pc - R;
        if (mbar_arrive_is_last(&empty[mo % NP])) {
          const int pnew = pc - R + NP;                             // plane that reuses this slot
          if (pnew < nplanes) issue(pnew);
        }
      }
      if (inxy) {
#pragma unroll
        for (int v = 0; v < NV; ++v) stage_emit(st, q + v * L.vstride, r[v], pr[v]);
      }
#pragma unroll
      for (int v = 0; v < NV; ++v) { pr[v] = n1[v]; n1[v] = n2[v]; }
      q += L.plane;
    }
    // release the 2R planes of the item that were never "oldest" (its last planes), so the next item can reuse them
    __syncwarp();
    if (lane == 0)
      for (int p = (k1 - k0); p < nplanes; ++p) mbar_arrive_is_last(&empty[(nbase + p) % NP]);
    n = nbase + nplanes;
  }
}

// ---- launch plans and layout test (pure host code: also compiled for the CTA emulator) ----------------------------
// what one launch of wave_tma_kernel issues, for the validator: one plane box per ring slot
template <int ORDER, bool KO, int TX, int TY, int NV>
static TmaPlan wv_plan(int xo) {
  using K = wv::Cfg<ORDER, KO, TX, TY, NV>;
  char name[80];
  snprintf(name, sizeof name, "wave_tma_kernel<order %d,ko %d,%dx%d,%d vars>", ORDER, (int)KO, TX, TY, NV);
  TmaPlan p;
  p.kernel = name;
  p.smem_bytes = K::SMEM;
  p.threads = K::THREADS;
  p.barrier_off = (size_t)K::NP * K::SLOT * 8;
  p.n_barriers = 2 * K::NP;
  for (int slot = 0; slot < K::NP; ++slot) {
    p.expect.push_back(K::BYTES);
    p.loads.push_back({"plane box", (size_t)slot * K::SLOT * 8, {(uint32_t)K::ROW, (uint32_t)K::COLS, 1, (uint32_t)NV}, slot, (xo - K::R) & 1});
  }
  return p;
}

// true when the TMA form can serve this layout: plane-box rows must start on 16-byte boundaries
bool wave_tma_ok(const Layout& L, int order, bool ko) {
  const int r0 = order / 2, r = (ko && r0 < 3) ? 3 : r0;
  return ((L.xo - r) % 2) == 0 && L.g >= r;
}

template <int ORDER, bool KO>
static void wv_plans_of(std::vector<TmaPlan>& out, int xo) {
  out.push_back(wv_plan<ORDER, KO, 32, 16, 2>(xo));
  out.push_back(wv_plan<ORDER, KO, 64, 8, 2>(xo));
  if (wv::Cfg<ORDER, KO, 16, 8, 5>::FITS) out.push_back(wv_plan<ORDER, KO, 16, 8, 5>(xo));
  if (wv::Cfg<ORDER, KO, 16, 16, 5>::FITS) out.push_back(wv_plan<ORDER, KO, 16, 16, 5>(xo));
  if (wv::Cfg<ORDER, KO, 32, 8, 5>::FITS) out.push_back(wv_plan<ORDER, KO, 32, 8, 5>(xo));
}
// every instance, on every ghost width wave_tma_ok admits (xo = g for the wave systems)
void plans_wave_tma(std::vector<TmaPlan>& out) {
  for (int g = 2; g <= 6; ++g) {
    Layout L{};
    L.xo = g; L.g = g;
    if (wave_tma_ok(L, 4, false)) wv_plans_of<4, false>(out, g);
    if (wave_tma_ok(L, 4, true)) wv_plans_of<4, true>(out, g);
    if (wave_tma_ok(L, 8, false)) wv_plans_of<8, false>(out, g);
    if (wave_tma_ok(L, 8, true)) wv_plans_of<8, true>(out, g);
  }
}

#ifndef CHM_EMULATE
// ---- host side ------------------------------------------------------------------------------------------------
typedef CUresult (*WvEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static WvEncodeFn wv_encode_fn() {
  static WvEncodeFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (WvEncodeFn)p;
  }
  return fn;
}

template <int ORDER, bool KO, int TX, int TY, int ZC, int NV = 2>
static cudaError_t wv_go(const Layout& L, const Coef& C, const Stage* st, cudaStream_t s, cudaFuncAttributes* a) {
  using K = wv::Cfg<ORDER, KO, TX, TY, NV>;
  if constexpr (!K::FITS) return cudaErrorInvalidConfiguration;   // ring does not fit: the caller falls back
  else {
  auto kern = wave_tma_kernel<ORDER, KO, TX, TY, ZC, NV>;
  if (a) return cudaFuncGetAttributes(a, kern);
  if (L.nvars != NV || !launch_allowed(wv_plan<ORDER, KO, TX, TY, NV>(L.xo), L, st->in, L.xo - K::R, K::R)) return cudaErrorInvalidValue;
  WvEncodeFn enc = wv_encode_fn();
  if (!enc) return cudaErrorNotSupported;
  CUtensorMap tm;
  cuuint64_t dims[4] = {(cuuint64_t)L.pitch, (cuuint64_t)L.tot_y, (cuuint64_t)L.tot_z, (cuuint64_t)L.nvars};
  cuuint64_t strides[3] = {(cuuint64_t)L.pitch * 8, (cuuint64_t)L.plane * 8, (cuuint64_t)L.vstride * 8};
  cuuint32_t box[4] = {(cuuint32_t)K::ROW, (cuuint32_t)K::COLS, 1, (cuuint32_t)NV};
  cuuint32_t estr[4] = {1, 1, 1, 1};
  if (enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(st->in), dims, strides, box, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  // per launch: function attributes are per device, and the call is cheap
  cudaError_t ea = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SMEM);
  if (ea != cudaSuccess) return ea;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int ntx = (L.nx + TX - 1) / TX, nty = (L.ny + TY - 1) / TY, ntz = (L.nz + ZC - 1) / ZC;
  const int nitems = ntx * nty * ntz;
  const int grid = nitems < sms ? nitems : sms;   // persistent, one CTA per SM
  kern<<<grid, dim3(TX, TY), K::SMEM, s>>>(tm, L, C, *st, ntx, nty, ntz);
  return cudaGetLastError();
  }
}

// which: 0 = 32x16 threads, 32-plane chunks; 1 = 32x16, 64-plane chunks; 2 = 64x8, 32-plane chunks
template <int ORDER, bool KO>
static cudaError_t wv_tile(int which, const Layout& L, const Coef& C, const Stage* st, cudaStream_t s,
                           cudaFuncAttributes* a) {
  switch (which) {
    case 0: return wv_go<ORDER, KO, 32, 16, 32>(L, C, st, s, a);
    case 1: return wv_go<ORDER, KO, 32, 16, 64>(L, C, st, s, a);
    case 2: return wv_go<ORDER, KO, 64, 8, 32>(L, C, st, s, a);
  }
  return cudaErrorInvalidValue;
}

// Sample-1 system (five variables): which: 0 = 16x8 threads, 1 = 16x16 (at 8th order with one plane of prefetch),
// 2 = 32x8 (fits at 4th order only); 64-plane chunks
// 64-plane chunks: measured 0.886 ms per launch at 256^3, 8th order (32: 0.914, 128: 1.006)
constexpr int kW1ZC = 64;
template <int ORDER, bool KO>
static cudaError_t wv1_tile(int which, const Layout& L, const Coef& C, const Stage* st, cudaStream_t s,
                            cudaFuncAttributes* a) {
  switch (which) {
    case 0: return wv_go<ORDER, KO, 16, 8, kW1ZC, 5>(L, C, st, s, a);
    case 1: return wv_go<ORDER, KO, 16, 16, kW1ZC, 5>(L, C, st, s, a);
    case 2: return wv_go<ORDER, KO, 32, 8, kW1ZC, 5>(L, C, st, s, a);
  }
  return cudaErrorInvalidValue;
}
static cudaError_t wv1_dispatch(int order, bool ko, int which, const Layout& L, const Coef& C, const Stage* st,
                                cudaStream_t s, cudaFuncAttributes* a) {
  if (order == 4) return ko ? wv1_tile<4, true>(which, L, C, st, s, a) : wv1_tile<4, false>(which, L, C, st, s, a);
  if (order == 8) return ko ? wv1_tile<8, true>(which, L, C, st, s, a) : wv1_tile<8, false>(which, L, C, st, s, a);
  return cudaErrorInvalidValue;
}
// true when plane-ring variant `which` of the Sample-1 system exists for this order / dissipation (its ring fits
// shared memory) and the layout suits TMA
bool wave1_tma_ok(const Layout& L, int order, bool ko, int which) {
  if (!wave_tma_ok(L, order, ko)) return false;
  cudaFuncAttributes fa;
  Layout L0{}; Coef C0{};
  return wv1_dispatch(order, ko, which, L0, C0, nullptr, 0, &fa) == cudaSuccess;
}
cudaError_t launch_wave1_tma(const Layout& L, const Coef& C, int order, int which, const Stage& st, cudaStream_t s) {
  return wv1_dispatch(order, C.ko != 0.0, which, L, C, &st, s, nullptr);
}
cudaError_t kernel_info_wave1_tma(int order, int which, cudaFuncAttributes* a) {
  Layout L{}; Coef C{};
  return wv1_dispatch(order, true, which, L, C, nullptr, 0, a);
}

static cudaError_t wv_dispatch(int order, bool ko, int which, const Layout& L, const Coef& C, const Stage* st,
                               cudaStream_t s, cudaFuncAttributes* a) {
  if (order == 4) return ko ? wv_tile<4, true>(which, L, C, st, s, a) : wv_tile<4, false>(which, L, C, st, s, a);
  if (order == 8) return ko ? wv_tile<8, true>(which, L, C, st, s, a) : wv_tile<8, false>(which, L, C, st, s, a);
  return cudaErrorInvalidValue;
}

cudaError_t launch_wave_tma(const Layout& L, const Coef& C, int order, int which, const Stage& st, cudaStream_t s) {
  return wv_dispatch(order, C.ko != 0.0, which, L, C, &st, s, nullptr);
}
cudaError_t kernel_info_wave_tma(int order, int which, cudaFuncAttributes* a) {
  Layout L{}; Coef C{};
  return wv_dispatch(order, true, which, L, C, nullptr, 0, a);
}

#endif   // CHM_EMULATE

}  // namespace chm
