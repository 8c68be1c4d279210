// cta_emu.hpp -- host emulation of the CUDA constructs libchemora's TMA kernels are written in, so that the KERNEL
// SOURCE ITSELF (csrc/kernels_bssn_tma.cu, csrc/kernels_wave_tma.cu, compiled by g++ with -DCHM_EMULATE) runs on a box
// without a GPU: one OS thread per CUDA thread, one CTA at a time.  Test infrastructure only.
//
// What is emulated, and how faithfully:
//   threadIdx / blockIdx / gridDim / blockDim   thread-local values
//   dynamic shared memory                       one 128-byte aligned heap block per CTA
//   __syncthreads, __syncwarp, bar.sync id,n    real barriers (mutex + condition variable); __syncwarp really waits
//                                               for the 32 threads of the warp (the kernels rely on nothing stronger)
//   mbarrier (init, arrive, arrive.expect_tx,   the PTX phase/parity semantics: a phase completes when the pending
//     complete_tx, try_wait.parity,             arrival count and the pending transaction bytes are both zero; the
//     pending_count of the returned state)      state returned by arrive holds the count BEFORE the arrival
//   cp.async.bulk.tensor.4d (TMA tile load)     a synchronous copy of the box (out-of-bounds elements = 0) at issue
//                                               time followed by complete_tx -- one of the timings the hardware may
//                                               produce; a protocol that is wrong for EVERY timing (slot, parity,
//                                               byte count, missing refill) shows up as wrong data or a timed-out wait
//   atomicCAS, clock64, __dadd_rn & co, __stcs  plain host equivalents
// Not emulated: timing, memory-model subtleties below the granularity of these barriers.
#pragma once
#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <condition_variable>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <map>
#include <memory>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

#define __global__
#define __device__
#define __host__
#define __forceinline__ inline
#define __launch_bounds__(...)
#define __grid_constant__
#define __align__(n) alignas(n)
#define __shared__ static   // static shared arrays: one CTA runs at a time, so one instance per kernel is per-CTA storage

using std::max;
using std::min;

struct alignas(16) int4 { int x, y, z, w; };
inline int4 make_int4(int x, int y, int z, int w) { return int4{x, y, z, w}; }

typedef int cudaError_t;
typedef void* cudaStream_t;
struct cudaFuncAttributes { int numRegs; size_t localSizeBytes, sharedSizeBytes; };
enum { cudaSuccess = 0, cudaErrorInvalidValue = 1 };

// the tensor map: what cuTensorMapEncodeTiled is given (doubles; strides in bytes for dimensions 1..3)
struct CUtensorMap {
  const double* base;
  uint64_t dims[4];
  uint64_t strides[3];
  uint32_t box[4];
};

namespace chm_emu {

struct Idx3 { unsigned x, y, z; };

class Barrier {   // reusable counting barrier for `n` participants (n fixed per use site)
 public:
  void wait(int n) {
    std::unique_lock<std::mutex> lk(m_);
    const unsigned gen = gen_;
    if (++count_ == n) { count_ = 0; ++gen_; cv_.notify_all(); return; }
    cv_.wait(lk, [&] { return gen_ != gen; });
  }
 private:
  std::mutex m_;
  std::condition_variable cv_;
  int count_ = 0;
  unsigned gen_ = 0;
};

struct MBar {
  std::mutex m;
  std::condition_variable cv;
  int expected = 0, pending = 0;
  long tx = 0;
  unsigned phase = 0;
  void settle() {   // with m held
    if (pending == 0 && tx == 0) { phase ^= 1u; pending = expected; cv.notify_all(); }
  }
};

struct Cta {
  unsigned char* smem = nullptr;
  size_t smem_bytes = 0;
  int nthreads = 0;
  Barrier all;
  std::vector<std::unique_ptr<Barrier>> warp, named;
  std::vector<double> shfl;                       // one slot per thread: warp shuffles
  std::mutex bars_m;
  std::map<size_t, std::unique_ptr<MBar>> bars;   // keyed by shared-memory offset
  long tma_loads = 0, tma_bytes = 0;              // statistics
  MBar& bar(const void* p) {
    const size_t off = (const unsigned char*)p - smem;
    if (off >= smem_bytes || off % 8) { fprintf(stderr, "cta_emu: mbarrier outside shared memory or misaligned\n"); abort(); }
    std::lock_guard<std::mutex> lk(bars_m);
    auto& u = bars[off];
    if (!u) u.reset(new MBar());
    return *u;
  }
};

inline thread_local Idx3 t_threadIdx, t_blockIdx, t_gridDim, t_blockDim;
inline thread_local Cta* t_cta = nullptr;

inline uint32_t smem_offset(const void* p) { return (uint32_t)((const unsigned char*)p - t_cta->smem); }
inline void* smem_at(uint32_t off) { return t_cta->smem + off; }

inline void mbar_init(void* bar, int count) {
  MBar& b = t_cta->bar(bar);
  std::lock_guard<std::mutex> lk(b.m);
  b.expected = b.pending = count; b.tx = 0; b.phase = 0;
}
inline uint64_t mbar_arrive(void* bar) {   // returns the pending count before this arrival
  MBar& b = t_cta->bar(bar);
  std::lock_guard<std::mutex> lk(b.m);
  const int before = b.pending;
  if (before <= 0) { fprintf(stderr, "cta_emu: more arrivals than the mbarrier expects\n"); abort(); }
  --b.pending;
  b.settle();
  return (uint64_t)before;
}
inline void mbar_expect_tx(void* bar, uint32_t bytes) {
  MBar& b = t_cta->bar(bar);
  std::lock_guard<std::mutex> lk(b.m);
  b.tx += bytes;
  if (b.pending <= 0) { fprintf(stderr, "cta_emu: arrive.expect_tx on a barrier with no pending arrival\n"); abort(); }
  --b.pending;
  b.settle();
}
inline void mbar_complete_tx(void* bar, uint32_t bytes) {
  MBar& b = t_cta->bar(bar);
  std::lock_guard<std::mutex> lk(b.m);
  b.tx -= bytes;
  b.settle();
}
inline bool mbar_try_wait(void* bar, uint32_t parity) {   // true once the phase of that parity has completed
  MBar& b = t_cta->bar(bar);
  std::unique_lock<std::mutex> lk(b.m);
  if ((b.phase & 1u) != (parity & 1u)) return true;
  b.cv.wait_for(lk, std::chrono::milliseconds(20));
  return (b.phase & 1u) != (parity & 1u);
}

// the tile load: box elements in x-fastest order, out-of-bounds = 0; then complete_tx on the barrier
inline void tma_load_4d(void* dst, const CUtensorMap* tm, void* bar, int x, int y, int z, int v) {
  Cta* c = t_cta;
  const size_t off = (unsigned char*)dst - c->smem;
  const size_t n = (size_t)tm->box[0] * tm->box[1] * tm->box[2] * tm->box[3];
  if (off % 128 || off + n * 8 > c->smem_bytes || (x & 1)) {
    fprintf(stderr, "cta_emu: TMA destination misaligned / out of shared memory, or odd x coordinate (%zu, %d)\n", off, x);
    abort();
  }
  double* d = (double*)dst;
  for (uint32_t l = 0; l < tm->box[3]; ++l)
    for (uint32_t k = 0; k < tm->box[2]; ++k)
      for (uint32_t j = 0; j < tm->box[1]; ++j)
        for (uint32_t i = 0; i < tm->box[0]; ++i) {
          const long cx = x + (long)i, cy = y + (long)j, cz = z + (long)k, cv = v + (long)l;
          const bool in = cx >= 0 && cy >= 0 && cz >= 0 && cv >= 0 && cx < (long)tm->dims[0] && cy < (long)tm->dims[1] &&
                          cz < (long)tm->dims[2] && cv < (long)tm->dims[3];
          *d++ = in ? *(const double*)((const char*)tm->base + cx * 8 + cy * tm->strides[0] + cz * tm->strides[1] +
                                       cv * tm->strides[2])
                    : 0.0;
        }
  {
    std::lock_guard<std::mutex> lk(c->bars_m);
    c->tma_loads += 1; c->tma_bytes += (long)n * 8;
  }
  mbar_complete_tx(bar, (uint32_t)(n * 8));
}

inline void sync_all() { t_cta->all.wait(t_cta->nthreads); }
inline void sync_warp() { t_cta->warp[(t_threadIdx.y * t_blockDim.x + t_threadIdx.x) / 32]->wait(32); }
#ifdef CHM_EMU_DROP_NAMED_BARRIERS   // self-test of the race detection: bar.sync id, n becomes a no-op
inline void sync_named(int, int) {}
#else
inline void sync_named(int id, int count) { t_cta->named[id]->wait(count); }
#endif
inline double shfl_down(double v, int delta) {   // all 32 threads of the warp call it together
  const int t = t_threadIdx.y * t_blockDim.x + t_threadIdx.x;
  t_cta->shfl[t] = v;
  sync_warp();
  const double r = (t & 31) + delta < 32 ? t_cta->shfl[t + delta] : v;
  sync_warp();
  return r;
}
inline double shfl_xor(double v, int lane_mask) {   // all 32 threads of the warp call it together
  const int t = t_threadIdx.y * t_blockDim.x + t_threadIdx.x;
  t_cta->shfl[t] = v;
  sync_warp();
  const double r = t_cta->shfl[(t & ~31) | ((t ^ lane_mask) & 31)];
  sync_warp();
  return r;
}

// run `grid` CTAs of `threads` (x * y) threads one after the other; body() is the kernel call
struct Stats { long tma_loads = 0, tma_bytes = 0; };
inline Stats run_grid(int grid, int bx, int by, size_t smem_bytes, const std::function<void()>& body, int grid_y = 1,
                      int grid_z = 1) {
  Stats st;
  for (int bz_ = 0; bz_ < grid_z; ++bz_)
  for (int by_ = 0; by_ < grid_y; ++by_)
  for (int b = 0; b < grid; ++b) {
    Cta cta;
    cta.smem_bytes = smem_bytes;
    cta.smem = (unsigned char*)aligned_alloc(128, (smem_bytes + 127) / 128 * 128);
    memset(cta.smem, 0xff, smem_bytes);   // NaN pattern: reading what was never loaded shows up
    cta.nthreads = bx * by;
    cta.shfl.assign(cta.nthreads, 0.0);
    for (int w = 0; w < (cta.nthreads + 31) / 32; ++w) cta.warp.emplace_back(new Barrier());
    for (int i = 0; i < 16; ++i) cta.named.emplace_back(new Barrier());
    std::vector<std::thread> th;
    for (int t = 0; t < cta.nthreads; ++t)
      th.emplace_back([&, t] {
        t_cta = &cta;
        t_threadIdx = Idx3{(unsigned)(t % bx), (unsigned)(t / bx), 0};
        t_blockIdx = Idx3{(unsigned)b, (unsigned)by_, (unsigned)bz_};
        t_gridDim = Idx3{(unsigned)grid, (unsigned)grid_y, (unsigned)grid_z};
        t_blockDim = Idx3{(unsigned)bx, (unsigned)by, 1};
        body();
      });
    for (auto& x : th) x.join();
    st.tma_loads += cta.tma_loads; st.tma_bytes += cta.tma_bytes;
    free(cta.smem);
  }
  return st;
}

// kernels without any inter-thread synchronisation (no barrier, no shuffle): every thread of every block in turn, on
// the calling OS thread
inline void run_grid_serial(int gx, int gy, int gz, int bx, int by, const std::function<void()>& body) {
  for (int z = 0; z < gz; ++z)
    for (int y = 0; y < gy; ++y)
      for (int x = 0; x < gx; ++x)
        for (int t = 0; t < bx * by; ++t) {
          t_cta = nullptr;
          t_threadIdx = Idx3{(unsigned)(t % bx), (unsigned)(t / bx), 0};
          t_blockIdx = Idx3{(unsigned)x, (unsigned)y, (unsigned)z};
          t_gridDim = Idx3{(unsigned)gx, (unsigned)gy, (unsigned)gz};
          t_blockDim = Idx3{(unsigned)bx, (unsigned)by, 1};
          body();
        }
}

}  // namespace chm_emu

#define threadIdx chm_emu::t_threadIdx
#define blockIdx chm_emu::t_blockIdx
#define gridDim chm_emu::t_gridDim
#define blockDim chm_emu::t_blockDim

inline void __syncthreads() { chm_emu::sync_all(); }
inline void __syncwarp() { chm_emu::sync_warp(); }
inline double __dadd_rn(double a, double b) { return a + b; }
inline double __dsub_rn(double a, double b) { return a - b; }
inline double __dmul_rn(double a, double b) { return a * b; }
template <class T> inline void __stcs(T* p, T v) { *p = v; }
template <class T> inline T __ldg(const T* p) { return *p; }
inline double __shfl_xor_sync(unsigned, double v, int lane_mask) { return chm_emu::shfl_xor(v, lane_mask); }
inline double __shfl_down_sync(unsigned, double v, int delta) { return chm_emu::shfl_down(v, delta); }
inline double atomicAdd(double* p, double v) {   // CTAs run one at a time and one thread per CTA adds: plain
  static std::mutex m;
  std::lock_guard<std::mutex> lk(m);
  const double old = *p;
  *p = old + v;
  return old;
}
inline double __longlong_as_double(long long x) { double d; memcpy(&d, &x, 8); return d; }
inline long long __double_as_longlong(double d) { long long x; memcpy(&x, &d, 8); return x; }
inline unsigned long long atomicMax(unsigned long long* p, unsigned long long v) {
  unsigned long long old = __atomic_load_n(p, __ATOMIC_SEQ_CST);
  while (old < v && !__atomic_compare_exchange_n(p, &old, v, false, __ATOMIC_SEQ_CST, __ATOMIC_SEQ_CST)) {}
  return old;
}
inline long long clock64() {
  return std::chrono::duration_cast<std::chrono::nanoseconds>(std::chrono::steady_clock::now().time_since_epoch()).count();
}
inline unsigned atomicCAS(unsigned* p, unsigned expect, unsigned val) {
  __atomic_compare_exchange_n(p, &expect, val, false, __ATOMIC_SEQ_CST, __ATOMIC_SEQ_CST);
  return expect;
}
