// tma_check.cuh -- host-side validation of every TMA launch of libchemora (no device needed).
// A cp.async.bulk.tensor whose shared-memory destination is not 128-byte aligned, whose box rows are not a multiple
// of 16 bytes, whose global coordinates do not start rows on 16-byte boundaries, or whose mbarrier expects a byte
// count other than what the loads deliver, is a device fault or a hung CTA -- on a shared, metered GPU that is
// unacceptable (the paper's own run-time path that edits, compiles and loads kernels has the same failure surface,
// PAPER.md:246).  So every launcher describes what its kernel instance will issue as a TmaPlan and launches only if
// check_tma_plan accepts it; chemora_selfcheck() walks the plans of ALL template instances without a device.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "common.cuh"

namespace chm {

struct TmaLoad {
  const char* what;
  size_t smem_off;      // destination, bytes from the (128-byte aligned) dynamic shared-memory base
  uint32_t box[4];      // box extents in elements (doubles), innermost first
  int barrier;          // index into TmaPlan::expect of the mbarrier it completes on
  int x_parity;         // parity (0/1) of every x coordinate this load is issued with (rows must start 16-byte aligned)
};
struct TmaPlan {
  std::string kernel;
  std::vector<TmaLoad> loads;
  std::vector<uint32_t> expect;   // bytes each barrier's arrive.expect_tx announces for one phase
  size_t barrier_off = 0;         // first mbarrier, bytes from the shared-memory base
  int n_barriers = 0;
  size_t smem_bytes = 0;          // dynamic shared memory of the launch
  int threads = 0;
};

constexpr size_t kSmemOptIn = 232448;   // 227 KB: the per-block opt-in limit of sm_100

// empty string = fine; otherwise the first violated rule
inline std::string check_tma_plan(const TmaPlan& p, size_t smem_limit = kSmemOptIn) {
  using std::to_string;
  const std::string k = std::string(p.kernel) + ": ";
  if (p.smem_bytes > smem_limit)
    return k + to_string(p.smem_bytes) + " bytes of dynamic shared memory > limit " + to_string(smem_limit);
  if (p.threads < 32 || p.threads > 1024 || p.threads % 32) return k + "bad thread count " + to_string(p.threads);
  if (p.barrier_off % 8) return k + "mbarrier offset " + to_string(p.barrier_off) + " not 8-byte aligned";
  if (p.barrier_off + 8 * (size_t)p.n_barriers > p.smem_bytes)
    return k + "mbarriers end beyond the " + to_string(p.smem_bytes) + " bytes of shared memory";
  std::vector<uint64_t> issued(p.expect.size(), 0);
  for (const TmaLoad& l : p.loads) {
    const std::string w = k + l.what + ": ";
    if (l.smem_off % 128) return w + "destination offset " + to_string(l.smem_off) + " not 128-byte aligned";
    uint64_t n = 1;
    for (int d = 0; d < 4; ++d) {
      if (l.box[d] < 1 || l.box[d] > 256) return w + "box extent " + to_string(l.box[d]) + " outside 1..256";
      n *= l.box[d];
    }
    if ((l.box[0] * 8) % 16) return w + "inner box extent " + to_string(l.box[0]) + " doubles is not a multiple of 16 bytes";
    if (l.x_parity != 0) return w + "odd x coordinates: rows would start off a 16-byte boundary";
    if (l.smem_off + n * 8 > p.barrier_off)
      return w + "box ends at " + to_string(l.smem_off + n * 8) + ", beyond the data area (" + to_string(p.barrier_off) + ")";
    if (l.barrier < 0 || l.barrier >= (int)p.expect.size()) return w + "barrier index out of range";
    issued[l.barrier] += n * 8;
  }
  for (size_t b = 0; b < p.expect.size(); ++b)
    if (issued[b] != p.expect[b])
      return k + "barrier " + to_string(b) + " expects " + to_string(p.expect[b]) + " bytes but its loads deliver " +
             to_string(issued[b]);
  return std::string();
}

// what a tensor map over a state buffer needs from the layout and the base address (cuTensorMapEncodeTiled rules)
inline std::string check_tma_layout(const Layout& L, const void* base, int x_origin) {
  if (reinterpret_cast<uintptr_t>(base) % 128) return "state buffer is not 128-byte aligned";
  if (L.pitch % 16) return "row pitch is not a multiple of 16 doubles (128 bytes)";
  if (L.pitch <= 0 || L.tot_y <= 0 || L.tot_z <= 0 || L.nvars <= 0) return "empty tensor";
  if (L.pitch > (1L << 31) || L.tot_y > (1 << 30) || L.tot_z > (1 << 30)) return "tensor dimension too large";
  if ((unsigned long long)L.vstride * 8ull >= (1ull << 40)) return "variable stride >= 2^40 bytes";
  if (x_origin % 2) return "box x origin " + std::to_string(x_origin) + " is odd: rows would start off a 16-byte boundary";
  return std::string();
}

// why the last launch on this thread was refused by the validator (empty: it was not)
inline std::string& last_refusal() {
  static thread_local std::string msg;
  return msg;
}
// true = go.  Records the reason otherwise.
inline bool launch_allowed(const TmaPlan& p, const Layout& L, const void* base, int x_origin, int need_ghost) {
  std::string why = L.err ? std::string() : std::string("no device error word in the layout");
  if (why.empty()) why = check_tma_plan(p);
  if (why.empty()) why = check_tma_layout(L, base, x_origin);
  if (why.empty() && L.g < need_ghost) why = p.kernel + ": ghost width " + std::to_string(L.g) + " < " + std::to_string(need_ghost);
  last_refusal() = why;
  return why.empty();
}

// the plans of every instance of a kernel family (implemented next to the kernels)
void plans_bssn_fused(std::vector<TmaPlan>& out);
void plans_wave_tma(std::vector<TmaPlan>& out);

}  // namespace chm
