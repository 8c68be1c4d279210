// Host-only probe of the launch validator (paper_1307_6488_b200/csrc/tma_check.cuh): a good plan passes, and each
// rule rejects a plan broken in exactly that way.  Prints one line per case: "<name> <0|1>" (1 = rejected).
#include <cstdio>

#include "../../paper_1307_6488_b200/csrc/tma_check.cuh"

using namespace chm;

static TmaPlan good() {
  TmaPlan p;
  p.kernel = "probe";
  p.smem_bytes = 64 * 1024;
  p.threads = 256;
  p.barrier_off = 32 * 1024;
  p.n_barriers = 4;
  p.expect = {22u * 10 * 10 * 8, 18u * 4 * 4 * 8};
  p.loads.push_back({"box", 0, {22, 10, 10, 1}, 0, 0});
  p.loads.push_back({"tile", 17664, {18, 4, 4, 1}, 1, 0});
  return p;
}

int main() {
  auto show = [](const char* name, const TmaPlan& p) { printf("%s %d\n", name, check_tma_plan(p).empty() ? 0 : 1); };
  TmaPlan p = good();
  show("good", p);
  p = good(); p.loads[1].smem_off = 17600 + 8; show("misaligned_destination", p);
  p = good(); p.loads[0].box[0] = 21; p.expect[0] = 21u * 10 * 10 * 8; show("odd_inner_extent", p);
  p = good(); p.loads[0].box[1] = 257; show("box_extent_over_256", p);
  p = good(); p.loads[0].x_parity = 1; show("odd_x_coordinate", p);
  p = good(); p.expect[1] += 8; show("expect_tx_mismatch", p);
  p = good(); p.smem_bytes = 300 * 1024; show("shared_memory_over_limit", p);
  p = good(); p.loads[1].smem_off = 32 * 1024 - 128; show("box_overruns_barriers", p);
  p = good(); p.barrier_off += 4; show("misaligned_barrier", p);
  p = good(); p.threads = 250; show("bad_thread_count", p);
  p = good(); p.loads[1].barrier = 7; show("barrier_index", p);
  Layout L{};
  L.pitch = 272; L.tot_y = 262; L.tot_z = 262; L.nvars = 25; L.vstride = 272L * 262 * 262;
  alignas(128) static char buf[256];
  printf("layout_good %d\n", check_tma_layout(L, buf, 0).empty() ? 0 : 1);
  printf("layout_odd_origin %d\n", check_tma_layout(L, buf, 1).empty() ? 0 : 1);
  printf("layout_misaligned_base %d\n", check_tma_layout(L, buf + 16, 0).empty() ? 0 : 1);
  L.pitch = 270;
  printf("layout_bad_pitch %d\n", check_tma_layout(L, buf, 0).empty() ? 0 : 1);
  return 0;
}
