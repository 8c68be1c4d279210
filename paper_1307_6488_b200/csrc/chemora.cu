// chemora.cu -- host side of libchemora.so: the C ABI declared in include/chemora.h.
// Handle, layout, parameter table, variant registry + runtime sweep, RK4 driver.  No CPU compute path exists:
// every compute entry point enqueues CUDA kernels and reports CHEMORA_ECUDA if that fails.
#include "../../include/chemora.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "common.cuh"
#include "tma_check.cuh"

using namespace chm;

struct chemora {
  Layout L;
  int order, system;
  double dx;
  double eps_diss, eta, sgc;
  int ko_order;          // 5, or 9 (8th-order BSSN only)
  cudaStream_t stream;
  void* (*alloc)(size_t, void*);
  void (*dealloc)(void*, void*);
  void* actx;
  double* buf[4];
  double* derivs;       // split variant scratch (lazy)
  double* staging;      // device packed staging for set/get_state (lazy)
  unsigned* dev_err;    // device error word the kernels' bounded waits write (Layout::err)
  int fused, tile;
  int boundary;         // CHEMORA_BC_PERIODIC (ghost fill) or CHEMORA_BC_RADIATIVE (ghost layers are evolved boundary points)
  int autotune_split;   // tuning: chemora_autotune also times the derivative-split variant
  int autotune_fused_ids;   // tuning: chemora_autotune times the fused tile ids below this bound
  chemora* nb_lo;        // z-neighbours of a linked block (chemora_link_z); nullptr: periodic in itself
  chemora* nb_hi;
  long launches;
  // optional per-kernel timing (chemora_timing): event pairs around every RHS evaluation / ghost fill
  bool timing;
  std::vector<cudaEvent_t> ev[2];   // [0] rhs, [1] fill: a fixed pool of kEvPool events, consecutive (start, stop) pairs
  int ev_used[2];                   // events of the pool recorded since the last drain
  double ev_ms[2];                  // time drained from the pool so far
  long ev_launches[2];
  std::string err;
};

namespace {

int fail(chemora_t* h, int code, const std::string& msg) {
  if (h) h->err = msg;
  return code;
}
int cuda_fail(chemora_t* h, cudaError_t e, const char* what) {
  std::string msg = std::string(what) + ": " + cudaGetErrorString(e);
  if (!last_refusal().empty()) { msg += " (launch refused by the validator: " + last_refusal() + ")"; last_refusal().clear(); }
  return fail(h, CHEMORA_ECUDA, msg);
}
#define CK(h, call, what)                                   \
  do {                                                      \
    cudaError_t e_ = (call);                                \
    if (e_ != cudaSuccess) return cuda_fail(h, e_, what);   \
  } while (0)

size_t state_bytes(const chemora_t* h) { return (size_t)h->L.nvars * h->L.vstride * sizeof(double); }
size_t packed_count(const chemora_t* h) { return (size_t)h->L.nvars * h->L.nx * h->L.ny * h->L.nz; }
long deriv_stride(const chemora_t* h) {
  long n = (long)h->L.nx * h->L.ny * h->L.nz;
  return (n + 15) / 16 * 16;
}

void* dev_alloc(chemora_t* h, size_t bytes) {
  if (h->alloc) return h->alloc(bytes, h->actx);
  void* p = nullptr;
  return cudaMalloc(&p, bytes) == cudaSuccess ? p : nullptr;
}
void dev_free(chemora_t* h, void* p) {
  if (!p) return;
  if (h->dealloc) h->dealloc(p, h->actx);
  else cudaFree(p);
}

Coef make_coef(const chemora_t* h) {
  Coef C;
  C.inv_h = 1.0 / h->dx;
  C.inv_h2 = 1.0 / (h->dx * h->dx);
  C.ko = h->eps_diss / (64.0 * h->dx);
  if (h->ko_order == 9) {
    const double k9 = h->eps_diss / (1024.0 * h->dx);
    const double w9[5] = {210.0, -120.0, 45.0, -10.0, 1.0};
    for (int k = 0; k < 5; ++k) C.kq[k] = k9 * w9[k];
  } else {
    const double w5[5] = {15.0, -6.0, 1.0, 0.0, 0.0};
    for (int k = 0; k < 5; ++k) C.kq[k] = C.ko * w5[k];
  }
  C.eta = h->eta;
  C.sgc = h->sgc;
  return C;
}

int ensure_derivs(chemora_t* h) {
  if (h->derivs) return CHEMORA_OK;
  size_t bytes = (size_t)kNumDerivArrays * deriv_stride(h) * sizeof(double);
  h->derivs = (double*)dev_alloc(h, bytes);
  if (!h->derivs) return fail(h, CHEMORA_ENOMEM, "derivative scratch allocation failed");
  return CHEMORA_OK;
}

constexpr int kEvPool = 512;   // 256 (start, stop) pairs per category

// add the recorded pairs' durations to ev_ms and make the pool empty again (waits for the last recorded event)
void drain(chemora_t* h, int cat) {
  const int n = h->ev_used[cat] & ~1;
  if (n >= 2 && cudaEventSynchronize(h->ev[cat][n - 1]) == cudaSuccess)
    for (int i = 0; i < n; i += 2) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, h->ev[cat][i], h->ev[cat][i + 1]) == cudaSuccess) h->ev_ms[cat] += ms;
    }
  h->ev_used[cat] = 0;
}

void tick(chemora_t* h, int cat) {
  if (!h->timing) return;
  if (h->ev_used[cat] == kEvPool) drain(h, cat);   // pool full: one wait per 256 timed launches
  cudaEventRecord(h->ev[cat][h->ev_used[cat]++], h->stream);
}

int run_rhs_inner(chemora_t* h, const Stage& st);

// one RHS evaluation with the given epilogue; counts launches
int run_rhs(chemora_t* h, const Stage& st) {
  tick(h, 0);
  long before = h->launches;
  int rc = run_rhs_inner(h, st);
  tick(h, 0);
  if (h->timing) h->ev_launches[0] += h->launches - before;
  return rc;
}

int run_rhs_inner(chemora_t* h, const Stage& st) {
  if (h->eps_diss != 0.0 && h->L.g < 3) return fail(h, CHEMORA_EINVAL, "eps_diss != 0 needs ghost >= 3 (KO order 5)");
  Coef C = make_coef(h);
  if (h->system == CHEMORA_SYS_WAVE) {
    if (h->tile >= 6 && h->tile < 9 && wave_tma_ok(h->L, h->order, C.ko != 0.0))
      CK(h, launch_wave_tma(h->L, C, h->order, h->tile - 6, st, h->stream), "wave plane-ring kernel launch");
    else
      CK(h, launch_wave(h->L, C, h->order, h->tile % 6, st, h->stream), "wave kernel launch");
    h->launches += 1;
  } else if (h->system == CHEMORA_SYS_WAVE1) {
    if (h->tile >= 6 && h->tile < 9 && wave1_tma_ok(h->L, h->order, C.ko != 0.0, h->tile - 6))
      CK(h, launch_wave1_tma(h->L, C, h->order, h->tile - 6, st, h->stream), "first-order wave plane-ring kernel launch");
    else
      CK(h, launch_wave1(h->L, C, h->order, h->tile % 6, st, h->stream), "first-order wave kernel launch");
    h->launches += 1;
  } else if (h->fused) {
    CK(h, launch_bssn_fused(h->L, C, h->order, h->tile, st, h->stream), "bssn fused kernel launch");
    h->launches += 1;
  } else {
    int rc = ensure_derivs(h);
    if (rc) return rc;
    CK(h, launch_bssn_derivs(h->L, C, h->order, h->tile % 6, st.in, h->derivs, h->stream), "bssn derivative kernel launch");
    CK(h, launch_bssn_from_derivs(h->L, C, h->tile % 6, h->derivs, st, h->stream), "bssn rhs kernel launch");
    h->launches += 2;
  }
  return CHEMORA_OK;
}

int fill(chemora_t* h, double* state) {
  FillLink link, *lp = nullptr;
  if (h->nb_lo || h->nb_hi) {
    // a linked block takes its ghost z-planes from the SAME buffer of its neighbours, so the state must be one of
    // the library's four buffers
    int which = -1;
    for (int b = 0; b < 4; ++b)
      if (state == h->buf[b]) which = b;
    if (which < 0) return fail(h, CHEMORA_ESTATE, "a z-linked block can fill only its own four buffers");
    chemora_t* lo = h->nb_lo ? h->nb_lo : h;
    chemora_t* hi = h->nb_hi ? h->nb_hi : h;
    link = FillLink{lo->buf[which], lo->L.vstride, lo->L.nz, hi->buf[which], hi->L.vstride};
    lp = &link;
  }
  tick(h, 1);
  CK(h, launch_fill_ghosts(h->L, state, h->stream, lp), "ghost fill launch");
  tick(h, 1);
  h->launches += 1;
  if (h->timing) h->ev_launches[1] += 1;
  return CHEMORA_OK;
}

// the radiative face kernel with the Runge-Kutta epilogue `st` (reading S16); u_inf = 1 on chi, gt11, gt22, gt33, alpha
int radiative(chemora_t* h, const Stage& st) {
  const unsigned mask = h->system == CHEMORA_SYS_BSSN ? (1u << 0) | (1u << 1) | (1u << 4) | (1u << 6) | (1u << 17) : 0u;
  tick(h, 1);
  CK(h, launch_radiative(h->L, st, h->dx, mask, h->stream), "radiative boundary launch");
  tick(h, 1);
  h->launches += 1;
  if (h->timing) h->ev_launches[1] += 1;
  return CHEMORA_OK;
}

}  // namespace

extern "C" {

int chemora_create(chemora_t** out, int nx, int ny, int nz, int ghost, int fd_order, int system_id, double dx,
                   void* cuda_stream, void* (*alloc)(size_t, void*), void (*dealloc)(void*, void*),
                   void* alloc_ctx) {
  if (!out) return CHEMORA_EINVAL;
  *out = nullptr;
  if (nx <= 0 || ny <= 0 || nz <= 0 || ghost < 0) return CHEMORA_EINVAL;
  if (fd_order != 4 && fd_order != 8) return CHEMORA_EINVAL;
  if (system_id != CHEMORA_SYS_WAVE && system_id != CHEMORA_SYS_BSSN && system_id != CHEMORA_SYS_WAVE1) return CHEMORA_EINVAL;
  if (!(dx > 0.0)) return CHEMORA_EINVAL;
  if ((alloc == nullptr) != (dealloc == nullptr)) return CHEMORA_EINVAL;
  const int need = system_id == CHEMORA_SYS_BSSN ? fd_order / 2 + 1 : fd_order / 2;
  if (ghost < need) return CHEMORA_EINVAL;
  if (nx < ghost || ny < ghost || nz < ghost) return CHEMORA_EINVAL;

  chemora_t* h = new (std::nothrow) chemora_t();
  if (!h) return CHEMORA_ENOMEM;
  Layout& L = h->L;
  L.nx = nx; L.ny = ny; L.nz = nz; L.g = ghost;
  L.nvars = system_id == CHEMORA_SYS_WAVE ? 2 : system_id == CHEMORA_SYS_WAVE1 ? 5 : 25;
  L.xo = (system_id == CHEMORA_SYS_BSSN && ((ghost - 3) & 1)) ? ghost + 1 : ghost;
  L.pitch = ((long)L.xo + nx + ghost + 15) / 16 * 16;
  L.tot_y = ny + 2 * ghost; L.tot_z = nz + 2 * ghost;
  L.plane = L.pitch * L.tot_y;
  L.vstride = L.plane * L.tot_z;
  L.col_rows = 32;
  h->order = fd_order; h->system = system_id; h->dx = dx;
  h->eps_diss = 0.0; h->eta = 1.0; h->sgc = 0.75;
  h->ko_order = 5;
  h->nb_lo = h->nb_hi = nullptr;
  h->stream = (cudaStream_t)cuda_stream;
  h->alloc = alloc; h->dealloc = dealloc; h->actx = alloc_ctx;
  h->derivs = nullptr; h->staging = nullptr; h->dev_err = nullptr;
  // 8th-order BSSN (the paper's configuration, 5 ghost zones): fused kernel on tile id 0 only
  h->fused = 1; h->tile = (system_id == CHEMORA_SYS_BSSN && fd_order == 8) ? 0 : 1;
  h->launches = 0;
  h->autotune_split = 0;
  h->autotune_fused_ids = CHEMORA_NUM_TILES;
  h->boundary = CHEMORA_BC_PERIODIC;
  h->timing = false;
  for (int c = 0; c < 2; ++c) { h->ev_used[c] = 0; h->ev_ms[c] = 0.0; h->ev_launches[c] = 0; }
  for (int b = 0; b < 4; ++b) h->buf[b] = nullptr;

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    delete h;
    return CHEMORA_ECUDA;   // no device: there is no CPU fallback
  }
  for (int b = 0; b < 4; ++b) {
    h->buf[b] = (double*)dev_alloc(h, state_bytes(h));
    if (!h->buf[b] || ((uintptr_t)h->buf[b] & 127)) {
      for (int c = 0; c <= b; ++c) dev_free(h, h->buf[c]);
      delete h;
      return CHEMORA_ENOMEM;
    }
    if (cudaMemsetAsync(h->buf[b], 0, state_bytes(h), h->stream) != cudaSuccess) {
      for (int c = 0; c <= b; ++c) dev_free(h, h->buf[c]);
      delete h;
      return CHEMORA_ECUDA;
    }
  }
  h->dev_err = (unsigned*)dev_alloc(h, 1024);   // [0] error word; from byte 16: the sweep guard's 2 x V norms
  if (!h->dev_err || cudaMemsetAsync(h->dev_err, 0, 1024, h->stream) != cudaSuccess) {
    dev_free(h, h->dev_err);
    for (int c = 0; c < 4; ++c) dev_free(h, h->buf[c]);
    delete h;
    return CHEMORA_ENOMEM;
  }
  L.err = h->dev_err;
  *out = h;
  return CHEMORA_OK;
}

int chemora_set_param(chemora_t* h, const char* name, double v) {
  if (!h || !name) return CHEMORA_EINVAL;
  if (!(v == v)) return fail(h, CHEMORA_EINVAL, "parameter value is NaN");
  if (!strcmp(name, "eps_diss")) {
    if (v < 0.0) return fail(h, CHEMORA_EINVAL, "eps_diss must be >= 0");
    if (v != 0.0 && h->L.g < 3) return fail(h, CHEMORA_EINVAL, "eps_diss != 0 needs ghost >= 3 (KO order 5)");
    h->eps_diss = v;
  } else if (!strcmp(name, "ko_order")) {
    if (v != 5.0 && v != 9.0) return fail(h, CHEMORA_EINVAL, "ko_order must be 5 or 9");
    if (v == 9.0 && !(h->system == CHEMORA_SYS_BSSN && h->order == 8))
      return fail(h, CHEMORA_EINVAL, "ko_order 9 is built for the 8th-order BSSN system only");
    h->ko_order = (int)v;
  } else if (!strcmp(name, "eta")) h->eta = v;
  else if (!strcmp(name, "shift_gamma_coeff")) h->sgc = v;
  else if (!strcmp(name, "col_rows")) {
    if (v < 1.0 || v > 1e6) return fail(h, CHEMORA_EINVAL, "col_rows must be >= 1");
    h->L.col_rows = (int)v;
  } else if (!strcmp(name, "autotune_split")) {
    if (v != 0.0 && v != 1.0) return fail(h, CHEMORA_EINVAL, "autotune_split must be 0 or 1");
    h->autotune_split = (int)v;
  } else if (!strcmp(name, "autotune_fused_ids")) {
    if (v != (double)(int)v || v < 1.0 || v > (double)CHEMORA_NUM_TILES) return fail(h, CHEMORA_EINVAL, "autotune_fused_ids must be 1..CHEMORA_NUM_TILES");
    h->autotune_fused_ids = (int)v;
  } else return fail(h, CHEMORA_EINVAL, std::string("unknown parameter: ") + name);
  return CHEMORA_OK;
}

int chemora_get_param(const chemora_t* h, const char* name, double* v) {
  if (!h || !name || !v) return CHEMORA_EINVAL;
  if (!strcmp(name, "eps_diss")) *v = h->eps_diss;
  else if (!strcmp(name, "ko_order")) *v = h->ko_order;
  else if (!strcmp(name, "eta")) *v = h->eta;
  else if (!strcmp(name, "shift_gamma_coeff")) *v = h->sgc;
  else if (!strcmp(name, "col_rows")) *v = h->L.col_rows;
  else if (!strcmp(name, "autotune_split")) *v = h->autotune_split;
  else if (!strcmp(name, "autotune_fused_ids")) *v = h->autotune_fused_ids;
  else return CHEMORA_EINVAL;
  return CHEMORA_OK;
}

int chemora_layout(const chemora_t* h, int* nvars, long* pitch, long* tot_y, long* tot_z, long* var_stride,
                   long* interior_offset) {
  if (!h) return CHEMORA_EINVAL;
  if (nvars) *nvars = h->L.nvars;
  if (pitch) *pitch = h->L.pitch;
  if (tot_y) *tot_y = h->L.tot_y;
  if (tot_z) *tot_z = h->L.tot_z;
  if (var_stride) *var_stride = h->L.vstride;
  if (interior_offset) *interior_offset = (long)h->L.g * h->L.plane + (long)h->L.g * h->L.pitch + h->L.xo;
  return CHEMORA_OK;
}

int chemora_state_ptr(chemora_t* h, int which, double** dev) {
  if (!h || !dev || which < 0 || which > 3) return CHEMORA_EINVAL;
  *dev = h->buf[which];
  return CHEMORA_OK;
}

static int ensure_staging(chemora_t* h) {
  if (h->staging) return CHEMORA_OK;
  // sized for the ghosted block too (chemora_set_state_ghosted / chemora_get_state_ghosted)
  const size_t ghosted = (size_t)h->L.nvars * (h->L.nx + 2 * h->L.g) * (h->L.ny + 2 * h->L.g) * (h->L.nz + 2 * h->L.g);
  h->staging = (double*)dev_alloc(h, ghosted * sizeof(double));
  return h->staging ? CHEMORA_OK : fail(h, CHEMORA_ENOMEM, "staging allocation failed");
}

int chemora_set_state_dev(chemora_t* h, const double* dev_packed) {
  if (!h || !dev_packed) return CHEMORA_EINVAL;
  CK(h, launch_pack(h->L, dev_packed, h->buf[0], true, h->stream), "unpack launch");
  h->launches += 1;
  return CHEMORA_OK;
}

int chemora_get_state_dev(chemora_t* h, double* dev_packed) {
  if (!h || !dev_packed) return CHEMORA_EINVAL;
  CK(h, launch_pack(h->L, dev_packed, h->buf[0], false, h->stream), "pack launch");
  h->launches += 1;
  return CHEMORA_OK;
}

int chemora_set_state_async(chemora_t* h, const double* host_packed) {
  if (!h || !host_packed) return CHEMORA_EINVAL;
  int rc = ensure_staging(h);
  if (rc) return rc;
  CK(h, cudaMemcpyAsync(h->staging, host_packed, packed_count(h) * sizeof(double), cudaMemcpyHostToDevice, h->stream),
     "H2D copy");
  return chemora_set_state_dev(h, h->staging);
}

int chemora_get_state_async(chemora_t* h, double* host_packed) {
  if (!h || !host_packed) return CHEMORA_EINVAL;
  int rc = ensure_staging(h);
  if (rc) return rc;
  rc = chemora_get_state_dev(h, h->staging);
  if (rc) return rc;
  CK(h, cudaMemcpyAsync(host_packed, h->staging, packed_count(h) * sizeof(double), cudaMemcpyDeviceToHost, h->stream),
     "D2H copy");
  return CHEMORA_OK;
}

int chemora_synchronize(chemora_t* h) {
  if (!h) return CHEMORA_EINVAL;
  unsigned code = 0;
  CK(h, cudaMemcpyAsync(&code, h->dev_err, sizeof code, cudaMemcpyDeviceToHost, h->stream), "error word D2H");
  CK(h, cudaStreamSynchronize(h->stream), "stream synchronisation");
  if (code != 0) {   // a bounded wait inside a kernel gave up: the results since the last synchronisation are invalid
    char msg[160];
    chemora_describe_device_error(code, msg, sizeof msg);
    cudaMemsetAsync(h->dev_err, 0, sizeof code, h->stream);
    return fail(h, CHEMORA_ECUDA, msg);
  }
  return CHEMORA_OK;
}

int chemora_describe_device_error(unsigned code, char* buf, size_t n) {
  if (!buf || n == 0) return CHEMORA_EINVAL;
  const unsigned family = code >> 16, where = code & 0xffffu;
  if (code == 0) snprintf(buf, n, "no device error");
  else if (family == 1 && where == 0x80) snprintf(buf, n, "fused BSSN kernel: wait for the point-value tiles timed out (code 0x%x)", code);
  else if (family == 1) snprintf(buf, n, "fused BSSN kernel: wait for the box of section %u timed out (code 0x%x)", where - 1, code);
  else if (family == 2) snprintf(buf, n, "wave plane-ring kernel: wait %u for a plane timed out (code 0x%x)", where, code);
  else snprintf(buf, n, "unknown device error code 0x%x", code);
  return CHEMORA_OK;
}

int chemora_selfcheck(char* buf, size_t n) {
  std::vector<TmaPlan> plans;
  plans_bssn_fused(plans);
  plans_wave_tma(plans);
  int bad = 0;
  std::string first;
  for (const TmaPlan& p : plans) {
    const std::string why = check_tma_plan(p);
    if (!why.empty() && bad++ == 0) first = why;
  }
  if (buf && n) snprintf(buf, n, "%zu launch plans checked, %d rejected%s%s", plans.size(), bad, bad ? ": " : "", first.c_str());
  return bad ? CHEMORA_EINVAL : (int)plans.size();
}

int chemora_set_state(chemora_t* h, const double* host_packed) {
  int rc = chemora_set_state_async(h, host_packed);
  return rc ? rc : chemora_synchronize(h);
}

int chemora_get_state(chemora_t* h, double* host_packed) {
  int rc = chemora_get_state_async(h, host_packed);
  return rc ? rc : chemora_synchronize(h);
}

int chemora_fill_ghosts(chemora_t* h, double* dev_state) {
  if (!h || !dev_state) return CHEMORA_EINVAL;
  return fill(h, dev_state);
}

int chemora_rhs(chemora_t* h, const double* dev_state, double* dev_rhs) {
  if (!h || !dev_state || !dev_rhs || dev_state == dev_rhs) return CHEMORA_EINVAL;
  Stage st{dev_state, nullptr, nullptr, dev_rhs, 0.0, MODE_RHS};
  return run_rhs(h, st);
}

// The steppers as stage tables: stage s fills buffer `in` (ghosts), then evaluates the right-hand side with the
// Runge-Kutta epilogue `st`.  One block: stage after stage.  A group of z-linked blocks: every block's fill of a
// stage, then every block's evaluation (a fill reads the neighbours' interiors of the same stage buffer).
struct StagePlan { int in; Stage st; };

static int rk4_plan(chemora_t* h, double dt, StagePlan* p) {
  double *U = h->buf[0], *Ya = h->buf[1], *Yb = h->buf[2], *S = h->buf[3];
  // stage 1: k1 = f(U);  S = k1;  Yb = U + dt/2 k1
  p[0] = {0, Stage{U, U, S, Yb, dt / 2.0, MODE_FIRST, 0.0, 0.0}};
  // stage 2: k2 = f(Yb); S += 2 k2; Ya = U + dt/2 k2
  p[1] = {2, Stage{Yb, U, S, Ya, dt / 2.0, MODE_MID, 0.0, 0.0}};
  // stage 3: k3 = f(Ya); S += 2 k3; Yb = U + dt k3
  p[2] = {1, Stage{Ya, U, S, Yb, dt, MODE_MID, 0.0, 0.0}};
  // stage 4: k4 = f(Yb); U = U + dt/6 (S + k4)
  p[3] = {2, Stage{Yb, U, S, nullptr, dt / 6.0, MODE_LAST, 0.0, 0.0}};
  return 4;
}

static int rk3_plan(chemora_t* h, double dt, StagePlan* p) {
  double *U = h->buf[0], *Ya = h->buf[1], *Yb = h->buf[2];
  // U1 = U + dt f(U)
  p[0] = {0, Stage{U, U, nullptr, Ya, dt, MODE_SSP, 0.0, 1.0}};
  // U2 = 3/4 U + 1/4 (U1 + dt f(U1))
  p[1] = {1, Stage{Ya, U, nullptr, Yb, dt, MODE_SSP, 3.0 / 4.0, 1.0 / 4.0}};
  // U+ = 1/3 U + 2/3 (U2 + dt f(U2)), written over U point by point
  p[2] = {2, Stage{Yb, U, nullptr, U, dt, MODE_SSP, 1.0 / 3.0, 2.0 / 3.0}};
  return 3;
}

static int step_one(chemora_t* h, double dt, bool rk3) {
  if (!h || !(dt == dt)) return CHEMORA_EINVAL;
  if (h->nb_lo || h->nb_hi) return fail(h, CHEMORA_ESTATE, "a z-linked block steps through the *_step_group calls");
  StagePlan p[4];
  const int ns = rk3 ? rk3_plan(h, dt, p) : rk4_plan(h, dt, p);
  for (int s = 0; s < ns; ++s) {
    int rc;
    if (h->boundary == CHEMORA_BC_RADIATIVE) {   // nothing is filled: the ghost layers are evolved by the face kernel
      if ((rc = run_rhs(h, p[s].st))) return rc;
      if ((rc = radiative(h, p[s].st))) return rc;
    } else {
      if ((rc = fill(h, h->buf[p[s].in]))) return rc;
      if ((rc = run_rhs(h, p[s].st))) return rc;
    }
  }
  return CHEMORA_OK;
}

static int step_group(chemora_t* const* hs, int n, double dt, bool rk3) {
  if (!hs || n < 1 || n > 64 || !(dt == dt)) return CHEMORA_EINVAL;
  for (int b = 0; b < n; ++b) {
    chemora_t* h = hs[b];
    if (!h) return CHEMORA_EINVAL;
    if (h->stream != hs[0]->stream) return fail(h, CHEMORA_EINVAL, "the blocks of a group share one stream");
    for (chemora_t* nb : {h->nb_lo, h->nb_hi}) {
      bool in_group = nb == nullptr;
      for (int c = 0; c < n; ++c) in_group = in_group || hs[c] == nb;
      if (!in_group) return fail(h, CHEMORA_EINVAL, "a block of the group is linked to a block outside it");
    }
  }
  StagePlan p[64][4];
  int ns = 0;
  for (int b = 0; b < n; ++b) ns = rk3 ? rk3_plan(hs[b], dt, p[b]) : rk4_plan(hs[b], dt, p[b]);
  for (int s = 0; s < ns; ++s) {
    int rc;
    for (int b = 0; b < n; ++b)
      if ((rc = fill(hs[b], hs[b]->buf[p[b][s].in]))) return rc;
    for (int b = 0; b < n; ++b)
      if ((rc = run_rhs(hs[b], p[b][s].st))) return rc;
  }
  return CHEMORA_OK;
}

int chemora_rk4_step(chemora_t* h, double dt) { return step_one(h, dt, false); }
int chemora_rk3_step(chemora_t* h, double dt) { return step_one(h, dt, true); }
int chemora_rk4_step_group(chemora_t* const* hs, int n, double dt) { return step_group(hs, n, dt, false); }
int chemora_rk3_step_group(chemora_t* const* hs, int n, double dt) { return step_group(hs, n, dt, true); }

int chemora_link_z(chemora_t* h, chemora_t* lower, chemora_t* upper) {
  if (!h) return CHEMORA_EINVAL;
  if ((lower || upper) && h->boundary != CHEMORA_BC_PERIODIC)
    return fail(h, CHEMORA_ESTATE, "a block with radiative boundaries cannot be z-linked");
  for (chemora_t* nb : {lower, upper}) {
    if (!nb) continue;
    if (nb->L.nx != h->L.nx || nb->L.ny != h->L.ny || nb->L.g != h->L.g || nb->system != h->system ||
        nb->order != h->order || nb->dx != h->dx)
      return fail(h, CHEMORA_EINVAL, "a z-neighbour has the same nx, ny, ghost width, system, order and spacing");
    if (nb->stream != h->stream) return fail(h, CHEMORA_EINVAL, "z-neighbours share the block's stream");
  }
  h->nb_lo = lower;
  h->nb_hi = upper;
  return CHEMORA_OK;
}

int chemora_set_boundary(chemora_t* h, int kind) {
  if (!h) return CHEMORA_EINVAL;
  if (kind != CHEMORA_BC_PERIODIC && kind != CHEMORA_BC_RADIATIVE) return fail(h, CHEMORA_EINVAL, "unknown boundary kind");
  if (kind == CHEMORA_BC_RADIATIVE && (h->nb_lo || h->nb_hi))
    return fail(h, CHEMORA_ESTATE, "a z-linked block cannot have radiative boundaries");
  if (kind == CHEMORA_BC_RADIATIVE && h->L.g < 2) return fail(h, CHEMORA_EINVAL, "radiative boundaries need ghost >= 2");
  h->boundary = kind;
  return CHEMORA_OK;
}

int chemora_get_boundary(const chemora_t* h, int* kind) {
  if (!h || !kind) return CHEMORA_EINVAL;
  *kind = h->boundary;
  return CHEMORA_OK;
}

int chemora_radiative_rhs(chemora_t* h, const double* dev_state, double* dev_rhs) {
  if (!h || !dev_state || !dev_rhs || dev_state == dev_rhs) return CHEMORA_EINVAL;
  if (h->L.g < 2) return fail(h, CHEMORA_EINVAL, "radiative boundaries need ghost >= 2");
  Stage st{dev_state, nullptr, nullptr, dev_rhs, 0.0, MODE_RHS};
  return radiative(h, st);
}

// the whole padded block as one packed array [V][nz+2g][ny+2g][nx+2g]: the pack kernel on a layout whose "interior" is
// the padded block (ghost width 0, first column xo - g)
static Layout ghosted_layout(const chemora_t* h) {
  Layout G = h->L;
  G.nx += 2 * G.g; G.ny += 2 * G.g; G.nz += 2 * G.g;
  G.xo -= G.g;
  G.g = 0;
  return G;
}

int chemora_set_state_ghosted(chemora_t* h, const double* host_ghosted) {
  if (!h || !host_ghosted) return CHEMORA_EINVAL;
  int rc = ensure_staging(h);
  if (rc) return rc;
  const Layout G = ghosted_layout(h);
  const size_t n = (size_t)G.nvars * G.nx * G.ny * G.nz;
  CK(h, cudaMemcpyAsync(h->staging, host_ghosted, n * sizeof(double), cudaMemcpyHostToDevice, h->stream), "H2D copy");
  CK(h, launch_pack(G, h->staging, h->buf[0], true, h->stream), "unpack launch");
  h->launches += 1;
  return chemora_synchronize(h);
}

int chemora_get_state_ghosted(chemora_t* h, double* host_ghosted) {
  if (!h || !host_ghosted) return CHEMORA_EINVAL;
  int rc = ensure_staging(h);
  if (rc) return rc;
  const Layout G = ghosted_layout(h);
  const size_t n = (size_t)G.nvars * G.nx * G.ny * G.nz;
  CK(h, launch_pack(G, h->staging, h->buf[0], false, h->stream), "pack launch");
  h->launches += 1;
  CK(h, cudaMemcpyAsync(host_ghosted, h->staging, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream), "D2H copy");
  return chemora_synchronize(h);
}

int chemora_enforce_constraints(chemora_t* h, double* dev_state) {
  if (!h) return CHEMORA_EINVAL;
  if (h->system != CHEMORA_SYS_BSSN) return fail(h, CHEMORA_EINVAL, "constraint enforcement is defined for the BSSN system only");
  CK(h, launch_enforce(h->L, dev_state ? dev_state : h->buf[0], h->stream), "constraint enforcement launch");
  h->launches += 1;
  return CHEMORA_OK;
}

int chemora_energy(chemora_t* h, const double* dev_state, double* dev_eps, double* host_sum) {
  if (!h) return CHEMORA_EINVAL;
  if (h->system != CHEMORA_SYS_WAVE1) return fail(h, CHEMORA_EINVAL, "the energy calculation belongs to the first-order wave system");
  int rc = ensure_staging(h);   // first 8 bytes of the staging buffer hold the sum
  if (rc) return rc;
  CK(h, cudaMemsetAsync(h->staging, 0, sizeof(double), h->stream), "energy memset");
  CK(h, launch_energy(h->L, dev_state ? dev_state : h->buf[0], dev_eps, h->staging, h->stream), "energy launch");
  h->launches += 1;
  if (host_sum) {
    CK(h, cudaMemcpyAsync(host_sum, h->staging, sizeof(double), cudaMemcpyDeviceToHost, h->stream), "energy D2H");
    CK(h, cudaStreamSynchronize(h->stream), "energy sync");
  }
  return CHEMORA_OK;
}

int chemora_set_variant(chemora_t* h, int fused, int tile_id) {
  if (!h || tile_id < 0 || tile_id >= CHEMORA_NUM_TILES || (fused != 0 && fused != 1)) return CHEMORA_EINVAL;
  if (!fused && h->system != CHEMORA_SYS_BSSN) return fail(h, CHEMORA_EINVAL, "wave systems have no split variant");
  if (!chemora_variant_available(h->system, h->order, fused, tile_id))
    return fail(h, CHEMORA_EINVAL, "no such kernel variant for this system and order (chemora_variant_available)");
  h->fused = fused;
  h->tile = tile_id;
  return CHEMORA_OK;
}

int chemora_variant_available(int system_id, int fd_order, int fused, int tile_id) {
  if (tile_id < 0 || tile_id >= CHEMORA_NUM_TILES || (fd_order != 4 && fd_order != 8)) return 0;
  if (system_id == CHEMORA_SYS_WAVE || system_id == CHEMORA_SYS_WAVE1) return fused == 1;   // ids 6..8: plane-ring kernel
  if (system_id != CHEMORA_SYS_BSSN) return 0;
  if (fused == 0) return tile_id < 6;                      // six split tiles, both orders
  if (fused != 1) return 0;
  return fd_order == 8 ? tile_id == 0 : tile_id < kNumFused;
}

int chemora_get_variant(const chemora_t* h, int* fused, int* tile_id) {
  if (!h) return CHEMORA_EINVAL;
  if (fused) *fused = h->fused;
  if (tile_id) *tile_id = h->tile;
  return CHEMORA_OK;
}

int chemora_tile_shape(int system_id, int fused, int tile_id, int* tx, int* ty, int* tz) {
  if (tile_id < 0 || tile_id >= CHEMORA_NUM_TILES) return CHEMORA_EINVAL;
  const bool f = system_id == CHEMORA_SYS_BSSN && fused;
  if (f && tile_id >= kNumFused) return CHEMORA_EINVAL;
  const TileShape T = f ? kTilesFused[tile_id]
                      : (system_id == CHEMORA_SYS_WAVE && tile_id >= 6 && tile_id < 9) ? kTilesWaveTma[tile_id - 6]
                      : (system_id == CHEMORA_SYS_WAVE1 && tile_id >= 6 && tile_id < 9) ? kTilesWave1Tma[tile_id - 6]
                                                                                        : kTilesMarch[tile_id % 6];
  if (tx) *tx = T.tx;
  if (ty) *ty = T.ty;
  if (tz) *tz = T.tz;
  return CHEMORA_OK;
}

// The paper's tile cost model for the uniform fused BSSN kernel; see include/chemora.h.
int chemora_tile_cost(int fd_order, int ghost, int tile_id, double* sigma, long* requests, long* points) {
  if (fd_order != 4 && fd_order != 8) return CHEMORA_EINVAL;
  if (tile_id < 0 || tile_id >= 5) return CHEMORA_EINVAL;   // the five tile shapes of the plain section layout
  if (fd_order == 8 && tile_id != 0) return CHEMORA_EINVAL;
  const int H = fd_order / 2 + 1;
  if (ghost < H) return CHEMORA_EINVAL;
  const TileShape T = kTilesFused[tile_id];
  const int xo = ((ghost - 3) & 1) ? ghost + 1 : ghost;   // the layout rule of chemora_create
  // 32-byte sectors (4 doubles) covered by `len` doubles from column x0 of a row (rows start 128-byte aligned)
  auto sectors = [](long x0, long len) { return (x0 + len - 1) / 4 - x0 / 4 + 1; };
  const long V = 25, rows_box = (long)(T.ty + 2 * H) * (T.tz + 2 * H), rows_tile = (long)T.ty * T.tz;
  const long r = V * rows_box * sectors(xo - H, T.tx + 2 * H)           // the halo boxes of the 25 variables
                 + 21 * rows_tile * sectors(xo - 1, T.tx + 2)           // point values needed ahead of their boxes
                 + 2 * V * rows_tile * sectors(xo - 1, T.tx + 2)        // Runge-Kutta operands U, S
                 + 2 * V * rows_tile * sectors(xo, T.tx);               // stores S, Y
  const long n = (long)T.tx * T.ty * T.tz;   // I = 1: one point per thread
  if (requests) *requests = r;
  if (points) *points = n;
  if (sigma) *sigma = ((double)r / (double)n) * (1.0 + 256.0 / (double)n);
  return CHEMORA_OK;
}

int chemora_autotune(chemora_t* h, int* fused_out, int* tile_out, float* ms_out) {
  if (!h) return CHEMORA_EINVAL;
  const int save_f = h->fused, save_t = h->tile;
  if (ms_out) for (int n = 0; n < 2 * CHEMORA_NUM_TILES; ++n) ms_out[n] = -1.f;
  float best = -1.f;
  int bf = save_f, bt = save_t;
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  for (int n = 0; n < 4; ++n)
    if (cudaEventCreate(&ev[n]) != cudaSuccess) {
      for (int m = 0; m < n; ++m) cudaEventDestroy(ev[m]);
      return cuda_fail(h, cudaGetLastError(), "event create");
    }
  int rc = fill(h, h->buf[0]);
  bool have_ref = false;
  // fused variants always; the derivative-split variant (about 18 GB of scratch at 256^3, never the pick in any
  // measured sweep) only when the tuning parameter "autotune_split" is 1
  for (int f = 1; f >= (h->autotune_split ? 0 : 1) && !rc; --f)
    for (int t = 0; t < CHEMORA_NUM_TILES && !rc; ++t) {
      if (!chemora_variant_available(h->system, h->order, f, t)) continue;
      if (f == 1 && t >= h->autotune_fused_ids) continue;                  // candidates bounded by the caller: ms stays -1
      h->fused = f; h->tile = t;
      // a middle RK4 stage (the common case) on scratch operands: k = f(U); S += 2k; Ya = U + a k.
      // S and Ya are scratch between steps (stage 1 overwrites them); U is only read.
      Stage st{h->buf[0], h->buf[0], h->buf[3], h->buf[1], 1e-3, MODE_MID};
      int vrc = run_rhs(h, st);                                            // warm-up
      for (int n = 0; n < 3 && !vrc; ++n) {                                // three timed runs, the median counts
        cudaEventRecord(ev[n], h->stream);
        vrc = run_rhs(h, st);
      }
      if (vrc == CHEMORA_ENOMEM || vrc == CHEMORA_EINVAL) continue;        // variant not usable here: ms stays -1
      if (vrc) { rc = vrc; break; }
      cudaEventRecord(ev[3], h->stream);
      if (cudaEventSynchronize(ev[3]) != cudaSuccess) { rc = cuda_fail(h, cudaGetLastError(), "autotune sync"); break; }
      // Guard (the paper's run-time path loads kernels it has just generated; here: a variant
      // is only eligible if it computes what the reference variant computes).  The fused BSSN tile ids evaluate
      // the same right-hand side (two-pass or one-pass mixed derivatives: rounding differs, nothing else), so their
      // Ya = U + a k must agree with the first one's -- kept in Yb, scratch between steps -- to 1e-11 in the norm
      // of reading S11, per variable.  A variant that disagrees, or whose bounded waits gave up, is disqualified.
      if (f == 1 && h->system == CHEMORA_SYS_BSSN) {
        const int V = h->L.nvars;
        unsigned long long* dnorm = reinterpret_cast<unsigned long long*>(h->dev_err) + 2;   // [2 V] after the error words
        unsigned long long host[2 + 2 * 25];
        cudaError_t ge = cudaSuccess;
        if (!have_ref) {
          ge = cudaMemcpyAsync(h->buf[2], h->buf[1], (size_t)V * h->L.vstride * sizeof(double), cudaMemcpyDeviceToDevice, h->stream);
        } else {
          ge = cudaMemsetAsync(dnorm, 0, 2 * V * sizeof(unsigned long long), h->stream);
          if (ge == cudaSuccess) ge = launch_maxdiff(h->buf[1], h->buf[2], h->L.vstride, V, dnorm, h->stream);
          h->launches += 1;
        }
        if (ge == cudaSuccess) ge = cudaMemcpyAsync(host, h->dev_err, sizeof host, cudaMemcpyDeviceToHost, h->stream);
        if (ge == cudaSuccess) ge = cudaStreamSynchronize(h->stream);
        if (ge != cudaSuccess) { rc = cuda_fail(h, ge, "autotune guard"); break; }
        if ((unsigned)host[0] != 0) {            // a wait timed out inside this variant: clear the word, disqualify
          cudaMemsetAsync(h->dev_err, 0, sizeof(unsigned), h->stream);
          if (ms_out) ms_out[f * CHEMORA_NUM_TILES + t] = -3.f;
          continue;
        }
        bool agree = true;
        for (int v = 0; have_ref && v < V; ++v) {
          double d, m;
          memcpy(&d, &host[2 + 2 * v], sizeof d);
          memcpy(&m, &host[2 + 2 * v + 1], sizeof m);
          if (!(d <= 1e-11 * m)) agree = false;
        }
        if (!agree) {
          if (ms_out) ms_out[f * CHEMORA_NUM_TILES + t] = -2.f;
          continue;
        }
        have_ref = true;
      }
      float m[3];
      for (int n = 0; n < 3; ++n) cudaEventElapsedTime(&m[n], ev[n], ev[n + 1]);
      const float lo = fminf(m[0], fminf(m[1], m[2])), hi = fmaxf(m[0], fmaxf(m[1], m[2]));
      const float ms = m[0] + m[1] + m[2] - lo - hi;
      if (best < 0.f || ms < best) { best = ms; bf = f; bt = t; }
      if (ms_out) ms_out[f * CHEMORA_NUM_TILES + t] = ms;
    }
  // Second axis for the fused BSSN kernel: the y-extent of the columns in which it visits its tiles ("col_rows";
  // decides how much of a box's halo is still in L2 when the neighbouring tile asks for it).  Any value computes the
  // same result; the picked variant is timed with half and twice the current extent and the fastest one stays.
  if (!rc && best > 0.f && bf == 1 && h->system == CHEMORA_SYS_BSSN) {
    const int base = h->L.col_rows;
    int keep = base;
    h->fused = bf; h->tile = bt;
    Stage st{h->buf[0], h->buf[0], h->buf[3], h->buf[1], 1e-3, MODE_MID};
    for (int cand : {base / 2, base * 2}) {
      if (cand < 2 || cand > 4 * h->L.ny) continue;
      h->L.col_rows = cand;
      int vrc = run_rhs(h, st);
      for (int n = 0; n < 3 && !vrc; ++n) { cudaEventRecord(ev[n], h->stream); vrc = run_rhs(h, st); }
      if (vrc) { rc = vrc; break; }
      cudaEventRecord(ev[3], h->stream);
      if (cudaEventSynchronize(ev[3]) != cudaSuccess) { rc = cuda_fail(h, cudaGetLastError(), "autotune sync"); break; }
      float m[3];
      for (int n = 0; n < 3; ++n) cudaEventElapsedTime(&m[n], ev[n], ev[n + 1]);
      const float ms = m[0] + m[1] + m[2] - fminf(m[0], fminf(m[1], m[2])) - fmaxf(m[0], fmaxf(m[1], m[2]));
      if (ms < 0.98f * best) { best = ms; keep = cand; }   // a change must pay at least 2 %
    }
    h->L.col_rows = keep;
  }
  for (int n = 0; n < 4; ++n) cudaEventDestroy(ev[n]);
  h->fused = rc ? save_f : bf;
  h->tile = rc ? save_t : bt;
  if (fused_out) *fused_out = h->fused;
  if (tile_out) *tile_out = h->tile;
  return rc;
}

int chemora_measure_box_fill(chemora_t* h, int tile_id, float* ms) {
  if (!h || !ms) return CHEMORA_EINVAL;
  if (h->system != CHEMORA_SYS_BSSN || h->order != 4 || !chemora_variant_available(h->system, h->order, 1, tile_id))
    return fail(h, CHEMORA_EINVAL, "the fill-only mode exists for the fused 4th-order BSSN tile ids");
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  for (int n = 0; n < 4; ++n)
    if (cudaEventCreate(&ev[n]) != cudaSuccess) {
      for (int m = 0; m < n; ++m) cudaEventDestroy(ev[m]);
      return cuda_fail(h, cudaGetLastError(), "event create");
    }
  int rc = fill(h, h->buf[0]);
  // what a middle RK4 stage loads: boxes of U, operand tiles of U and S; nothing is written
  Stage st{h->buf[0], h->buf[0], h->buf[3], h->buf[1], 1e-3, MODE_MID};
  const Coef C = make_coef(h);
  cudaError_t e = rc ? cudaSuccess : launch_bssn_fill(h->L, C, tile_id, st, h->stream);   // warm-up
  for (int n = 0; n < 3 && !rc && e == cudaSuccess; ++n) {
    cudaEventRecord(ev[n], h->stream);
    e = launch_bssn_fill(h->L, C, tile_id, st, h->stream);
  }
  if (!rc && e != cudaSuccess) rc = cuda_fail(h, e, "fill-only kernel launch");
  if (!rc) {
    h->launches += 4;
    cudaEventRecord(ev[3], h->stream);
    if (cudaEventSynchronize(ev[3]) != cudaSuccess) rc = cuda_fail(h, cudaGetLastError(), "fill-only sync");
  }
  if (!rc) {
    float m[3];
    for (int n = 0; n < 3; ++n) cudaEventElapsedTime(&m[n], ev[n], ev[n + 1]);
    *ms = m[0] + m[1] + m[2] - fminf(m[0], fminf(m[1], m[2])) - fmaxf(m[0], fmaxf(m[1], m[2]));
  }
  for (int n = 0; n < 4; ++n) cudaEventDestroy(ev[n]);
  return rc ? rc : chemora_synchronize(h);
}

long chemora_launch_count(const chemora_t* h) { return h ? h->launches : 0; }

static void drop_events(chemora_t* h) {
  for (int c = 0; c < 2; ++c) {
    for (cudaEvent_t e : h->ev[c]) cudaEventDestroy(e);
    h->ev[c].clear();
    h->ev_used[c] = 0;
    h->ev_ms[c] = 0.0;
    h->ev_launches[c] = 0;
  }
}

int chemora_timing(chemora_t* h, int enable) {
  if (!h) return CHEMORA_EINVAL;
  h->timing = false;
  drop_events(h);
  if (!enable) return CHEMORA_OK;
  for (int c = 0; c < 2; ++c)
    for (int i = 0; i < kEvPool; ++i) {
      cudaEvent_t e;
      if (cudaEventCreate(&e) != cudaSuccess) {
        drop_events(h);
        return cuda_fail(h, cudaGetLastError(), "event create");
      }
      h->ev[c].push_back(e);
    }
  h->timing = true;
  return CHEMORA_OK;
}

int chemora_timing_read(chemora_t* h, double* rhs_ms, long* rhs_launches, double* fill_ms, long* fill_launches) {
  if (!h) return CHEMORA_EINVAL;
  CK(h, cudaStreamSynchronize(h->stream), "timing sync");
  for (int c = 0; c < 2; ++c) drain(h, c);
  if (rhs_ms) *rhs_ms = h->ev_ms[0];
  if (fill_ms) *fill_ms = h->ev_ms[1];
  if (rhs_launches) *rhs_launches = h->ev_launches[0];
  if (fill_launches) *fill_launches = h->ev_launches[1];
  return CHEMORA_OK;
}

int chemora_kernel_info(const chemora_t* h, int* regs, int* local_bytes, int* smem_bytes) {
  if (!h) return CHEMORA_EINVAL;
  cudaFuncAttributes a;
  cudaError_t e = h->system == CHEMORA_SYS_WAVE && h->tile >= 6 && h->tile < 9 ? kernel_info_wave_tma(h->order, h->tile - 6, &a)
                  : h->system == CHEMORA_SYS_WAVE ? kernel_info_wave(h->order, h->tile % 6, &a)
                  : h->system == CHEMORA_SYS_WAVE1 && h->tile >= 6 && h->tile < 9 &&
                            wave1_tma_ok(h->L, h->order, true, h->tile - 6)
                      ? kernel_info_wave1_tma(h->order, h->tile - 6, &a)
                  : h->system == CHEMORA_SYS_WAVE1 ? kernel_info_wave1(h->order, h->tile % 6, &a)
                  : !h->fused              ? kernel_info_bssn_split(1, h->tile % 6, &a)
                                           : kernel_info_bssn_fused(h->order, h->tile, &a);
  if (e != cudaSuccess) return cuda_fail(const_cast<chemora_t*>(h), e, "cudaFuncGetAttributes");
  if (regs) *regs = a.numRegs;
  if (local_bytes) *local_bytes = (int)a.localSizeBytes;
  if (smem_bytes) *smem_bytes = (int)a.sharedSizeBytes;
  return CHEMORA_OK;
}

int chemora_measure_fp64_peak(chemora_t* h, double* gflops) {
  if (!h || !gflops) return CHEMORA_EINVAL;
  int dev = 0, sms = 0;
  CK(h, cudaGetDevice(&dev), "get device");
  CK(h, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "get SM count");
  const int blocks = sms * 8, threads = 256, iters = 1 << 15;
  cudaEvent_t e0, e1;
  CK(h, cudaEventCreate(&e0), "event create");
  CK(h, cudaEventCreate(&e1), "event create");
  double* sink = h->buf[3];
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, h->stream);
    cudaError_t e = launch_dfma_peak(blocks, threads, iters, sink, h->stream);
    cudaEventRecord(e1, h->stream);
    if (e != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess) {
      cudaEventDestroy(e0); cudaEventDestroy(e1);
      return cuda_fail(h, e != cudaSuccess ? e : cudaGetLastError(), "fp64 probe");
    }
    float ms;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
    h->launches += 1;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *gflops = (double)blocks * threads * iters * 8.0 * 2.0 / (best * 1e-3) / 1e9;
  return CHEMORA_OK;
}

const char* chemora_last_error(const chemora_t* h) { return h ? h->err.c_str() : "null handle"; }

int chemora_destroy(chemora_t* h) {
  if (!h) return CHEMORA_OK;
  cudaStreamSynchronize(h->stream);
  drop_events(h);
  for (int b = 0; b < 4; ++b) dev_free(h, h->buf[b]);
  dev_free(h, h->derivs);
  dev_free(h, h->staging);
  dev_free(h, h->dev_err);
  delete h;
  return CHEMORA_OK;
}

}  // extern "C"
