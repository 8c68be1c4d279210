/* chemora.h -- C ABI of libchemora.so: the B200-native (sm_100a, fp64) method-of-lines right-hand-side
 * path of the codes the Chemora framework generates (arXiv:1307.6488).
 *
 * What the path is (citations are PAPER.md lines): a "calculation" applied to all grid points of a
 * block-structured grid (:133, :187, :218-220) -- high-order finite differences (:9, :194, :338) followed by
 * the pointwise right-hand-side expression -- driven by a method-of-lines integrator (:338, :408) with a
 * ghost-zone synchronisation before every evaluation (:105, :354, :382).  The paper prints no equations or
 * coefficients; DESIGN.md "Readings" (S1-S14) fixes them.
 *
 * Conventions
 *  - All functions return int: 0 = CHEMORA_OK, negative = error (below).  No exceptions cross the ABI.
 *    chemora_last_error() gives a handle-owned, NUL-terminated message for the last failing call.
 *  - A handle is used from one host thread at a time.  All device work is enqueued on the stream given at
 *    creation and is asynchronous with respect to the host unless stated otherwise.
 *  - "dev" pointers are CUDA device pointers, "host" pointers ordinary host memory.
 *  - Device state layout (SoA): V variables; each variable is tot_z x tot_y rows of
 *    `pitch` doubles (pitch = roundup(xo + nx + g, 16): 128-byte rows), x fastest; variable stride
 *    var_stride = pitch*tot_y*tot_z; buffers are 128-byte aligned.  Interior point (i,j,k) of variable v is
 *    at  v*var_stride + ((k+g)*tot_y + (j+g))*pitch + (i+xo), where xo = g except for BSSN with even g,
 *    where xo = g+1 (keeps the fused kernel's TMA halo boxes 16-byte aligned).  Always take the offsets
 *    from chemora_layout (interior_offset = (g*tot_y + g)*pitch + xo).
 *  - Packed host layout: V x nz x ny x nx doubles, x fastest, no ghosts.
 *  - There is no CPU fallback: every entry point that computes needs a CUDA device and fails with
 *    CHEMORA_ECUDA otherwise.
 */
#ifndef CHEMORA_H
#define CHEMORA_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct chemora chemora_t; /* opaque, owned by the library */

enum { CHEMORA_OK = 0, CHEMORA_EINVAL = -1, CHEMORA_ENOMEM = -2, CHEMORA_ECUDA = -3, CHEMORA_ESTATE = -4 };

/* system_id.  WAVE: (phi, pi), d_t phi = pi, d_t pi = delta^ij d_i d_j phi (reading S1; PAPER.md:152-169 is
 * the paper's own wave example).  BSSN: 25 variables, chi-variant vacuum BSSN with 1+log
 * lapse and Gamma-driver shift (readings S3-S6), slots: chi, gt11 gt12 gt13 gt22 gt23 gt33, trK,
 * At11..At33, Gt1..3, alpha, beta1..3, B1..3, A.  WAVE1: the paper's Sample 1 itself, the wave
 * equation in fully first-order form, 5 variables (u, rho, v_1, v_2, v_3): D_t u = rho, D_t rho = delta^ij D_i v_j,
 * D_t v_i = D_i rho, with centred first derivatives of order fd_order (needs ghost >= fd_order/2). */
enum { CHEMORA_SYS_WAVE = 0, CHEMORA_SYS_BSSN = 1, CHEMORA_SYS_WAVE1 = 2 };

/* boundary kind of a block (chemora_set_boundary): periodic ghost fill (reading S8, the default) or radiative outer
 * boundary (reading S16) */
enum { CHEMORA_BC_PERIODIC = 0, CHEMORA_BC_RADIATIVE = 1 };

/* which buffer of the four RK4 buffers (reading S9) */
enum { CHEMORA_BUF_U = 0, CHEMORA_BUF_YA = 1, CHEMORA_BUF_YB = 2, CHEMORA_BUF_S = 3 };

/* kernel variant axes (PAPER.md:215-216 fused vs derivative-split; :248-266 tile shape) */
enum { CHEMORA_NUM_TILES = 9 };

/* Create a handle for an nx x ny x nz interior block with `ghost` ghost layers per face, centred FD order
 * fd_order (4 or 8), system system_id and grid spacing dx (same in x, y, z).
 * Rejects (CHEMORA_EINVAL): non-positive dims, dims < ghost (periodic images would overlap),
 * fd_order not in {4,8}, ghost < fd_order/2 (wave), ghost < fd_order/2 + 1 (BSSN: upwinded advection,
 * 5 ghost zones at 8th order, the paper's configuration), dx <= 0.  For 8th-order BSSN the fused kernel
 * exists for tile id 0 only (other fused ids are rejected by chemora_set_variant); all six split tiles work.  Dissipation (eps_diss != 0, KO order 5)
 * needs ghost >= 3; that is checked when the parameter is set and again at launch.
 * cuda_stream: a cudaStream_t (may be NULL = default stream).
 * alloc/dealloc: optional device allocator callbacks (e.g. torch's caching allocator); alloc(bytes, ctx)
 * returns a device pointer aligned to >= 128 bytes or NULL.  NULL callbacks -> cudaMalloc/cudaFree.
 * The library owns the four state buffers (+ derivative scratch of the split variant) until destroy. */
int chemora_create(chemora_t** out, int nx, int ny, int nz, int ghost, int fd_order, int system_id, double dx,
                   void* cuda_stream, void* (*alloc)(size_t, void*), void (*dealloc)(void*, void*),
                   void* alloc_ctx);

/* Named parameters: "eps_diss" (KO strength, default 0), "eta" (default 1), "shift_gamma_coeff"
 * (default 0.75), "ko_order" (5, the default, or 9: the 11-point operator (eps/1024h) h^10 (D+D-)^5 that goes
 * with the paper's 8th-order, 5-ghost-zone configuration; accepted for the 8th-order BSSN
 * system only); tuning: "col_rows" (default 32: y-extent in grid rows of the columns in which the fused BSSN
 * kernel visits its tiles, chosen so the halo planes shared by z-neighbour tiles stay in L2), "autotune_split"
 * (default 0; 1: chemora_autotune also times the derivative-split variant, which allocates its derivative scratch),
 * "autotune_fused_ids" (default CHEMORA_NUM_TILES; 1..CHEMORA_NUM_TILES: chemora_autotune times only the fused tile
 * ids below this bound, e.g. 5 = the five tile shapes of the plain section layout).
 * Unknown name or invalid value -> CHEMORA_EINVAL. */
int chemora_set_param(chemora_t* h, const char* name, double value);

/* The paper's tile cost model re-targeted at this design, for the uniform fused BSSN kernel
 * (fused tile ids 0..4; 8th order: id 0).  Host arithmetic only, no device needed.
 *   requests r = the 32-byte L2 sectors one interior tile of a middle RK4 stage requests: the (tx+2H)(ty+2H)(tz+2H)
 *     halo boxes of the 25 variables (H = fd_order/2 + 1), the point-value and Runge-Kutta operand boxes
 *     ((tx+2) x ty x tz, 21 + 2*25 of them) and the 2*25 stored tiles, every row counted with its alignment in
 *     the padded layout ("all lines survive" is exact here: each sector is staged once per tile);
 *   points = I tx ty tz with I = 1 iteration per thread;
 *   sigma = (r / points) * (1 + 256 / (tx ty tz)): the request size per grid point, divided by the paper's
 *     empirical efficiency 1 / (1 + 256/(tx ty tz)) of small tiles (reading S15: the printed formula
 *     divides by (1 + 256/...), which would favour small tiles against the sentence that introduces it).
 * Any out pointer may be NULL.  CHEMORA_EINVAL for ids the model does not cover. */
int chemora_tile_cost(int fd_order, int ghost, int tile_id, double* sigma, long* requests, long* points);
int chemora_get_param(const chemora_t* h, const char* name, double* value);

/* Layout in units of doubles; any out pointer may be NULL.  interior_offset = offset of interior (0,0,0)
 * inside one variable. */
int chemora_layout(const chemora_t* h, int* nvars, long* pitch, long* tot_y, long* tot_z, long* var_stride,
                   long* interior_offset);

/* Borrowed device pointer to one of the four buffers (valid until destroy). */
int chemora_state_ptr(chemora_t* h, int which, double** dev);

/* Copy a packed host state into U's interior / U's interior out to the host.  Synchronous (the stream is
 * synchronised before returning).  Ghosts of U are left untouched by set_state. */
int chemora_set_state(chemora_t* h, const double* host_packed);
int chemora_get_state(chemora_t* h, double* host_packed);
/* The same two copies without the final synchronisation, for pipelining independent handles on different
 * streams (one handle's copies run under another's kernels): host_packed should be page-locked (with pageable
 * memory the copy degrades to a synchronous one), must stay valid and, for set, unmodified until
 * chemora_synchronize(h) returns; each handle stages through its own device buffer, so a handle has at most one
 * such copy in flight per direction between two synchronisations of the same kind.  chemora_synchronize waits
 * for everything queued on the handle's stream and returns the first asynchronous error, if any. */
int chemora_set_state_async(chemora_t* h, const double* host_packed);
int chemora_get_state_async(chemora_t* h, double* host_packed);
int chemora_synchronize(chemora_t* h);
/* Same for a device buffer in the padded layout: pack/unpack between a DEVICE packed array and U
 * (asynchronous on the stream; used by the device-resident benchmark path). */
int chemora_set_state_dev(chemora_t* h, const double* dev_packed);
int chemora_get_state_dev(chemora_t* h, double* dev_packed);

/* Periodic ghost-zone fill of all V variables of a device state in the padded layout (reading S8):
 * ghost (i,j,k) <- interior (i mod nx, j mod ny, k mod nz), faces, edges and corners.  In place. */
int chemora_fill_ghosts(chemora_t* h, double* dev_state);

/* dev_rhs interior <- RHS(dev_state); ghosts of dev_state must be filled; ghosts of dev_rhs untouched.
 * Both in the padded layout; must not alias.  Uses the current variant. */
int chemora_rhs(chemora_t* h, const double* dev_state, double* dev_rhs);

/* U <- U(t + dt): classical RK4 with the association of reading S9; fills ghosts itself before each of
 * the four RHS evaluations; asynchronous on the stream. */
int chemora_rk4_step(chemora_t* h, double dt);

/* U <- U(t + dt) with the third-order Shu-Osher Runge-Kutta scheme (reading S9b; the paper's own runs use RK3,
 * PAPER.md:338): U1 = U + dt f(U); U2 = 3/4 U + 1/4 (U1 + dt f(U1)); U+ = 1/3 U + 2/3 (U2 + dt f(U2)); ghost fill
 * before each of the three RHS evaluations; uses buffers U, YA, YB; asynchronous on the stream. */
int chemora_rk3_step(chemora_t* h, double dt);

/* Multi-block interface, the second boundary kind (the paper's domains are sets of blocks whose ghost zones are
 * synchronised from their neighbours): slab decomposition along z.  After
 * chemora_link_z(h, lower, upper) the ghost z-planes of block h are copied from the top `ghost` interior planes of
 * `lower` and the bottom `ghost` interior planes of `upper` (the same one of the four buffers), x and y stay
 * periodic; NULL = the block's own periodic image on that side.  Neighbours have the same nx, ny, ghost width,
 * system, order, spacing and stream (else CHEMORA_EINVAL) and their own nz >= ghost.  The library keeps the
 * pointers: unlink (NULL, NULL) before destroying a neighbour.
 * Linked blocks step together: chemora_rk4_step_group / chemora_rk3_step_group run, stage by stage, every block's
 * ghost fill and then every block's right-hand side (n <= 64 blocks, all links inside the group, one stream);
 * chemora_rk4_step / chemora_rk3_step / chemora_fill_ghosts of a foreign buffer return CHEMORA_ESTATE on a linked
 * block.  A ring of blocks linked periodically gives bit for bit the single-block result. */
int chemora_link_z(chemora_t* h, chemora_t* lower, chemora_t* upper);
int chemora_rk4_step_group(chemora_t* const* blocks, int n, double dt);
int chemora_rk3_step_group(chemora_t* const* blocks, int n, double dt);

/* Radiative (Sommerfeld) outer boundary, the outer-face half of the second boundary kind (the paper's
 * blocks have outer faces as well as inter-block faces, and it prints no boundary condition:
 * DESIGN.md reading S16).  With CHEMORA_BC_RADIATIVE the g ghost layers of the block are evolved BOUNDARY POINTS:
 * chemora_rk4_step / chemora_rk3_step fill nothing and run, after every interior right-hand side, a face kernel that
 * applies  d_t u = -[ n^i D_i u + (u - u_inf)/r ]  (n^i = x^i/r, block centred on the origin, x^i = (i - (N_i-1)/2) dx,
 * u_inf = 1 on chi, gt11, gt22, gt33, alpha of the BSSN system and 0 elsewhere, D_i second order: centred, one-sided
 * three-point at the two ends of the padded array) with the same Runge-Kutta stage update.  Needs ghost >= 2; not
 * combinable with chemora_link_z (CHEMORA_ESTATE).  The caller provides the boundary-point values of the initial state
 * (chemora_set_state_ghosted, or chemora_fill_ghosts once after chemora_set_state).
 * chemora_radiative_rhs: dev_rhs boundary points <- the radiative right-hand side of dev_state (interior untouched).
 * chemora_set_state_ghosted / chemora_get_state_ghosted: U's whole padded block as one packed host array
 * V x (nz+2g) x (ny+2g) x (nx+2g), x fastest.  Synchronous. */
int chemora_set_boundary(chemora_t* h, int kind);
int chemora_get_boundary(const chemora_t* h, int* kind);
int chemora_radiative_rhs(chemora_t* h, const double* dev_state, double* dev_rhs);
int chemora_set_state_ghosted(chemora_t* h, const double* host_ghosted);
int chemora_get_state_ghosted(chemora_t* h, double* host_ghosted);

/* Algebraic constraint enforcement on the interior of a BSSN state in the padded layout (dev_state == NULL: U):
 * gt_ij <- gt_ij + gt_ij (det(gt)^(-1/3) - 1), the bracket evaluated as expm1(-log(det)/3) and det in a fixed
 * association without FMA contraction (reading S10b: mathematically gt_ij / det^(1/3); this form rounds the O(1)
 * values identically in any implementation), then At_ij <- At_ij - 1/3 gt_ij gtu^kl At_kl with the new metric.
 * In place, asynchronous.
 * CHEMORA_EINVAL for the wave systems. */
int chemora_enforce_constraints(chemora_t* h, double* dev_state);

/* The "Energy" calculation of the paper's Sample 1 for the first-order wave system:
 * eps = 1/2 (rho^2 + delta^ij v_i v_j) at every interior point of dev_state (padded layout; NULL: U).
 * dev_eps, if not NULL, receives the field packed nz x ny x nx (device); host_sum, if not NULL, the sum of eps over
 * the grid (then the call synchronises the stream).  CHEMORA_EINVAL for the other systems. */
int chemora_energy(chemora_t* h, const double* dev_state, double* dev_eps, double* host_sum);

/* Kernel variant: fused (1: derivatives + RHS + RK stage update in one kernel) or split (0: derivatives
 * written to global arrays by one kernel, RHS + stage update by a second), and tile_id in
 * [0, CHEMORA_NUM_TILES); chemora_variant_available says (host only, 1/0) which ids exist for a system and order.
 * chemora_tile_shape reports the (x, y, z) extent of a tile id.  Fused BSSN kernel: a 3-D tile with one grid point
 * per thread, staged with an (order/2 + 1)-cell halo by TMA; ids 0..4 = 16x4x4, 16x8x2, 8x4x8, 16x2x8, 16x4x2 at 4th
 * order, id 5 = 16x4x4 with the interleaved section layout (the cheap advection-only stencils evaluated between the
 * expensive sections, box-less emit sections at the end of a tile), id 6 = id 5 with a full
 * variable's own right-hand side emitted before the plane barrier of its mixed derivatives, id 7 = id 6 with a six-slot box ring
 * (a box section of that layout needs two operand tiles, not four: six slots fit the shared memory of five); id 0 only
 * at 8th order.  Split BSSN kernels (ids 0..5) and the L1-path wave kernels (ids 0..5): an x*y thread
 * block marching z planes.  Ids 6..8 of the wave systems: the TMA plane-ring kernel (CHEMORA_SYS_WAVE: 32x16x32,
 * 32x16x64, 64x8x32; CHEMORA_SYS_WAVE1, five variables a plane: 16x8x64, 16x16x64, 32x8x64; runs id - 6 instead
 * when the layout does not give 16-byte aligned plane boxes or the ring of planes does not fit shared memory,
 * as 32x8x64 at 8th order).  chemora_set_variant returns CHEMORA_EINVAL for an id that does not exist. */
int chemora_set_variant(chemora_t* h, int fused, int tile_id);
int chemora_get_variant(const chemora_t* h, int* fused, int* tile_id);
int chemora_variant_available(int system_id, int fd_order, int fused, int tile_id);
int chemora_tile_shape(int system_id, int fused, int tile_id, int* tx, int* ty, int* tz);

/* Runtime sweep (the paper's model-based choice, replaced by measurement): times every available
 * fused tile id below the parameter "autotune_fused_ids" (default: all; and, with the parameter "autotune_split" = 1,
 * the six split tiles) on the handle's own grid -- one
 * middle RK4 stage evaluated on the current U, results into the scratch buffers S and Ya; one warm-up run, then the
 * median of three timed runs -- keeps the fastest, returns it.  A variant that cannot run here (CHEMORA_ENOMEM for
 * its scratch, CHEMORA_EINVAL from its launch check) is skipped, not fatal.  Guard: every fused BSSN tile id evaluates
 * the same right-hand side, so a candidate whose result (Ya) differs from the first fused id's (kept in Yb for the
 * duration of the sweep) by more than 1e-11 in the norm of reading S11, or whose bounded waits gave up, is
 * disqualified: ms_out = -2 / -3.
 * For the fused BSSN kernel the pick is then timed with half and twice the current "col_rows" and the fastest
 * extent is kept (chemora_get_param tells which; results do not depend on it).
 * ms_out, if not NULL, receives 2*CHEMORA_NUM_TILES timings in milliseconds ([fused*NUM_TILES + tile];
 * negative = variant unavailable or not timed).  U is not modified.  Synchronous. */
int chemora_autotune(chemora_t* h, int* fused, int* tile_id, float* ms_out);

/* Launch safety (the paper's run-time path that edits, compiles and loads kernels is its failure surface,
 * PAPER.md:246; here the equivalent is a TMA launch with a bad box or byte count).
 * chemora_selfcheck: host only, no device: builds the launch plan (shared-memory destinations, box extents, x-coordinate
 * parity, mbarrier byte counts, shared-memory total, threads) of EVERY TMA kernel instance in the library for every
 * ghost width and Runge-Kutta mode and validates it with the same checker every launcher runs before <<<>>>.
 * Returns the number of plans checked (> 0), or CHEMORA_EINVAL if one is rejected; buf (may be NULL) gets a one-line
 * report.  A launch whose plan or layout is rejected is never issued: the call returns CHEMORA_ECUDA and
 * chemora_last_error names the rule.
 * Device error word: every wait on a TMA mbarrier inside the kernels is bounded (seconds); a wait that gives up records
 * a code in the handle's device error word and the kernel runs on without the data (memory-safe: no address depends on
 * loaded values).  chemora_synchronize (and chemora_get_state) read the word: non-zero -> CHEMORA_ECUDA, the message
 * from chemora_describe_device_error(code) (host only), and the word is cleared. */
int chemora_selfcheck(char* buf, size_t n);
int chemora_describe_device_error(unsigned code, char* buf, size_t n);

/* Benchmark mode: the cost of moving one launch's data into shared memory.  Runs the fused 4th-order BSSN kernel of
 * tile_id in FILL-ONLY mode on the current U: every TMA box, Runge-Kutta operand tile and point-value tile of a middle
 * RK4 stage is requested, awaited, released and refilled by the code the full kernel uses (same launch plan, same
 * validator), and no arithmetic is done and nothing is written.  *ms = median of three launches after a warm-up.
 * This is the tracked form of the stand-alone probe behind DESIGN.md section 6.5's box-fill floor.  Fills U's ghosts;
 * S and YA are not modified.  CHEMORA_EINVAL for other systems / orders / ids.  Synchronous. */
int chemora_measure_box_fill(chemora_t* h, int tile_id, float* ms);

/* Number of kernel launches issued through this handle so far (for benchmarks' gpu_launches). */
long chemora_launch_count(const chemora_t* h);

/* Per-kernel device timing for benchmarks: chemora_timing(h, 1) starts recording a CUDA-event pair on the
 * handle's stream around every RHS evaluation (all kernels of the current variant) and around every ghost
 * fill, and resets the totals; chemora_timing(h, 0) stops.  chemora_timing_read synchronises the stream
 * and returns the summed durations in milliseconds and the number of kernels launched inside them. */
int chemora_timing(chemora_t* h, int enable);
int chemora_timing_read(chemora_t* h, double* rhs_ms, long* rhs_launches, double* fill_ms, long* fill_launches);

/* Static kernel resource usage of the current variant's main kernel (from cudaFuncGetAttributes):
 * registers per thread, local (spill) bytes per thread, static+dynamic shared bytes per block. */
int chemora_kernel_info(const chemora_t* h, int* regs, int* local_bytes, int* smem_bytes);

/* Sustained FP64 FMA rate of the device in GFLOP/s (register-resident DFMA chains on all SMs); used as
 * the measured FP64 roofline denominator.  Synchronous; ~50 ms. */
int chemora_measure_fp64_peak(chemora_t* h, double* gflops);

const char* chemora_last_error(const chemora_t* h);

/* Waits for the stream, frees buffers.  NULL-safe. */
int chemora_destroy(chemora_t* h);

#ifdef __cplusplus
}
#endif
#endif /* CHEMORA_H */
