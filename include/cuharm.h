/* cuharm.h — C ABI of libcuharm.so: the per-zone HARM conservative update of ideal GR-MHD on a fixed
 * Kerr-Schild / modified-Kerr-Schild grid (cuHARM, arXiv 2205.02484), fp64, one NVIDIA B200 (sm_100a).
 *
 * Citations: "P:L<n>" = line n of the paper text with the equation it falls in; "A<n>" = a
 * reading of the paper listed in DESIGN.md where the text is silent, garbled or self-contradictory.
 *
 * General rules
 *   - Every function returns int: 0 = OK, <0 = one of the CUHARM_E* codes.  Nothing throws or aborts.
 *     Physics trouble (a failed inversion, a floor hit) is NOT an error: see cuharm_get_stats.
 *   - Pointers named d_* are DEVICE pointers, everything else is a HOST pointer.
 *   - The caller owns every device byte.  The library borrows d_prim / d_workspace from cuharm_bind until
 *     cuharm_destroy or the next cuharm_bind; it never allocates or frees device memory.
 *   - All work is enqueued on the CUDA stream given to cuharm_grid_init.  Only the calls that return host
 *     scalars (cuharm_cfl_dt, cuharm_last_cfl_dt, cuharm_divb, cuharm_get_stats) synchronise that stream.
 *   - There is no CPU fallback: without a CUDA device every compute call returns CUHARM_ECUDA.
 *   - The context belongs to the CUDA device that is current when cuharm_grid_init is called; every later call
 *     makes that device current for its own duration and restores the caller's.
 *   - Geometry: Kerr-Schild in the (diagonal-Jacobian) MKS coordinates of eq. 39, or Minkowski.  The kernels
 *     store and contract only the metric entries that do not vanish identically there (00 01 03 11 13 22 33 of
 *     g_{mu nu} and g^{mu nu}; g^{t phi} = 0), use u_i = g_ij utilde^j and beta^2 = beta^3 = 0, and drop the nu = t,
 *     phi source terms (the metric depends on neither).  `coords` in {0, 1} is the only geometry the library
 *     accepts; a metric with another zero pattern needs other kernels.
 *
 *   - One environment switch, read by cuharm_grid_init: CUHARM_NO_TMAP=1 makes the update kernel stage its tiles with
 *     one-dimensional bulk copies instead of tensor-map copies (the path taken anyway when the driver's tensor-map
 *     encoder is unavailable); results are bit-identical (tests/test_gpu_parity_wide.py compares the two).
 *
 * Array layout (device, fp64, C order, the last index fastest):
 *   prim[8][n1+2ng][n2+2ng][n3+2ng], variables (rho, u, utilde^1, utilde^2, utilde^3, B^1, B^2, B^3)
 *   (eq. 10).  All vector components are coordinate components in (X^1, X^2, X^3).  Zone (I,J,K) has its
 *   centre at X^d = X^d_min + (index + 1/2) dx^d; array index = zone index + ng.
 */
#ifndef CUHARM_H
#define CUHARM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CUHARM_OK 0
#define CUHARM_EINVAL (-1) /* bad argument / shape / struct size            */
#define CUHARM_ESTATE (-2) /* called out of order (e.g. step before bind)   */
#define CUHARM_ECUDA (-3)  /* a CUDA call failed; text via cuharm_strerror  */
#define CUHARM_ENOMEM (-4) /* workspace too small                           */

typedef struct cuharm_ctx* cuharm_handle; /* opaque, host side; owns no device memory */

/* Plain-old-data parameter block; struct_bytes = sizeof(cuharm_params) guards against layout drift. */
typedef struct {
  int32_t struct_bytes;
  int32_t n1, n2, n3, ng; /* interior zones per direction (n3 == 1 allowed); ghost layers, 3 <= ng <= 8     */
  int32_t coords;         /* 0 = MKS (eq. 39; A14); 1 = Minkowski-Cartesian (tests; A39)        */
  double a, gam;          /* black-hole spin (eq. 38); adiabatic index of p = (gam-1) u     */
  double r_in, r_out, R0, hslope; /* MKS: X1 in [ln(r_in-R0), X1(r_out)], X2 in [-1,1], X3 in [0,2pi)         */
  double xmin[3], xmax[3];        /* Minkowski box                                                          */
  int32_t recon;   /* 0 = PLM + MC limiter (eqs. 15-16; A2); 1 = PPM (A20)              */
  int32_t riemann; /* 0 = local Lax-Friedrichs (eq. 17); 1 = HLL (eq. 20)                   */
  int32_t bc_x1, bc_x2, bc_x3; /* 0 outflow (+ inflow check in MKS X1; A15), 1 periodic, 2 polar reflection
                                  with utilde^2, B^2 sign flip, 3 fixed (ghosts never overwritten) */
  double rho_fl_coef, rho_fl_pow, rho_fl_abs; /* rho >= max(abs, coef * r^pow)  (eq. 35; A9)    */
  double u_fl_coef, u_fl_pow, u_fl_abs;       /* u   >= max(abs, coef * r^pow)                              */
  double sigma_max, b2_over_u_max, gamma_max; /* b^2/rho, b^2/u ceilings (eqs. 36-37; A10, A11) and Lorentz
                                                 factor cap (A12); <= 0 disables                    */
  double newton_tol;                          /* |dW/W| criterion of the 2D Newton-Raphson (A8)     */
  int32_t newton_maxit, newton_extra;         /* iteration cap; extra iterations after the criterion is met */
  int32_t fixup_max_passes;                   /* Jacobi passes of the eq. 34 repair (A13), 0..21           */
  int32_t n_x;     /* hyper-exponential radial branch of eq. 39: r = R0 + exp(X + (X - x_b)^n_x) for */
  double r_break;  /* X >= x_b = ln(r_break - R0) (the paper: n_x = 4, r_break = 400 M, r_out = 5e3 M); the grid    */
                   /* stays uniform in X1 from ln(r_in - R0) to the X1 of r_out.  Off unless n_x >= 2, r_break > R0 */
  int32_t inv_chain;   /* 1: the inversion fallback chain of P:L233-239 on the zones the 2D Newton method fails in:
                          no result -> 1D method for W by Brent; non-physical result, or 1D failed too -> the
                          entropy method (eq. 32 in eq. 29, by Brent; eq. 11 advanced for those zones); what still
                          fails goes to the eq. 34 repair.  0: failures go straight to eq. 34 (A33)               */
  int32_t brent_maxit; /* iteration cap of the Brent solver                                                       */
  double beta_min;     /* eq. 33 (A37): zones with p_g / (p_g + b^2/2) < beta_min at the previous time
                          level take the entropy method as first and only choice; <= 0 disables; needs inv_chain  */
  double brent_tol;    /* relative tolerance of the Brent solver (A40)                                            */
  int32_t polar_damp;  /* 1: after inversion + floors of every substep utilde^2 of the two zones nearest each pole is
                          replaced by the straight line in X^2 through zero at the pole and the third zone's value
                          ("interpolation to zero at the pole"; A16).  Needs bc_x2 = 2 and n2 >= 6.  0: off     */
  int32_t n1_global;   /* Slab decomposition along X1 (P:L271-273 splits the grid among GPUs).  > 0: this   */
  int32_t i_offset;    /* grid is the slab of zones i_offset .. i_offset + n1 - 1 of a grid with n1_global zones in X1:  */
  int32_t slab_lo;     /* coordinates, spacing and geometry are the full grid's.  slab_lo / slab_hi = 1: the lower /     */
  int32_t slab_hi;     /* upper X1 side is internal: its ghost zones are never written by the ghost fill -- the caller  */
                       /* copies the neighbouring slab's outermost ng interior planes there (halo exchange) after every */
                       /* cuharm_substep.  0 everywhere: the whole grid (default)                                       */
  int32_t reserved;    /* must be 0                                                                               */
} cuharm_params;

/* Create a context for the grid and scheme described by *p (the statement of the problem: spin a, adiabatic
 * index, MKS parameters, resolution — P:L285-311).  cuda_stream is a cudaStream_t (NULL = default stream).
 * Errors: EINVAL (null pointers, struct_bytes mismatch, n < 1, ng < 3, bad enum, polar reflection with n2 < ng),
 * ECUDA (no usable device). */
int cuharm_grid_init(cuharm_handle* out, const cuharm_params* p, void* cuda_stream);

/* Bytes of device workspace cuharm_bind needs: geometry tables, face fluxes F^1..3, edge EMFs, the half-step
 * primitives, the fail mask, counters (and, with inv_chain = 1, the updated conserved variables of every zone).
 * 0 if h is NULL. */
size_t cuharm_workspace_bytes(cuharm_handle h);

/* Borrow the caller's primitive array d_prim (layout above) and workspace (256-byte aligned, ws_bytes >=
 * cuharm_workspace_bytes).  If the geometry is already computed the ghost zones of d_prim are filled.
 * Errors: EINVAL (null / misaligned), ENOMEM (ws_bytes too small). */
int cuharm_bind(cuharm_handle h, double* d_prim, void* d_workspace, size_t ws_bytes);

/* Geometry precompute (eqs. 38-39): g_cov, g_con, sqrt(-g), lapse at zone centres, 1-faces and
 * 2-faces (3-faces equal centres: the metric is phi-independent), and the connection coefficients at
 * centres from closed-form derivatives (A19) together with the source weights sqrt(-g) (1/2 | 1) d_nu g_kl that
 * the update kernel contracts with T^kl (the same S_nu as eq. 7), plus the floor profiles of eq. 35.  Then fills the ghost
 * zones of the bound d_prim.  Errors: ESTATE (not bound). */
int cuharm_metric_precompute(cuharm_handle h);

/* The step size is kept in a device scalar that the kernels read, so one recorded CUDA graph (cuharm_use_graph)
 * serves every dt.
 *
 * One full RK2 (midpoint predictor / corrector) step of size dt, in place (eq. 25; A5): each substep
 * = reconstruction (eqs. 15-16 / PPM) -> LLF/HLL face fluxes (eqs. 17-20) -> flux-CT (eqs. 21-22; A3) -> source
 * (eq. 14) -> update -> Noble 2D inversion (eqs. 27-31; A6-A8) -> floors (eqs. 35-37) -> ghost fill -> repair of
 * failed zones (eq. 34; A13) -> ghost fill.  d_prim has valid ghosts on entry and on exit.  Asynchronous.
 * Errors: ESTATE (not bound / no geometry), EINVAL (dt not finite or <= 0). */
int cuharm_step(cuharm_handle h, double dt);

/* The same step with dt taken ON THE DEVICE from eq. 26 (A17) applied to the face speeds the predictor
 * of the previous step saw ("the next time step"): dt = min(dt_max, 1 / sum_l max c_w^l / (xi dx^l))
 * (dt_max <= 0: no cap) -- the value cuharm_last_cfl_dt would return, bit for bit, without the read-back and the
 * synchronisation, including its guard: where that value is not finite and positive (a non-finite face speed; no
 * speed at all and no cap) dt = 0, the step leaves the state unchanged and cuharm_get_time reports dt_last = 0.
 * Asynchronous.  Errors: ESTATE (no previous step since bind), EINVAL (xi not finite or <= 0). */
int cuharm_step_cfl(cuharm_handle h, double xi, double dt_max);

/* The same step in two calls, for a caller that exchanges halo planes between slabs (n1_global > 0): cuharm_set_dt
 * puts the step size into the device scalar (and advances the integrated time); cuharm_substep(h, 0) is the predictor
 * (P^n -> the half-step array, which lives in the workspace at byte offset cuharm_half_offset, layout of d_prim);
 * cuharm_substep(h, 1) is the corrector (in place into d_prim).  After substep 0 the halo planes of the half-step array,
 * after substep 1 those of d_prim must be refreshed from the neighbouring slabs before the next call.  The sequence
 * set_dt, substep 0, substep 1 enqueues exactly what cuharm_step(h, dt) enqueues (plain launches).
 * Errors: as cuharm_step; cuharm_substep(h, 1) before (h, 0): ESTATE.
 *
 * The eq. 34 repair (A13) reads neighbours across an internal boundary, and a zone repaired in one Jacobi pass is a
 * donor in the next.  For slabs whose failed zones may lie next to an internal boundary the substep therefore comes in
 * pieces as well, with a halo exchange of the substep's array AND of the flag array (int32 [n1g][n2g][n3g] in the
 * workspace at byte offset cuharm_flag_offset; flags ride with the halo) between them:
 *   cuharm_substep_update(h, which)        fluxes, update, inversion, floors, first ghost fill
 *   [exchange array + flags]
 *   cuharm_repair_pass(h, which, pass, out) for pass = 0, 1, ... <= fixup_max_passes: ONE Jacobi pass over this slab's
 *                                          failed zones; out[0] = failed zones of this slab in this substep, out[1] =
 *                                          zones still waiting (HOST pointer; synchronises); [exchange array + flags]
 *                                          after every pass in which any slab had failed zones; stop when the sum of
 *                                          out[1] over the slabs is 0 (or after pass fixup_max_passes, the last-resort one)
 *   cuharm_substep_finish(h, which)        second ghost fill (needed only if any slab had failed zones); [exchange array]
 * With the exchanges in place every pass sees across an internal boundary what the single-domain repair sees there.
 * Exception: a periodic X1 wrap that coincides with a cut.  The single-domain repair counts ghost zones as good donors
 * (their flags are 0), so the periodic image of a failed zone donates its unrepaired value; slabs exchange the real flags
 * and skip it.  With failed zones on both sides of such a wrap the results differ in the repaired zones. */
int cuharm_set_dt(cuharm_handle h, double dt);
int cuharm_substep(cuharm_handle h, int32_t which);
int cuharm_substep_update(cuharm_handle h, int32_t which);
int cuharm_repair_pass(cuharm_handle h, int32_t which, int32_t pass, int64_t out[2]);
int cuharm_substep_finish(cuharm_handle h, int32_t which);
size_t cuharm_half_offset(cuharm_handle h);
size_t cuharm_flag_offset(cuharm_handle h);

/* Maxima of the face speeds c_w per direction: of the predictor of the last step (cuharm_last_cw), or of the bound
 * primitives (cuharm_cfl_cw; overwrites the flux workspace) -- what cuharm_last_cfl_dt / cuharm_cfl_dt reduce; and eq. 26
 * from a given triple (cuharm_dt_of_cw; host arithmetic only), so that a caller can take the maximum over slabs in
 * between.  cw: HOST pointer to 3 doubles (+infinity where a speed was not finite).  The first two synchronise. */
int cuharm_last_cw(cuharm_handle h, double cw[3]);
int cuharm_cfl_cw(cuharm_handle h, double cw[3]);
int cuharm_dt_of_cw(cuharm_handle h, double xi, const double cw[3], double* dt_out);

/* Integrated time since cuharm_bind (*t, the sum of the step sizes) and the size of the last step (*dt_last);
 * either pointer may be NULL.  HOST pointers.  Synchronises. */
int cuharm_get_time(cuharm_handle h, double* t, double* dt_last);

/* Pure inversion (eqs. 27-31) on full-grid arrays of the prim layout: d_U holds the 8 conserved variables
 * sqrt(-g)(rho u^t, T^t_t, T^t_i, B^i) (A18); d_prim_inout carries the Newton guess in and the answer out;
 * d_flag[zone] (int32, [n1g][n2g][n3g], may be NULL) = 0 ok, 1 D<=0 / non-finite input, 2 no convergence,
 * 3 W<=0 or non-finite, 4 v^2 outside [0,1), 5 rho<=0, 6 u<0.  No floors, no repairs.  Asynchronous. */
int cuharm_cons_to_prim(cuharm_handle h, const double* d_U, double* d_prim_inout, int32_t* d_flag);

/* One of the two fallback inversions of P:L229-233 on full-grid arrays, like cuharm_cons_to_prim (test helper):
 * method 1 = the 1D method (v^2 from eq. 30 put into eq. 29, solved for W by Brent), method 2 = the entropy
 * method (eq. 32 in eq. 29, solved for v^2 by Brent; A36) with d_US[zone] ([n1g][n2g][n3g]) the conserved entropy
 * sqrt(-g) S u^t, S = p_g / rho^(gam-1) (eq. 11).  Brent's tolerance and iteration cap are
 * brent_tol / brent_maxit of the parameter block (EINVAL if those are not set).  d_flag as in cuharm_cons_to_prim
 * (2 also: no bracket / Brent did not converge).  Asynchronous. */
int cuharm_invert_fallback(cuharm_handle h, int32_t method, const double* d_U, const double* d_US, double* d_prim_inout,
                           int32_t* d_flag);

/* Primitive -> conserved on full-grid arrays.  Test helper.  Asynchronous. */
int cuharm_prim_to_cons(cuharm_handle h, const double* d_prim, double* d_U);

/* Time step of eq. 26 (A17) from the bound primitives: dt^l = xi dx^l / max_faces c_w^l,
 * 1/dt = sum_l 1/dt^l.  Overwrites the flux workspace.  Synchronises.  *dt_out = 0 if a wave speed anywhere is
 * not finite (physics trouble is not an error code; cuharm_step rejects dt = 0). */
int cuharm_cfl_dt(cuharm_handle h, double xi, double* dt_out);

/* Same formula from the face speeds the predictor of the last cuharm_step saw ("the next time step",
 * P:L198) — costs one 24-byte read-back, no extra kernel.  Synchronises.  ESTATE before the first step. */
int cuharm_last_cfl_dt(cuharm_handle h, double xi, double* dt_out);

/* Corner-centred discrete divergence of sqrt(-g) B (eq. 23; A4) over the corners whose cells are
 * interior: *max_abs = max |D|, *max_norm = max |D| / (sum of the magnitudes of D's own terms), the latter over
 * the corners where that sum exceeds 1e-290 (below it the terms are in the subnormal range).  Synchronises. */
int cuharm_divb(cuharm_handle h, double* max_abs, double* max_norm);

/* The same two numbers for a caller that cannot allocate device memory and so has no context (a context needs a
 * workspace of cuharm_workspace_bytes): an in-situ monitor, analysis or I/O plug-in running inside another code's time
 * loop, where the host application has given the whole device to its own memory pool, hands the plug-in its arrays and
 * nothing else, and where cudaMalloc / cudaFree may fail on the full device and would stall every stream of the process.
 * Needs no handle and no workspace, and calls no cudaMalloc, cudaFree or allocating library routine.
 *   d_prim       DEVICE, prim[8][n1+2ng][n2+2ng][n3+2ng] (layout above); only B^1..3 are read.  With periodic_x3 != 0 the
 *                first X3 ghost layer must hold the periodic image (as after cuharm_bind / cuharm_step / cuharm_apply_bc)
 *   d_sqrtg      DEVICE, sqrt(-g) at zone centres, [n1+2ng][n2+2ng] (component 20 of cuharm_get_geom(h, 0, .), or the
 *                caller's own table); only interior entries are read
 *   dx           HOST, the three coordinate spacings; periodic_x3: bc_x3 == 1; 1 <= ng <= 8
 *   cuda_stream  cudaStream_t (NULL = default stream) of the device that is CURRENT at the call
 *   d_out        DEVICE, 2 doubles: max |D|, max |D| / (sum of the magnitudes of D's own terms) as cuharm_divb defines
 *                them; written by a kernel on cuda_stream.  Asynchronous: nothing is synchronised or copied to the host
 * The reduction's scratch (one pair of partial maxima per (i, j) corner row) is a fixed static device array of
 * CUHARM_DIVB_NOALLOC_MAX_ROWS rows (2 MiB), present on every GPU that loads the library until the process exits.
 * Limit: (n1 - 1) * (n2 - 1) <= CUHARM_DIVB_NOALLOC_MAX_ROWS (n3 is unlimited; 362 x 362 and 512 x 257 both fit);
 * beyond it the call returns CUHARM_ENOMEM, launches nothing and leaves d_out alone.
 * All calls on one device share that array: two calls whose kernels can overlap on the GPU (different streams with no
 * ordering between them) race and both results are void -- keep the calls on one stream or order them with events.  The
 * array keeps the previous call's contents; no call depends on them (each overwrites every slot it later reads).
 * The FIRST call on each device also looks up the array's device address (cudaGetSymbolAddress); make that first call
 * outside any stream capture.  Thread-safe on the host side.
 * Errors: EINVAL (null pointer, bad shape, dx not finite and positive), ENOMEM (grid beyond the limit), ECUDA; the text
 * of the last failure of this call on the calling thread: cuharm_divb_noalloc_errtext(). */
#define CUHARM_DIVB_NOALLOC_MAX_ROWS 131072
int cuharm_divb_noalloc(const double* d_prim, const double* d_sqrtg, int32_t n1, int32_t n2, int32_t n3, int32_t ng,
                        const double dx[3], int32_t periodic_x3, void* cuda_stream, double* d_out);
const char* cuharm_divb_noalloc_errtext(void);

/* Fluxes through the coordinate shell of zone centres of radial index i (0 <= i < n1), the paper's horizon
 * diagnostics when i is the shell nearest r_h (eqs. 43-46): out[0] = Mdot = sum sqrt(-g) rho u^1,
 * out[1] = phi_B = 1/2 sum sqrt(-g) |B^1| (*F^{rt} = B^r), out[2] = Ldot = sum sqrt(-g) T^1_phi,
 * out[3] = Edot = -sum sqrt(-g) T^1_t, each summed over the interior (j, k) with weight dX2 dX3 (the integrand
 * sqrt(-g) J^1 dX2 dX3 is coordinate invariant).  Mdot is negative for inflow, as eq. 43 is printed.  Sums are
 * deterministic (fixed-order trees).  out: HOST pointer to 4 doubles.  Needs geometry and bound primitives with
 * valid interior; synchronises.  CUHARM_EINVAL for i out of range. */
int cuharm_shell_fluxes(cuharm_handle h, int32_t i, double out[4]);

/* Copy a geometry table to a caller array d_out[comp][n1g][n2g]: loc 0 centre, 1 = 1-face (I-1/2,J), 2 = 2-face
 * (I,J-1/2): 22 comps = g_cov (00 01 02 03 11 12 13 22 23 33), g_con (same order), sqrt(-g), lapse; loc 3: the 40
 * connection coefficients Gamma^l_{nk}, l-major, (n,k) in the same 10-pair order.  Test helper.  Asynchronous. */
int cuharm_get_geom(cuharm_handle h, int32_t loc, double* d_out);

/* Fill the ghost zones of an arbitrary primitive array of the bound shape.  Asynchronous. */
int cuharm_apply_bc(cuharm_handle h, double* d_prim);

/* Floors, ceilings and Lorentz cap (eqs. 35-37; A9-A12) as a stage of their own on the interior zones
 * of an arbitrary primitive array of the bound shape, in place; d_mask[zone] (int32, [n1g][n2g][n3g], may be NULL)
 * = bit mask: 1 rho floor, 2 u floor, 4 ceiling applied, 8 Lorentz cap, 16 ceiling re-inversion failed.  Test
 * helper.  Asynchronous. */
int cuharm_apply_floors(cuharm_handle h, double* d_prim, int32_t* d_mask);

/* The eq. 34 repair (A13) as a stage of its own on an arbitrary primitive array of the bound shape, in
 * place: the interior zones with d_flag[zone] > 0 (int32, [n1g][n2g][n3g]) are the failed ones; ghost zones count
 * as good and must hold valid values.  Counters 0, 1, 7 of cuharm_get_stats advance.  Test helper.  Asynchronous. */
int cuharm_repair(cuharm_handle h, double* d_prim, const int32_t* d_flag);

/* Stage-level test helpers (asynchronous; arrays have the prim layout unless stated):
 * face fluxes of direction dir (1..3) BEFORE flux-CT, d_F[8][zones] stored at the zone whose LOWER dir-face it
 * is, valid on faces 0..N_dir and transverse zones -1..N (eqs. 15-20); d_cw[zones] (may be NULL) = c_w. */
int cuharm_flux_dir(cuharm_handle h, const double* d_prim, int32_t dir, double* d_F, double* d_cw);

/* out[8] (HOST): 0 failed inversions, 1 zones repaired, 2 rho-floor hits, 3 u-floor hits, 4 ceilings applied,
 * 5 Lorentz caps, 6 Newton iterations, 7 zones repaired by the last-resort rule.  Synchronises. */
int cuharm_get_stats(cuharm_handle h, int64_t out[8]);

/* out[4] (HOST), the fallback chain of P:L229-239 (inv_chain = 1): 0 zones the 2D method failed in that went down
 * the chain, 1 of them recovered by the 1D method, 2 zones recovered by the entropy method (from the chain or as an
 * eq. 33 zone), 3 zones that took the entropy method first and only (eq. 33).  Synchronises. */
int cuharm_get_chain_stats(cuharm_handle h, int64_t out[4]);

/* Record the two substeps of cuharm_step into a CUDA graph and replay it on later calls (on != 0), or go back
 * to plain launches (on == 0).  Purely a launch-overhead optimisation; results are identical. */
int cuharm_use_graph(cuharm_handle h, int32_t on);

/* Number of kernel launches the library has enqueued since grid_init (graph replays count their nodes). */
int64_t cuharm_launch_count(cuharm_handle h);

/* Kernel classes of the per-class timing below. */
#define CUHARM_K_FLUX1 0  /* reconstruct + flux, direction 1 */
#define CUHARM_K_FLUX2 1
#define CUHARM_K_FLUX3 2
#define CUHARM_K_EMF 3    /* flux-CT edge EMFs               */
#define CUHARM_K_UPDATE 4 /* source + update + inversion + floors */
#define CUHARM_K_BC 5     /* one ghost fill (up to 3 launches)    */
#define CUHARM_K_FIXUP 6  /* eq. 34 repair                        */
#define CUHARM_NCLASS 8

/* Measurement aid: when on, a pair of CUDA events on the library's stream brackets every launch of the classes
 * above (plain launches only; ignored while a graph replays).  cuharm_get_timing synchronises and returns, per
 * class, the summed device milliseconds and the number of bracketed launches since cuharm_set_timing(h, 1). */
int cuharm_set_timing(cuharm_handle h, int32_t on);
int cuharm_get_timing(cuharm_handle h, double ms[CUHARM_NCLASS], int64_t count[CUHARM_NCLASS]);

int cuharm_destroy(cuharm_handle h);

/* Static text for a CUHARM_E* code; for CUHARM_ECUDA the text of the last CUDA error seen by this thread. */
const char* cuharm_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* CUHARM_H */
