/*
 * clt.h -- C ABI of libclt: the B200-native (sm_100a, FP64) hot path of CLTx, arxiv 1812.00525.
 *
 * What the library computes (citations are PAPER.md line numbers / equation numbers):
 *   the full resistive-MHD right-hand side in the equilibrium-subtracted form, eqs (11)-(14)
 *   [L105-115], with J = curl B, eq (6) [L79], and E = -v x B + eta (J - J0), eq (5) [L77] with
 *   d_i = 0, for the 8 fields rho, p, v_R, v_phi, v_Z, B_R, B_phi, B_Z [L139, L191-196] on a uniform
 *   cylindrical (R, phi, Z) grid [L121-125] with 4th-order central finite differences in all three
 *   directions [L125], advanced by the classical 4th-order Runge-Kutta scheme [L125, L139]
 *   ("DERIVATIVES", "J, E", "RIGHT HANDS OF EQUATIONS", "STEP ON" modules of Fig. 2 [L139-141]),
 *   with fixed values on two node layers per R/Z side [L123, L187-189] and phi periodic, plus the
 *   DIAGN-type reductions (kinetic / magnetic energy [L430], max |div B|) and the SETDT CFL
 *   time step of Fig. 4 [L180-215].  The exact discrete definitions are in DESIGN.md section 3.
 *
 * Conventions
 *   - Every function returns CLT_OK (0) or a negative clt_status.  No exceptions, no aborts, nothing
 *     is printed.  clt_strerror() gives a static string for a code.
 *   - All floating-point data is IEEE binary64.  Array arguments may be HOST or DEVICE pointers; the
 *     library finds out with cudaPointerGetAttributes.  The caller owns every buffer it passes; the
 *     library copies in or out and keeps no pointer to it after the call returns, with one
 *     exception: the workspace given to clt_create(), which the context sub-allocates and the
 *     caller must keep alive (and not touch) until clt_destroy().
 *   - User-visible array layout (dense, C order, R fastest -- the C image of CLTx's X(JX,JZ,JY,M)):
 *        state / dUdt : double[8][nphi][nZ][nR]   fields rho, p, v_R, v_phi, v_Z, B_R, B_phi, B_Z
 *        equilibrium  : double[8][nZ][nR]          axisymmetric
 *        vector field : double[3][nphi][nZ][nR]    components R, phi, Z
 *     Inside the workspace the library uses its own padded layout.
 *   - One context = one CUDA stream (given at creation; NULL = the legacy default stream).  All work
 *     is enqueued on that stream.  Calls are asynchronous with respect to the host except where
 *     noted (a host destination pointer, or clt_diagnostics / clt_suggest_dt, which return scalars).
 *     A context is not thread-safe.
 *   - Call order: clt_create -> [clt_set_equilibrium] -> clt_set_state -> { clt_rhs | clt_step |
 *     clt_curl_J1 | clt_diagnostics | clt_suggest_dt | clt_get_state | clt_set_dt }*  -> clt_destroy.
 *     A call out of order returns CLT_ESTATE.
 *   - There is no CPU fallback: without a usable CUDA device every compute entry point fails with
 *     CLT_ECUDA.
 */
#ifndef CLT_H
#define CLT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    CLT_OK = 0,
    CLT_EINVAL = -1,     /* bad argument, shape or parameter                         */
    CLT_ENOMEM = -2,     /* workspace too small / misaligned                         */
    CLT_ESTATE = -3,     /* call out of order (e.g. clt_step before clt_set_state)   */
    CLT_ECUDA = -4,      /* a CUDA runtime error (sticky: see clt_last_cuda_error)   */
    CLT_ENONFINITE = -5  /* clt_diagnostics found a non-finite sum                   */
} clt_status;

typedef struct clt_ctx clt_ctx;  /* opaque */

/* Grid [L121-125].  Node counts include the two fixed layers per R/Z side, and the box edge is a
 * node:  R_i = Rmin + i*(Rmax-Rmin)/(nR-1), i = 0..nR-1 (computed on the host in plain double
 * arithmetic, no FMA), Z_k likewise; phi_j = j*dphi, dphi = L/nphi, L = phi_extent (0 means 2*pi),
 * periodic.  Requirements: nR >= 9, nZ >= 9, nphi >= 5, Rmin > 0, Rmax > Rmin, Zmax > Zmin.     */
typedef struct {
    int32_t nR, nphi, nZ;
    double Rmin, Rmax, Zmin, Zmax;
    double phi_extent;
} clt_grid;

/* Physics and run parameters [L67-81]: ratio of specific heats Gamma, and the uniform dissipation
 * coefficients eta (resistivity), nu (viscosity), D (density diffusion), kappa (heat conduction).
 * dt > 0 is the fixed RK4 time step used by clt_step.  cfl is only used by clt_suggest_dt when its
 * cfl argument is <= 0.  flags: reserved, must be 0.  d_i >= 0 is the ion inertial length of the Hall
 * term (d_i/rho)(J x B - grad p) of eq (5) [L77]; 0 (the measured configs) = resistive MHD.  With
 * d_i > 0 the curl pass also forms G = (J1 x B + J0 x B1 - grad p1)/rho - (rho1/rho)(v0.grad)v0 on
 * interior nodes and E1 gains d_i G (reading R11); this needs the default kernel variant and
 * tile height (clt_rhs / clt_step return CLT_EINVAL otherwise).                                   */
typedef struct {
    double gamma, eta, nu, D, kappa;
    double dt;
    double cfl;
    uint32_t flags;
    double d_i;
} clt_params;

/* Diagnostics [L139, L149, L430]; sums run over interior nodes with weight R_i dR dphi dZ:
 *   kinetic       = sum 1/2 rho |v|^2          magnetic      = sum 1/2 |B|^2
 *   magnetic_pert = sum 1/2 |B - B0|^2         magnetic_n1   = energy of the n = 1 toroidal Fourier
 *   harmonic of B - B0;  max_divB = max over the deep interior (i in [4,nR-5], k in [4,nZ-5]) of
 *   |div_c B|, the conservative discrete divergence that the discrete curl annihilates.          */
typedef struct {
    double kinetic, magnetic, magnetic_pert, magnetic_n1, max_divB;
    int64_t step;   /* RK4 steps taken since clt_set_state */
    double time;    /* sum of the dt's of those steps      */
} clt_diag;

/* Device bytes clt_create() needs for this grid (38 padded fields + equilibrium tables + reduction
 * scratch).  Returns 0 for an invalid grid.                                                      */
size_t clt_workspace_bytes(const clt_grid *grid);

/* Creates a context.  d_workspace: DEVICE memory, at least clt_workspace_bytes(grid) bytes, 256-byte
 * aligned, owned by the caller (e.g. a torch tensor), zero-initialised or not.  cuda_stream: a
 * cudaStream_t (NULL = default stream).  The equilibrium starts as all-zero.
 * Errors: CLT_EINVAL (NULL pointers, bad grid, gamma/dt not finite, negative coefficients, flags),
 * CLT_ENOMEM (bytes too small, pointer misaligned or not device memory), CLT_ECUDA.               */
int clt_create(const clt_grid *grid, const clt_params *params, void *d_workspace, size_t bytes,
               void *cuda_stream, clt_ctx **out);

/* Releases the context (not the workspace).  Synchronises the stream.  NULL is allowed.           */
int clt_destroy(clt_ctx *ctx);

/* Sets the axisymmetric reference state U0[8][nZ][nR] of eqs (11)-(14) (host or device pointer;
 * NULL = all zero, which makes the path evaluate eqs (1)-(4) directly).  Also computes J0 = curl B0
 * and the other time-independent tables.  Must be called before clt_set_state (it invalidates the
 * state: a later compute call returns CLT_ESTATE until clt_set_state is called again).            */
int clt_set_equilibrium(clt_ctx *ctx, const double *U0);

/* Sets the state U[8][nphi][nZ][nR] (host or device pointer), resets step/time to 0 and freezes the
 * two boundary node layers per R/Z side at these values for all later steps [L123, L187-189].     */
int clt_set_state(clt_ctx *ctx, const double *U);

/* Copies the current state out (host or device pointer).  Synchronous if U is host memory.        */
int clt_get_state(clt_ctx *ctx, double *U);

/* dUdt[8][nphi][nZ][nR] = right-hand side of eqs (11)-(14) at the current state; exactly 0 on the
 * boundary layers.  Does not change the state.  Synchronous if dUdt is host memory.  CLT_ESTATE
 * between clt_step_stage(1) and clt_step_stage(4) (the call uses U_b as scratch).                  */
int clt_rhs(clt_ctx *ctx, double *dUdt);

/* J1[3][nphi][nZ][nR] = curl(B - B0) of the current state (eq (6)); 0 on the boundary layers.     */
int clt_curl_J1(clt_ctx *ctx, double *J1);

/* G[3][nphi][nZ][nR] = Hall field (J1 x B + J0 x B1 - grad p1)/rho - (rho1/rho)(v0.grad)v0 of the current
 * state (eq (5) [L77], reading R11); 0 on the boundary layers.  CLT_EINVAL if params.d_i = 0
 * or with the plain-load kernel variant.                                                         */
int clt_hall_G(clt_ctx *ctx, double *G);

/* n >= 0 classical RK4 steps with the fixed time step params.dt (or the last clt_set_dt value).
 * Asynchronous.                                                                                  */
int clt_step(clt_ctx *ctx, int n);

/* NEXT-4, slab decomposition [L127, L250-256, L337]: the pieces a caller needs to run one sub-domain per GPU and
 * exchange ghost rows between RK stages (paper_1812_00525_b200/slab.py does exactly that).
 * A sub-domain is an ordinary context whose grid is a Z-slab of the global grid with 4 ghost rows per cut; the
 * kernels never write the two outer rows, recompute rows 2-3 (and nZ-4, nZ-3) from the ghost data, and the caller
 * overwrites all 4 ghost rows after every stage.
 *   clt_step_stage : stage = 1..4 of one RK4 step (curl + fused kernel), in order; stage 4 completes the step.
 *                    The stage's output buffer is  1 (U_a), 2 (U_b), 1 (U_a), 0 (U^n)  for stage 1, 2, 3, 4.
 *                    CLT_ESTATE if called out of order (clt_step is refused in the middle of a step).
 *   clt_get_rows / clt_set_rows : rows k0 .. k0+nrows-1 of buffer 0 = U^n, 1 = U_a, 2 = U_b as a dense array
 *                    double[8][nphi][nrows][nR] (host or device pointer; synchronous for host pointers).
 *   clt_set_owned_rows : the rows this context is responsible for (default 2 .. nZ-3): the rows a stage writes, the
 *                    diagnostics sums and the SETDT minimum run over them; and the rows of max |div_c B| (default
 *                    4 .. nZ-5; first > last = none), so that slabs can be reduced without counting ghost rows twice. */
int clt_step_stage(clt_ctx *ctx, int stage);
int clt_get_rows(clt_ctx *ctx, int buffer, int k0, int nrows, double *dst);
int clt_set_rows(clt_ctx *ctx, int buffer, int k0, int nrows, const double *src);
int clt_set_owned_rows(clt_ctx *ctx, int k_first, int k_last, int deep_first, int deep_last);

/* Adaptive time step [L139, Fig. 3-4] for a GROUP of contexts that share one dt (the slabs of one grid), with dt kept on
 * the device as in clt_step_cfl -- no host round trip per step:
 *   clt_cfl_open(ctx, cfl)        enters adaptive mode: SETDT of the current state over the context's owned rows
 *                                 (cfl <= 0: params.cfl).  CLT_ESTATE inside a step or if already open.
 *   clt_cfl_commit(ctxs, n, init) one single-thread kernel: the minimum over the n contexts (init = 1: of the SETDT values
 *                                 clt_cfl_open computed; init = 0: of the minima stage 4 collected over the owned rows
 *                                 of the new state, after advancing every clock by the dt just used) becomes every
 *                                 context's dt.  All contexts on one device; n <= 64; stream-ordered (events).
 *   clt_step_stage(ctx, 1..4)     runs with the committed dt; the caller exchanges ghost rows in between.
 *   clt_cfl_close(ctx, ..)        leaves adaptive mode; returns the dt the next step would use and the time advanced
 *                                 since clt_cfl_open (synchronises).  CLT_ENONFINITE like clt_step_cfl.
 * One context alone: open, commit(init = 1), { four stages, commit(init = 0) } x steps, close == clt_step_cfl, bit for bit.
 * Between open and close clt_step and clt_step_cfl return CLT_ESTATE; clt_set_state ends the sequence.               */
int clt_cfl_open(clt_ctx *ctx, double cfl);
int clt_cfl_commit(clt_ctx *const *ctxs, int n, int init);
int clt_cfl_close(clt_ctx *ctx, double *dt_next, double *time_advanced);

/* A slab of a larger grid carries the GLOBAL spacing: dZ replaces (Zmax - Zmin)/(nZ - 1) of this context's own grid in
 * every stencil weight, table and diagnostic weight, so that a decomposed run reproduces the undivided run bit for bit
 * (the method has no other use for Z than its spacing).  Call it right after clt_create: it invalidates the
 * equilibrium tables and the state (set them again).  dZ must be finite and > 0.  Asynchronous.            */
int clt_set_z_spacing(clt_ctx *ctx, double dZ);

/* Ghost-row hand-over between two contexts of one process [L127 "message passing between every two neighboring
 * blocks"]: rows k0_src .. k0_src+nrows-1 of `buffer` (0 = U^n, 1 = U_a, 2 = U_b; all 8 fields, all planes) of `src`
 * are written straight into rows k0_dst .. of the same buffer of `dst` by ONE kernel -- no dense staging array, no host
 * wait.  Both contexts must have the same nR and nphi.  Stream order: the copy runs on dst's stream after everything
 * enqueued on src's stream so far, and src's stream waits for it (events; nothing to do when both contexts share one
 * stream).  Contexts on different devices need peer access (CLT_ECUDA otherwise).                         */
int clt_push_rows(clt_ctx *src, int buffer, int k0_src, int nrows, clt_ctx *dst, int k0_dst);

/* Compute and exchange in ONE kernel [L250-256: the paper hands device pointers to MPI; here the neighbour's memory is
 * written directly]: after clt_link_rows(ctx, side, peer, k0, nrows, k0_peer) every stage kernel of `ctx` stores rows
 * k0 .. k0+nrows-1 (owned rows of ctx) of its output also into rows k0_peer .. of the same buffer of `peer` -- the
 * peer's ghost rows -- straight from the RK4 epilogue, tile by tile, while the rest of the stage is still being computed.
 * side = 0 (lower neighbour) or 1 (upper); peer = NULL removes the link.  A stage writes a context's owned rows only
 * (clt_set_owned_rows, to be called first), so the peer's own kernels never touch its ghost rows.  Same nR and nphi;
 * contexts on different devices need peer access (CLT_ECUDA otherwise).  clt_sync_peers(a, b) orders the two contexts'
 * streams after each other's work so far (call it between stages; nothing happens when they share one stream).  A
 * link holds a pointer into the peer's workspace: remove it before the peer is destroyed.                          */
int clt_link_rows(clt_ctx *ctx, int side, clt_ctx *peer, int k0, int nrows, int k0_peer);
int clt_sync_peers(clt_ctx *a, clt_ctx *b);

/* NEXT-1 in the loop [L139 "the time step ... is calculated based on the latest rho, p, v, B"; Fig. 3: STEPON then
 * SETDT; Fig. 4]: n RK4 steps, each with dt = SETDT(cfl) of the state at its start.  The time step lives on the
 * device: the first one comes from the reduction kernel of clt_suggest_dt, the following ones are collected by the
 * stage-4 epilogue of the fused kernel (no extra pass over the state, no host round trip per step).  cfl <= 0 means
 * params.cfl.  Synchronises once at the end to report *dt_last (SETDT of the final state, i.e. the step the next call
 * would start with) and *time_advanced (sum of the n steps); either pointer may be NULL.  params.dt is unchanged.
 * Slabs need the global minimum instead: slab.py's step_cfl reduces clt_suggest_dt over the slabs every step.
 * CLT_ENONFINITE if a state of the call had a non-finite signal speed (NaN / Inf in rho, p, v or B): the device
 * clock then holds dt = 0 for the remaining steps of the call instead of stepping on with a meaningless dt.  */
int clt_step_cfl(clt_ctx *ctx, int n, double cfl, double *dt_last, double *time_advanced);

/* Changes the fixed time step (dt > 0, finite).  Stream-ordered: steps already enqueued keep their dt; the CUDA
 * graph of the step is kept (the kernels read dt/2, dt/3, dt/6 from device memory).             */
int clt_set_dt(clt_ctx *ctx, double dt);

/* Reductions over the current state; synchronises the stream.  CLT_ENONFINITE if a sum is not
 * finite (out is still filled).                                                                  */
int clt_diagnostics(clt_ctx *ctx, clt_diag *out);

/* The same reductions for callers that cannot allocate or synchronise (code under CUDA graph capture, tight serving
 * loops): the ONE entry point of the library that uses no memory but its own.  The block partials of the reduction go
 * to a file-scope device array inside the library instead of the caller's workspace (768 KiB = 16384 reduction CTAs
 * x 6 doubles, held by every GPU that loads the library until the process exits); the call allocates nothing, copies
 * nothing to the host and does not synchronise.
 *   d_out6 : DEVICE pointer to 6 doubles, written on the context's stream:
 *            { kinetic, magnetic, magnetic_pert, magnetic_n1, max |div_c B|, SETDT(cfl) }  (cfl <= 0: params.cfl, else 0.5)
 * Limit: grids with more than 16384 reduction CTAs, ceil((nR-4)/32) * (nZ-4) > 16384, are refused with CLT_ENOMEM and a
 * text in clt_last_cuda_error (512 x 64 x 512 needs 8128).  CLT_EINVAL if d_out6 is not device memory.
 * Every call on a device shares the array: calls that overlap on the GPU (contexts on different streams) race; calls
 * on one stream are safe.  Nothing in the array has to be zero and nothing a previous call left there is read.       */
int clt_diagnostics_static(clt_ctx *ctx, double cfl, double *d_out6);

/* SETDT of Fig. 4 [L180-215]: dt = min(100, min over interior nodes of min(dR/(|v_R|+c),
 * dZ/(|v_Z|+c), R dphi/(|v_phi|+c)) * cfl), c = sqrt(|Gamma p/rho + |B|^2/rho|).  cfl <= 0 means
 * params.cfl.  Synchronises the stream.  Does not change the context's dt.                        */
int clt_suggest_dt(clt_ctx *ctx, double cfl, double *dt_out);

/* phi scheme [L125: "either 4th order finite difference or pseudo-spectrum method can be used"].
 * scheme 0 (default) = 4th-order central differences; 1 = pseudo-spectral: every d/dphi and d2/dphi2 of the
 * path (curl, gradients, divergences, Laplacians, curl E, div_c B of the diagnostics) is the exact derivative
 * of the trigonometric interpolant through the nphi samples (Nyquist mode: first derivative 0, second
 * derivative -(pi nphi/L)^2; reading R12).  It needs a second caller-owned DEVICE scratch buffer of
 * clt_spectral_workspace_bytes(grid) bytes (256-byte aligned; 14 padded fields), kept alive until the scheme is
 * set back to 0 or the context is destroyed, nphi <= 256, and the default kernel variant
 * (clt_rhs / clt_step return CLT_EINVAL otherwise).  Synchronises the stream.
 * Errors: CLT_EINVAL (scheme, nphi > 256), CLT_ENOMEM (scratch missing, small, misaligned, not device).   */
size_t clt_spectral_workspace_bytes(const clt_grid *grid);
int clt_set_phi_scheme(clt_ctx *ctx, int scheme, void *d_scratch, size_t bytes);

/* Launch-shape knobs for measurement (all optional; 0 = library default): tile height in Z of the
 * fused RHS kernel (one shape is built: 0 or 8, anything else is CLT_EINVAL), number of phi chunks per tile
 * (default: 1, more on grids with fewer tiles than the
 * device has SMs), use of a CUDA graph for the 8 launches of a clt_step step (0 = default: yes, unless
 * per-kernel profiling is on; 1 = always; 2 = never).  None of them changes a bit of the result.   */
int clt_set_tuning(clt_ctx *ctx, int tile_z, int phi_chunks, int use_graph);

/* Selects the implementation of the fused RHS kernel: 0 (default) = shared-memory tiles fed by TMA
 * (cp.async.bulk.tensor + mbarrier), 1 = the same arithmetic fed by plain global loads (kept as the A/B
 * measurement and as a parity cross-check; no Hall term, no pseudo-spectral scheme).  The two agree to
 * round-off (separate template instantiations: the compiler may contract FMAs differently).       */
int clt_set_kernel_variant(clt_ctx *ctx, int variant);

/* Per-kernel device timing for the roofline report.  With profiling enabled (and use_graph != 1)
 * every hot-path launch of clt_step / clt_rhs is bracketed by CUDA events on the context's stream;
 * clt_get_profile() synchronises, sums the elapsed times per kernel kind since profiling was
 * (re-)enabled, and resets the record.  rhs index = RK4 stage 1..4, 0 = clt_rhs' K-only variant.
 * At most 8192 launches are recorded; later ones are counted in `dropped`.                       */
typedef struct {
    double ms_curl;  int64_t n_curl;
    double ms_rhs[5]; int64_t n_rhs[5];
    int64_t dropped;
    double ms_phi;   int64_t n_phi;      /* pseudo-spectral phi pre-passes */
} clt_profile;
int clt_set_profiling(clt_ctx *ctx, int enable);
int clt_get_profile(clt_ctx *ctx, clt_profile *out);

/* Number of kernels launched by this context so far (for bench.py's gpu_launches).               */
int64_t clt_launch_count(const clt_ctx *ctx);

/* The stream-ordered device time of the kernels is measured by the caller with CUDA events on the
 * context's stream; the library offers the stream back for that.                                 */
void *clt_stream(const clt_ctx *ctx);

const char *clt_strerror(int code);
/* Text of the last CUDA error seen by this context ("" if none).                                 */
const char *clt_last_cuda_error(const clt_ctx *ctx);
/* Library version string, e.g. "clt-b200 0.1 (sm_100a)".                                         */
const char *clt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CLT_H */
