/* fvnl.h -- C ABI of the B200-native finite-volume step for nonlinear thermoviscous acoustics.
 *
 * Implements the per-time-step 2-D high-resolution finite-volume update of arXiv 1311.3004
 * (Velasco-Segura & Rendon), Sections II-III.  "PAPER.md:<line>" cites /root/reference/PAPER.md.
 *
 *   conservation system (19a,b) in the dimensionless form (21)-(23)
 *   fractional steps: x-sweep (24) -> y-sweep (25) -> source step (26)
 *   wave-propagation update (27), fluctuations (28),(29), MC-limited F~ (30)
 *   Roe matrix of the arithmetic-mean primitive state, eigenvalues (32)-(34)
 *   CFL number nu and lagged time-step control towards nu_W
 *   boundary cells: analytic (41), focused source (43), zero-order extrapolation,
 *   reflecting border
 *
 * General conventions
 *   - Every function returns an int status (0 = FVNL_OK) unless noted.  No exceptions, no aborts, no output.
 *   - The library runs on the CUDA device that is current when fvnl_create is called and on the CUDA stream
 *     passed to it.  There is NO CPU fallback: without a usable device fvnl_create returns FVNL_ECUDA.
 *   - The caller owns every buffer it passes.  The library copies in / out and never keeps a caller pointer,
 *     except `workspace` (fvnl_create), which must stay valid until fvnl_destroy.
 *   - State = the paper's dimensionless conserved vector q of (22), PAPER.md:133:
 *         q1 = rho/rho0,  q2 = q1*u/c0,  q3 = q1*v/c0        (equilibrium: 1, 0, 0)
 *     as three separate contiguous planes of nx*ny values, index = j*nx + i, i = x index (fastest).
 *   - Pointers named `*_dev_or_host` are device pointers when `where & FVNL_ON_DEVICE`, host pointers otherwise.
 *   - SI units at the boundary (m, s, Hz); only lambda = c0 dt/dx, kappa = delta dt/dx^2 and beta enter the update.
 */
#ifndef FVNL_H
#define FVNL_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fvnl_ctx fvnl_ctx;

/* Host-side status codes (returned as such) and sticky device flags (OR-ed together, returned by fvnl_step). */
enum {
    FVNL_OK = 0,
    FVNL_EARG = 1,      /* bad argument                                                    */
    FVNL_EALLOC = 2,    /* workspace too small / allocation failed                         */
    FVNL_ECUDA = 3,     /* CUDA runtime error or no device                                 */
    FVNL_ESTATE = 4,    /* call order (e.g. step before set_state)                         */
    FVNL_ESIZE = 5,     /* grid larger than the static scratch array of fvnl_step_noalloc  */
    FVNL_ECFL = 16,     /* a step ran with nu > 1 or kappa_x + kappa_y > 1/2 */
    FVNL_ENONREAL = 32, /* square-root argument of (32),(33) negative        */
    FVNL_ENONPOS = 64,  /* q1 <= 0 met in a primitive conversion                            */
    FVNL_ENAN = 128     /* NaN met                                                          */
};

/* Medium of (19): small-signal sound speed [m/s], equilibrium density [kg/m^3], coefficient of nonlinearity
 * beta = 1 + B/(2A), sound diffusivity delta [m^2/s] (18). */
typedef struct { double c0, rho0, beta, delta; } fvnl_medium;

/* Edge kinds.  PERIODIC must be set on both sides of an axis.  REFLECT mirrors the interior and negates the
 * normal momentum (the paper's reflecting bottom border).  EXTRAP is zero-order extrapolation
 * ("simplified absorbing").  SOURCE prescribes the ghost cells analytically (below). */
enum { FVNL_BC_EXTRAP = 0, FVNL_BC_PERIODIC = 1, FVNL_BC_REFLECT = 2, FVNL_BC_SOURCE = 3 };
enum { FVNL_SIDE_XLO = 0, FVNL_SIDE_XHI = 1, FVNL_SIDE_YLO = 2, FVNL_SIDE_YHI = 3 };

/* Source shapes.  With d = (coordinate of the ghost cell's centre along the edge, from the low corner) - centre_m,
 * lambda_w = c0/freq_hz, and, when 0 < focus_m < inf,  R = sqrt(d^2 + focus_m^2):
 *     tau = freq_hz*(t + t0_s) + d^2/(2*focus_m*lambda_w)          [periods]      tau of (43)
 *     SINE  : g = amp*sin(2 pi tau) for tau >= 0, else 0           (plane piston = SINE with focus_m <= 0)
 *     PACKET: g = amp*sin(2 pi tau)*exp(-(tau/4)^10)               (43d), PAPER.md:417 (exponent sign: DESIGN.md A13)
 *     q1 = 1 + g ; inward-normal momentum = g*focus_m/R ; along-edge momentum = -g*d/R      (43a-c)
 *     (focus_m <= 0 or infinite: plane wave, tau has no d term, normal momentum = g, along-edge momentum = 0).
 *   Both ghost layers of the edge take the same values (they sample (43) at the edge, A14).  Cells with
 *   |d| > half_aperture_m (> 0) behave as FVNL_BC_EXTRAP; half_aperture_m <= 0: the whole edge.
 *     TANH  : q1 = 1 - amp*tanh(steep*(xi - c0*(t + t0_s))), (q2, q3) = (q1 - 1)*(cos theta, sin theta)   (41)
 *   with xi = x*cos(theta) + y*sin(theta), (x, y) = the ghost cell's OWN centre measured from the x-lo / y-lo edge
 *   (negative in the low ghosts; x in the frame that fvnl_shift moves): (41) is a field, the same on whichever side it is
 *   attached to.  theta = theta_T, the propagation angle from the x axis (0: q2 = q1 - 1, q3 = 0 as printed).
 *   steep [1/m].
 *   Sources are evaluated at t_n, the time at the start of the step. */
enum { FVNL_SRC_SINE = 0, FVNL_SRC_PACKET = 1, FVNL_SRC_TANH = 2 };
typedef struct {
    int shape;
    double amp;             /* dimensionless: u0/c0 = p'/(rho0 c0^2)                                   */
    double freq_hz;
    double focus_m;         /* F of (43); <= 0 or inf: plane wave                                      */
    double centre_m;        /* aperture centre along the edge, from the low corner                     */
    double half_aperture_m; /* a of PAPER.md:405; <= 0: whole edge                                     */
    double t0_s;
    double steep;           /* TANH only                                                               */
    double theta;           /* TANH only: propagation angle theta_T [rad]                              */
} fvnl_source;

/* Precision of a context.  64: the paper's, state planes of double holding q.  32: the single-precision
 * variant ("sometimes ... as good", faster), PERTURBATION FORM: the state planes are float and hold
 * (rho' = q1 - 1, q2, q3), so that fp32 round-off is relative to the acoustic perturbation and not to the unit background;
 * all arithmetic of the step is fp32, the clock (t, dt, M) and the analytic boundary cells stay fp64.  Everything else
 * (edges, sources, modes, flags) is the same; the comparison kernels (fvnl_set_option) exist in fp64 only.
 *
 * Bytes of device memory the context needs for an nx x ny grid (two states, clock, analytic ghost cells); 0 for bad
 * arguments. */
size_t fvnl_workspace_bytes(int nx, int ny, int precision);

/* Create a context.  nx, ny >= 4; dx, dy, c0, rho0 > 0; beta >= 1; delta >= 0; precision = 64 or 32.
 * cuda_stream: a cudaStream_t (NULL = default stream); all work of this context is issued on it.
 * workspace: DEVICE memory of at least fvnl_workspace_bytes() bytes, 256-byte aligned, owned by the caller (e.g. a
 * torch tensor) and kept alive until fvnl_destroy; or NULL, then the library cudaMallocs it itself.
 * Initial state: equilibrium (1,0,0), all edges EXTRAP, t = 0.
 * Errors: FVNL_EARG, FVNL_EALLOC (workspace_bytes too small / cudaMalloc failed), FVNL_ECUDA. */
int fvnl_create(fvnl_ctx** out, int nx, int ny, double dx, double dy, const fvnl_medium* medium, int precision,
                void* cuda_stream, void* workspace_dev, size_t workspace_bytes);

/* Release the context (and its workspace if the library allocated it).  NULL is allowed. */
void fvnl_destroy(fvnl_ctx* ctx);

/* Set the rule for one edge.  src is read for FVNL_BC_SOURCE only (copied).  FVNL_EARG on bad side/kind/shape or
 * missing src.  A lone PERIODIC side is reported by fvnl_step (FVNL_EARG). */
int fvnl_set_bc(fvnl_ctx* ctx, int side, int kind, const fvnl_source* src_or_null);

/* Where the planes passed to fvnl_set_state / fvnl_get_state live and what they hold (OR-ed):
 *   FVNL_ON_DEVICE   device pointers (else host pointers);
 *   FVNL_PLANES_F64  fp32 contexts only, device pointers only: the planes are double and hold the standard state q; the
 *                    library converts to / from its stored form (rho', q2, q3) in a kernel.  Ignored by fp64 contexts.
 * Without FVNL_PLANES_F64 the planes are in the context's own form: double q (precision 64), float (rho', q2, q3) (32). */
enum { FVNL_ON_HOST = 0, FVNL_ON_DEVICE = 1, FVNL_PLANES_F64 = 2 };

/* Copy a state in (three planes of nx*ny values, see above).  Resets the sticky flags and the lagged maximum M (the next
 * CFL-mode step starts with the pre-pass), keeps t.  Device input: asynchronous, everything (copies and the clock reset)
 * is queued on the stream and the call returns at once.  Host input: the call synchronises the stream, so the buffers may
 * be reused when it returns. */
int fvnl_set_state(fvnl_ctx* ctx, const void* q1_dev_or_host, const void* q2_dev_or_host,
                   const void* q3_dev_or_host, int where);

/* Moving domain, the second stage of PAPER.md:281-287 ("the domain moves with the propagation wave"): move the domain by
 * `cells` >= 0 cells in +x.  The state is re-indexed, Q_new(i, j) = Q_old(i + cells, j); the columns that enter on the right
 * are the x-hi ghost cells of the old state by the x-hi rule at the current time (EXTRAP: copies of the last column;
 * SOURCE: the analytic cell at its own centre, inside the aperture), and the frame in which TANH sources are written
 * moves along.  t and the lagged M are untouched.  Asynchronous (one kernel on the stream).  The caller decides when to
 * move (e.g. one cell each time c0*t has advanced by dx) and which rule the x-lo edge follows in this stage (the paper:
 * zero-order extrapolation).
 * Errors: FVNL_EARG (cells < 0 or >= nx; x edges PERIODIC, x-hi REFLECT), FVNL_ESTATE. */
int fvnl_shift(fvnl_ctx* ctx, int cells);

/* Set the clock: simulation time t [s] and the lagged maximum M [1/m] of the previous step.
 * last_M <= 0: M unknown -- the next CFL-mode step recomputes it by the pre-pass on the state as it is then, unless a
 * fixed-dt step has been taken in between (M is then that step's).  Asynchronous (queued on the stream).
 * (t, M) from fvnl_get_info + the state from fvnl_get_state restart a run bit-exactly. */
int fvnl_set_clock(fvnl_ctx* ctx, double t_s, double last_M);

/* Advance nsteps time steps.  Each step: ghost rule -> x-sweep (24) -> y-sweep (25) -> source step (26), (27)-(34).
 *   mode 0: value = dt [s], fixed.
 *   mode 1: value = nu_W; dt_n = nu_W/(c0*M_{n-1}), M = max over all x-interfaces of |s|/dx and y-interfaces of
 *           |s|/dy met during the previous step; first step: a pre-pass over the current state.
 *           No step is rejected; a step that ran with nu_n = c0*dt_n*M_n > 1 sets FVNL_ECFL.
 * The steps are queued on the stream without host synchronisation, ONE kernel launch per time step: dt lives on the
 * device, and the thread block of the step kernel that finishes last ends the step (M_n, nu_n, t, the next dt, the
 * analytic ghost cells of the next step).  On grids of at most 2^18 cells pairs of steps are replayed from a CUDA graph
 * captured on first use.  The call then reads back the clock {flags, t, dt, M, steps} and returns the OR of the sticky
 * device flags (0 = clean).  With flags set the state is undefined but readable.
 * Errors: FVNL_EARG (nsteps < 0, value <= 0, bad mode, lone PERIODIC, mode 0 with delta*dt*(1/dx^2+1/dy^2) > 1/2),
 * FVNL_ECUDA. */
int fvnl_step(fvnl_ctx* ctx, long nsteps, double value, int mode);

/* Copy the current state out (three planes of nx*ny values, `where` as for fvnl_set_state).  Synchronises the stream for
 * host output. */
int fvnl_get_state(fvnl_ctx* ctx, void* q1_dev_or_host, void* q2_dev_or_host, void* q3_dev_or_host, int where);

/* Clock and step statistics after the last fvnl_step: time [s], last dt [s], CFL number of the last step
 * nu = c0*dt*M, last M [1/m], number of steps taken since fvnl_create.  Any pointer may be NULL.  Synchronises. */
int fvnl_get_info(fvnl_ctx* ctx, double* t_s, double* last_dt_s, double* last_cfl, double* last_M,
                  long* steps_done);

/* Kernel selection (tuning and cross-check aid; results agree to rounding for every choice).
 * FVNL_OPT_KERNEL:  FVNL_KERNEL_DEFAULT = the one-pass step kernel (each state array read once and written once per
 *   step); FVNL_KERNEL_UNFUSED = the three-pass form (x-sweep, y-sweep, source step as separate kernels through HBM;
 *   allocates one more y-extended state with cudaMalloc on first use) -- the measured "what fusion buys" point.
 * FVNL_OPT_VARIANT (one-pass kernel): 0 = warp-specialised kernel k_step_ws (default), 1 = single-role kernel
 *   k_step_fused (one thread does both sweeps of its column; evaluates analytic edge cells in place).
 * FVNL_OPT_ROWS_PER_BLOCK: rows one thread block of the one-pass kernel marches over (0 = automatic).
 * FVNL_OPT_KERNEL_TIMING: see fvnl_get_kernel_time.
 * FVNL_OPT_SMALL_GRID: 1 (default) = a double-precision grid of at most 16384 cells runs ALL steps of a fvnl_step call in
 *   one launch of one thread-block cluster (up to 16 CTAs; the time loop, the CFL clock and the analytic edge cells inside
 *   the kernel) instead of one launch per step -- such grids are bound by launches and latency (C1: 512 x 4 cells);
 *   0 = always one launch per step.  Ignored while FVNL_OPT_KERNEL_TIMING is on or another kernel / variant is selected. */
enum { FVNL_OPT_KERNEL = 0, FVNL_OPT_ROWS_PER_BLOCK = 1, FVNL_OPT_KERNEL_TIMING = 2, FVNL_OPT_VARIANT = 3,
       FVNL_OPT_SMALL_GRID = 4 };
enum { FVNL_KERNEL_DEFAULT = 0, FVNL_KERNEL_UNFUSED = 1 };
int fvnl_set_option(fvnl_ctx* ctx, int option, int value);

/* Per-kernel device time, for the roofline figures of bench.py.  With FVNL_OPT_KERNEL_TIMING set to 1, fvnl_step
 * records a CUDA event pair on the context's stream around every launch of the kernels below (no host
 * synchronisation is added; at most 65536 launches are kept between two reads).  fvnl_get_kernel_time
 * synchronises the stream, returns the summed device time [ms] and the number of launches of kernel `which`
 * since the previous read of that kernel, and resets both.  FVNL_EARG on a bad `which`.
 *   FVNL_TIMED_STEP  : the fused one-pass step kernel (default path)
 *   FVNL_TIMED_XSWEEP / _YSWEEP / _SOURCE : the three kernels of the unfused path */
enum { FVNL_TIMED_STEP = 0, FVNL_TIMED_XSWEEP = 1, FVNL_TIMED_YSWEEP = 2, FVNL_TIMED_SOURCE = 3, FVNL_TIMED_KINDS = 4 };
int fvnl_get_kernel_time(fvnl_ctx* ctx, int which, double* total_ms, long* launches);

/* Number of kernels this context has launched so far (step kernels, pre-pass, clock, boundary); for bench accounting. */
long fvnl_kernel_launches(const fvnl_ctx* ctx);

/* ---- MEASUREMENT AID, not part of the method --------------------------------------------------------------------------
 * FP64-pipe probe for the roofline denominator of bench.py: runs a register-only kernel of independent DFMA chains (16
 * warps per SM, 8 chains per thread) on the current device and stream and returns the achieved rate in TFLOP/s (FMA = 2
 * flop), best of three.  Needs no context, touches no state.  Errors: FVNL_EARG, FVNL_ECUDA. */
int fvnl_probe_fp64(void* cuda_stream, double* tflops);

/* ---- ALLOCATION-FREE ENTRY POINT -------------------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 * ONE fixed-dt time step Q(t) -> Q(t + dt) of the whole path (ghost rules, x-sweep (24), y-sweep (25), source step (26);
 * PAPER.md:147-279) by the three-pass kernels, with no context and no workspace.  The three-pass form needs scratch memory --
 * Q* on the y-extended mesh, Q**, and the clock block (dt, lambda, kappa, running maxima, flags): here it lives in a
 * file-scope `static __device__` array of FVNL_NOALLOC_MAX_BYTES = 16 MiB that every GPU that loads the library holds until
 * the process exits.  The call launches five kernels on `cuda_stream` and returns without synchronising; it calls no
 * cudaMalloc, cudaFree, cudaMemcpy or allocating library routine (the first call on a device resolves the array's device
 * address with cudaGetSymbolAddress: make that call outside a graph capture).
 *   q*_in / q*_out   DEVICE pointers, nx*ny doubles each (layout of fvnl_set_state), in != out; the caller owns them.
 *   bc_kind[4]       FVNL_BC_* per side (FVNL_SIDE_* order); bc_source[s] is read for FVNL_BC_SOURCE sides only (may be NULL
 *                    otherwise, and bc_source itself may be NULL when no side is a SOURCE).
 *   t, dt            time at the start of the step and the time step [s] (fvnl_step's mode 0).
 *   flags_dev        DEVICE pointer to one int that receives the step's flag word (FVNL_ECFL ... FVNL_ENAN, 0 = clean), or NULL.
 * Limit: 6 nx ny + 12 nx + 64 doubles must fit the array (e.g. 512 x 512 or 580 x 580 cells); larger grids are rejected with
 * FVNL_ESIZE before anything is launched.  fp64 only.
 * Sharing: every call on a device uses the same array, which keeps the previous call's contents; the call itself resets what
 * must start at zero (running maxima, flags).  Calls that OVERLAP on one GPU (different streams, or graphs replayed
 * concurrently) race on it: serialise them.
 * Errors: FVNL_EARG (as fvnl_create / fvnl_set_bc / fvnl_step, or in == out), FVNL_ESIZE, FVNL_ECUDA. */
#define FVNL_NOALLOC_MAX_BYTES (16u << 20)
int fvnl_step_noalloc(int nx, int ny, double dx, double dy, const fvnl_medium* medium, const int bc_kind[4],
                      const fvnl_source* const bc_source[4], double t, double dt, const double* q1_in, const double* q2_in,
                      const double* q3_in, double* q1_out, double* q2_out, double* q3_out, int* flags_dev, void* cuda_stream);

/* Text for a status code or flag word (static storage). */
const char* fvnl_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* FVNL_H */
