/*
 * wave2d.h -- C ABI of libwave2d.so: B200-native (sm_100a) ADI time stepping for the 2D acoustic
 * wave equation
 *
 *     u_tt - c(t) (u_xx + u_yy) = f(t,x,y)  on [0,T] x [0,l]^2,   u(0) = phi, u_t(0) = psi,
 *     u = 0 on the boundary                                     (eqs (2.1)-(2.5))
 *
 * discretised on the grid t_k = k tau, x_i = i h1, y_j = j h2, h_d = l/N_d ((2.6)-(2.7))
 * by the split implicit scheme (2.11)-(2.12) and stepped by Algorithm 1
 * (PAPER.md:99-118): per time step one batched family of tridiagonal solves along x (one per grid
 * row), one along y (one per grid column), and a rotation of the time levels.  Every step of that
 * path runs in hand-written CUDA kernels; there is no CPU fallback.
 *
 * Conventions (all entry points):
 *   - extern "C"; every function returns an int status (WAVE2D_OK == 0, errors < 0) and never throws
 *     or aborts.  wave2d_strerror() names a status, wave2d_last_error() gives detail (CUDA error text).
 *   - N1, N2 >= 2 are the paper's INTERVAL counts; a line along x has n1 = N1-1 unknowns, along y
 *     n2 = N2-1.  Boundary nodes are never stored, read or written: (2.10) fixes them to 0.
 *   - Field arrays (phi, psi, s, u_out) are INTERIOR arrays of n2 rows x n1 columns: node (i,j),
 *     1 <= i <= n1, 1 <= j <= n2, lives at [(j-1)*ld + (i-1)], ld >= n1 in ELEMENTS.  The element type
 *     is the handle's dtype (double for WAVE2D_F64, float for WAVE2D_F32).
 *   - Field pointers may be HOST or DEVICE pointers (detected with cudaPointerGetAttributes; a torch
 *     tensor passes .data_ptr()).  Inputs are copied during the call: the caller keeps ownership and may
 *     free them on return.  Time-sample arrays (c_half, g_half) are HOST double arrays for both dtypes.
 *   - Half-level index n = 0,1,2,...: t = n tau/2; the half-step n -> n+1 is implicit in x for even n and
 *     in y for odd n.  c_half[n] = c(n tau/2), g_half[n] = g(n tau/2).
 *   - The handle owns all device memory it allocates (three pitched field buffers, the optional source
 *     field, a per-half-step scalar table, the work plan) and frees it in wave2d_destroy().
 *   - One handle is single-threaded; distinct handles are independent.  Work is asynchronous on the
 *     handle's stream unless stated otherwise.
 *
 * State machine: create -> (set_* in any order; set_initial required) -> run* -> get.
 *   run before set_initial                      -> WAVE2D_ERR_STATE
 *   cumulative steps > M                        -> WAVE2D_ERR_RANGE
 *   set_speed / set_source / set_option after the first run -> WAVE2D_ERR_STATE
 *   set_initial at any time resets the step count k to 0.
 */
#ifndef WAVE2D_H
#define WAVE2D_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wave2d_s wave2d_t; /* opaque */

enum { WAVE2D_F64 = 0, WAVE2D_F32 = 1 };

enum {
    WAVE2D_OK = 0,
    WAVE2D_ERR_ARG = -1,         /* NULL / out-of-range argument                                  */
    WAVE2D_ERR_STATE = -2,       /* call not allowed in the handle's current state                */
    WAVE2D_ERR_ALLOC = -3,       /* host or device allocation failed                              */
    WAVE2D_ERR_CUDA = -4,        /* a CUDA call failed; see wave2d_last_error()                   */
    WAVE2D_ERR_UNSUPPORTED = -5, /* no solver path can handle this size / option on this device   */
    WAVE2D_ERR_RANGE = -6        /* more than M steps requested                                   */
};

/* Solver selection for wave2d_set_option(h, "solver", v). */
enum {
    WAVE2D_SOLVER_AUTO = 0,     /* LINE on small grids; else streamed kernels where the decay bound
                                 * rho^H <= tol allows, else EXACT                                        */
    WAVE2D_SOLVER_EXACT = 1,    /* whole lines on chip, nothing truncated (any tau/h); a line must fit one CTA's shared
                                 * memory: x lines up to 24576 unknowns in fp64 (49152 in fp32), y lines up to 22752
                                 * (45504); longer ones give ERR_UNSUPPORTED at the first plan, with the limit in the text */
    WAVE2D_SOLVER_STREAM = 2,   /* force the streamed kernels; ERR_UNSUPPORTED if the bound fails        */
    WAVE2D_SOLVER_LINE = 3      /* small grids (at most 256 unknowns per line in both directions): the whole step
                                 * loop in one launch of one thread-block cluster, every line solved whole and
                                 * exactly on chip by a warp-shuffle scan (any tau/h); AUTO picks it when the grid
                                 * fits; forcing it on a larger grid gives ERR_UNSUPPORTED                        */
};

/* =====================================================================================================
 * STABLE INTERFACE: the calls of the paper's problem statement.  Everything from here to the
 * banner "DIAGNOSTICS AND TUNING" below keeps its meaning between versions.
 * ===================================================================================================== */

/*
 * Create a solver for the grid of (2.6)-(2.7): N1 x N2 intervals on [0,l]^2, time step tau, at most M
 * steps (T = M tau), dtype WAVE2D_F64 or WAVE2D_F32.  Defaults: c == 1, no source, gamma = 2,
 * kappa = 1/2 (see wave2d_set_option).  Uses the current CUDA device and a non-blocking stream of its own.
 * Errors: ERR_ARG (N < 2, l <= 0, tau <= 0, M < 0, bad dtype, out == NULL), ERR_ALLOC, ERR_CUDA
 * (no device, or not an sm_100 device).  Whether a solver path can take the grid depends on options and speed samples
 * that are set later, so a line too long for every path is reported by the first plan instead: wave2d_run or
 * wave2d_get_info return ERR_UNSUPPORTED, never this call.
 */
int wave2d_create(wave2d_t **out, int N1, int N2, double l, double tau, int M, int dtype);

/* Free the handle and everything it owns.  NULL-safe.  Synchronises the handle's stream first. */
void wave2d_destroy(wave2d_t *h);

/* Use `cuda_stream` (a cudaStream_t) for all later work; NULL returns to the handle's own stream.  On the
 * legacy default stream the step loop falls back from graph replay to plain launches. */
int wave2d_set_stream(wave2d_t *h, void *cuda_stream);

/*
 * Options (before the first run only):
 *   "gamma"  time-quotient constant, > 0.  Default 2.   | gamma = 2, kappa = 1/2 is the consistent
 *   "kappa"  source weight.              Default 0.5.   | locally-one-dimensional form of (2.11)-(2.12);
 *                                                       | gamma = kappa = 1 is the scheme as printed
 *                                                       |, which solves u_tt = 2c Lap u + 4f.
 *   "ly"     extent in y of this grid (h2 = ly / N2); default 0 = l.  For row blocks of a larger domain (wave2d_get_rows).
 *   "sigma"  weight of the implicit operator in the split scheme, in (0, 1].  Default 0.5 = (2.11)-(2.12):
 *            alpha+ = sigma tau^2 c_{n+1} / h_d^2 on w_{n+1}, alpha- = (1 - sigma) tau^2 c_{n-1} / h_d^2 on w_{n-1}.
 *            sigma = 1 with gamma = 1 and c = 1 is the tridiagonal system Listing 1 prints (PAPER.md:157-162:
 *            a = c = tau^2, b = 2 tau^2 + h^2, f = h^2 u^{k-1} - 2 h^2 u^k), the fully implicit three-level step.
 *            Scheme 0 only (ERR_UNSUPPORTED with scheme 1, whose weight is 1/2 by definition).
 *   "start"  scheme 1 only.  1 (default): (2.9) as printed, u^1 = phi + tau psi (first order).
 *            2: u^1 = phi + tau psi + (tau^2 / 2) (c^0 Lap_h phi + g^0 s), the Taylor value with u_tt from (2.1): the
 *            three-level scheme (2.8) is then second order in tau also for psi != 0 or f != 0.  The extra term needs
 *            the final speed and source samples, so it is added by the first wave2d_run with steps > 0: until then
 *            -- after wave2d_run(h, 0) too, and always when M = 1, where no step can be run -- wave2d_get returns
 *            the first-order phi + tau psi.  With scheme 0, wave2d_run returns ERR_UNSUPPORTED.
 *   "scheme" 0 (default): the split scheme (2.11)-(2.12) driven by Algorithm 1.
 *            1: the factorised form of the unsplit three-level scheme (2.8),
 *                 (I - ax+ Dx)(I - ay+ Dy) u^{k+1} = 2 u^k - (I - ax- Dx)(I - ay- Dy) u^{k-1} + tau^2 f^k,
 *               a_d^+- = tau^2 c^{k+-1} / (2 h_d^2): one x solve and one y solve per step, 5 field passes
 *               instead of 6.  Uses c_half[2k], g_half[2k] only; gamma and kappa do not apply.  Start (2.9) as
 *               printed: u^0 = phi, u^1 = phi + tau psi, so wave2d_set_initial leaves the handle at time level 1
 *               (wave2d_steps_done = 1, wave2d_get = u^1; needs M >= 1) and wave2d_run(M - 1) reaches level M.
 *               wave2d_get_prev is available only before the first solve (it returns u^0), then
 *               ERR_UNSUPPORTED: the ring carries (I - ay Dy) u^{k-1}, not u^{k-1}.  Must be set before
 *               wave2d_set_initial (ERR_ARG afterwards).  Uses a fourth field buffer.
 *   "solver" one of WAVE2D_SOLVER_*.     Default AUTO.
 *   "graph"  1 (default): the step loop is replayed as CUDA Graphs; 0: the same kernel sequence launched directly.
 *            The loop runs in chunks of 2^i time steps, longest first (20 steps = 16 + 4); one graph per chunk length is
 *            captured, instantiated and uploaded when the plan is made (first wave2d_run / wave2d_get_info after the
 *            last set_* call; wave2d_run(h, 0) forces it), never inside a later run call.  The kernels take the buffer
 *            roles of the time-level ring from the device step counter, so every graph serves every phase of the
 *            ring and no step of any run call is launched outside a graph.
 *   "graph_steps"  longest chunk in time steps: 1, 2, 4, 8, 16 or 32 (default 32).
 *   "shape_x", "shape_y"   tuning: kernel shape variant 0..3 (units per stage = consumer warps / stages).
 *   "pdl"    1 (default): sweep kernels are launched with programmatic stream serialization, so that a kernel's
 *            prologue overlaps the tail of the previous one (it waits for it before touching the fields).
 *   "early"  1 (default): early start -- a CTA that becomes resident while the previous sweep is still finishing its
 *            last drawn pieces begins with a piece of its share that touches only grid lines that sweep completed in
 *            its static part; needs "pdl".  0: every CTA waits for the whole previous sweep.
 *   "resident"  1 (default): small grids of the split scheme keep the time levels in the cluster's distributed shared
 *            memory for a whole run call; 0: the small-grid kernel that goes through global memory.
 *   "trace"  1: sweep kernels record per-CTA timing (see wave2d_get_trace).  Default 0.
 *   "static_frac"          tuning: share of a sweep's work dealt out statically (0..1; default 0.70 in fp64, 0.75 in fp32); the rest is
 *                          drawn from the ticket counter in short pieces.
 *   "tail_min", "tail_max", "tail_div"   tuning of the drawn pieces: shortest / longest length in stages (tail_min 0 =
 *                          planned from the stage size; tail_max default 6) and the divisor d of the guided length
 *                          remaining / (d * CTAs) (default 2).
 *   "quota_x", "quota_y"   tuning: length in stages of every piece of work a line is cut into (0 = planned:
 *                          guided self-scheduling, long pieces first, short ones last).
 * Errors: ERR_ARG (unknown name / bad value), ERR_STATE.
 */
int wave2d_set_option(wave2d_t *h, const char *name, double value);

/*
 * Caller-owned memory for the time levels (SURVEY.md 8b "Memory"; optional).  By default the handle cudaMallocs its
 * ring of time levels (three fields, four with scheme 1: all but a few KB of what it owns).  A caller that manages
 * device memory itself -- PyTorch's caching allocator, an arena -- can hand the library a block instead:
 * wave2d_workspace_bytes gives the size for the handle's current scheme, wave2d_set_workspace attaches a DEVICE block of
 * at least that size, 256-byte aligned (ERR_ARG otherwise; a torch allocation is).  The handle frees its own fields,
 * zeroes the block and keeps every time level in it; the caller must keep the block alive and untouched until
 * wave2d_destroy or wave2d_set_workspace(h, NULL, 0) (back to memory of its own).  The small tables and counters stay
 * handle-owned.  Allowed before wave2d_set_initial only (ERR_STATE afterwards), and after the scheme is chosen:
 * wave2d_set_option(h, "scheme", 1) on a handle with a three-field workspace gives ERR_STATE.
 * For a step loop that allocates nothing at all on small grids see wave2d_small_steps_static.
 */
int wave2d_workspace_bytes(const wave2d_t *h, unsigned long long *bytes);
int wave2d_set_workspace(wave2d_t *h, void *workspace, unsigned long long bytes);

/*
 * Initial data (2.2)-(2.3), discretised as in (2.9) adapted to half-levels:
 *   u^0 = phi,  u^{-1/2} = phi - (tau/2) psi     (psi == NULL means psi = 0, i.e. Algorithm 1's "u = U0").
 * Resets the step count to 0.  Synchronous for host pointers.
 */
int wave2d_set_initial(wave2d_t *h, const void *phi, const void *psi, long ld);

/*
 * Checkpoint / resume (scheme 0): the state of Algorithm 1 is the pair (u, U0) = (u^{k-1/2}, u^k),
 * which wave2d_get_prev / wave2d_get return.  wave2d_set_state puts a handle at time level k with that pair, so
 * that a run continued from a checkpoint is bit-identical to the uninterrupted one (same speed / source samples).
 * Errors: ERR_ARG (k outside 0..M), ERR_UNSUPPORTED (scheme 1).  Synchronous for host pointers.
 */
int wave2d_set_state(wave2d_t *h, int k, const void *u_prev_half, const void *u, long ld);

/*
 * Speed samples c_half[n] = c(n tau/2), n = 0..2M (count == 2M+1), or one constant (count == 1).
 * Every value must be > 0 ("positive speed function"), else ERR_ARG.  c_{-1} := c_0.
 */
int wave2d_set_speed(wave2d_t *h, const double *c_half, int count);

/*
 * Spatially varying speed: c(t,x,y) = c_half[n] * cs(x,y), separable like the source below.
 * cs: interior array, every value > 0 (else ERR_ARG); NULL returns to c = c(t).  Algorithm 1 computes the tridiagonal
 * elements a_i, b_i, c_i point by point: the weights of (2.11)/(2.12) are taken at the point of the
 * equation, a_p = tau^2 c_{n+1} cs_p / (2 h_d^2).  The systems are then no longer Toeplitz: every line computes its own
 * elimination pivots (a scan of linear-fractional maps, csrc/exact.cuh) inside the whole-line solvers, which read one
 * more field per sweep (32 instead of 24 bytes per point in fp64).  Split scheme only (scheme 1: ERR_UNSUPPORTED), lines
 * of at most 4096 unknowns (ERR_UNSUPPORTED at the first run otherwise), solver AUTO or EXACT.  Before the first run.
 * The field is checked before anything changes: a call that fails with ERR_ARG leaves a previously accepted field (or
 * c = c(t)) in force.
 */
int wave2d_set_speed_field(wave2d_t *h, const void *cs, long ld);

/*
 * Source f(t,x,y) = g(t) s(x,y).  s: interior array (NULL clears the source);
 * g_half[n] = g(n tau/2), n = 0..2M-1 (count >= 2M), or NULL for g == 1 (a time-independent full-grid
 * source).  Half-step n uses g_half[n]: f^k in (2.11), f^{k+1/2} in (2.12).
 */
int wave2d_set_source(wave2d_t *h, const void *s, long ld, const double *g_half, int count);

/*
 * Advance `steps` time steps (Algorithm 1's loop body: x-sweep (2.11), y-sweep (2.12), rotate levels).
 * Asynchronous on the handle's stream.  Errors: ERR_STATE, ERR_RANGE, ERR_UNSUPPORTED, ERR_CUDA.
 */
int wave2d_run(wave2d_t *h, int steps);

/* Copy u^k (k = steps done so far) / u^{k-1/2} to u_out (host or device).  Synchronises the stream. */
int wave2d_get(wave2d_t *h, void *u_out, long ld);
int wave2d_get_prev(wave2d_t *h, void *u_out, long ld);

/*
 * Row blocks of a time level (split scheme only; ERR_UNSUPPORTED with scheme 1): rows [j0, j0 + count) of level 0 = u^k or
 * level 1 = u^{k-1/2}, `count` rows of n1 values, row stride ld >= n1, host or device pointer.  wave2d_get_rows copies
 * them out, wave2d_set_rows overwrites them (both synchronise the handle's stream).  With option "ly" (the extent in y of
 * THIS grid, h2 = ly / N2, default l) a handle can hold a row block of a larger domain plus halo rows: the step of the
 * block is exact up to rho^G in its interior when G halo rows per side are refreshed from the neighbouring blocks after
 * every step (paper_2006_10142_b200/sharded.py).  Errors: ERR_ARG, ERR_STATE (no initial data).
 */
int wave2d_get_rows(wave2d_t *h, int level, int j0, int count, void *out, long ld);
int wave2d_set_rows(wave2d_t *h, int level, int j0, int count, const void *in, long ld);

/* Number of completed time steps k. */
int wave2d_steps_done(const wave2d_t *h, int *k);

/* Block until all work queued on the handle's stream has finished. */
int wave2d_sync(wave2d_t *h);

const char *wave2d_strerror(int status);
const char *wave2d_last_error(const wave2d_t *h);

/*
 * Small grids without any allocation: `steps` time steps of Algorithm 1 (split scheme (2.11)-(2.12),
 * PAPER.md:79-85, gamma = 2, kappa = 1/2, constant speed c, no source) in ONE kernel launch and nothing else -- no
 * handle, no cudaMalloc / cudaFree, no host allocation, no copy, no synchronisation.
 *
 * Who needs this.  Everything else in this header works on a wave2d_create handle, and a handle cudaMallocs its time
 * levels, counters and scalar table.  That is not possible for every caller: code that runs inside a framework whose
 * caching allocator has already taken the GPU's memory (a raw cudaMalloc from a library then fails while the framework
 * still reports free space), a service whose device-memory budget is fixed at start-up, or a loop that shares the GPU
 * with other streams (cudaMalloc and cudaFree synchronise the whole device and stall them).  Here the working memory of
 * the small-grid kernel -- the ring of three time levels and two scalar rows -- is a fixed array inside the library
 * image: 1 581 184 bytes (1.5 MiB) on every GPU that loads libwave2d.so, held from module load until the process exits.
 *
 * The limit.  Lines of at most 256 unknowns in each direction: N1, N2 <= 257.  Anything larger is refused with
 * WAVE2D_ERR_UNSUPPORTED and a message in errbuf; use a handle then.
 *
 * Arguments.  N1, N2, l, tau, dtype as in wave2d_create; c > 0 the constant speed.  The state of Algorithm 1 is the pair
 * (u^{k-1/2}, u^k): u_prev_half and u are read, u_out receives u^{k+steps} and u_prev_out (may be NULL)
 * u^{k+steps-1/2}, so a second call continues where the first stopped.  A start from (2.9) with psi = 0 passes phi as both
 * inputs.  All four are DEVICE arrays of the current device (host pointers are refused with ERR_ARG: staging them would
 * need a buffer), interior layout, n2 = N2-1 rows of n1 = N1-1 values of the dtype, one row stride ld >= n1 in elements
 * for all of them; the caller owns them.  The outputs may be the inputs (the kernel reads both inputs completely before
 * it writes an output).  cuda_stream: the cudaStream_t to launch into (NULL = the default stream); the call returns as
 * soon as the kernel is queued.  errbuf / errbuf_len: optional caller-owned buffer for the detail of a failure.
 *
 * Shared scratch.  There is ONE array per device for the whole process.  It keeps what the previous call left in it; each
 * call rewrites every byte it later reads (the pad columns that must be zero included), so calls of any sizes and dtypes
 * may follow each other.  But two calls whose kernels can overlap on the same GPU -- different streams with no event
 * between them, or two host threads -- race on it and both results are garbage: order them on one stream or with events.
 * Handles are not affected (they own their memory).
 *
 * First call on a device.  It does the one-time set-up for that device (looks up the array's device address -- every
 * device has its own copy -- and opts the kernels in to their shared-memory size), with that device current; if the
 * library's module was not loaded yet, this is also when the driver loads it and the array comes into being.  Make
 * this first call during start-up, before any stream capture.
 *
 * Errors: ERR_ARG (bad size / NULL / host pointer / ld < n1), ERR_UNSUPPORTED (beyond the limit; device ordinal >= 64),
 * ERR_CUDA (no sm_100 device, set-up or launch failed).
 */
int wave2d_small_steps_static(int N1, int N2, double l, double tau, double c, int steps, int dtype,
                              const void *u_prev_half, const void *u, void *u_out, void *u_prev_out, long ld,
                              void *cuda_stream, char *errbuf, int errbuf_len);

/* =====================================================================================================
 * DIAGNOSTICS AND TUNING: not part of the stable interface.  Used by bench.py, the tests and the profiles; names,
 * keys and record layouts may change with the kernels.  Of the options of wave2d_set_option the METHOD options are
 * stable ("gamma", "kappa", "sigma", "start", "scheme", "solver", "ly"); "graph", "graph_steps", "pdl", "early",
 * "resident", "trace", "shape_*", "static_frac", "tail_*", "quota_*" are tuning / diagnostic switches that never
 * change a result beyond rounding.
 * ===================================================================================================== */

/*
 * Introspection for benchmarks and tests.  name:
 *   "solver_x", "solver_y"   solver path in use per direction (WAVE2D_SOLVER_EXACT / _STREAM / _LINE), after planning
 *   "halo_x", "halo_y"       look-ahead H (points) with rho^H <= 1e-17 (fp64) / 1e-8 (fp32)
 *   "rho_x", "rho_y"         largest decay ratio rho over all half-steps
 *   "nbk_*"                  carry series length in units (halo = nbk * unit)
 *   "kb_*"                   leading units solved with the tabulated boundary pivots
 *   "chunks_*" (pieces of work), "grid_*", "ctas_per_sm_*", "smem_*", "threads_*", "unit_*", "quota_*",
 *   "upc_*" (units per CTA)  launch geometry
 *   "source_window"          points kept of the source field (its non-zero bounding box)
 *   "launches"               kernels launched by this handle so far (graph nodes count individually)
 *   "graph_launches"         graph replays issued by wave2d_run so far
 *   "plain_sweeps"           sweep kernels launched outside a graph so far (0 unless "graph" = 0 or
 *                            wave2d_profile_sweeps was used)
 *   "static_*", "safe_*"     pieces dealt out statically / of those, pieces that may start before the previous
 *                            sweep has ended (early start)
 *   "pitch"                  internal row pitch in elements
 *   "device_bytes"           device memory owned by the handle
 * The plan is (re)computed by this call if needed.  Errors: ERR_ARG.
 */
int wave2d_get_info(wave2d_t *h, const char *name, double *value);

/*
 * Time the two sweeps separately: runs `steps` time steps with plain launches and CUDA events around
 * every kernel on the handle's stream, returning the mean milliseconds per launch of the x-sweep and
 * y-sweep kernels.  Synchronous.  Counts toward the step total like wave2d_run.
 */
int wave2d_profile_sweeps(wave2d_t *h, int steps, double *ms_x, double *ms_y);

/*
 * Tracing (option "trace" = 1, before the first run): every CTA of a sweep kernel records its start and end
 * time (GPU global timer, ns), the SM it ran on and the number of pieces of work it had.
 * Copies the records of the most recent launch of direction dir (0 = x, 1 = y) to the host array
 * out[16 * capacity], 16 values per CTA: start_ns, end_ns, sm_id, pieces of work, 12 reserved;
 * *count = CTAs in the grid.
 * Errors: ERR_ARG (capacity < *count), ERR_STATE (tracing off or nothing planned).  Synchronises the stream.
 */
int wave2d_get_trace(wave2d_t *h, int dir, unsigned long long *out, int capacity, int *count);

/*
 * Host-only planning logic, exposed for inspection and tests; no device is touched.
 *
 * wave2d_host_scalars: the per-half-step scalar row for alpha+ = tau^2 c_{n+1}/(2 h^2),
 * alpha- = tau^2 c_{n-1}/(2 h^2), q = kappa tau^2 g_n ((2.11)-(2.12) times tau^2).  out[0..7] =
 * alpha-, q, rho, 1/(beta - alpha+ rho), -(gamma + 2 alpha-), alpha+, beta = gamma + 2 alpha+, 0; then K boundary
 * values cp_p = alpha+/u_pp and K values inv_p = 1/u_pp, u_pp the LU pivots of tridiag(-alpha+, beta, -alpha+),
 * K = (*count - 8) / 2.  Errors: ERR_ARG (also capacity < *count).
 *
 * wave2d_host_plan: how a sweep over `nlines` lines of n unknowns is cut into pieces of work for `slots` CTAs
 * (DESIGN.md 8.1): pieces[4 i ..] = (panel of 32 lines, first output unit, end output unit, stages); pieces
 * [0, *nstatic) are dealt out statically, CTA c owning [cta_off[c], cta_off[c+1]) (cta_off has slots + 1
 * entries), the rest is drawn at run time.  fixed_stages > 0: every piece that many stages, nothing static.
 */
int wave2d_host_scalars(double gamma, double alpha_plus, double alpha_minus, double q, double *out, int capacity,
                        int *count);
/*
 * wave2d_host_decay: the decay ratio rho of a sweep's systems tridiag(-alpha+, gamma + 2 alpha+, -alpha+) for lines of mesh
 * width extent / N at the speed sample c: alpha+ = sigma tau^2 c / (extent / N)^2 ((2.11)-(2.12) times tau^2,
 * PAPER.md:79-85), rho = the small root of alpha+ z^2 - (gamma + 2 alpha+) z + alpha+ -- the number the handle reports as
 * "rho_x" / "rho_y" once it exists.  A line may be cut where G further points are available with rho^G below the rounding
 * unit: the row-block driver (paper_2006_10142_b200/sharded.py) sizes its halo with it before any handle is created, so
 * that no arithmetic of the method lives outside the library.  Errors: ERR_ARG.
 */
int wave2d_host_decay(int N, double extent, double tau, double c, double gamma, double sigma, double *rho);
int wave2d_host_plan(int n, int nlines, int unit, int units_per_stage, int units_per_tile, int nbk, int slots,
                     int fixed_stages, double static_frac, int *pieces, int capacity, int *npieces, int *nstatic,
                     int *cta_off);

#ifdef __cplusplus
}
#endif
#endif /* WAVE2D_H */
