/*
 * dd4dvar.h -- C-ABI of the B200-native space-time decomposed 4D-Var (DD-4DVar) library.
 *
 * Method: arXiv 2205.06649 (text: /root/reference/PAPER.md; "l.N" below = PAPER.md line N).
 * The library evaluates, on every overlapping space-time subdomain Delta_j x Omega_i at once,
 * the regularised local functional J_ji (Def 13 eq (23)-(25), l.326-344) and its gradient by a
 * forward sweep of the discretised shallow-water model (eq (60)-(62) l.945-954, discretisation
 * l.971-989) and an adjoint backward sweep (eq (3)-(4) l.91-98), and drives a batched
 * per-subdomain L-BFGS (Remark 3 l.595; l.941) inside the outer loop of Algorithm 1 (l.443-472).
 * The readings of the paper that fix every constant and convention are listed in DESIGN.md.
 *
 * Conventions
 *   - Every `d_*` pointer is DEVICE memory owned by the caller (e.g. a torch tensor's data_ptr());
 *     every `h_*` pointer is HOST memory owned by the caller.  The library keeps no pointer to
 *     caller memory after a call returns, except the workspaces handed over with
 *     dd4dvar_set_workspace / dd4dvar_set_observations, which must outlive the handle.
 *   - Fields are ordered (h, u, v).  A global state is fp64 [3][nlat][nlon], longitude fastest;
 *     row j is the cell-centred latitude theta_j = -pi/2 + (j + 1/2) pi/nlat.
 *   - A subdomain's control / gradient is fp64 [3][ey][ex] on its extended tile (owned range
 *     plus `overlap` cells on every interior side, periodic in longitude, cut at the pole
 *     walls).  "All subdomains" arrays are the concatenation of these in subdomain order
 *     k = (window * p_lat + tile_row) * p_lon + tile_col; offsets from dd4dvar_subdomain_info.
 *   - All work is queued on the CUDA stream given to dd4dvar_create; calls that return host
 *     values synchronise that stream before returning.
 *   - Return value: 0 on success, otherwise
 *       -1 invalid argument            -2 decomposition does not fit the grid / window
 *       -3 called out of order         -4 CUDA error          -5 non-finite cost or gradient
 *       -6 problem larger than the built-in scratch array (dd4dvar_forecast_static only)
 *     Nothing is thrown across the ABI; dd4dvar_last_error gives the text of the last failure.
 *   - There is no CPU fallback: without a CUDA device every compute call returns -4.
 *   - Handles share nothing: every table and buffer a kernel reads belongs to one handle, so
 *     several live handles may work concurrently on different streams (one host thread per handle
 *     at a time; a handle itself is not re-entrant).  One side effect reaches beyond the handle:
 *     when the row-marching adjoint kernel is in use (paths 2 and 4), dd4dvar_set_workspace raises
 *     the device's cudaLimitPersistingL2CacheSize (never lowers it) and puts a persisting
 *     access-policy window for its scratch on the caller's stream; dd4dvar_destroy restores the
 *     stream's previous window, releases the persisting lines and resets the limit to the value
 *     found at set_workspace.  Two handles on the SAME stream would overwrite each other's window
 *     (performance only, never results).
 */
#ifndef DD4DVAR_H
#define DD4DVAR_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dd4dvar_s* dd4dvar_t; /* opaque, library-owned */

/* Grid and model constants: eq (60)-(62) l.945-954 (a, Omega, g), index ranges eq (67) l.976-980.
 * cos_clamp: lower bound of the cos(theta) metric factor (R3); diffusion: the
 * dimensionless index-space diffusion kappa of stage A (R3). */
typedef struct {
    int nlon, nlat;
    double radius, omega, gravity;
    double cos_clamp;
    double diffusion;
} dd4dvar_grid;

/* Uniform space-time decomposition, Def 3 l.128-154 and Def 16 l.755-763: p_lon x p_lat tiles
 * times q_time windows; `overlap` cells are added on each interior side (eq (70) l.1024).
 * mu = weight of the overlap term (25c) l.344; lambda = weight of the observation term eq (6)
 * l.111. */
typedef struct {
    int p_lon, p_lat, q_time;
    int overlap;
    double mu, lambda;
} dd4dvar_decomp;

/* Assimilation window: nsteps model steps of dt seconds, time levels 0..nsteps (Def 1 l.78-87). */
typedef struct {
    double dt;
    int nsteps;
} dd4dvar_window;

/* Local minimiser (L-BFGS, R10): history length, iterations per outer iteration,
 * maximum number of step halvings, Armijo constant.
 * path: 0 = choose automatically (5 where eligible, else 2, else 1), 1 = force the generic kernels (one block-tiled
 *       launch per step, any tile size), 2 = force the fused row-marching kernels (create fails with -2 if a tile does
 *       not fit), 3 = force the per-stage generic kernels (cross-check), 4 = wavefront forward kernel (tile resident in
 *       shared memory, one time step per warp, TMA-staged rows) + row-marching adjoint kernel, 5 = wavefront forward +
 *       wavefront adjoint kernels.  On 4 and 5 the cost terms (25a)-(25c) run in the kernel ck_cost between the two
 *       sweeps.  4 and 5: create fails with -2 unless every tile has a ghost ring in longitude, an even number of
 *       columns, at most 100 padded columns, an extended tile of at most 49 rows (80 rows up to 68 padded columns),
 *       and every window at least 4 steps. */
typedef struct {
    int lbfgs_m, n_inner, max_backtrack;
    double armijo_c1;
    int path;
} dd4dvar_opts;

/* Build the handle: row tables, decomposition, device descriptors.  `cuda_stream` is a
 * cudaStream_t (NULL = the legacy default stream).  Fails with -2 if a tile is narrower than its
 * ghost ring allows, a window has no step, or overlap regions would cover a cell more than 4x4
 * times. */
int dd4dvar_create(const dd4dvar_grid* grid, const dd4dvar_decomp* decomp,
                   const dd4dvar_window* window, const dd4dvar_opts* opts, void* cuda_stream,
                   dd4dvar_t* out);

/* Device memory the library needs besides the observations; the caller allocates it (256-byte
 * aligned) and hands it over before set_background. */
size_t dd4dvar_workspace_bytes(dd4dvar_t h);
int dd4dvar_set_workspace(dd4dvar_t h, void* d_buf, size_t bytes);

/* Background u_0^b and B = diag(sigma_b^2 per field) (Def 1 l.82, eq (6) l.111).  Runs the model
 * from d_xb over the whole window (Alg 1 l.452: u^b = M(u_0^b)), sets every local control to
 * the restricted background (l.455) and all frozen neighbour data to the background trajectory. */
int dd4dvar_set_background(dd4dvar_t h, const double* d_xb, const double h_sigma_b[3]);

/* Observations v_k, H = selection of grid values, R = diag(sigma_o^2 per field) (Def 1 l.83-85;
 * DESIGN.md R20).  h_levels: n_times strictly ascending time levels in [0, nsteps];
 * h_offsets[n_times+1]: start of each level's block in d_index / d_value; d_index: flat index
 * into [3][nlat][nlon], strictly ascending inside a level; d_value: observed values.
 * The restriction of H to each subdomain (Def 8 l.239) is built here.  d_obs_ws: device
 * workspace of at least dd4dvar_obs_workspace_bytes(h, total) bytes, total = h_offsets[n_times]. */
size_t dd4dvar_obs_workspace_bytes(dd4dvar_t h, long long n_obs_total);
int dd4dvar_set_observations(dd4dvar_t h, int n_times, const int* h_levels,
                             const long long* h_offsets, const int* d_index,
                             const double* d_value, const double h_sigma_o[3], void* d_obs_ws,
                             size_t obs_ws_bytes);

/* Algorithm 1 l.443-472: `outer_iters` additive (Jacobi) outer iterations, each = n_inner
 * L-BFGS iterations on every subdomain at once followed by the exchange of overlap / boundary
 * data (l.465).  Continues from the current local controls (fresh after set_background).
 * d_analysis [3][nlat][nlon]: gathered analysis at t_0 (eq (12)-(13) l.194-201).
 * h_history [(outer_iters+1)][3]: row l = J(gathered analysis after iteration l) by eq (6),
 * sum_ji J_ji at the end of iteration l (row 0: at the start of iteration 1),
 * delta_l = max_ji ||u_ji^l - u_ji^(l-1)||_inf (l.466; row 0: 0). */
int dd4dvar_run(dd4dvar_t h, int outer_iters, double* d_analysis, double* h_history);

/* Algorithm 1 with the paper's own local minimiser (Algorithms 5-7, l.568-696): n_gn incremental Gauss-Newton
 * iterations per outer iteration; each linearises the model about the current local trajectory (TLM, Alg 6
 * l.14-16) and solves the normal equations (42)-(43) l.620-626 in w = V^+ (u - u^b), V = diag(sigma_b)
 * (eq (44)-(46) l.630-649, "B-preconditioned") by exactly n_cg conjugate-gradient iterations from dw = 0, then
 * takes the full step (Alg 5 l.8).  One CG iteration = one tangent-linear sweep + one adjoint sweep (ADJ, Alg 6
 * l.17-19) on every subdomain.  Arguments and history as dd4dvar_run.  Served by the wavefront kernels
 * (dd4dvar_active_path == 5) and by the generic kernels (paths 1, 3: any layout; they keep the tangent-linear
 * trajectory in a second trajectory-sized store); -2 on the row-marching paths 2 and 4. */
int dd4dvar_run_gn(dd4dvar_t h, int outer_iters, int n_gn, int n_cg, double* d_analysis, double* h_history);

/* Test hook: the Gauss-Newton operator H_GN = 2 grad F^T grad F of every J_ji (F = stacked residuals of eq (25)
 * l.338-344) about the given controls, applied to d_p; d_controls, d_p, d_out in the "all subdomains" control
 * layout, d_p and d_out in w-space.  Runs a forward sweep at d_controls first (uses the current frozen data). */
int dd4dvar_gn_hessvec(dd4dvar_t h, const double* d_controls, const double* d_p, double* d_out);

/* eq (6) l.111 and its gradient by one forward + one adjoint sweep over the whole grid.
 * d_x0 [3][nlat][nlon]; h_cost[1]; d_grad [3][nlat][nlon] or NULL. */
int dd4dvar_eval_global(dd4dvar_t h, const double* d_x0, double* h_cost, double* d_grad);

/* The hot path: J_ji (eq (25) l.338-344) and dJ_ji/dx of EVERY subdomain at the given controls,
 * with the current frozen neighbour data: forward sweep + trajectory store, misfit / background /
 * overlap terms, adjoint sweep.  d_controls, d_grads: "all subdomains" arrays (physical units);
 * d_grads may be NULL (forward sweep and costs only).  h_costs[nsub]; h_parts[nsub][5] or NULL =
 * background (25a), observation (25b), spatial-overlap, predecessor and successor terms (25c). */
int dd4dvar_eval_local(dd4dvar_t h, const double* d_controls, double* h_costs, double* h_parts,
                       double* d_grads);

/* The same evaluation end to end with HOST buffers: h_controls is copied to the device, the
 * gradient sweep runs, costs and (if h_grads != NULL) gradients are copied back; the copies are inside the call.
 * The overlap of copies and sweeps described next needs PINNED (page-locked) host buffers: with pageable memory every
 * copy blocks the host until it is done, the next chunk's sweep is queued late, and the call is correct but no faster
 * than copy + sweep + copy in sequence.
 * With 64 or more subdomains the evaluation runs in six chunks of consecutive subdomains (they are independent:
 * all neighbour data is frozen) so that the copies of one chunk overlap the sweeps of the others (on the wavefront
 * path the chunks are whole rounds of the persistent grid, 1, 2, .. rounds from either end); the library
 * creates two non-blocking copy streams for this on first use and destroys them with the handle.  Results are
 * identical to dd4dvar_eval_local. */
int dd4dvar_eval_local_host(dd4dvar_t h, const double* h_controls, double* h_costs, double* h_grads);

/* Same evaluation, queued on the stream without host synchronisation or host output, at the
 * library's own current controls: used for timing the gradient sweep (bench.py).
 * mode 0: forward sweep + trajectory store + cost terms (a1-a3); 1: the whole gradient sweep
 * (a1-a4); 2: adjoint sweep only (a4), on the trajectories the last forward sweep stored. */
/* (mode 2, the adjoint sweep alone, belongs to the forward sweep before it: on wavefront layouts it ADDS lambda^0 to the
 * control-level part of the gradient that the forward sweep's cost kernel left behind; one adjoint sweep per forward sweep.) */
int dd4dvar_sweep_async(dd4dvar_t h, int mode);

/* Copy the current local controls of all subdomains ("all subdomains" array, physical units). */
int dd4dvar_get_controls(dd4dvar_t h, double* d_controls);

/* Gathered state at a time level from the stored local trajectories: weighted extension-sum
 * with weights 1/multiplicity (Def 4 l.164-170, eq (12) l.196).  d_out [3][nlat][nlon]. */
int dd4dvar_get_trajectory(dd4dvar_t h, int level, double* d_out);

/* Local trajectory of subdomain `sub` as stored by the last sweep: d_out [(W+1)][3][ey][ex]. */
int dd4dvar_get_local_trajectory(dd4dvar_t h, int sub, double* d_out);

/* Model only: run the forecast from d_x0 and return the states at the given ascending levels,
 * d_out [n_levels][3][nlat][nlon] (used to generate twin-experiment observations, l.993-995). */
int dd4dvar_forecast(dd4dvar_t h, const double* d_x0, int n_levels, const int* h_levels,
                     double* d_out);

/* Forecast for callers that cannot give the library any device memory of their own making.
 *
 * Every other entry point works out of a workspace that the caller allocates (dd4dvar_set_workspace).  Some callers
 * have no allocator to turn to at the moment they need a forecast: code that runs after a framework has claimed the
 * whole device for its own pool and hands out nothing to plug-ins; a monitoring or fail-over path that must still
 * produce the background trajectory when the device is full and cudaMalloc would fail; host code in a latency-bound
 * loop, where cudaMalloc / cudaFree would stall every stream of the device.  For them this call runs the model
 * (the same step kernel code as dd4dvar_forecast, on the undecomposed grid) without a handle and without a
 * workspace.  It calls no cudaMalloc, cudaFree or other allocating routine, on any path.
 *
 * The scratch it needs -- the six row tables and the time levels between which the model steps -- is one array of
 * DD4DVAR_STATIC_SCRATCH_BYTES compiled into the library.  That memory is taken on EVERY GPU on which the process
 * loads libdd4dvar.so and is held until the process exits, whether this call is used or not; that is the price, and
 * why the array is small.  Limit: 8 * (32 * ceil(6 nlat / 32) + 2 * 3 nlon nlat) <= DD4DVAR_STATIC_SCRATCH_BYTES,
 * i.e. up to about 349 000 grid cells (720 x 360 fits, 1440 x 720 does not).  Larger grids are refused with -6 and a
 * message that names the two sizes; nothing is launched in that case.  nsteps is not limited: when the array holds
 * fewer levels than the window has, the newest level is moved to the front and the stepping continues.
 *
 * grid, window: as for dd4dvar_create.  d_x0: DEVICE, fp64 [3][nlat][nlon], read only.  h_levels: HOST, n_levels
 * ascending time levels in [0, nsteps].  d_out: DEVICE, fp64 [n_levels][3][nlat][nlon], caller-owned, written in full.
 * cuda_stream: a cudaStream_t (NULL = legacy default stream); all work is queued there and the call returns after
 * synchronising it.  h_err / err_len: optional HOST buffer that receives the text of a failure (there is no handle
 * to ask); may be NULL / 0.  Returns 0, -1, -2, -4 or -6 as listed at the top.
 *
 * First call on each device: the library looks up the device address of its array (once per device, with the
 * caller's current device; the result is kept).  Make that first call at set-up time, outside any stream capture.
 * All calls in a process share the one array per device, and it keeps whatever the last call left there.  Nothing in
 * it has to start at zero -- each call rewrites the tables and writes every level in full before reading it -- but
 * two calls whose work overlaps on the same GPU (two streams, or two host threads) race on it and both results are
 * then undefined: run them one after the other. */
#define DD4DVAR_STATIC_SCRATCH_BYTES (16u << 20)
int dd4dvar_forecast_static(const dd4dvar_grid* grid, const dd4dvar_window* window, const double* d_x0,
                            int n_levels, const int* h_levels, double* d_out, void* cuda_stream,
                            char* h_err, size_t err_len);

int dd4dvar_num_subdomains(dd4dvar_t h);
/* out[16] = tile_col, tile_row, window, owned i0,i1,j0,j1, ext i0 (may be < 0: wraps), ext j0,
 * ex, ey, ghost width lon, ghost south, ghost north, first level s, last level e. */
int dd4dvar_subdomain_info(dd4dvar_t h, int sub, int out[16]);
/* offset (in doubles) of subdomain `sub` inside an "all subdomains" array; sub = nsub gives the
 * total length. */
long long dd4dvar_control_offset(dd4dvar_t h, int sub);
/* which kernels serve the local sweeps: the value of dd4dvar_opts.path in effect, 1 .. 5 (see there) */
int dd4dvar_active_path(dd4dvar_t h);

/* Weight of the background term (25a) l.338 in the time windows j > 0 (R7).  The paper is
 * at odds with itself here: (25a) is printed for every window, but eq (19) l.288 (J = sum of the
 * local functionals) only holds beyond the background state if the term is counted where eq (6)
 * l.111 has it, at t_0.  Default 0 (only window 0 carries (25a); the windows j > 0 are anchored by
 * the predecessor term of (25c) instead); 1 = as printed.  Takes effect at the next evaluation;
 * returns 0 or -1 (negative weight). */
int dd4dvar_set_bg_weight(dd4dvar_t h, double w_later);

/* Column 0 of the history of dd4dvar_run / dd4dvar_run_gn, J of eq (6) l.111 at the gathered analysis, costs one
 * undecomposed forecast over the whole assimilation window per outer iteration (it is a diagnostic, not part of
 * Algorithm 1).  on = 0: skip it, column 0 is NaN; default on. */
int dd4dvar_set_history_global(dd4dvar_t h, int on);

/* Where the time of dd4dvar_run goes (the L-BFGS passes and the exchange are timed separately and
 * reported).  on = 1: dd4dvar_run records CUDA events on its stream at every change of phase; after it returns,
 * dd4dvar_get_phase_ms gives the device time of that run per phase, in ms: [0] gradient / trial sweeps (a1-a4),
 * [1] L-BFGS kernels, resets and the host round trips of the line search (a5), [2] exchange (a6), [3] the J_global
 * diagnostic (dd4dvar_set_history_global), [4] final gather.  Idle time of the stream while the host decides (the
 * check of the line search, the sums of the history) falls into the phase that was open.  Default off: nothing is
 * recorded.  The events are created on first use and destroyed with the handle. */
int dd4dvar_set_phase_timing(dd4dvar_t h, int on);
int dd4dvar_get_phase_ms(dd4dvar_t h, double h_out[5]);

/* Sharded runs, one process per GPU: within an outer iteration the local problems are independent
 * (eq (37) l.433) and there is one exchange step per outer iteration (Alg 1 l.465).  Every process holds the whole
 * problem and OWNS the subdomains of the time windows [j0, j1): dd4dvar_run moves only those; its exchange freezes the
 * controls of the owned subdomains and the end states of the owned windows.  After every dd4dvar_run(h, 1, ...) the
 * caller completes the exchange between the processes on the two buffers of dd4dvar_exchange_buffer (device pointers
 * into the workspace, "all subdomains" control layout): which = 0 frozen controls, owner = the subdomain's own window;
 * which = 1 predecessor end states, owner = the window BEFORE the subdomain's.  Spatial neighbours share a window, so
 * the ghost-ring store never crosses processes.  In a sharded run the history rows of dd4dvar_run are local (column 0
 * needs dd4dvar_set_history_global(h, 0)); dd4dvar_get_local_stats returns J_ji and |u_ji^l - u_ji^(l-1)|_inf per
 * subdomain (valid for the owned ones) for the caller's reductions, dd4dvar_gather_analysis the analysis (eq (12)-(13)
 * l.194-201) from the frozen controls.  paper_2205_06649_b200/parallel.py drives this with torch.distributed.
 * set_owned_windows: after set_workspace; (0, q_time) switches sharding off.  dd4dvar_run_gn is not sharded (-2). */
int dd4dvar_set_owned_windows(dd4dvar_t h, int j0, int j1);
int dd4dvar_exchange_buffer(dd4dvar_t h, int which, void** d_ptr, long long* count);
int dd4dvar_get_local_stats(dd4dvar_t h, double* h_J, double* h_dmax);
int dd4dvar_gather_analysis(dd4dvar_t h, double* d_analysis);

/* The spatial overlap penalty (25c) case 1 l.310-314 acts on the control level of the window (R12, the
 * default).  on = 1: on every level of the window, eq (21) l.300 read literally (O_ik maps onto Delta_j x (Omega_i n
 * Omega_k)); the neighbours' frozen trajectories on the overlap rectangles are then kept in a second store,
 * refreshed at every exchange.  Served by the generic kernels only: create with opts.path = 1, else -2; call
 * before dd4dvar_set_background, else -3.  dd4dvar_run_gn and dd4dvar_gn_hessvec return -2 while it is on. */
int dd4dvar_set_overlap_levels(dd4dvar_t h, int on);

/* Measurement aid ("which roofline binds"): microbenchmarks of the device's
 * fp64 FMA rate, fp64 ADD rate, shared-memory load bandwidth and 64-bit warp-shuffle rate, the
 * secondary bounds of the stencil sweep next to HBM (SURVEY.md section 8(d) asks for the fp64 peak to
 * be measured on the box).  h_out: [0] fp64 FMA TFLOP/s, [1] fp64 ADD 1e12 instr/s, [2] LDS.64
 * bytes/s over all SMs, [3] 64-bit shuffles/s (per thread), [4] SM count, [5] SM clock MHz.
 * Needs no handle; runs ~0.1 s on `cuda_stream`; returns 0, -1 (null argument) or -4. */
int dd4dvar_measure_peaks(void* cuda_stream, double h_out[6]);
/* number of kernel launches issued by this handle so far (bench.py's gpu_launches) */
long long dd4dvar_launch_count(dd4dvar_t h);

const char* dd4dvar_last_error(dd4dvar_t h);
void dd4dvar_destroy(dd4dvar_t h);

#ifdef __cplusplus
}
#endif
#endif /* DD4DVAR_H */
