/*
 * tf.h -- C-ABI of the B200-native ADI sweep for the thin-film equation
 *
 *     h_t + div[ h^3 grad( lap h + Pi(h) ) ] = 0,   Pi(h) = kappa[(hstar/h)^n - (hstar/h)^m]
 *
 * i.e. eq (1.1)/(2.1) of Lam, Cummings, Kondic (arXiv:1806.10550) with
 * f0 = h^3, f1 = h^3 Pi'(h) (eqs (1.7)-(1.8)), no-flux boundaries (2.28)
 * (PAPER.md:297-302), Crank-Nicolson in time (2.14), solved by the ADI
 * pseudo-Newton iteration (2.19)-(2.21).  All arithmetic is fp64 and runs
 * in hand-written sm_100a CUDA kernels; there is NO CPU fallback: every entry point that
 * needs the GPU returns TF_ERR_CUDA when no device / kernel image is usable.
 *
 * Layout: a field is nx*ny doubles, row-major h[j*nx + i], i along x (contiguous), j along y;
 * cell centre ((i+1/2)dx, (j+1/2)dy).
 * Ownership: the context owns its device buffers (tf_create) or borrows the caller's
 * workspace for its lifetime (tf_create_with_workspace).  No pointer passed to any other
 * call is retained after the call returns.
 * Errors: every call returns a tf_status; nothing throws or aborts across this boundary.
 * CUDA errors map to TF_ERR_CUDA with text in tf_last_error().
 * Threading: one context is used from one host thread at a time; all work of a context is
 * ordered on its stream.
 */
#ifndef TF_B200_H
#define TF_B200_H
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tf_ctx tf_ctx;   /* opaque */

typedef enum {
    TF_OK = 0,
    TF_NOT_CONVERGED = 1,       /* soft: step rejected, state still u^n   */
    TF_REJECTED = 2,            /* soft: converged, but an extra solution criterion failed (PAPER.md:252 Note 2); state still u^n */
    TF_ERR_INVALID_ARG = -1,
    TF_ERR_UNSUPPORTED = -2,
    TF_ERR_CUDA = -3,
    TF_ERR_ALLOC = -4,
    TF_ERR_STATE = -5
} tf_status;

typedef enum { TF_BC_NOFLUX = 0 } tf_bc;   /* (2.28): h_n = h_nnn = 0 on all four sides */

/* Bytes of device workspace a context for an nx*ny grid needs (so the caller, e.g. PyTorch,
 * can allocate it).  0 if nx or ny < 5. */
size_t tf_workspace_bytes(int nx, int ny);

/*
 * Create a context (problem statement: PAPER.md:47 (1.1), 86-91 (1.7)-(1.8), 297-302 (2.28)).
 *   nx, ny >= 5 and (nx+1)*(ny+1) < 2^31 (the kernels index a field with 32-bit element offsets);
 *   dx, dy, kappa, hstar > 0; integer exponents 16 >= n > m >= 1 (the powers are formed by repeated multiplication;
 *   a larger n is TF_ERR_INVALID_ARG); bc = TF_BC_NOFLUX
 *   (anything else: TF_ERR_UNSUPPORTED -- the paper defines no other boundary condition).
 * tf_create allocates tf_workspace_bytes() of device memory itself and uses the legacy
 * default stream.  tf_create_with_workspace borrows `dev_ws` (device pointer, 256-byte
 * aligned, `bytes` >= tf_workspace_bytes) and launches on `cuda_stream` (a cudaStream_t
 * cast to void*; NULL = default stream).
 */
tf_status tf_create(tf_ctx** out, int nx, int ny, double dx, double dy,
                    double kappa, double hstar, int n, int m, tf_bc bc);
tf_status tf_create_with_workspace(tf_ctx** out, int nx, int ny, double dx, double dy,
                                   double kappa, double hstar, int n, int m, tf_bc bc,
                                   void* dev_ws, size_t bytes, void* cuda_stream);
void tf_destroy(tf_ctx* ctx);

/* Disjoining pressure behind the same sweep.  With (1.7), in the form
 * f0 = cap0 h^3, f1 = cap1 h^3 Pi'(h) (the printed placement of the capillary number is cap0 = C, cap1 = 1/C;
 * both prefactors are the caller's):
 *   TF_PI_POWER    Pi = kappa[(hstar/h)^n - (hstar/h)^m] of tf_create, cap0 = cap1 = 1 (default; params ignored)
 *   TF_PI_NLC      (1.8)-(1.9): Pi = K[(b/h)^3 - (b/h)^2] + (N/2)[m(h)/h]^2,
 *                  m = g h^2/(h^2 + beta^2), g = (1 + tanh((h - 2b)/w))/2;
 *                  params[7] = {cap0, cap1, K, b, N, beta, w}   (host pointer; (1.11) lists the paper's values)
 *   TF_PI_POLYMER  (1.12): Pi = -d psi/dh, psi = C/h^8 - A_SiOx/(12 pi h^2) + (A_SiOx - A_Si)/(12 pi (h+d)^2);
 *                  params[6] = {cap0, cap1, C, A_SiOx, A_Si, d}
 * Takes effect from the next tf_step; the state is kept.  TF_ERR_INVALID_ARG for a wrong count, non-finite values or
 * non-positive cap0, cap1, b, w, d; TF_ERR_UNSUPPORTED for another kind. */
typedef enum { TF_PI_POWER = 0, TF_PI_NLC = 2, TF_PI_POLYMER = 3 } tf_pressure;
tf_status tf_set_pressure(tf_ctx* ctx, tf_pressure kind, const double* params, int nparams);

/* Newton controls, (2.22) and Notes 1-2.  Defaults: tol = 1e-10,
 * max_iter = 10, fixed_iters = 0 (off).  tol >= 1e-14;
 * 1 <= max_iter <= 4096; 0 <= fixed_iters <= 4096.  fixed_iters = K > 0 (parity mode): exactly K
 * iterations per step, no convergence test; the step is accepted unless one of the K iterates was
 * non-finite or non-positive (then TF_NOT_CONVERGED, state unchanged, *residual = NaN if a residual was NaN). */
tf_status tf_set_newton(tf_ctx* ctx, double tol, int max_iter, int fixed_iters);

/* Host decision of Fig. 1 (PAPER.md:256-258; the paper reads one flag per 16x16 block per iteration, :675-683).
 * batch = 0: the host reads the residual after every iteration before launching the next.  batch > 0 (default 2):
 * speculative launch-ahead -- iterations are enqueued in batches (the first as long as the last accepted step's
 * iteration count, then `batch` at a time) and the residual records of a batch are read at once; iterations enqueued
 * past the deciding one return immediately on the device, so iterates, iteration count and residual are exactly
 * those of batch = 0.  0 <= batch <= 64. */
tf_status tf_set_launch_ahead(tf_ctx* ctx, int batch);

/* Launch-ahead batches through CUDA graphs (default on): a batch {first iteration, count, which buffer holds u^n, dt}
 * that recurs is captured once (at its second occurrence) and replayed from then on -- the same launches with the same
 * arguments, so results are bit-identical; what changes is the launch cost (per step on a 128^2 grid: about a dozen
 * iterations of four ~10 us kernels).  Setters that change a launch argument (tf_set_newton, tf_set_pressure) drop the
 * captured graphs; profiled steps (tf_set_profiling) and fixed_iters steps are launched plainly.  At most 16 graphs are
 * kept per context (least recently used goes).  tf_graph_replays: how many batches were replayed so far. */
tf_status tf_set_cuda_graphs(tf_ctx* ctx, int on);
tf_status tf_graph_replays(tf_ctx* ctx, unsigned long long* replays);

/* Copy nx*ny doubles into the context as u^n.  `h` is a device pointer if is_device_ptr != 0,
 * else a host pointer.  Rejects non-finite or non-positive values (Pi is singular at h = 0)
 * with TF_ERR_INVALID_ARG; the previous state is then kept. */
tf_status tf_set_state(tf_ctx* ctx, const double* h, int is_device_ptr);

/* Copy the current state u^n out (nx*ny doubles, same layout). */
tf_status tf_get_state(tf_ctx* ctx, double* h_out, int is_device_ptr);

/*
 * One Crank-Nicolson time step of size dt > 0 by the ADI pseudo-Newton iteration:
 *   b^n = u^n - (dt/2) D(u^n);  u_(0) = u^n;  for k = 0, 1, ...:
 *     (I + dt/2 J_y(u_k)) w = b^n - u_k - (dt/2) D(u_k)          (2.19)  y-sweep
 *     (I + dt/2 J_x(u_k)) v = w                                  (2.20)  x-sweep
 *     res = max |v / u_k|;  u_(k+1) = u_k + v                    (2.22), (2.21)
 * until res < tol (TF_OK, state advanced) or max_iter iterations were done or an iterate
 * became non-finite / non-positive (TF_NOT_CONVERGED, state unchanged).  *newton_iters
 * (>= 1) and *residual (last res) are filled in both cases; either may be NULL.
 */
tf_status tf_step(tf_ctx* ctx, double dt, int* newton_iters, double* residual);

/*
 * Extra "solution criteria" (PAPER.md:252 Note 2: "Other restrictions besides the convergence of the iterative scheme
 * may be placed on accepting the solution ... e.g. sufficiently small truncation error").  The paper fixes none; this
 * build offers one: a converged step is accepted only if  max_ij |u^{n+1} - u^n| / u^n  <= max_rel_change, else
 * tf_step returns TF_REJECTED and the state stays u^n.  0 switches the criterion off (default).
 */
tf_status tf_set_solution_criteria(tf_ctx* ctx, double max_rel_change);

/*
 * The criterion the paper names (PAPER.md:252 Note 2: "e.g. sufficiently small truncation error"), reading R25 of
 * the local truncation error of the Crank-Nicolson / trapezoidal step (2.14) is -(dt^3/12) u_ttt.  It is
 * estimated from quantities the step already holds: with u_t^n = -D(u^n) = 2 (b^n - u^n)/dt and the scheme's own relation
 * u_t^{n+1} = 2 (u^{n+1} - u^n)/dt - u_t^n, the second time derivative at the middle of the step is
 *     a_{n+1/2} = (u_t^{n+1} - u_t^n)/dt = 2 (u^{n+1} + u^n - 2 b^n)/dt^2,
 * and u_ttt ~ (a_{n+1/2} - a_{n-1/2}) / ((dt + dt_prev)/2), a_{n-1/2} being kept from the previous accepted step (one
 * field of the workspace).  A converged step is accepted only if
 *     max_ij (dt^3/12) |u_ttt| / |u^{n+1}|  <=  max_rel_truncation,
 * else tf_step returns TF_REJECTED with the state (and the stored a_{n-1/2}) untouched.  The first step after
 * tf_set_state or tf_accept has no history and is not tested.  0 = off (default).
 * tf_last_truncation_estimate: the estimate of the last converged step that was tested (0 if none).
 * One fused pass over four fields per step (40 B per grid point), order-independent max.
 */
tf_status tf_set_truncation_criterion(tf_ctx* ctx, double max_rel_truncation);
tf_status tf_last_truncation_estimate(tf_ctx* ctx, double* estimate);

/*
 * Adaptive time stepping of Fig. 1: take a step of size dt; if the solution criteria are met
 * (status TF_OK) advance time and, after `grow_after` consecutive accepted steps, multiply dt by `grow` (bounded by
 * dt_max); otherwise multiply dt by `shrink` and retry; fail (TF_NOT_CONVERGED) when dt falls below dt_min or after
 * max_attempts steps (<= 0: 50 * n_accept).  Runs until n_accept steps were accepted.  ctl->dt is the first step on
 * entry and the step to continue with on return; *t_advanced = sum of the accepted steps; the first hist_cap attempts
 * are recorded in hist, *nhist = number of attempts (all optional, may be NULL / 0).  A negative status of a step
 * stops the run and is returned.  The paper gives no constants; BASELINE.json config 2 uses shrink 0.5, grow 1.1,
 * grow_after 1.  tf_adaptive_run is the controller over any step function (tf_advance_adaptive = over tf_step).
 */
typedef struct { double dt, shrink, grow; int grow_after; double dt_min, dt_max; } tf_adaptive;
typedef struct { double dt; int status; int newton_iters; double residual; } tf_step_record;
typedef int (*tf_step_fn)(void* user, double dt, int* newton_iters, double* residual);   /* returns a tf_status */
tf_status tf_adaptive_run(tf_step_fn step, void* user, tf_adaptive* ctl, int n_accept, int max_attempts,
                          double* t_advanced, tf_step_record* hist, int hist_cap, int* nhist);
tf_status tf_advance_adaptive(tf_ctx* ctx, tf_adaptive* ctl, int n_accept, int max_attempts,
                              double* t_advanced, tf_step_record* hist, int hist_cap, int* nhist);

/*
 * The same controller with every decision taken ON THE DEVICE (the paper's controller is host
 * code that reads a flag array after every iteration): attempts are enqueued in chunks without a
 * host round trip -- per attempt a control kernel opens the attempt and publishes dt/2, max_iter gated iterations run
 * (those past the deciding one return at once), a control kernel takes the decision of Fig. 1 from the residual
 * records (accept / shrink / grow, dt_min, attempt cap) and a copy kernel commits u^{n+1} if the step was accepted.
 * The host reads the control block once per chunk.  Same arguments, same results as tf_advance_adaptive: the sequence
 * of (dt, status, iterations, residual) and the films are identical bit for bit, for any number of attempts (the device
 * records them in a ring of 1024 entries that the host drains between chunks).
 * Both extra solution criteria (tf_set_solution_criteria, tf_set_truncation_criterion) are decided on the device too:
 * their reductions run behind a converged attempt and read dt, dt_prev and the history flag from device memory; a
 * rejected attempt is recorded as TF_REJECTED and shrinks dt as on the host.  The stored a_{n-1/2} carries over from
 * and to tf_step.  TF_ERR_UNSUPPORTED with fixed_iters > 0.
 */
tf_status tf_advance_adaptive_device(tf_ctx* ctx, tf_adaptive* ctl, int n_accept, int max_attempts,
                                     double* t_advanced, tf_step_record* hist, int hist_cap, int* nhist);

/*
 * The rows of the path one at a time, for callers that put an exchange step between the sweeps (a film distributed over
 * several devices).  tf_step is: for k = 0, 1, ...: tf_sweep(ctx, dt, k, 3); decide on
 * tf_residual(ctx, k); on acceptance tf_accept(ctx).
 *   tf_field     device address of a field the context owns: 0 = u^n (the state), 1 = the iterate buffer (u_(k) for
 *                k >= 1 on input of a sweep, u_(k+1) on output of the x-sweep), 2 = b^n, 3 = w; 4 = the residual records,
 *                2 doubles {res, bad} per iteration, 4096 iterations.  The addresses of 0 and 1 swap on tf_accept / an
 *                accepted tf_step: ask again afterwards.
 *   tf_sweep     which = 1: y-sweep of iteration k (S1-S4; reads field 0 if k == 0 else field 1, and b^n; k == 0 also
 *                writes b^n; writes w); which = 2: x-sweep (S5-S7; reads the same source field and w; writes field 1 and
 *                the residual record of iteration k); which = 3: both.  Adding 4 gates the sweep on the record of
 *                iteration k-1 (k >= 1): its kernels return at once if that record says res < tol, bad iterate or NaN --
 *                a caller that launches iterations ahead of its decisions (tf_set_launch_ahead does the same inside
 *                tf_step) and, across devices, writes the all-reduced record back into field 4 first.  Enqueues only.
 *   tf_residual  (2.22) of iteration k and the bad-iterate flag; synchronises the stream.
 *   tf_accept    u^{n+1} = u_(k+1): swaps fields 0 and 1.
 */
tf_status tf_field(tf_ctx* ctx, int which, double** dev_ptr);
tf_status tf_sweep(tf_ctx* ctx, double dt, int k, int which);
tf_status tf_residual(tf_ctx* ctx, int k, double* res, int* bad);
tf_status tf_accept(tf_ctx* ctx);

/*
 * Exchange steps of a time step whose film is spread over several devices (the paper names a multi-GPU
 * implementation as future work).  The caller (paper_1806_10550_b200/dist_step.py) owns the collective;
 * the library moves the blocks and applies the boundary condition:
 *   tf_blocks_gather   buf[offset_k + r*ncols_k + c] = field[(row0_k + r)*ld + col0_k + c] for every block k -- the send
 *                      buffer of an all-to-all in ONE kernel;
 *   tf_blocks_scatter  the reverse, from the receive buffer into a field of row pitch ld; in the same pass the ghost
 *                      columns of a halo'd column block at a domain edge are filled by the reflection of (2.28),
 *                      reflect_left != 0: columns 1, 0 := columns 2, 3 (h_{-1} = h_0, h_{-2} = h_1);
 *                      reflect_right_at = g >= 0: columns g, g+1 := columns g-1, g-2; g < 0: none;
 *   tf_record_sanitize the residual record {res, bad} of iteration k before it is max-reduced over the ranks: a NaN
 *                      (or +inf) residual becomes {+inf, 1}, so that it wins the max and closes the gates.
 * field, buf: DEVICE pointers; rects: HOST array of nrect <= 64 blocks (copied into the launch); offsets in doubles.
 * Blocks must lie inside the field (col0 + ncols <= ld).  All four enqueue on a stream and return (no host sync).
 *   tf_block_copy      one block straight from field to field (what a rank keeps for itself never enters the buffers):
 *                      dst[(drow0 + r)*dld + dcol0 + c] = src[(srow0 + r)*sld + scol0 + c], ghost columns as in scatter.
 */
typedef struct { int row0, nrows, col0, ncols; long long offset; } tf_rect;
tf_status tf_block_copy(const double* src, int sld, int srow0, int scol0, double* dst, int dld, int drow0, int dcol0,
                        int nrows, int ncols, int reflect_left, int reflect_right_at, void* cuda_stream);
tf_status tf_blocks_gather(const double* field, int ld, const tf_rect* rects, int nrect, double* buf, void* cuda_stream);
tf_status tf_blocks_scatter(const double* buf, const tf_rect* rects, int nrect, double* field, int ld,
                            int reflect_left, int reflect_right_at, void* cuda_stream);
tf_status tf_record_sanitize(tf_ctx* ctx, int k);

/* mass = dx*dy*sum(h)  ((3.2), times the domain area); fixed-order fp64 tree. */
tf_status tf_mass(tf_ctx* ctx, double* mass);

/*
 * Isolated batched pentadiagonal solve (LU without pivoting, (A.5)).
 * Seven DEVICE arrays, each nrow*ncol doubles, row-major [r*ncol + c]; row i of a system is
 *   e_i x_{i-2} + c_i x_{i-1} + d_i x_i + a_i x_{i+1} + b_i x_{i+2} = rhs_i,
 * band entries that fall outside a system are ignored.
 *   dir = 0: system s = row s    (contiguous; nsys = nrow, len = ncol)   -- the x-sweep shape
 *   dir = 1: system s = column s (strided;   nsys = ncol, len = nrow)   -- the y-sweep shape
 * dev_ws: device scratch of tf_penta_workspace_bytes(nrow, ncol) bytes.  x may not alias inputs.
 * len >= 3.  Runs on cuda_stream; returns after enqueueing (no host sync).
 * Pivots: no pivoting, and the reciprocal of every pivot is formed from a hardware seed
 * (rcp.approx.ftz.f64) plus one cubic correction, <= 1 ulp for pivots with |mu| in [1e-290, 1e290]; pivots outside
 * that range (or zero) give inf / NaN in the affected system, as a division would for a zero pivot.
 */
size_t    tf_penta_workspace_bytes(int nrow, int ncol);
tf_status tf_penta_solve(int nrow, int ncol, int dir,
                         const double* e, const double* c, const double* d,
                         const double* a, const double* b, const double* rhs, double* x,
                         void* dev_ws, void* cuda_stream);

/*
 * tf_penta_solve for callers that have no device scratch to hand over and no way to get any.
 *
 * tf_penta_solve needs three scratch arrays (the LU factors alpha, beta and the intermediate z of (A.5),
 * PAPER.md:729-734) and leaves their allocation to the caller.  Some callers cannot allocate at the moment of the call:
 *   - a service that, at start-up, gave all free HBM to its own memory pool: a later cudaMalloc fails for lack of memory;
 *   - a latency-bound loop: cudaMalloc / cudaFree synchronise the whole device and take an unbounded time, which stalls
 *     the work other streams have in flight;
 *   - a plug-in inside a host application whose rules forbid CUDA allocations after initialisation.
 * For them the library itself carries the scratch: one fixed array in the device image of libtf_b200.so
 * (3 * TF_PENTA_STATIC_MAX_ELEMS doubles = 24 MiB).  The price is paid by everybody: every GPU on which this library's
 * device code gets loaded holds those 24 MiB from then until the process exits, whether or not this call is ever made.
 *
 * Same arguments, same kernels, same result (bit for bit) as tf_penta_solve without dev_ws; e ... rhs and x are DEVICE
 * arrays on the CURRENT device, owned by the caller, x may not alias an input.
 *   Limit:     nrow * ncol <= TF_PENTA_STATIC_MAX_ELEMS (tf_penta_static_max_elems() returns it at run time); a larger
 *              shape is refused with TF_ERR_INVALID_ARG and a message naming the limit, before any CUDA call.
 *   No allocation: neither this call nor anything below it calls cudaMalloc, cudaFree or a library routine that allocates.
 *   First call on each device: looks up the device address of the array (once per device, that device being current)
 *              and raises the shared-memory limit of the kernels it launches.  Make this first call during set-up,
 *              before any stream capture is started; later calls only enqueue kernels on cuda_stream and return.
 *   Sharing:   every call on a device uses the SAME array and finds in it whatever the previous call left.  Nothing in
 *              it has to start at zero -- the forward elimination writes every entry before the back substitution
 *              reads it -- so no clearing is done.  Two calls whose kernels can overlap on the GPU (different streams,
 *              or different host threads, without an ordering between them) race on the array and both results are
 *              garbage: keep all calls on one stream or order them with events.
 */
#define TF_PENTA_STATIC_MAX_ELEMS (1u << 20)
size_t    tf_penta_static_max_elems(void);
tf_status tf_penta_solve_static(int nrow, int ncol, int dir,
                                const double* e, const double* c, const double* d,
                                const double* a, const double* b, const double* rhs, double* x,
                                void* cuda_stream);

/*
 * The same solve with a selectable algorithm (PAPER.md:647 names "the SPIKE method or
 * cyclical reduction" as the way to parallelise a single system):
 *   TF_PENTA_LU         one thread per system, two-sided LU (what tf_penta_solve runs);
 *   TF_PENTA_PARTITION  every system is cut into nparts chunks of rows (nparts = 0: chosen from the shape so that
 *                       about four marching warps per SM exist): (1) per chunk, elimination from both ends with the
 *                       two coupling columns as extra right-hand sides gives exact relations between the chunk's
 *                       four end unknowns and the four unknowns outside it, (2) the reduced system of 4*nparts end
 *                       unknowns per system is solved, (3) all chunks are solved independently with corrected
 *                       right-hand sides.  Same solution up to rounding; for few, long systems (nsys << 20 000).
 *   TF_PENTA_PCR        parallel cyclic reduction (PAPER.md:647 names "cyclical reduction"), systems along rows only
 *                       (dir = 0): one CTA holds one system in shared memory as a block-tridiagonal system of 2 x 2
 *                       blocks, one thread per pair of unknowns, ceil(log2(len/2)) levels; global traffic is the
 *                       compulsory 56 B per unknown, ~76 fp64 operations per pair and level.  64 <= ncol <= 2048, ncol
 *                       even, 16-byte aligned arrays; TF_ERR_UNSUPPORTED otherwise.  The x-sweep alternative measured
 *                       against the LU; not used by tf_step.
 * tf_penta_partition_chunks returns the chunk count that will be used (1 = the shape falls back to TF_PENTA_LU:
 * odd nrow or ncol, fewer than 32 systems, or systems shorter than 192); 0 for invalid arguments.
 * dev_ws needs tf_penta_workspace_bytes_ex(nrow, ncol, dir, variant, nparts) bytes.  Arrays must be 16-byte
 * aligned for TF_PENTA_PARTITION (TF_ERR_UNSUPPORTED otherwise).
 */
typedef enum { TF_PENTA_LU = 0, TF_PENTA_PARTITION = 1, TF_PENTA_PCR = 2 } tf_penta_variant;
int       tf_penta_partition_chunks(int nrow, int ncol, int dir, int nparts);
size_t    tf_penta_workspace_bytes_ex(int nrow, int ncol, int dir, int variant, int nparts);
tf_status tf_penta_solve_ex(int nrow, int ncol, int dir, int variant, int nparts,
                            const double* e, const double* c, const double* d,
                            const double* a, const double* b, const double* rhs, double* x,
                            void* dev_ws, void* cuda_stream);

/*
 * The partition variant across devices (slab decomposition with a reduced-interface solve
 * instead of a transpose).  Every system is cut into `nslabs` slabs of consecutive rows (dir = 1; columns for dir = 0),
 * one slab per device, each slab into `nparts` chunks (the same nparts on every device).  Per device:
 *   1. tf_penta_slab_interface on the LOCAL arrays (the slab only: nrow x ncol is the local shape) writes the local
 *      interface values, tf_penta_slab_interface_doubles(...) doubles (device);
 *   2. the caller gathers them from all devices in slab order (an all-gather of 20 * nparts doubles per system and
 *      device: the one exchange step) into iface_all;
 *   3. tf_penta_slab_solve solves the reduced system of all nslabs * nparts chunks (redundantly on every device) and
 *      then the local chunks -> x (local shape).
 * Band entries that point outside the WHOLE system are ignored; entries at slab seams are used.  Same constraints as
 * TF_PENTA_PARTITION: local length / nparts >= 96, at least 32 systems, even nrow and ncol, 16-byte aligned arrays.
 * dev_ws of tf_penta_slab_solve: tf_penta_slab_workspace_bytes(local nrow, local ncol, dir, nparts, nslabs) bytes.
 * With nslabs = 1 the two calls are the single-device partition variant.
 */
size_t    tf_penta_slab_interface_doubles(int nrow, int ncol, int dir, int nparts);
size_t    tf_penta_slab_workspace_bytes(int nrow, int ncol, int dir, int nparts, int nslabs);
tf_status tf_penta_slab_interface(int nrow, int ncol, int dir, int nparts, int slab, int nslabs,
                                  const double* e, const double* c, const double* d,
                                  const double* a, const double* b, const double* rhs,
                                  double* iface_local, void* cuda_stream);
tf_status tf_penta_slab_solve(int nrow, int ncol, int dir, int nparts, int slab, int nslabs,
                              const double* e, const double* c, const double* d,
                              const double* a, const double* b, const double* rhs,
                              const double* iface_all, double* x, void* dev_ws, void* cuda_stream);

/*
 * Betti numbers of the thresholded film ("b0 counts the number of mountain peaks
 * (components) above H*, and b1 counts the number of valleys (loops) surrounding the peaks"; the paper uses CHomP on
 * cubical sets).  For every threshold H* = thresholds[t] (host array), with X = the closed unit squares of the cells
 * with h > H*:  b0[t] = connected components of X (cells connect through edges and corners), b1[t] = holes of X =
 * components of the complement (cells connect through edges only) that do not reach the border of the image.
 * h: DEVICE pointer, nx*ny doubles, row-major; b0, b1: HOST arrays of nthr entries; dev_ws: device scratch of
 * tf_betti_workspace_bytes(nx, ny, nthr) bytes (256-byte aligned).  nx*ny < 2^31, ny <= 65535.  Synchronises the
 * stream before returning (the counts are read back).  One union-find labelling per threshold, exact integers.
 */
size_t    tf_betti_workspace_bytes(int nx, int ny, int nthr);
tf_status tf_betti(const double* h, int nx, int ny, const double* thresholds, int nthr,
                   long long* b0, long long* b1, void* dev_ws, void* cuda_stream);

/*
 * Radial Fourier transform, steps one to four of Appendix B:
 *   1. |DFT2(h - H0)| on the nx x ny samples (the FFT itself is cuFFT, loaded at run time: TF_ERR_UNSUPPORTED if
 *      libcufft.so.11 cannot be found);
 *   2. convolution with a Gaussian of standard deviation `sigma` in DFT-index units, truncated at ceil(3 sigma) <= 64,
 *      normalised, periodic, separable (sigma = 0: no filter);
 *   3./4. eq. (B.1): for every radius that occurs, the mean over the points of equal radius and their number N_k.
 * The domain must be square, nx dx = ny dy = L: equal radius then means equal kx^2 + ky^2 of the signed DFT indices;
 * radii up to kmax index units are reported (the paper restricts q to [0, 5 q_m]).
 * h: DEVICE pointer (nx*ny doubles, row-major).  q, zeta, count: HOST arrays of `cap` entries, filled in ascending q
 * with q_r = 2 pi sqrt(kx^2 + ky^2) / L, the mean magnitude and N_k; *nk = number of distinct radii (may exceed cap:
 * then only the first cap are stored).  dev_ws: tf_spectrum_workspace_bytes(nx, ny, kmax) bytes of device scratch.
 * Synchronises the stream.  Steps five and six of the appendix (least-squares fit, moving average, maxima) are 1-D
 * post-processing of this output: tf_radial_peaks below.
 */
size_t    tf_spectrum_workspace_bytes(int nx, int ny, int kmax);
tf_status tf_radial_spectrum(const double* h, int nx, int ny, double L, double H0, double sigma, int kmax,
                             double* q, double* zeta, long long* count, int cap, int* nk,
                             void* dev_ws, void* cuda_stream);

/*
 * Steps five and six of Appendix B and the extraction of the maxima, on the HOST (a few thousand
 * numbers): (B.2) least-squares fit of a continuous piecewise-linear function with value 0 at q = 0 whose intervals
 * hold `per_interval` points each (paper: 10; the last interval takes what is left; points with q = 0 are left out);
 * evaluation on `ngrid` equispaced points of [0, q_last] (paper: 400); (B.3) moving average with P = 3, 2, 1 (the
 * window is cut off at the ends of the grid); derivative by second-order differences, roots by sign change and linear
 * interpolation, kept if the second difference is negative.  q (strictly ascending), zeta: nk host values, e.g. the
 * output of tf_radial_spectrum.  qgrid, zsmooth: ngrid host values each, or NULL.  peak_q, peak_z: the first peak_cap
 * maxima in ascending q; *npeaks = number found.  No GPU work.
 */
tf_status tf_radial_peaks(const double* q, const double* zeta, int nk, int per_interval, int ngrid,
                          double* qgrid, double* zsmooth, double* peak_q, double* peak_z, int peak_cap, int* npeaks);

/* Text of the last error on this context ("" if none); ctx == NULL: last error of a failed
 * tf_create* / tf_penta_solve on this thread.  Valid until the next call. */
const char* tf_last_error(const tf_ctx* ctx);

/*
 * Per-kernel device timing of the Newton iteration (for bench.py's roofline object).  When on,
 * tf_step brackets each of its four kernels with CUDA events on the context's stream and
 * accumulates the elapsed times.  Slots: 0 = y forward (assembly + elimination), 1 = y backward,
 * 2 = x forward, 3 = x backward + update + residual.  tf_get_profile copies the accumulated
 * milliseconds and launch counts (either may be NULL) and does not reset them;
 * tf_set_profiling(ctx, on) resets them.  Only steps with a per-iteration host decision
 * (fixed_iters = 0) or fixed_iters <= 64 are profiled.
 */
#define TF_PROFILE_SLOTS 4
tf_status tf_set_profiling(tf_ctx* ctx, int on);
tf_status tf_get_profile(tf_ctx* ctx, double ms[TF_PROFILE_SLOTS], unsigned long long launches[TF_PROFILE_SLOTS]);

/*
 * Measured fp64 arithmetic peak of the current device, the denominator of bench.py's "alu" roofline (SURVEY.md section 6:
 * the fp64 peak is not in MEASURED_PEAKS.json and has to be measured).  Launches `launches` >= 1 times (after one untimed
 * launch) a kernel in which every thread runs 8 independent chains of dependent DFMAs, 16 CTAs of 256 threads per SM
 * (2048 threads, 16 384 chains per SM: the fp64 pipe is the only limit), each launch timed with CUDA events on
 * cuda_stream.  *best_dfma_per_s / *mean_dfma_per_s: thread-level DFMA instructions per second of the fastest launch /
 * over all launches (either may be NULL); 2 flops each.  A launch takes about 2 ms.  Synchronises the stream.
 */
tf_status tf_fp64_peak(int launches, double* best_dfma_per_s, double* mean_dfma_per_s, void* cuda_stream);

/* Number of kernels this library has launched since load (all contexts); for bench.py's
 * gpu_launches claim. */
unsigned long long tf_kernel_launches(void);

#ifdef __cplusplus
}
#endif
#endif /* TF_B200_H */
