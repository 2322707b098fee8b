/*
 * kratos_hydro.h -- C-ABI boundary of the B200-native Kratos hydrodynamics hot path.
 *
 * The library advances the compressible Euler equations (Eq. 2)
 *     d_t rho + div(rho v) = 0,  d_t(rho v) + div(rho v v + p I) = 0,  d_t eps + div[(eps+p) v] = 0,
 *     eps = p/(gamma-1) + rho v^2/2
 * on ONE uniform Cartesian block on ONE GPU (several such blocks can be stacked along z, one per GPU, through
 * communication boundaries: see the end of this file) with the paper's default scheme: primitive
 * recovery (Sec. 3.1), ghost zones by the paper's boundary rules
 * (Sec. 3.1.1), minmod-limited PLM (Eq. 3), the
 * subtraction-safe HLLC solver (Eq. 4-5), a flux-difference update inside
 * the Heun integrator (Sec. 3.3), the CFL time-step reduction
 * and the mixed-precision split float_t / float2_t (Sec. 3.2.2,
 * PAPER.md:230-240).  Every step runs in hand-written sm_100a CUDA kernels; there is no CPU
 * fallback: without a CUDA device every call that computes fails with KRATOS_ERR_CUDA.
 *
 * Conventions
 *  - State layout: conserved U = (rho, m_x, m_y, m_z, eps), struct of arrays
 *    U[5][nz][ny][nx] of double, x fastest, INTERIOR cells only (the library keeps no ghost
 *    storage: boundary rules are applied as the stencil is loaded).
 *  - An axis is active when its extent is > 1 (nz = 1: 2D, ny = nz = 1: 1D).  Active axes
 *    need extent >= 4.  Inactive axes carry no flux; their bc entries are ignored and their
 *    momentum stays exactly as given (normally 0).
 *  - Cell centres x_i = (i + 1/2) dx; default spacing 1/n per active axis (unit box).
 *  - Every function returning int returns KRATOS_OK (0) or a negative error code; the message
 *    is available from kratos_hydro_last_error() (thread-local).  The handle owns all device
 *    memory; the caller owns every buffer it passes.  A handle is not thread-safe.
 *  - "host"/"device" below says where a pointer must live.  Device pointers must belong to
 *    the current CUDA device of the calling thread at create time.
 *  - All work is enqueued on the stream given by kratos_hydro_set_stream (default: the
 *    legacy default stream 0).  Calls documented as "asynchronous" return before the GPU
 *    has finished; all others synchronise that stream before returning.
 *  - The handle remembers the CUDA device that was current at create; every entry point makes
 *    that device current for its duration and restores the caller's device before returning.
 *  - Mixed precision only: the fp32 Riemann solver carries the pressure as the deviation from a
 *    reference pressure p_ref (reading S14).  p_ref = fp32(min(mean p, 2 min p)) of the
 *    state last given to kratos_hydro_set_state; it is computed by the first cfl_dt / step / run
 *    after set_state (one extra read of the state) and then kept until the next set_state, so what
 *    step(dt) computes depends on the state and on dt only, not on which other calls were made.
 *    With p_ref > 0 the pressure floor of the primitives is max(1e-30, p_ref 2^-22).
 */
#ifndef KRATOS_HYDRO_H
#define KRATOS_HYDRO_H

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define KRATOS_API __attribute__((visibility("default")))
#else
#define KRATOS_API
#endif

typedef struct kratos_hydro kratos_hydro_t; /* opaque */

/* error codes */
#define KRATOS_OK 0
#define KRATOS_ERR_ARG (-1)       /* bad argument (see each call) */
#define KRATOS_ERR_ALLOC (-2)     /* device or host allocation failed */
#define KRATOS_ERR_CUDA (-3)      /* CUDA runtime error / no device */
#define KRATOS_ERR_NONFINITE (-4) /* non-finite state or time step detected */

/* scheme word: bits 0-1 precision, bits 4-5 integrator.
 * Reconstruction is PLM-minmod and the Riemann solver HLLC (the paper's defaults; no other choice). */
#define KRATOS_PREC_MIXED 0 /* float_t = fp32 (reconstruction, Riemann), float2_t = fp64 (state, update) */
#define KRATOS_PREC_FP64 1  /* float_t = float2_t = fp64 */
#define KRATOS_PREC_SINGLE 2 /* float_t = float2_t = fp32 ("Single" of Tables 1-2): the handle stores the state as
                               floats (half the memory and traffic); the boundary still carries doubles, converted on the way in
                               and out.  Conservation holds to fp32 rounding only.  Heun integrator only. */
#define KRATOS_INTEGRATOR_HEUN (0 << 4)
#define KRATOS_INTEGRATOR_VANLEER (1 << 4) /* predictor-corrector of Sec. 3.3: predictor kept as float_t
                                             primitives (20 B per cell in mixed precision instead of a second fp64 state);
                                             both sub-steps run on the TMA kernel where KRATOS_KERNEL_TMA applies, else on
                                             general one-thread-per-cell kernels (KRATOS_KERNEL_SIMPLE) */

/* boundary codes, the paper's list order */
#define KRATOS_BC_PERIODIC 0 /* communication boundary onto the same block: wrap copy */
#define KRATOS_BC_FREE 1     /* q(-i-1/2) = q(1/2) */
#define KRATOS_BC_OUTFLOW 2  /* Free, but inward normal velocity v(-i-1/2) = min(v(1/2), 0) */
#define KRATOS_BC_REFLECT 3  /* q(-i-1/2) = q(i+1/2), normal velocity negated */
#define KRATOS_BC_COMM 4     /* communication boundary onto ANOTHER block (Sec. 3.1.2: "c-boundaries"): the two
                                ghost planes beyond the face are supplied by the block on the other side.  z faces only;
                                mixed precision, Heun, blocks the TMA kernel serves (nx % 32 == 0, ny % 16 == 0), nz >= 4.
                                See "Communication boundaries" below. */

/* kernel variants (kratos_hydro_set_kernel) */
#define KRATOS_KERNEL_AUTO 0   /* x,y active: TMA (mixed, 3D, nx % 32 == 0, ny % 16 == 0), strip (mixed, 2D, even extents),
                                  else paired (mixed) or tiled (all-fp64); otherwise simple */
#define KRATOS_KERNEL_SIMPLE 1 /* one thread per cell, stencil from global memory (any axes) */
#define KRATOS_KERNEL_TILED 2  /* shared-memory tile + halo, z marched in registers, each face once */
#define KRATOS_KERNEL_PAIRED 3 /* mixed precision only: two cells per thread, packed fp32x2 arithmetic,
                                  halo warps, fp64 flux exchange (x,y active) */
#define KRATOS_KERNEL_TMA 5    /* the paired scheme with all global traffic moved by TMA boxes (a producer warp loads
                                  tile, halo and U0 planes onto mbarriers and stores each updated plane): mixed
                                  precision, three active axes, nx % 32 == 0, ny % 16 == 0 */

#define KRATOS_KERNEL_STRIP 6  /* 2D blocks (nz = 1, nx and ny even; all-fp32 mode: nx % 4 == 0), mixed precision or all-fp32, Heun: one warp per 28-column strip
                                  marching along y, x neighbours by warp shuffles, row pairs by per-warp TMA boxes; no
                                  block barriers */

/* Create a solver for an nx*ny*nz block.  gamma > 1.  bc (host, 6 ints) =
 * {x-lo, x-hi, y-lo, y-hi, z-lo, z-hi}; periodic must be set on both sides of an axis or
 * neither.  Allocates two copies of the state plus small work buffers on the current device.
 * Returns NULL on error (bad argument, no device, out of memory): see kratos_hydro_last_error(). */
KRATOS_API kratos_hydro_t *kratos_hydro_create(int nx, int ny, int nz, double gamma, int scheme, const int bc[6]);

/* Free everything the handle owns.  NULL is allowed. */
KRATOS_API void kratos_hydro_destroy(kratos_hydro_t *h);

/* Cell sizes (> 0, finite); entries of inactive axes are ignored.  Default 1/n. */
KRATOS_API int kratos_hydro_set_spacing(kratos_hydro_t *h, double dx, double dy, double dz);

/* Stream (a cudaStream_t passed as void*) used by all later calls.  The caller keeps ownership. */
KRATOS_API int kratos_hydro_set_stream(kratos_hydro_t *h, void *cuda_stream);

/* Choose the kernel variant (KRATOS_KERNEL_*).  KRATOS_ERR_ARG if the variant does not
 * support this block's active axes. */
KRATOS_API int kratos_hydro_set_kernel(kratos_hydro_t *h, int variant);

/* The kernel variant (KRATOS_KERNEL_*, never AUTO) that step / run launch for this handle.  variant: host. */
KRATOS_API int kratos_hydro_get_kernel(kratos_hydro_t *h, int *variant);

/* z-extent of the slab one thread block of the marching 3D kernels works through; for the 2D strip kernel the number
 * of rows (rounded up to even) one warp marches through (0 = automatic). */
KRATOS_API int kratos_hydro_set_zchunk(kratos_hydro_t *h, int planes);

/* Copy a state in.  U: 5*nx*ny*nz doubles in the layout above; on_device = 0: host pointer
 * (pageable or pinned), 1: device pointer.  Synchronises the stream when U is on the host. */
KRATOS_API int kratos_hydro_set_state(kratos_hydro_t *h, const double *U, int on_device);

/* Copy the current state out (same layout and rules).  KRATOS_ERR_NONFINITE is NOT checked here. */
KRATOS_API int kratos_hydro_get_state(kratos_hydro_t *h, double *U, int on_device);

/* CFL time step of the current state:
 *   dt = cfl / max_cells sum_{active d} (|v_d| + c)/dx_d,  c = sqrt(gamma p / rho),
 * evaluated in fp64 in every precision mode by a min-reduction kernel.  dt_out: host.
 * Synchronises.  KRATOS_ERR_NONFINITE if the result is not finite and positive. */
KRATOS_API int kratos_hydro_cfl_dt(kratos_hydro_t *h, double cfl, double *dt_out);

/* One full step of length dt (> 0, finite; else KRATOS_ERR_ARG).  Heun:
 *   U1 = U + dt L(U);  U <- 1/2 U + 1/2 (U1 + dt L(U1))
 * van Leer (reading S15): W = prim(U + dt/2 L_1(U)); U <- U + dt L(W).
 * Asynchronous; a non-finite result is reported by kratos_hydro_status, not here. */
KRATOS_API int kratos_hydro_step(kratos_hydro_t *h, double dt);

/* nsteps Heun steps with the time step kept on the device (no host round trip per step):
 * before each step dt = cfl / (rate maximum of the current state), the maximum having been
 * reduced inside the previous step's final kernel (first step: by the cfl_dt kernel).  In mixed
 * precision that fused rate is evaluated in float_t from the freshly updated float2_t state.
 * t_inout (host): time before / after.  Synchronises at the end. */
KRATOS_API int kratos_hydro_run(kratos_hydro_t *h, double cfl, int nsteps, double *t_inout);

/* As run, but every dt is clipped so that t lands exactly on t_end; stops when t == t_end or
 * after max_steps.  steps_done (host, may be NULL). */
KRATOS_API int kratos_hydro_run_until(kratos_hydro_t *h, double cfl, double t_end, int max_steps,
                           double *t_inout, int *steps_done);

/* Compensated (double-double) sums of the five conserved fields over the interior, not
 * multiplied by the cell volume.  out: host.  Synchronises. */
KRATOS_API int kratos_hydro_totals(kratos_hydro_t *h, double out[5]);

/* Number of times a primitive floor (rho, p >= 1e-30) fired since create.  n: host.  Synchronises. */
KRATOS_API int kratos_hydro_floor_hits(kratos_hydro_t *h, long long *n);

/* Health of the run so far: KRATOS_OK, or KRATOS_ERR_NONFINITE when a time step of run / run_until came out
 * non-finite or the state left by the last step / run holds a NaN or an infinite wave speed (the final kernel of
 * every step reduces the CFL rate of the new state, and maps NaN onto +inf), or KRATOS_ERR_CUDA
 * when an asynchronous launch failed.  Synchronises.  step() itself is asynchronous and cannot report this. */
KRATOS_API int kratos_hydro_status(kratos_hydro_t *h);

/* Number of kernel launches this handle has issued since create.  n: host.  No synchronisation. */
KRATOS_API int kratos_hydro_launch_count(kratos_hydro_t *h, long long *n);

/* Per-kernel timing with CUDA events on the handle's stream.  enable != 0 switches event
 * recording on for step / run: around every launch (enable = 1), or around the launches of every
 * enable-th step only (enable > 1: two event records cost about 2.5 us of stream time each, which
 * shows on grids whose step takes a fraction of a millisecond); kratos_hydro_get_timing then returns, since the last call to
 * set_profiling, the summed duration [ms] and launch count of: slot 0 stage-1 kernel,
 * slot 1 stage-2 kernel, slot 2 all other kernels (dt bookkeeping, reductions).
 * ms, launches: host arrays of 3.  Synchronises. */
KRATOS_API int kratos_hydro_set_profiling(kratos_hydro_t *h, int enable);
KRATOS_API int kratos_hydro_get_timing(kratos_hydro_t *h, double ms[3], long long launches[3]);

/* ---- Communication boundaries: one block per GPU, blocks stacked along z (Sec. 3.1.2; Table 2's
 * two-GPU splits).
 *
 * A z face with KRATOS_BC_COMM has a ghost array per state array, [5][2][ny][nx] doubles (field, plane, y, x; plane 0 is
 * the one further from the block on the low side and the one next to it on the high side: ghost planes in ascending z),
 * which the block on the other side fills: its stage kernels store every updated plane that lies within two planes of the
 * common face a second time, straight into this array (peer memory: the same process, or another process through a CUDA IPC
 * handle; over NVLink between GPUs) -- the halo exchange is fused into the stage kernel, there is no pack / send / unpack.
 * What remains for the driver (paper_2501_02317_b200/slab.py) is ordering: a block may start stage 2 only after its
 * neighbours have finished stage 1, and the next step's stage 1 only after their stage 2; and the time step is the minimum
 * over all blocks.  Hence the step is cut into pieces:
 *
 *     set_state on every block; get_/set_reference_pressure (one value for all blocks); push_halo; <sync>
 *     begin_run(cfl, t0)                       local CFL rate
 *     repeat:  get_rate -> <max over blocks> -> set_rate;  substep(PREPARE);  substep(STAGE1);  <sync>;  substep(STAGE2);  <sync>
 *     end_run
 *
 * <sync> = every block's stream has passed this point before any continues (stream order within a process, a collective
 * of the process group across processes).  kratos_hydro_step / run / run_until refuse blocks with communication boundaries.
 * array: 0 = the current state, 1 = the predictor of the Heun step.  side: 0 = low z face, 1 = high z face. */
#define KRATOS_PHASE_PREPARE 0 /* dt = cfl / rate (the rate set by set_rate, or left by the last stage 2), t += dt */
#define KRATOS_PHASE_STAGE1 1
#define KRATOS_PHASE_STAGE2 2

/* Device pointer of this block's ghost array (owned by the handle).  ptr: host. */
KRATOS_API int kratos_hydro_ghost_array(kratos_hydro_t *h, int array, int side, double **ptr);

/* CUDA IPC handle (64 bytes, cudaIpcMemHandle_t) of that ghost array, for a neighbour in another process.  handle: host. */
KRATOS_API int kratos_hydro_ghost_ipc_handle(kratos_hydro_t *h, int array, int side, unsigned char handle[64]);

/* The block beyond z face `side`: its ghost arrays that hold THIS block's planes (its high-side arrays for side 0, its
 * low-side arrays for side 1) of the current state and of the predictor, as device pointers valid on this handle's device
 * (the caller keeps them alive).  open_peer takes the neighbour's IPC handles instead and maps them (unmapped at destroy). */
KRATOS_API int kratos_hydro_set_peer(kratos_hydro_t *h, int side, double *peer_ghost_state, double *peer_ghost_pred);
KRATOS_API int kratos_hydro_open_peer(kratos_hydro_t *h, int side, const unsigned char handle_state[64],
                                      const unsigned char handle_pred[64]);

/* Copy the two planes of the current state next to each communication boundary into the neighbours' ghost arrays (after
 * set_state; during a run the stage kernels do this themselves).  Asynchronous. */
KRATOS_API int kratos_hydro_push_halo(kratos_hydro_t *h);

/* The pieces of kratos_hydro_run (see above).  begin_run: Courant number and start time, CFL rate of the current state if
 * none is at hand.  substep: one KRATOS_PHASE_*; asynchronous.  end_run: time reached and steps taken (host; steps_done may
 * be NULL); synchronises; KRATOS_ERR_NONFINITE as for run.  Heun integrator, mixed or all-fp64 precision; also valid for
 * blocks without communication boundaries (then equal to run). */
KRATOS_API int kratos_hydro_begin_run(kratos_hydro_t *h, double cfl, double t0);
KRATOS_API int kratos_hydro_substep(kratos_hydro_t *h, int phase);
KRATOS_API int kratos_hydro_end_run(kratos_hydro_t *h, double *t, int *steps_done);

/* The CFL rate maximum max_cells sum_d (|v_d| + c)/dx_d of the current state as left by begin_run, cfl_dt or
 * the last stage 2, and its replacement by the maximum over all blocks.  rate: one double, host (synchronises) or device
 * (asynchronous, on the handle's stream). */
KRATOS_API int kratos_hydro_get_rate(kratos_hydro_t *h, double *rate, int on_device);
KRATOS_API int kratos_hydro_set_rate(kratos_hydro_t *h, const double *rate, int on_device);

/* Reference pressure of the mixed-precision solver (see the top of this file; 0 in the other modes).  get computes it from
 * the current state if that has not happened yet.  set replaces it (rounded to fp32; >= 0) until the next set_state: blocks
 * of one decomposed domain must share one value (reading S17).  p_ref: host.  get synchronises; set is asynchronous
 * (stream-ordered like set_state from a device pointer). */
KRATOS_API int kratos_hydro_get_reference_pressure(kratos_hydro_t *h, double *p_ref);
KRATOS_API int kratos_hydro_set_reference_pressure(kratos_hydro_t *h, double p_ref);

/* ---- Conserved totals without any allocation.
 *
 * Who this is for.  Everything above works on a handle, and kratos_hydro_create calls cudaMalloc for the handle's state
 * and work buffers.  Some hosts of this library cannot afford that call, or cannot make it succeed:
 *   - a simulation framework (Kratos' own mesh manager is one) or a tensor library that has reserved the
 *     whole device for its own memory pool at start-up: a cudaMalloc issued later by a guest library either fails with
 *     "out of memory" or takes pages the pool's owner believed it had;
 *   - code between the steps of a running simulation that must not stall the device: cudaMalloc and cudaFree wait for all
 *     outstanding work on the device, so one diagnostic call would serialise every stream of the application.
 * Such a caller keeps the state in its own device memory already.  It can still ask for the conserved totals (the
 * conservation diagnostic of PAPER.md:232-238: mass, momentum and energy conserved to machine accuracy) with the call
 * below, which needs no handle and calls neither cudaMalloc, cudaFree nor any library routine that allocates.
 *
 * How.  The per-block partial sums that kratos_hydro_totals keeps in a buffer of the handle live here in an array that is
 * part of the library image itself (a file-scope __device__ array, KRATOS_TOTALS_STATIC_SCRATCH_BYTES = 47 424 bytes).  Every
 * GPU on which this library has been loaded by the CUDA runtime holds one copy of it until the process exits, whether the
 * call is ever used or not.  The size is fixed: the grid is capped at 592 thread blocks, each leaving one double-double
 * per field.
 *
 *   U        device pointer, on the calling thread's current device: 5*ncell doubles, U[5][ncell] (the layout at the top
 *            of this file; only the field stride matters here).  Not modified.
 *   ncell    1 <= ncell <= KRATOS_TOTALS_STATIC_MAX_CELLS, else KRATOS_ERR_ARG and nothing is launched.
 *   out      5 doubles, owned by the caller: out_on_device = 1: device pointer on the same device, the call is
 *            asynchronous on the stream; out_on_device = 0: host pointer, the call synchronises the stream.
 *   stream   a cudaStream_t passed as void* (NULL: the legacy default stream).
 * The result is, bit for bit, what kratos_hydro_totals returns for a handle holding the same state (same kernels, same
 * grid, same order of summation).  Returns KRATOS_OK, KRATOS_ERR_ARG (NULL pointer, ncell out of range, U or a device
 * `out` that is not device memory of the current device) or KRATOS_ERR_CUDA.
 *
 * Things to know.
 *  - The first call on each device looks up the device address of the scratch array (cudaGetSymbolAddress, which may make the
 *    runtime load the library's device code onto that GPU).  Make that first call once at start-up, outside any stream
 *    capture; later calls on that device only launch the two kernels.
 *  - All calls on one device share the one array.  Nothing in it needs clearing between calls (each call overwrites every
 *    slot it later reads, whatever an earlier call with another ncell left there), but two calls whose kernels can be on the
 *    GPU at the same time -- different streams without an ordering between them, or two host threads -- race on it and
 *    both return garbage.  Order them (one stream, or an event) yourself; the library does not.
 *  - The call is thread-safe on the host side only in the sense that the one-time set-up is locked. */
#define KRATOS_TOTALS_STATIC_MAX_CELLS (1LL << 31)  /* 2 147 483 648 cells: an 80 GiB fp64 state */
#define KRATOS_TOTALS_STATIC_SCRATCH_BYTES 47424
KRATOS_API int kratos_hydro_totals_static(const double *U, long long ncell, double *out, int out_on_device,
                                          void *cuda_stream);

/* Message of the last error raised on this thread ("" if none).  Never NULL. */
KRATOS_API const char *kratos_hydro_last_error(void);

/* Library version string, e.g. "kratos-hydro-b200 0.1 (sm_100a)". */
KRATOS_API const char *kratos_hydro_version(void);

#ifdef __cplusplus
}
#endif
#endif /* KRATOS_HYDRO_H */
