/*
 * hydro.h -- C-ABI boundary of the B200-native RK2 step of the 3D compressible-Euler
 * finite-volume update (the hot path of the GenASiS RiemannProblem example,
 * arXiv 1812.07977).
 *
 * The calls follow the paper's statement of the problem: Algorithm 1 "Fluid Evolution"
 * -- Initialize / ComputeTimeStep / two Runge-Kutta substeps of
 * {ComputeDifferences, ComputeReconstruction, ComputeFluxes, ComputeUpdate} separated by
 * GhostExchange -- over persistently device-allocated storage with explicit, rare transfers
 * (PAPER.md:23, 130, 247).  The numerics the paper does not print (limiter, Riemann solver,
 * EOS, time-step formula) are BASELINE.json:north_star's, under the readings R1-R20 listed in
 * DESIGN.md section 3.
 *
 * Conventions
 *  - Every call returns an int status (HYDRO_OK = 0); results come back through out-pointers.
 *  - Packed state layout for set/get: double U[5][nz][ny][nx], x fastest, ACTIVE cells only,
 *    variable order (rho, m_x, m_y, m_z, E) ("Value(nCells,nVariables)").
 *  - A `U` pointer may be a HOST pointer (pageable or pinned) or a DEVICE pointer on the
 *    handle's device; the library detects which (cudaPointerGetAttributes).  The caller owns
 *    `U` and may free or reuse it as soon as the call returns (hydro_set_state and
 *    hydro_get_state synchronise the handle's stream for host and device pointers alike; a device
 *    `U` written by work on ANOTHER stream must be complete, or ordered before the handle's stream
 *    by the caller, when the call is made).
 *  - The handle owns all device memory it allocates (two ghost-padded SoA buffers + scalars).
 *  - Work is enqueued on the handle's stream (default: the legacy default stream; see
 *    hydro_set_stream).  hydro_step / hydro_run_steps only enqueue; hydro_cfl_dt,
 *    hydro_max_signal_speed, hydro_evolve, hydro_get_state and hydro_get_time synchronise
 *    that stream.
 *  - A handle is not thread-safe; distinct handles are independent.
 *  - Deterministic: same inputs => bit-identical outputs run to run (the only atomic is an
 *    integer max on the bit pattern of a non-negative double).
 *  - There is no CPU fallback: without a CUDA device every call that needs one returns
 *    HYDRO_ERR_CUDA.
 */
#ifndef HYDRO_B200_H
#define HYDRO_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hydro hydro_t;   /* opaque */

/* Boundary rule per face (R9; replaces the physical-boundary part of the paper's
 * GhostExchange). */
enum { HYDRO_BC_OUTFLOW = 0, HYDRO_BC_REFLECT = 1, HYDRO_BC_PERIODIC = 2,
       /* z faces only: the face is an interface to a neighbouring slab of a domain decomposed along
        * z; its two ghost layers are written by the halo exchange (hydro_halo_*), never by the
        * library's boundary code.  Set by hydro_create_slab. */
       HYDRO_BC_NEIGHBOUR = 3 };

enum {
    HYDRO_OK = 0,
    HYDRO_ERR_ARG = 1,        /* bad argument (see each call) */
    HYDRO_ERR_ALLOC = 2,      /* device or host allocation failed */
    HYDRO_ERR_CUDA = 3,       /* a CUDA call failed; text in hydro_last_error() */
    HYDRO_ERR_UNPHYSICAL = 4, /* rho <= 0, p <= 0 or a non-finite signal speed was seen */
    HYDRO_ERR_NOSTATE = 5     /* step/evolve/cfl_dt/get_state before set_state */
};

/* ---- the calls BASELINE.json:north_star names -------------------------------------- */

/* Algorithm 1 line 1, "Initialize": allocate the persistent device state for an
 * nx*ny*nz grid of cubic cells of edge dx (R13) with 2 ghost layers per side,
 * ideal gas with adiabatic index gamma (R1).
 *   bc[6]: HYDRO_BC_* for faces xlo,xhi,ylo,yhi,zlo,zhi (host pointer, copied).
 * Defaults: CFL 0.7, limiter theta 1.4.
 * Performance note: the stage kernels tile x in units of 32 cells and y in units of 8 or 16 and march
 * along z, so a grid with one awkward extent (33) is cheapest with that extent as nz; the library holds
 * such a run with its axes relabelled by itself (hydro_get_axis_order below).
 * HYDRO_ERR_ARG if nx,ny,nz < 2, gamma <= 1, dx <= 0 or non-finite, unknown bc value,
 * periodic on only one face of an axis, or a NULL pointer.  *out is NULL on failure. */
int hydro_create(int nx, int ny, int nz, double gamma, double dx, const int bc[6],
                 hydro_t **out);

/* The paper's RiemannProblem also runs in one and two dimensions (Fig. 1, PAPER.md:138:
 * "an extension of the classic 1D Sod shock tube ... to 2D and 3D"): hydro_create_nd makes a run of
 * dimension ndim = 1, 2 or 3 whose first ndim axes are active, with cell edges d[0..ndim-1]
 * (R21-R24).  An inactive axis has n[a] == 1, no ghost layers, no ghost exchange and no
 * differences, reconstruction or fluxes (its d[a] and bc entries are ignored); all five variables
 * are still carried.  The update is -(dt/dx) [dFx + (dx/dy) dFy + (dx/dz) dFz] over the active axes
 * and hydro_cfl_dt returns (cfl/ndim) * min_d(d[a]) / max(|v| + c_s).  hydro_create(nx,ny,nz,..,dx,..)
 * is hydro_create_nd(3, {nx,ny,nz}, {dx,dx,dx}, ..).  The packed layout stays U[5][nz][ny][nx].
 * HYDRO_ERR_ARG if ndim is not 1..3, an active axis has n[a] < 2 or d[a] <= 0, an inactive axis has
 * n[a] != 1, or the bc of an active axis is invalid. */
int hydro_create_nd(int ndim, const int n[3], const double d[3], double gamma, const int bc[6],
                    hydro_t **out);

/* Copy a packed state (host or device pointer, layout above) into the device state; resets the
 * time to 0 and the step count to 0.  Synchronises the handle's stream. */
int hydro_set_state(hydro_t *h, const double *U);

/* Algorithm 1 line 5, "ComputeTimeStep": reduction over active cells,
 *   *dt = (cfl/3) * (dx / max(|v| + c_s))      (R8; |v| Euclidean, c_s = sqrt(gamma p/rho);
 *                                               in general (cfl/ndim) * min_d(d[a]) / max, R22).
 * dt: host pointer.  Synchronises.  HYDRO_ERR_UNPHYSICAL if any active cell has rho <= 0,
 * p <= 0 or a non-finite speed. */
int hydro_cfl_dt(hydro_t *h, double *dt);

/* One RK2 step of size dt: Algorithm 1 lines 6-21:
 *   U1 = U0 + dU(U0);  U(n+1) = 0.5*(U0 + U1 + dU(U1)),  ghost fill before each substep.
 * Asynchronous (enqueue only).  HYDRO_ERR_ARG if dt <= 0 or non-finite. */
int hydro_step(hydro_t *h, double dt);

/* Algorithm 1 lines 3-4, 23: while t < t_final { dt = cfl_dt; clip the
 * last step to land on t_final exactly (R14); step }.  *nsteps (host, may be NULL) receives the
 * number of steps taken.  The time step, the clipping and the clock stay on the device: steps are
 * enqueued in batches (at most 64) between host reads of the device scalars, and a step enqueued
 * past t_final runs with dt = 0, which leaves the state numerically identical (U + 0 and
 * 0.5*((U + U) + 0): every value keeps its bits except that a conserved value of -0.0 may come back
 * as +0.0).  Synchronises.
 * HYDRO_ERR_ARG if t_final < t or non-finite; HYDRO_ERR_UNPHYSICAL as hydro_cfl_dt, and when the
 * time step stops advancing the clock (dt underflows to 0 or t + dt == t). */
int hydro_evolve(hydro_t *h, double t_final, long long *nsteps);

/* Copy the device state out into a packed array (host or device pointer).  Synchronises.
 * Returns HYDRO_ERR_UNPHYSICAL (after copying) if the sticky unphysical flag is set. */
int hydro_get_state(hydro_t *h, double *U);

/* ---- needed but not named in north_star -------------------------------------------- */

int hydro_destroy(hydro_t *h);
int hydro_set_cfl(hydro_t *h, double cfl);               /* > 0; configs use 0.7 / 0.5 */
int hydro_set_limiter_theta(hydro_t *h, double theta);   /* in [1,2]; default 1.4 (R5) */
int hydro_get_time(hydro_t *h, double *t, long long *step);   /* either may be NULL */
/* Raw reduction max(|v| + c_s) over active cells (test hook; same error rule as cfl_dt). */
int hydro_max_signal_speed(hydro_t *h, double *smax);
/* Run on this cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream).  NULL = default. */
int hydro_set_stream(hydro_t *h, void *cuda_stream);
/* Process-wide allocator hook used by handles created afterwards (e.g. torch's caching
 * allocator).  alloc(bytes, stream) returns a device pointer or NULL; release(ptr) frees it.
 * Pass NULL, NULL to restore cudaMalloc / cudaFree. */
int hydro_set_allocator(void *(*alloc)(size_t bytes, void *stream), void (*release)(void *ptr));
/* n steps with the time step kept on the device: each step uses
 * dt = (cfl/3)*dx/smax with smax reduced by the previous step's last kernel (or by a
 * stand-alone reduction after set_state).  No host round trip; asynchronous.  On a non-default
 * stream the step is captured once as a CUDA graph and replayed (rebuilt when the stream, CFL,
 * theta or the kernel variant changes).  The benchmark path (Algorithm 1's loop body without the
 * host-side ComputeTimeStep of Algorithm 2). */
int hydro_run_steps(hydro_t *h, long long n);
/* ---- host mirror with explicit, selective, overlapped transfers -------------------------------
 * The paper's StorageForm keeps a host copy of the device storage and moves "all the selected fields
 * ... en masse with a single call.  Alternatively, individual fields can be specified",
 * from page-locked host memory for 1.7-2.0x faster transfers.  Same here, with
 * the transfers off the compute stream:
 * hydro_host_alloc: a pinned host buffer of one packed state U[5][nz][ny][nx], owned by the handle
 *   (freed by hydro_destroy).  Any pinned or pageable host pointer works with the calls below; pinned
 *   memory is what makes them asynchronous.
 * hydro_update_device(h, fields, U_host): field v (bit v of `fields`: 1 rho, 2 m_x, 4 m_y, 8 m_z,
 *   16 E) of the device state <- U_host, host-to-device on the handle's copy-in stream; work already
 *   enqueued on the compute stream keeps running during the transfer, work enqueued afterwards sees
 *   the new fields.  Keeps the clock (unlike hydro_set_state); the first update of a handle must bring
 *   all five fields.
 * hydro_update_host(h, fields, U_host): U_host <- selected fields of the state as of the work
 *   enqueued so far: a device-side snapshot on the compute stream, then device-to-host on the copy-out
 *   stream, so steps enqueued next overlap the transfer (and a following hydro_update_device's
 *   transfer runs concurrently in the other direction).  U_host is valid after hydro_transfer_sync.
 * hydro_transfer_sync: wait for the outstanding transfers of both directions.
 * HYDRO_ERR_ARG for an empty or unknown field mask. */
int hydro_host_alloc(hydro_t *h, double **U_host);
int hydro_update_device(hydro_t *h, unsigned fields, const double *U_host);
int hydro_update_host(hydro_t *h, unsigned fields, double *U_host);
int hydro_transfer_sync(hydro_t *h);

/* ---- domain decomposition into z-slabs ----------------------------------------------------
 * The paper runs the problem decomposed over MPI ranks, one GPU each, 256^3 cells per rank, with a
 * ghost exchange after every Runge-Kutta substep and a reduction of the time step every step
 * (PAPER.md:172, 186, 245, 264, 325, 357); its exchange goes through the host, and device-to-device
 * exchange is named as future work.  Here a slab is an ordinary handle whose z faces
 * towards neighbouring slabs have kind HYDRO_BC_NEIGHBOUR; a driver (paper_1812_07977_b200/slab.py)
 * alternates hydro_substep with the exchange of the two boundary planes per interface and all-reduces
 * the maximum signal speed.  Results are bit-identical to the single-domain run.
 *
 * hydro_create_slab: the handle of slab `rank` of `nranks` for a global nx*ny*nz_global grid with
 * physical boundaries bc (cubic cells).  Planes are dealt out evenly, the first nz_global % nranks
 * slabs getting one more; *k_first / *nz_local (may be NULL) receive the slab's first global plane
 * and its plane count.  A periodic z boundary becomes a neighbour interface between the last and the
 * first slab.  HYDRO_ERR_ARG if a slab would have fewer than 2 planes.
 * hydro_substep: one substep (stage 1: U1 = U0 + dU(U0) into the second buffer; stage 2:
 * U(n+1) = 0.5 (U0 + U1 + dU(U1)) in place, with the fused max-signal-speed reduction) on
 * part 0 = all planes, 1 = the planes next to neighbour interfaces (launch these first, exchange
 * them while part 2 runs), 2 = the remaining planes.  dt > 0: host-supplied step; dt == 0: the
 * device-resident step (cfl/3) dx / smax formed at the start of stage 1 from the running maximum
 * at hydro_smax_device, which the driver has all-reduced (MAX) over the slabs (hydro_reduce_smax
 * computes the local value after hydro_set_state).  Asynchronous.
 * hydro_halo_count: doubles in one packed face = 5 * 2 * ny * nx.  hydro_halo_pack copies the two
 * ACTIVE planes next to face `side` (0 = z low, 1 = z high) of buffer `which` (0 = state, 1 = stage-1
 * result) into dst[5][2][ny][nx] (device pointer); hydro_halo_unpack writes src into the two GHOST
 * planes of that face.  hydro_halo_push does both at once as direct stores into the neighbour's
 * state (device pointer from hydro_state_base on the neighbour, mapped on this device: same process,
 * peer access or CUDA IPC) -- over NVLink when the neighbour lives on another GPU.  All asynchronous
 * on the handle's stream; ordering between slabs (events, barriers) is the driver's. */
int hydro_create_slab(int nx, int ny, int nz_global, double gamma, double dx, const int bc[6],
                      int rank, int nranks, hydro_t **out, int *k_first, int *nz_local);
int hydro_substep(hydro_t *h, int stage, double dt, int part);
int hydro_halo_count(hydro_t *h, size_t *doubles);
int hydro_halo_pack(hydro_t *h, int which, int side, double *dst);
int hydro_halo_unpack(hydro_t *h, int which, int side, const double *src);
int hydro_halo_push(hydro_t *h, int which, int side, double *peer_base, int peer_nz,
                    long long peer_var_stride);
int hydro_state_base(hydro_t *h, int which, double **base, int *nz_local, long long *var_stride);
int hydro_smax_device(hydro_t *h, double **smax);
int hydro_reduce_smax(hydro_t *h);

/* Test hooks: run only the ghost fill on the current state, and read the padded buffer
 * [5][nz+4][ny+4][nx+4] (x fastest, row pitch removed; no +4 on an inactive axis) into a host or
 * device array. */
int hydro_ghost_fill(hydro_t *h);
int hydro_get_padded(hydro_t *h, double *Upad);
/* Tuning hooks of the fused stage kernel (tests and measurement; defaults are chosen per grid).
 * hydro_set_tiling: tile_rows = 8 | 16 (rows of 32 cells per block; 0 = chosen by the library),
 * planes_per_chunk = z-planes a block marches over (for a 2D run: 32 x 16 tiles a block walks down y);
 * 0 = chosen by the library: uniform chunks that fill whole waves of the SMs, or "balanced layers" --
 * chunks that put one block on every resident slot of the device plus thinner remainder chunks for
 * the slots left over ("Launch geometry").  hydro_get_tiling reports the geometry
 * in use -- planes_per_chunk is the (primary) chunk length -- and the number of blocks per stage launch
 * (any out-pointer may be NULL).  hydro_tiling_partition is the host logic behind it, callable without a
 * device: the z partition of a launch over the active planes [kb, ke) of an nx x ny x nz grid on a device
 * with `sms` multiprocessors, out = { lz, km, nprim, lzr, nlayer }: layers 0 .. nprim-1 are the chunks of
 * lz planes of [kb, km), layers nprim .. nlayer-1 the chunks of lzr planes of [km, ke).
 * hydro_set_graph_replay(h, 0) makes hydro_run_steps /
 * hydro_evolve enqueue plain launches instead of replaying the captured one-step CUDA graph. */
int hydro_set_tiling(hydro_t *h, int tile_rows, int planes_per_chunk);
int hydro_get_tiling(hydro_t *h, int *tile_rows, int *planes_per_chunk, long long *blocks);
int hydro_tiling_partition(int nx, int ny, int nz, int tile_rows, int planes_per_chunk, int sms, int kb, int ke,
                           int out[5]);
int hydro_set_graph_replay(hydro_t *h, int enable);
/* The library may hold a 3D run of cubic cells with its axes relabelled when the launch-geometry cost
 * model says another order is at least 12 % cheaper (a grid 33 cells wide costs two 32-wide tile columns;
 * as nz it costs nothing): the scheme is symmetric under relabelling, and only the copies in and out of
 * the handle know.  Every call keeps the caller's axis order; hydro_get_axis_order reports the internal
 * axis of the caller's axes x, y, z (0, 1, 2 = not relabelled).  hydro_get_padded is not available on
 * a relabelled handle (HYDRO_ERR_ARG). */
int hydro_get_axis_order(hydro_t *h, int order[3]);
/* Select the stage-kernel implementation:
 * 0 = reference-structured simple kernel (one thread per
 * cell, everything recomputed, ghost layers filled in memory before each substep); 1 = fused tiled
 * kernel (default).  2D and 3D runs: the boundary rules are applied in the kernel (ghost layers are
 * written to memory only for periodic x / y faces, and not at all otherwise -- three launches per
 * step); 1D runs: each slope and flux once per cell, every boundary kind applied in the kernel.
 * 2 = the fused 2D / 3D kernel reading every ghost layer from memory (cross-check of 1; not for 1D
 * runs).  3 = 2D runs only: the "warp column" kernel -- a warp owns a 32-lane strip and marches down y
 * with the y direction in registers and the x direction exchanged by warp shuffles (no shared memory,
 * no barriers, every boundary kind applied on the way in); within 2 % of variant 1 on large grids,
 * 10-15 % faster around 1024^2 - 2048^2, slower below 768^2; the default of 2D
 * runs of 2^20 cells and more. */
int hydro_set_kernel_variant(hydro_t *h, int variant);
/* Measurement hooks (bench.py): when enabled, every kernel launch of this handle is bracketed by
 * CUDA events on the handle's stream.  hydro_get_kernel_time synchronises and returns the summed
 * duration (ms) and launch count since profiling was enabled, for which = 0 ghost fill,
 * 1 stage-1 kernel, 2 stage-2 kernel, 3 start-of-step kernel (time step and accumulator reset, when
 * the step has no ghost fill to carry them), 4 stand-alone CFL reduction. */
int hydro_set_profiling(hydro_t *h, int enable);
int hydro_get_kernel_time(hydro_t *h, int which, double *ms, long long *count);
/* ---- allocation-free entry point ---------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): Algorithm 1 line 5, "ComputeTimeStep" -- the reduction
 * max(|v| + c_s) over the cells of a packed state (R8; the same arithmetic as hydro_max_signal_speed) --
 * without a handle and without any allocation: no cudaMalloc, cudaFree or allocating library routine is
 * called.  The scratch of the reduction (one partial maximum per block of 2048 cells and a ticket) is a
 * file-scope device array of HYDRO_NOALLOC_SCRATCH_BYTES (1 MiB + 256 B) that every GPU loading this
 * library holds until the process exits; its capacity sets the limit HYDRO_NOALLOC_MAX_CELLS = 2^27
 * cells (512^3, the largest configuration).
 *   U_dev:    DEVICE pointer (current device), packed double U[5][ncells] (rho, m_x, m_y, m_z, E; the
 *             layout of hydro_get_state with ncells = nx*ny*nz); read only, the caller keeps ownership.
 *   smax_dev: DEVICE pointer to one double, receives max(|v| + c_s) (0 if no cell has a positive speed).
 *   flag_dev: DEVICE pointer to one int, receives 1 if any cell has rho <= 0, p <= 0 or a non-finite
 *             speed (HYDRO_ERR_UNPHYSICAL's condition), else 0.
 *   cuda_stream: the cudaStream_t to enqueue on (NULL = default stream).  Asynchronous: the outputs are
 *             valid once the stream has run the call; the time step is (cfl/ndim) * min_d(d[a]) / *smax_dev.
 * Every call on a device shares the one scratch array, which keeps the last call's contents (the call
 * clears what must start at zero itself): calls that overlap on the GPU -- two streams, two threads --
 * race on it and give wrong results; calls on one stream, or otherwise ordered, are safe.  The first call
 * on a device looks up the array's address (cudaGetSymbolAddress); make that call outside graph capture.
 * HYDRO_ERR_ARG (before any CUDA call) for a NULL pointer, ncells < 1, ncells > HYDRO_NOALLOC_MAX_CELLS
 * (use a handle and hydro_max_signal_speed for larger states) or gamma <= 1; HYDRO_ERR_ARG for a host
 * pointer; HYDRO_ERR_CUDA if a CUDA call fails.  Not counted by hydro_get_kernel_time. */
#define HYDRO_NOALLOC_MAX_CELLS 134217728LL
#define HYDRO_NOALLOC_SCRATCH_BYTES 1048832
int hydro_max_signal_speed_noalloc(const double *U_dev, long long ncells, double gamma,
                                   double *smax_dev, int *flag_dev, void *cuda_stream);
/* Number of kernels this library has launched since load (for bench.py's gpu_launches). */
long long hydro_launch_count(void);
/* 1 if this library was compiled with -fmad=false (verification build), else 0. */
int hydro_is_verification_build(void);
/* Text of the last error on this thread (never NULL). */
const char *hydro_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* HYDRO_B200_H */
