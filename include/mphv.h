/*
 * mphv.h -- C ABI of the B200-native (sm_100a) kinetic Vlasov hot path of muphyII
 * (arXiv 2305.01487): dimensionally split, conservative, positivity-preserving
 * third-order semi-Lagrangian (PFC) sweeps of f(x,v) plus the velocity moments n, j, P.
 *
 * Citations: "P:Lnnn" = PAPER.md line nnn; "R1..R14" = the readings listed in DESIGN.md
 * (= SURVEY.md sec. 8(c)); BJ = BASELINE.json.
 *
 * Conventions (all calls)
 * -----------------------
 *  - Plain C, no torch types. "dev" pointers are CUDA device pointers owned by the
 *    CALLER (the library allocates only O(spatial cells) workspace); they must stay
 *    valid until the context's stream has drained. "host" pointers are host memory.
 *  - Layouts, C order, fastest index LAST, interior cells only (no stored halo):
 *        f    [nz][ny][nx][nvz][nvy][nvx]                  fp64
 *        E, B [3][nz][ny][nx]   component-major, CELL-CENTRED (R8)
 *        n    [nz][ny][nx];  j [3][nz][ny][nx];  P [6][nz][ny][nx] in order xx,xy,xz,yy,yz,zz
 *  - Units: j = int v f d3v, P = int v v f d3v (no q, no m: the API carries only q/m; R10).
 *  - Async: every *device* call only enqueues work on the context's stream and returns;
 *    outputs are valid after the caller synchronises that stream. Host-buffer calls
 *    (mphv_run_host) synchronise before returning.
 *  - Errors: int status, 0 = MPHV_OK. No exception or abort crosses the ABI. A call that
 *    fails with ARG/STATE/RANGE leaves f untouched. Text: mphv_strerror / mphv_last_error.
 *  - Inactive dimension = extent 1. Inactive velocity dim: v == 0, dv == 1 in dV.
 *    An active dimension needs extent >= 4 (two boundary cells per side).
 *  - There is NO CPU fallback: without a CUDA device of compute capability 10.x
 *    mphv_create fails (MPHV_ERR_ARCH / MPHV_ERR_CUDA through mphv_last_error(NULL)).
 */
#ifndef MPHV_H
#define MPHV_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mphv_ctx mphv_ctx;      /* opaque; created/destroyed by the library */

typedef struct {
    int32_t nx[3];                     /* spatial extents x,y,z; 1 = inactive                    */
    int32_t nv[3];                     /* velocity extents vx,vy,vz; 1 = inactive                */
    int32_t bc[3];                     /* per spatial dim: MPHV_BC_PERIODIC or MPHV_BC_OUTFLOW   */
} mphv_grid;

typedef struct {                       /* cell-centred finite volumes tile [lo,hi) (R1)          */
    double xlo[3], xhi[3], vlo[3], vhi[3];
} mphv_box;

enum { MPHV_BC_PERIODIC = 0, MPHV_BC_OUTFLOW = 1 };

enum {
    MPHV_OK        = 0,
    MPHV_ERR_ARG   = 1,  /* null pointer, dim out of range or inactive, non-finite dt, extent < 1,
                            hi <= lo, active extent < 4, bad bc                                    */
    MPHV_ERR_STATE = 2,  /* f or fields not bound                                                  */
    MPHV_ERR_RANGE = 3,  /* |s| >= 1 on a non-periodic axis (outflow or velocity), or |s| >= 1 on a
                            periodic axis with no scratch bound                                    */
    MPHV_ERR_CUDA  = 4,  /* CUDA runtime / launch error; text in mphv_last_error                   */
    MPHV_ERR_ARCH  = 5   /* device is not compute capability 10.x (sm_100)                         */
};

/* Create a context for one species on one GPU (the current CUDA device).
 * Grid/box per R1; q_over_m multiplies (E + v x B) in eq. (1).
 * Returns NULL on error (reason: mphv_last_error(NULL)). BJ north_star: mphv_create. */
mphv_ctx *mphv_create(const mphv_grid *grid, const mphv_box *box, double q_over_m);
int mphv_destroy(mphv_ctx *ctx);

/* CUDA stream (cudaStream_t passed as void*) all later calls enqueue on; NULL = legacy
 * default stream (the default after create). */
int mphv_set_stream(mphv_ctx *ctx, void *cuda_stream);

/* Number of doubles in f = prod(nx) * prod(nv). 0 if ctx is NULL. */
size_t mphv_f_count(const mphv_ctx *ctx);
/* Number of spatial cells prod(nx). */
size_t mphv_space_count(const mphv_ctx *ctx);

/* Bind the distribution function (device, f_count doubles, 16-byte aligned) and an optional
 * scratch buffer of the same size (device; NULL allowed). Scratch is only used when a
 * periodic spatial sweep is asked for |s| >= 1 (whole-cell shifts, semi-Lagrangian part
 * R3/R11); without it such a call returns MPHV_ERR_RANGE. All sweeps are in place. */
int mphv_bind_f(mphv_ctx *ctx, double *f_dev, double *scratch_dev);

/* E, B: device, [3][nz][ny][nx] each, cell-centred, borrowed until the next set_fields.
 * The call also enqueues a small reduction that records max |a_d| bounds used for the
 * MPHV_ERR_RANGE check of velocity sweeps; it synchronises the stream once to read the
 * three bounds back (fields change once per step, sweeps do not sync). */
int mphv_set_fields(mphv_ctx *ctx, const double *E_dev, const double *B_dev);

/* Spatial sweep S_d(dt), d = dim in 0..2: every pencil of f along spatial axis d is remapped
 * by the 1-D PFC-3 scheme with Courant number s = v_d dt / dx_d, v_d the velocity cell
 * centre (term v.grad_x f of eq. (1); scheme P:L135; readings R1-R3, R6, R11, R12).
 * Boundary: periodic = index wrap, outflow = zero-gradient ghosts (a1 of SURVEY 8(a)).
 * dt < 0 is legal. Errors: ARG (dim inactive / out of range, dt not finite), STATE,
 * RANGE (see above). */
int mphv_sweep_x(mphv_ctx *ctx, int dim, double dt);

/* Velocity sweep V_d(dt), d = dim in 0..2: every pencil along velocity axis d is remapped
 * with s = a_d dt / dv_d, a_d = (q/m)(E_d + (v x B)_d) at the spatial cell, using the cell
 * centres of the other two velocity components (eq. (1)). The velocity box is
 * closed: empty ghosts and zero flux through the two wall faces (R7). |s| >= 1 anywhere
 * => MPHV_ERR_RANGE (checked against the bound recorded by mphv_set_fields). */
int mphv_sweep_v(mphv_ctx *ctx, int dim, double dt);

/* Full split step (R4, R5): S_x, S_y, S_z, V_vx, V_vy, V_vz in that order, each with
 * the full dt, inactive dimensions skipped, fields frozen. All range checks are done
 * before the first sweep is enqueued. The library may fuse consecutive sweeps into one
 * kernel; the result is that of the unfused sequence up to fp64 rounding. */
int mphv_step(mphv_ctx *ctx, double dt);

/* The X stage of mphv_step alone: S_x, S_y, S_z in that order (fused as in mphv_step), inactive
 * dimensions skipped; range checks as mphv_sweep_x, all before the first sweep is enqueued. With
 * mphv_stage_v this gives callers true Strang splitting, X(dt/2) V(dt) X(dt/2). */
int mphv_stage_x(mphv_ctx *ctx, double dt);

/* The X stage of a block that is decomposed along x ONLY (the other spatial axes are whole and follow
 * grid.bc): S_x with its ghost cells from lo_dev / hi_dev (as mphv_sweep_x_halo(0, ...); NULL = global
 * outflow end), then S_y, S_z; S_x and S_y fused into one pass as in mphv_step where the grid allows.
 * Same checks as mphv_sweep_x_halo for axis 0 and mphv_sweep_x for the others. */
int mphv_stage_x_halo(mphv_ctx *ctx, double dt, const double *lo_dev, const double *hi_dev);

/* The V stage of mphv_step alone: V_vx, V_vy, V_vz in that order (fused as in mphv_step), and, when
 * n_dev is not NULL, the moments of the result (then j_dev and P_dev must be given too). With
 * mphv_sweep_x / mphv_sweep_x_halo for the X stage this is mphv_step[_moments] taken apart, for callers
 * that exchange boundary cells between the spatial sweeps (spatial block decomposition). */
int mphv_stage_v(mphv_ctx *ctx, double dt, double *n_dev, double *j_dev, double *P_dev);

/* ---- spatial block decomposition over several GPUs (the paper's MPI domain decomposition with
 * boundary cells; "two boundary cells"). A context then describes ONE block; along a
 * decomposed spatial axis its ghost cells come from the neighbouring blocks instead of the bc rule.
 *
 * mphv_halo_count: doubles in one halo slab of axis dim = 2 layers x (cells of the block / nx[dim]).
 * mphv_pack_halo:  copies the two boundary layers of f at the low (side 0) or high (side 1) end of
 *                  spatial axis dim into buf_dev (device, halo_count doubles), laid out as f with
 *                  extent 2 along dim, layers in ascending index order. What a block packs at its
 *                  high end is its upper neighbour's lo halo and vice versa.
 * mphv_sweep_x_halo: S_dim(dt) as mphv_sweep_x, with the two ghost layers below the block read from
 *                  lo_dev and the two above from hi_dev (device or peer-mapped memory, layout as
 *                  packed). A NULL pointer marks a global OUTFLOW end (zero-gradient ghosts, R6);
 *                  on a periodic axis both must be given (the wrap-around neighbour's layers).
 *                  Needs max |s| < 1 (else MPHV_ERR_RANGE: whole-cell shifts would reach past the
 *                  two boundary cells). The result on the block equals the sweep of the whole grid. */
size_t mphv_halo_count(const mphv_ctx *ctx, int dim);
int mphv_pack_halo(mphv_ctx *ctx, int dim, int side, double *buf_dev);
int mphv_sweep_x_halo(mphv_ctx *ctx, int dim, double dt, const double *lo_dev, const double *hi_dev);

/* Velocity moments by the midpoint rule at velocity cell centres (R9, R10):
 * n = sum f dV, j_a = sum v_a f dV, P_ab = sum v_a v_b f dV, dV = dvx dvy dvz.
 * Outputs: device, n [nz][ny][nx], j [3][...], P [6][...] (xx,xy,xz,yy,yz,zz). */
int mphv_moments(mphv_ctx *ctx, double *n_dev, double *j_dev, double *P_dev);

/* mphv_step followed by mphv_moments of the new f, with the moments accumulated inside
 * the last velocity sweep's kernel when that is possible (f is then read once less).
 * Same result as the two calls up to fp64 summation order. */
int mphv_step_moments(mphv_ctx *ctx, double dt, double *n_dev, double *j_dev, double *P_dev);

/* Host-buffer convenience path (used for end-to-end timing): copies f_host (f_count doubles,
 * ideally pinned) to the bound device f, runs nsteps x mphv_step(dt), computes the moments
 * into library-owned device workspace, copies f back to f_host and the moments to
 * n_host [ns], j_host [3 ns], P_host [6 ns] (any of the three may be NULL), and
 * synchronises the stream. Requires bind_f and set_fields. On grids of 16 MiB and more (plain V mode, |s| < 1 along
 * the outermost active spatial axis) f is cut into up to 16 slabs along that axis and the copy in, the first step,
 * the last step and the copy out are overlapped slab by slab on three streams (each slab is swept as a block of a
 * spatial decomposition, with the neighbouring slabs' boundary layers as ghost cells): a call then costs about one
 * PCIe transfer of f instead of two. Same result up to fp64 rounding.
 * What the slab path needs and costs: (1) f_host must be PINNED (cudaHostAlloc / cudaHostRegister) for the overlap
 * to happen; with pageable memory every copy blocks the host and the call costs about what the plain path costs.
 * (2) It is taken only when |s| < 1 on EVERY active spatial axis (the slabs have no scratch buffer; a whole-cell shift
 * on a periodic axis takes the plain path, which needs the scratch bound by mphv_bind_f). (3) Device memory, allocated
 * at the first such call and kept until mphv_destroy: up to 16 slab contexts (O(spatial cells) each), a copy of the
 * fields, and 4 boundary layers per slab -- K*4/n of f for n cells along the slab axis, i.e. a FULL extra copy of f
 * when n = 64 and K = 16. If that allocation fails the failure is remembered and this context uses the plain path from
 * then on. (4) With mphv_set_timing on, the kernels of pipelined steps run in the slab contexts and are NOT recorded in
 * this context's timing slots (mphv_get_timing then under-counts; bench.py times mphv_step, not this call).
 * (5) On a context in deferred mode (mphv_set_fields_deferred, mphv_step_fields_host) the plain path is taken and the
 * call ends with mphv_deferred_status: MPHV_ERR_RANGE if a velocity sweep since the last query had |s| >= 1. */
int mphv_run_host(mphv_ctx *ctx, double *f_host, int nsteps, double dt,
                  double *n_host, double *j_host, double *P_host);

/* One step of a COUPLED run with f resident on the device (the way the paper's framework drives a Vlasov
 * model: the field solver hands over E, B, the Vlasov model hands back its moments):
 * copies E_host, B_host ([3][nz][ny][nx] each, ideally pinned) to library-owned device memory,
 * mphv_set_fields_deferred, mphv_step_moments(dt), copies n, j, P to n_host [ns], j_host [3 ns], P_host [6 ns] and
 * synchronises the stream ONCE, at the end. f stays in the bound device buffer. Requires bind_f. The velocity RANGE
 * check is the deferred one: MPHV_ERR_RANGE is returned after the step has run, and f is then lost (see
 * mphv_set_fields_deferred); the context stays in deferred mode until mphv_set_fields is called. */
int mphv_step_fields_host(mphv_ctx *ctx, const double *E_host, const double *B_host, double dt,
                          double *n_host, double *j_host, double *P_host);

/* Sum of all entries of the bound f (device reduction, deterministic order), written to
 * *sum_dev (device, 1 double). Used for the mass checks of BJ (1e-13 relative). */
int mphv_sum_f(mphv_ctx *ctx, double *sum_dev);

/* The same total for callers that cannot allocate device memory: no context, and no cudaMalloc,
 * cudaFree or allocating library routine anywhere inside. It is meant for a host code whose own memory
 * manager already holds all of HBM (a cudaMalloc from inside a library would fail there), and for a
 * caller inside its time loop, where cudaMalloc / cudaFree would synchronise the device and stall the
 * other streams. (mphv_create, and therefore mphv_sum_f, gets its workspace from cudaMalloc.)
 *
 *   x_dev   [count] fp64, device memory of the CURRENT device, 8-byte aligned, read only
 *   sum_dev 1 double, device memory of the current device: receives sum_i x_dev[i] (0 for count = 0)
 *   stream  a cudaStream_t of the current device (NULL = the default stream); the call enqueues two
 *           kernels on it and returns, *sum_dev is valid once that stream has drained
 *   err     optional host buffer [err_cap] for the text of a failure (this call has no context, so
 *           mphv_last_error does not see it); may be NULL
 *
 * The per-block partial sums that mphv_sum_f keeps in its context's workspace live here in a static
 * __device__ array of MPHV_SUM_NOALLOC_MAX_COUNT / MPHV_SUM_NOALLOC_CHUNK = 16384 doubles (128 KiB),
 * part of the library image: every GPU on which the library is used holds it until the process exits.
 * Block b sums the fixed chunk x[b*CHUNK, (b+1)*CHUNK), so the result depends on (x, count) only, is
 * the same bits on every call, and differs from mphv_sum_f's (another summation order) by rounding:
 * both are Kahan-compensated, |difference| <~ 1e-15 sum|x|.
 *  - count > MPHV_SUM_NOALLOC_MAX_COUNT (2^30 doubles = 8 GiB of f): MPHV_ERR_RANGE, nothing launched.
 *    Sum a larger array in pieces, or use mphv_sum_f.
 *  - The FIRST call on each device looks up the array's device address (cudaGetSymbolAddress, which may
 *    load the library's kernels on that device) and caches it; make that call during set-up, before any
 *    stream capture begins. Later calls only launch.
 *  - All calls on one device share the one array. Nothing in it has to start at zero (each call
 *    overwrites the entries it reads; what a previous call left beyond them is never read), but two
 *    calls that may run on the GPU at the same time -- different streams without an ordering between
 *    them, or several host threads -- race on it and return garbage: order them (same stream, or an
 *    event). Calls on different devices do not interfere.
 *  - Errors: MPHV_ERR_ARG (NULL or misaligned pointer), MPHV_ERR_RANGE (above), MPHV_ERR_ARCH (the
 *    current device is not sm_100), MPHV_ERR_CUDA; outputs untouched on any of them. */
#define MPHV_SUM_NOALLOC_CHUNK 65536
#define MPHV_SUM_NOALLOC_MAX_COUNT ((size_t)1 << 30)
int mphv_sum_noalloc(const double *x_dev, size_t count, double *sum_dev, void *stream,
                     char *err, size_t err_cap);

/* Number of kernel launches enqueued through this context since creation (for the
 * bench's gpu_launches figure). */
uint64_t mphv_launch_count(const mphv_ctx *ctx);

/* Per-kernel device timing. When enabled, every kernel launch of this context is bracketed by
 * two CUDA events on the context's stream; durations accumulate per slot. Enabling (again)
 * clears the records. mphv_get_timing synchronises the stream, then reports slot `slot`
 * (0 <= slot < mphv_timing_slots()): its name (copied into name[name_cap]), the summed device
 * time in ms, the number of launches, and the ALGORITHMIC bytes of one launch (f read once +
 * written once per sweep it performs, f read once per moments pass). */
int mphv_set_timing(mphv_ctx *ctx, int enabled);
int mphv_timing_slots(void);
int mphv_get_timing(mphv_ctx *ctx, int slot, char *name, size_t name_cap, double *total_ms,
                    uint64_t *launches, double *alg_bytes_per_launch);
/* The bytes ONE launch of slot `slot` has to move through HBM whatever it fuses: f read once and written
 * once per PASS over f (16 B/cell for a fused stage of several sweeps, 8 for a moments pass). This is the
 * numerator of the physical HBM roofline fraction; the algorithmic figure above counts every fused sweep. */
int mphv_get_timing_moved(mphv_ctx *ctx, int slot, double *moved_bytes_per_launch);

/* ---- model coupling at a Vlasov / ten-moment border (sec. 4.3; readings R16, R17).
 * mphv_maxwellian: f_out_dev[c][nvel] = the ten-moment Maxwellian ("a multivariate normal distribution",
 * P:L185) of cell c < count: with u = j/n and C_ab = P_ab/n - u_a u_b (moment conventions of
 * mphv_moments: j = int v f, P = int v v f),
 *     M(v) = n (2 pi)^(-D/2) det(C)^(-1/2) exp(-(v-u)^T C^-1 (v-u) / 2)
 * at the velocity cell centres, D = number of active velocity dimensions. n <= 0 or C not positive
 * definite gives M = 0 for that cell. Layouts: n_dev [count], j_dev [3][count], P_dev [6][count]
 * (xx, xy, xz, yy, yz, zz), f_out_dev [count][nvz][nvy][nvx]; all device memory of the caller.
 * mphv_exchange_maxwellian: "exchanging Maxwellians" in the two boundary cells at one end
 * (side 0 = low, 1 = high index) of spatial axis dim of the bound f, in place: for every column,
 *     ghost_i = M[fluid data of boundary cell i] + sigma_i (f_ext - M[moments of f_ext]),
 * f_ext = the last interior cell (third from the end; zero-gradient extension), sigma = 2/3 in the
 * boundary cell next to the interior and 1/3 in the outer one. Fluid data n_fl_dev [2][plane],
 * j_fl_dev [3][2][plane], P_fl_dev [6][2][plane]: layer 0 = lower index along dim, plane = the other two
 * spatial indices in C order. Needs nx[dim] >= 4. Both calls only enqueue. */
int mphv_maxwellian(mphv_ctx *ctx, size_t count, const double *n_dev, const double *j_dev,
                    const double *P_dev, double *f_out_dev);
int mphv_exchange_maxwellian(mphv_ctx *ctx, int dim, int side, const double *n_fl_dev,
                             const double *j_fl_dev, const double *P_fl_dev);

/* Matching the ten moments of the bound f to given ones by exchanging Maxwellians, in every spatial
 * cell, in place ("matched-moments Vlasov solver", "exchanging Maxwellians"; reading R18):
 *     f <- M[n_t, j_t, P_t] + (f - M[moments of f]).
 * n_t_dev [ns], j_t_dev [3][ns], P_t_dev [6][ns] in the layouts of mphv_moments. The time-step order of the
 * paper's Algorithm 1 and its density correction are missing from PAPER.md and not reproduced;
 * positivity of the result is the caller's concern. Only enqueues. */
int mphv_match_moments(mphv_ctx *ctx, const double *n_t_dev, const double *j_t_dev, const double *P_t_dev);

/* Mode of the V stage. MPHV_V_PLAIN (default; BASELINE.json north_star): three plain 1-D sweeps with
 * the Courant numbers a_d dt / dv_d, a = (q/m)(E + v x B) at the cell centres. MPHV_V_BACKSUB: "The
 * velocity space splitting is realized via backsubstitution" (sec. 4.1; reading R15 of
 * DESIGN.md): the three sweeps vx, vy, vz displace every cell FACE to the foot coordinate of the Boris
 * map of the cell (half kick, rotation about B, half kick over dt), each sweep knowing the coordinates
 * the later sweeps have already made final, so that their composition is the exact characteristic foot
 * and no O((q/m)|B| dt) splitting error remains. Same limiter and flux polynomial; closed velocity box;
 * every face needs |s_face| < 1 (MPHV_ERR_RANGE otherwise). Needs all three velocity dimensions
 * active (MPHV_ERR_ARG otherwise). It applies to mphv_sweep_v (call dims 0, 1, 2 in that order with the
 * same dt), mphv_stage_v, mphv_step, mphv_step_moments and mphv_run_host. The face coefficients depend
 * on (fields, dt): the first call with a new dt after mphv_set_fields or mphv_set_vmode runs one small
 * kernel and synchronises the stream once; later calls with the same dt only enqueue. */
enum { MPHV_V_PLAIN = 0, MPHV_V_BACKSUB = 1 };
int mphv_set_vmode(mphv_ctx *ctx, int mode);

/* Tuning knob for experiments and tests. level 0 = one kernel per sweep; 1 = pairwise fused
 * kernels (V_vx+V_vy per velocity plane, V_vz+moments);
 * 2 = the whole V stage (three sweeps and the moments) in one pass over f; 3 = level 2 plus the
 * spatial sweeps S_x and S_y in one pass over f (the default, fastest measured on B200). Levels 1..3 fall back to lower-level kernels for
 * grids their kernels do not cover (nvx, nvy not multiples of 4 resp. 2, fewer than 3 velocity
 * dimensions; nx not a multiple of 4 or above 256, nvel not a multiple of 8, |s| >= 1 on a periodic axis).
 * Results agree up to fp64 rounding at every level. */
int mphv_set_fusion(mphv_ctx *ctx, int level);

/* For tests and experiments: the newest generation of the whole-V-stage kernel (fusion levels 2 and 3) this context may
 * use. 4 (the default) = vstage3_kernel / vstage3_bs_kernel where the grid allows, else the older ones; 3 = at most
 * vstage2_kernel (backsubstitution mode: vstage_bs_kernel); 2 = vstage_kernel / vstage_bs_kernel. Same results up to
 * fp64 rounding. The library reads no environment variable. Errors: ARG (generation outside 2..4). */
int mphv_set_vstage_generation(mphv_ctx *ctx, int generation);

/* mphv_set_fields without the host round trip, for coupled runs that change the fields every step (P:L109,
 * P:L141): the max |a_d| reduction is enqueued as in mphv_set_fields but its result stays on the device, and the
 * MPHV_ERR_RANGE check of every later velocity sweep / V stage / step is made ON THE DEVICE when that call is
 * enqueued (one 1-thread kernel in front of it) and raises a sticky device flag instead of failing the call.
 * mphv_deferred_status synchronises the stream and returns MPHV_ERR_RANGE if the flag was raised since the last
 * query (and clears it), else MPHV_OK. A sweep enqueued with |s| >= 1 computes a wrong remap of f (no out-of-bounds
 * access): after MPHV_ERR_RANGE from mphv_deferred_status f must be considered lost. mphv_set_fields switches back
 * to the immediate check. E_dev, B_dev are borrowed as in mphv_set_fields; if they are changed in place, one of the
 * two set_fields calls MUST be made again before the next velocity sweep. */
int mphv_set_fields_deferred(mphv_ctx *ctx, const double *E_dev, const double *B_dev);
int mphv_deferred_status(mphv_ctx *ctx);

/* ---- closing the loop: Maxwell's equations fed by the species' currents, and the coupled step.
 * eq. (9): curl E = -dB/dt, curl B = mu0 j + mu0 eps0 dE/dt, j = sum_s q_s n_s u_s; "solved via the finite
 * difference time domain (FDTD) method", div B = 0 by construction; "The Maxwell solver itself uses Strang
 * splitting between E and B". Readings R19..R22 of DESIGN.md:
 *   R19  Yee lattice on the Vlasov cells, integer indices = cell centres: array element [k][j][i] of
 *        Ex at (i+1/2, j, k), Ey at (i, j+1/2, k), Ez at (i, j, k+1/2)   (faces normal to the component),
 *        Bx at (i, j+1/2, k+1/2), By at (i+1/2, j, k+1/2), Bz at (i+1/2, j+1/2, k)   (edges along the component);
 *        no derivative and no staggering along an inactive axis.
 *   R20  E_d at a centre = mean of its 2 faces along d; B_d at a centre = mean of its 4 edges in the plane normal
 *        to d; the current on the face of E_d = mean of the two adjacent cell-centred values.
 *   R21  periodic axis = index wrap, bounded axis (MPHV_BC_OUTFLOW) = zero-gradient ghost value.
 * All field arrays: device, [3][nz][ny][nx], component-major, owned by the caller. Calls only enqueue. */
typedef struct mphv_maxwell mphv_maxwell;

typedef struct {
    int32_t nx[3];                     /* spatial extents (as mphv_grid.nx)                                */
    int32_t bc[3];                     /* MPHV_BC_PERIODIC or MPHV_BC_OUTFLOW (zero-gradient ghosts, R21)   */
    double dx[3];                      /* cell widths; ignored along inactive axes                          */
    double c2;                         /* c^2 = 1 / (mu0 eps0)                                              */
    double inv_eps0;                   /* 1 / eps0                                                          */
} mphv_field_grid;

mphv_maxwell *mphv_maxwell_create(const mphv_field_grid *grid);     /* NULL on error: mphv_last_error(NULL)  */
int mphv_maxwell_destroy(mphv_maxwell *m);
int mphv_maxwell_set_stream(mphv_maxwell *m, void *cuda_stream);
/* The staggered fields (R19) the later calls update in place. */
int mphv_maxwell_bind(mphv_maxwell *m, double *E_dev, double *B_dev);
/* B <- B - dt curl E (Faraday). */
int mphv_maxwell_faraday(mphv_maxwell *m, double dt);
/* E <- E + dt (c^2 curl B - J / eps0) (Ampere-Maxwell); J_dev = cell-centred charge current or NULL (vacuum). */
int mphv_maxwell_ampere(mphv_maxwell *m, const double *J_dev, double dt);
/* One Maxwell step with J frozen: B(dt/2), E(dt; J), B(dt/2). One launch on grids up to 65536 cells. */
int mphv_maxwell_step(mphv_maxwell *m, const double *J_dev, double dt);
/* Fields at the cell centres (R20): what mphv_set_fields takes (R8). */
int mphv_maxwell_centre(mphv_maxwell *m, double *Ec_dev, double *Bc_dev);
/* Charge current J = sum_s q_s j_s (eq. (9)); q_host[nspecies], j_dev_ptrs = HOST array of nspecies device
 * pointers to the species' number fluxes j = int v f d3v ([3][ns] each, as mphv_moments writes them); nspecies <= 4. */
int mphv_maxwell_current(mphv_maxwell *m, int nspecies, const double *q_host, const double *const *j_dev_ptrs,
                         double *J_dev);
const char *mphv_maxwell_last_error(const mphv_maxwell *m);

/* A set of kinetic species coupled through Maxwell's equations: the paper's Scheme {Vlasov e, Vlasov i, Maxwell}
 * (P:L109). The species contexts (each with f bound, created on the same device with the spatial grid of
 * the field solver) and the field solver (fields bound) belong to the caller and must outlive the plasma object;
 * q_host[s] is the charge that weights species s in the current (its q/m lives in its context).
 * mphv_plasma_step: nsteps steps of the coupled scheme R22 (leapfrog-like Strang between plasma and fields, P:L135,
 * P:L145), per step
 *        J = sum_s q_s j_s[f_s];  Maxwell(dt/2; J);  E_c, B_c = centred fields;
 *        every species: f_s <- mphv_step(dt) with E_c, B_c frozen, moments of the new f_s;
 *        J' = sum_s q_s j_s[f_s];  Maxwell(dt/2; J').
 * By default everything is enqueued on the field solver's stream (mphv_maxwell_set_stream). With
 * mphv_plasma_set_concurrent(p, 1) every species runs on a CUDA stream of its own, ordered against the field update
 * by events. Measured on B200 (profiles/r02b_two_species.md) that gains nothing (6.26 - 6.51 vs 6.32 ms per step for
 * ions 40^3 + electrons 36^3 on 128x64): the spatial-sweep kernel and the V-stage kernel each fill an SM's register file,
 * so two species never share an SM, and two spatial sweeps at once split the L2 their row rings live in. Either way
 * the host never waits inside the loop (velocity RANGE checks are deferred, see mphv_set_fields_deferred). The call
 * returns after the last step has been enqueued (the species' streams joined on the field solver's stream);
 * mphv_plasma_sync waits for it and reports a deferred RANGE error. The species contexts are left on the streams
 * the last call used.
 * The first call computes the moments of the initial f_s itself; later calls reuse the moments the previous call
 * ended with for their opening Maxwell half step. If a species' f is changed between two calls by anything but
 * mphv_plasma_step (mphv_exchange_maxwellian or mphv_match_moments at a model border, a re-bind, a direct sweep),
 * call mphv_plasma_invalidate_moments first: the next mphv_plasma_step then recomputes every species' moments from
 * the f it finds (one moments pass per species), instead of using the stale current.
 * mphv_plasma_destroy: while a plasma object lives, its species read the cell-centred fields from buffers the
 * plasma owns (bound inside mphv_plasma_step). Destroying it un-binds those fields from every species that still
 * uses them and ends their deferred mode: such a context must get fields again (mphv_set_fields) before its next
 * sweep, step or mphv_run_host, which otherwise return MPHV_ERR_STATE. Fields the caller bound since are kept.
 * mphv_plasma_moments: device pointers to the latest moments of species s (n [ns], j [3][ns], P [6][ns], owned by
 * the plasma object, valid after mphv_plasma_sync). */
typedef struct mphv_plasma mphv_plasma;
mphv_plasma *mphv_plasma_create(mphv_maxwell *m, int nspecies, mphv_ctx *const *species, const double *q_host);
int mphv_plasma_destroy(mphv_plasma *p);
int mphv_plasma_set_concurrent(mphv_plasma *p, int concurrent);
int mphv_plasma_step(mphv_plasma *p, double dt, int nsteps);
int mphv_plasma_sync(mphv_plasma *p);
int mphv_plasma_invalidate_moments(mphv_plasma *p);
int mphv_plasma_moments(mphv_plasma *p, int s, double **n_dev, double **j_dev, double **P_dev);
/* centred fields of the last step (device, [3][ns] each, owned by the plasma object) */
int mphv_plasma_centred_fields(mphv_plasma *p, double **Ec_dev, double **Bc_dev);
const char *mphv_plasma_last_error(const mphv_plasma *p);

const char *mphv_strerror(int code);
/* Last error text of this context, or of the last failed mphv_create when ctx is NULL.
 * The returned pointer is owned by the library and valid until the next failing call. */
const char *mphv_last_error(const mphv_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* MPHV_H */
