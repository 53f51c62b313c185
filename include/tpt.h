/*
 * tpt.h — C ABI of the B200 (sm_100a) tensor-product–Thomas Poisson/Helmholtz solver.
 *
 * The library solves, in FP64 on one GPU,
 *      T phi = f                  (Poisson,   helmholtz_alpha == 0)      PAPER.md:139, Eq. 7
 *      (I - alpha T) u = f        (Helmholtz, helmholtz_alpha  > 0)      PAPER.md:68,  Eq. 2b
 * with T = Tx (x) Iy (x) Iz + Ix (x) Ty (x) Iz + Ix (x) Iy (x) Tz the second-order finite-difference
 * Laplacian of Eq. 3–4 on a staggered, non-uniform Cartesian grid, by the paper's
 * tensor-product–Thomas procedure (steps 1.1–1.3 at plan time, 2.1–2.5 per solve).
 *
 * Conventions (all entry points):
 *   - plain C, no torch types; every function returns a tpt status code (0 = TPT_OK) and never
 *     throws or aborts across the ABI.  tpt_strerror() names a code.
 *   - fields are FP64 arrays of nx*ny*nz elements, element (i,j,k) at  i + nx*(j + ny*k)
 *     (x contiguous, z slowest — the paper's "leading dimension N_x").
 *   - "HOST" / "DEVICE" below says where a pointer must live.  Device pointers must be 16-byte
 *     aligned (any cudaMalloc / torch allocation is).
 *   - the CUDA device is the one current at tpt_plan_create; the same device must be current in
 *     later calls on that plan (TPT_EINVAL otherwise).  There is no CPU fallback: without a usable CUDA device
 *     tpt_plan_create fails with TPT_ECUDA.
 */
#ifndef TPT_H
#define TPT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tpt_plan tpt_plan; /* opaque */

/* Homogeneous, the same at both ends of a direction.  PERIODIC (PAPER.md:102 "cyclic corners", :211 dense cyclic
 * operator; the paper's benchmark BCs are periodic x, Neumann y and z): x and y, the diagonalised
 * directions, take it through their eigenbasis; a periodic z makes the sweep a cyclic tridiagonal solve — the
 * ordinary sweep on a corner-modified matrix followed by a Sherman-Morrison correction whose column vectors are swept
 * once at plan time (one extra field of device memory; natural layout; >= 3 cells).  Not available with periodic z:
 * the sharded solve (TPT_EINVAL) and the one-launch small-grid path (the separate kernels run instead). */
enum { TPT_BC_NEUMANN = 0, TPT_BC_DIRICHLET = 1, TPT_BC_PERIODIC = 2 };

/* Implicitly treated directions L_I of the Helmholtz problem, Eq. 2b: bit 0 = x, 1 = y, 2 = z. */
enum { TPT_DIRS_Z = 4, TPT_DIRS_YZ = 6, TPT_DIRS_XYZ = 7 };

enum {
    TPT_OK = 0,
    TPT_EINVAL = -1,   /* bad argument (sizes, faces, bc, alpha, null/misaligned pointer) */
    TPT_ENOMEM = -2,   /* host or device allocation failed */
    TPT_ECUDA = -3,    /* CUDA runtime error (no device, launch failure, ...) */
    TPT_ENUMERIC = -4, /* plan-time eigen-solver did not reach its accuracy rule */
    TPT_ELIMIT = -5    /* grid beyond the fixed capacity of tpt_solve_static_scratch (TPT_STATIC_SCRATCH_POINTS) */
};

/* Kernel slots, in execution order (used by tpt_plan_get_kernel_times / tpt_stage). */
enum {
    TPT_K_FWD_X = 0,  /* step 2.1, Eq. 10a */
    TPT_K_FWD_Y = 1,  /* step 2.2, Eq. 10b */
    TPT_K_THOMAS = 2, /* step 2.3, PAPER.md:183 (+ null-mode gauge) */
    TPT_K_INV_Y = 3,  /* step 2.4, Eq. 12a */
    TPT_K_INV_X = 4,  /* step 2.5, Eq. 12b */
    TPT_K_COUNT = 5
};

/*
 * tpt_plan_create — initialisation, steps 1.1–1.3.  Untimed, synchronous.
 *   For x and y: build T_d (Eq. 3–4 with boundary rows), symmetrise T~ = D^{1/2} T D^{-1/2} (Eq. 5),
 *   eigendecompose T~ = Q~ Lambda Q~^T on the host (implicit-shift QL + guarded factored-form
 *   refinement), form the pre-scaled transform matrices Q^{-1} = Q~^T D^{1/2}, Q = D^{-1/2} Q~
 *   (Eq. 6) and upload them; for z: the tridiagonal coefficients of T_z.
 *   nx, ny, nz >= 2 cells.  xf, yf, zf: HOST, face coordinates, lengths nx+1, ny+1, nz+1, finite and
 *   strictly increasing.  bc: HOST, {bc_x, bc_y, bc_z}.  helmholtz_alpha: 0 selects Poisson, > 0
 *   Helmholtz; negative / non-finite is TPT_EINVAL.
 *   No Dirichlet direction (every bc Neumann or periodic) with alpha == 0 gives a SINGULAR plan: tpt_solve then returns the solution
 *   with zero cell-volume-weighted mean; following PAPER.md:219 the last z-equation of mode (0,0)
 *   is replaced by "unknown = 0", so an incompatible rhs is not projected.
 *   Ownership: the plan owns its device matrices, coefficient vectors and ONE field-sized
 *   workspace (nx*ny*nz doubles).  *plan_out is untouched on failure.
 */
int tpt_plan_create(tpt_plan **plan_out, int nx, int ny, int nz,
                    const double *xf, const double *yf, const double *zf,
                    const int bc[3], double helmholtz_alpha);

/*
 * tpt_plan_create_dirs — the same with a choice of the implicitly treated directions L_I of Eq. 2b
 * (PAPER.md:59 "four choices for L_I", :209): the plan then solves (I - alpha L_I) u = f with
 *   TPT_DIRS_XYZ  L_I = L                 all five steps (what tpt_plan_create builds),
 *   TPT_DIRS_YZ   L_I = L_y + L_z         "the yz option omits the x transforms": steps 2.2, 2.3, 2.4,
 *   TPT_DIRS_Z    L_I = L_z               "the z option performs only the tridiagonal solve": step 2.3.
 * The partial choices need helmholtz_alpha > 0 (the pressure equation, Eq. 2c, always carries the full
 * Laplacian): TPT_EINVAL otherwise.  No eigendecomposition is made for a direction that is not diagonalised.
 */
int tpt_plan_create_dirs(tpt_plan **plan_out, int nx, int ny, int nz,
                         const double *xf, const double *yf, const double *zf,
                         const int bc[3], double helmholtz_alpha, int implicit_dirs);

/*
 * tpt_plan_create_ex — the same with the transform type chosen per diagonalised direction ("the transform
 * type is selected independently in each diagonalized direction.  A uniform direction may use either FFT-based
 * transforms or numerical eigenbasis transforms evaluated with GEMM, whereas a non-uniform direction uses the latter";
 * "for a uniform direction, the analytical eigenvalues are stored"; O(N log N) per line).
 *   transform: HOST, {transform_x, transform_y}.  TPT_TRANSFORM_FFT needs a direction that is diagonalised, has
 *   2^m cells with 16 <= n <= 2048 and is uniform (every width within rounding of (x_n - x_0)/n; the plan then solves
 *   the exactly uniform operator of that spacing); for y also nx % 16 == 0.  TPT_EINVAL otherwise.  All three boundary
 *   types are taken: cosine transforms (Neumann), sine transforms (Dirichlet), the real DFT (periodic), each as one
 *   complex FFT per pair of lines in shared memory.  tpt_plan_get_eigen returns the analytical eigenvalues of such a
 *   direction; its basis is not stored (qtilde_host must be NULL).
 * Combinations: GEMM/GEMM = the paper's GG variant, FFT/GEMM = FG, GEMM/FFT = GF, FFT/FFT = FF.
 */
enum { TPT_TRANSFORM_GEMM = 0, TPT_TRANSFORM_FFT = 1 };
int tpt_plan_create_ex(tpt_plan **plan_out, int nx, int ny, int nz,
                       const double *xf, const double *yf, const double *zf,
                       const int bc[3], double helmholtz_alpha, int implicit_dirs, const int transform[2]);

/*
 * tpt_solve — steps 2.1–2.5: five kernels (+ one tiny gauge kernel on a singular
 * plan) enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy default stream).
 * Asynchronous: returns after enqueueing; no host synchronisation, no allocation.
 *   rhs_dev: DEVICE, nx*ny*nz doubles, read only (unless rhs_dev == out_dev, which is allowed).
 *   out_dev: DEVICE, nx*ny*nz doubles, overwritten with phi (or u).
 * A plan is not re-entrant (one workspace): order concurrent solves on one stream or use two plans.
 */
int tpt_solve(tpt_plan *plan, const double *rhs_dev, double *out_dev, void *cuda_stream);

/*
 * tpt_solve_static_scratch — the same solve (steps 2.1–2.5 + the null-mode gauge) for callers
 * that may not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  It is
 * the one-launch cluster kernel of the small-grid path (TPT_PATH_FUSED_SMALL) with its mode-space scratch — the field
 * between the two changes of ownership — in a file-scope static device array instead of the plan's workspace.  Nothing
 * on this call path calls cudaMalloc, cudaFree, or any allocating routine (no events, no streams); the plan, created
 * earlier, is only read.
 *   rhs_dev / out_dev / cuda_stream: as tpt_solve (DEVICE, nx*ny*nz doubles each, 16-byte aligned, rhs_dev == out_dev
 *   allowed); asynchronous.
 * Limits: nx*ny*nz <= TPT_STATIC_SCRATCH_POINTS (16384 points: 128 KiB, held by every GPU that loads the library until
 *   the process exits) — TPT_ELIMIT beyond it, nothing launched (also when the two transform matrices of a very flat
 *   grid, nx*nx + ny*ny doubles, do not fit in shared memory beside the field).  The plan must diagonalise x and/or y with GEMM
 *   transforms and have a non-periodic z (what that kernel computes): TPT_EINVAL otherwise.  The debug switches
 *   tpt_plan_set_fused_small / _gemm_variant / _thomas_variant do not apply; profiling records nothing for it.
 * Sharing: ALL calls on one GPU — any plan, any stream, any host thread — use the same array.  Calls that may overlap
 *   on the GPU race on it: order them on one stream (or with events).  The array keeps the last call's contents; no
 *   call depends on them (every element read is written earlier in the same launch), so there is nothing to clear.
 * First call on a device: resolves the array's device address (cudaGetSymbolAddress) and sets the kernel's dynamic
 *   shared-memory attribute, once, thread-safe; neither allocates, but both are set-up calls — a caller that captures
 *   a CUDA graph makes one call before the capture starts.
 * Result: the same kernel and arithmetic as tpt_solve on a plan that takes the small-grid path (bitwise equal to it).
 */
#define TPT_STATIC_SCRATCH_POINTS 16384
int tpt_solve_static_scratch(tpt_plan *plan, const double *rhs_dev, double *out_dev, void *cuda_stream);

/*
 * tpt_solve_batch — nrhs right-hand sides of the same plan in one call ("the resulting eigenvalues and forward/inverse
 * transform matrices are reused for every right-hand side"; the three velocity components of Eq. 2b):
 * fields stacked densely, field r at rhs_dev + r*nx*ny*nz.  Each transform runs as ONE launch over all fields of a
 * chunk (the stack is just a longer z axis for steps 2.1, 2.2, 2.4, 2.5); the sweep runs once per field.  A chunk is
 * as many fields as the workspace holds: 1 unless tpt_plan_reserve_batch grew it.  Same rules as tpt_solve
 * (asynchronous, no allocation, rhs_dev == out_dev allowed).
 * tpt_plan_reserve_batch — grows the plan workspace to nrhs fields (synchronises the device; never shrinks).
 */
int tpt_solve_batch(tpt_plan *plan, const double *rhs_dev, double *out_dev, int nrhs, void *cuda_stream);
int tpt_plan_reserve_batch(tpt_plan *plan, int nrhs);

/*
 * tpt_solve_host — the same solve for HOST buffers, synchronous: returns after the result is in out_host.
 * The transforms act plane by plane in z (Eq. 10, 12 at PAPER.md:154–169), so the field crosses the bus in up to
 * 16 z-slabs: slab s is transformed (steps 2.1, 2.2) while slab s+1 is still being copied in, the sweep (2.3) runs
 * once every slab has arrived, and slab s is copied out while slab s+1 is transformed back (2.4, 2.5).  The copies
 * run on two plan-owned streams ordered after earlier work on `cuda_stream`; the kernels run on `cuda_stream`.
 * Uses a plan-owned staging field allocated on first use.  rhs_host / out_host: HOST, nx*ny*nz doubles each
 * (pinned memory makes the copies asynchronous and fast; pageable memory works).  May alias.
 */
int tpt_solve_host(tpt_plan *plan, const double *rhs_host, double *out_host, void *cuda_stream);

/*
 * tpt_solve_host_async / tpt_plan_wait — the same solve (steps 2.1–2.5 of PAPER.md:181–185 between the two copies),
 * split into "enqueue" and "wait": tpt_solve_host_async returns as soon as the copies and kernels are enqueued
 * (truly asynchronous only for pinned HOST buffers, which must stay valid and untouched until tpt_plan_wait returns);
 * tpt_plan_wait blocks until the plan's most recent host solve has delivered its result.  A second call on the same
 * plan queues behind the first.  Two plans on two streams overlap one solve's device-to-host copy with the next
 * one's host-to-device copy (the bus is full duplex): that is how bench.py measures its end-to-end throughput.
 */
int tpt_solve_host_async(tpt_plan *plan, const double *rhs_host, double *out_host, void *cuda_stream);
int tpt_plan_wait(tpt_plan *plan);

/*
 * Pressure projection of the fractional-step method on the staggered grid, Eq. 2c–2e (staggered
 * arrangement PAPER.md:57; "applying the pressure-projection step to a white-noise velocity field produces a
 * discretely divergence-free field to machine precision").
 *   Velocity components live on cell faces: u_dev (nz, ny, nx+1) on x-faces, v_dev (nz, ny+1, nx) on y-faces,
 *   w_dev (nz+1, ny, nx) on z-faces, each dense with x contiguous; face f of a direction lies between cells f-1 and f.
 *   Divergence D (cells) and gradient G (faces) are the second-order differences whose product D G is the Laplacian
 *   of Eq. 3 with the plan's boundary rows.  Boundary faces follow the pressure BC of their direction: NEUMANN = wall
 *   (G Phi = 0 there; the face keeps its prescribed normal velocity), DIRICHLET = ghost value -Phi one cell width
 *   away, PERIODIC = faces 0 and n are one face (entry n is ignored on input and written as a copy of entry 0).
 *
 * tpt_divergence      out = scale * D(u, v, w)                    (right-hand side of Eq. 2c with scale = 1/(gamma_k dt))
 * tpt_gradient_correct u -= c G phi  (Eq. 2d);  if p_dev != NULL:  p += phi - alpha_p L_I phi  (Eq. 2e), L_I the 1-D
 *                     Laplacians of the directions in implicit_dirs (TPT_DIRS_*; alpha_p = gamma_k nu dt / 2;
 *                     alpha_p == 0 is the fully explicit choice L_I = 0), evaluated in flux form.
 * tpt_project         Eq. 2c, 2d, 2e in order: phi_dev = L^{-1} (D u / gamma_dt) through tpt_solve, then the correction.
 *                     The plan must be a Poisson plan of the full operator (helmholtz_alpha == 0, TPT_DIRS_XYZ):
 *                     TPT_EINVAL otherwise.  On a singular plan the velocity field must be compatible (zero net flux
 *                     through the walls), as in the paper's solver; Phi then has zero volume-weighted mean.
 * All DEVICE pointers, no aliasing between arguments; phi_dev / out_dev: nx*ny*nz doubles.  Alignment: 8 bytes is
 * enough for tpt_divergence and tpt_gradient_correct (a view into a larger buffer is fine: arrays that are not 16-byte
 * aligned take the one-cell-per-thread kernels instead of the two-cell ones); tpt_project needs a 16-byte aligned
 * phi_dev because it runs tpt_solve on it.  Anything less is TPT_EINVAL, never a fault.
 * Asynchronous on cuda_stream, no allocation, no host synchronisation.  gamma_dt, c > 0; alpha_p >= 0.
 */
int tpt_divergence(tpt_plan *plan, const double *u_dev, const double *v_dev, const double *w_dev, double scale,
                   double *out_dev, void *cuda_stream);
int tpt_gradient_correct(tpt_plan *plan, const double *phi_dev, double c, double *u_dev, double *v_dev, double *w_dev,
                         double *p_dev, double alpha_p, int implicit_dirs, void *cuda_stream);
int tpt_project(tpt_plan *plan, double *u_dev, double *v_dev, double *w_dev, double gamma_dt, double *phi_dev,
                double *p_dev, double alpha_p, int implicit_dirs, void *cuda_stream);

/* tpt_plan_destroy — frees everything the plan owns (synchronises the device). NULL is a no-op. */
int tpt_plan_destroy(tpt_plan *plan);

/* ---- the solve sharded across the GPUs of one NVLink domain ------------------------------------------
 *
 * PAPER.md:197-207 (pencil layouts, collective transposes between them), Algorithm 1 steps 2, 4, 6, 8.
 * The paper moves the field between x-, y- and z-aligned pencils with four all-to-alls per solve.  Here rank r of
 * nranks (<= 8, one process per GPU) owns
 *   - the z-SLAB [k0, k1) of the physical field: rhs and solution are nx*ny*(k1-k0) doubles, element (i, j, k - k0) at
 *     i + nx*(j + ny*(k - k0)).  Steps 2.1, 2.2, 2.4, 2.5 act plane by plane, so both transforms are local to a slab;
 *   - the y-MODE rows [m0, m1) (all kx, all z) of the mode-space field, on which it runs step 2.3.
 * The two remaining exchanges are the STORES of kernels that touch the data anyway: the forward-y GEMM's epilogue writes
 * each mode row into its owner's memory, the z sweep's TMA store writes each z-range of a solved tile into its slab
 * owner's memory — peer-mapped pointers over NVLink, no pack/unpack kernel, no collective.  Per solve a rank sends
 * nvlink_bytes_per_solve bytes (2 * 8 * nx * (m1-m0) * (nz - (k1-k0))), two device-side flag barriers order the phases.
 *
 * Shapes: nx a multiple of 128; ny a multiple of 128 (GEMM y transform) or a power of two >= 16 (fast y transform,
 * tpt_shard_create_ex); 2*nranks <= nz <= 1056; ny/16 >= nranks; x and y by GEMM or fast transform — all four variants
 * GG / FG / GF / FF of PAPER.md:294, the y transform (GEMM epilogue or the fast transform's own stores) carrying exchange 1;
 * bc and alpha as tpt_plan_create (periodic z: TPT_EINVAL); anything else TPT_EINVAL.  Slab boundaries are even numbers.
 *
 * tpt_shard_layout      HOST only, needs no device: the split every rank computes identically.
 * tpt_shard_create      plan-time setup of rank `rank` on the current device (full-grid eigenproblems: every rank solves
 *                       the same ones — they are tiny beside a solve and avoid a broadcast) + one "symmetric" allocation
 *                       of sym_bytes: [mode buffer | slab buffer | signal pad], same offsets on every rank.
 * tpt_shard_sym         that allocation (DEVICE pointer) and its size.
 * tpt_shard_set_peers   sym_dev[r] = rank r's allocation as addressable from THIS device (HOST array of nranks DEVICE
 *                       pointers): same-process peers ("virtual ranks" on one device, or cudaDeviceEnablePeerAccess), or
 *                       pointers the caller mapped itself.  sym_dev[rank] must be the shard's own.
 * tpt_shard_ipc_export  writes the TPT_IPC_HANDLE_BYTES-byte CUDA IPC handle of the allocation to handle_out (HOST);
 * tpt_shard_ipc_import  takes the nranks handles (HOST, rank-major, own entry ignored) all-gathered by the caller over
 *                       its own control plane (torch.distributed) and maps the peers; closes them at destroy.
 * tpt_solve_sharded     the whole solve of this rank's slab: rhs_slab_dev -> out_slab_dev (DEVICE, 16-byte aligned, may
 *                       alias), asynchronous on cuda_stream.  EVERY rank must call it the same number of times; the
 *                       barrier kernels spin until all ranks arrive (so all ranks' kernels must be able to run
 *                       concurrently: one GPU per rank).
 * tpt_shard_solve_phase one phase without any waiting kernel (0: steps 2.1-2.2 + exchange 1; 1: step 2.3 + exchange 2;
 *                       2: steps 2.4-2.5), for callers that order the phases themselves — run phase p of every rank, then
 *                       phase p+1 (virtual ranks sharing one device and stream, the tests' setting).  Unused slab
 *                       arguments may be NULL.
 * tpt_shard_barrier     one flag barrier on cuda_stream (exposed for tests and for callers composing their own phases).
 * tpt_shard_barrier_all  the flag barrier of ALL n = nranks virtual ranks of one device (shards[r] = rank r, peers set to one
 *                       another's allocations) as ONE cooperative launch, block r acting as rank r — kernels that wait on
 *                       one another must not be separate launches on one GPU.  HOST array of handles.  Test / one-GPU use.
 * tpt_shard_launches    kernels the last solve / phase call launched.
 * tpt_shard_destroy     synchronises, unmaps peers, frees.  Call it on every rank only after all ranks' solves are done.
 */
#define TPT_IPC_HANDLE_BYTES 64
typedef struct tpt_shard tpt_shard; /* opaque */
typedef struct tpt_shard_layout_t {
    int rank, nranks;
    int k0, k1;                     /* owned z-planes */
    int m0, m1;                     /* owned y-mode rows */
    size_t mode_bytes, slab_bytes;  /* the two parts of the symmetric allocation (sized for the largest rank) */
    size_t sym_bytes;
    size_t slab_points;             /* nx * ny * (k1 - k0) */
    size_t nvlink_bytes_per_solve;  /* bytes this rank writes into OTHER ranks' memory per solve (both exchanges) */
} tpt_shard_layout_t;
int tpt_shard_layout(int nranks, int rank, int nx, int ny, int nz, tpt_shard_layout_t *out);
int tpt_shard_create(tpt_shard **shard_out, int rank, int nranks, int nx, int ny, int nz, const double *xf, const double *yf,
                     const double *zf, const int bc[3], double helmholtz_alpha, int transform_x);
int tpt_shard_create_ex(tpt_shard **shard_out, int rank, int nranks, int nx, int ny, int nz, const double *xf, const double *yf,
                        const double *zf, const int bc[3], double helmholtz_alpha, const int transform_xy[2]);
int tpt_shard_get_layout(const tpt_shard *shard, tpt_shard_layout_t *out);
int tpt_shard_sym(const tpt_shard *shard, void **sym_dev_out, size_t *bytes_out);
int tpt_shard_set_peers(tpt_shard *shard, void *const *sym_dev);
int tpt_shard_ipc_export(const tpt_shard *shard, void *handle_out);
int tpt_shard_ipc_import(tpt_shard *shard, const void *handles);
int tpt_solve_sharded(tpt_shard *shard, const double *rhs_slab_dev, double *out_slab_dev, void *cuda_stream);
int tpt_shard_solve_phase(tpt_shard *shard, int phase, const double *rhs_slab_dev, double *out_slab_dev, void *cuda_stream);
int tpt_shard_barrier(tpt_shard *shard, void *cuda_stream);
int tpt_shard_barrier_all(tpt_shard *const *shards, int n, void *cuda_stream);
int tpt_shard_launches(const tpt_shard *shard);
int tpt_shard_destroy(tpt_shard *shard);

/* ---- inspection / test entry points ------------------------------------------------------------ */

/* Eigen-decomposition of direction dir (0 = x, 1 = y) as used by the plan: lambda_host[n]
 * (descending, mode 0 smoothest) and qtilde_host[n*n] row-major, qtilde[i*n + m] = component i of
 * mode m of the orthogonal Q~ (Eq. 5).  Either output may be NULL.  HOST pointers. */
int tpt_plan_get_eigen(const tpt_plan *plan, int dir, double *lambda_host, double *qtilde_host);

/* The plan-time eigen-solver alone, on the HOST (no device needed): steps 1.1-1.2 of PAPER.md:175-176 for one direction —
 * operator of Eq. 3-4 from the n+1 faces, symmetrisation (Eq. 5), base solver, two guarded factored-form refinement
 * steps (A9) — with the output conventions of tpt_plan_get_eigen.  base_kind 0 = the plan's implicit-QL base
 * solver; 1 = a deliberately crude one (normwise deflation, 64x looser): the accuracy rule says the refinement must
 * absorb the difference (SURVEY 8(c.5) cross-solver check).  tpt_debug_set_eigen_base selects the base solver of every
 * plan created afterwards in this process (test only; 0 restores the default).  HOST pointers; either output may be NULL. */
int tpt_host_eigen(int n, const double *faces_host, int bc, int base_kind, double *lambda_host, double *qtilde_host);
int tpt_debug_set_eigen_base(int base_kind);

/* Launch geometry of the on-chip z sweep (step 2.3) for columns of nz rows, on the HOST (no device needed;
 * test only): blocked != 0: the tile-blocked mode-space layout (or a launch that asks for its partition), sharded != 0:
 * the sharded store (needs blocked).  out12 (HOST, 12 ints) = { rows per segment M, columns per tile, thread limit, CTAs per
 * SM, coefficient table in shared memory (0/1), segments S, TMA boxes per tile, rows per box, rows per tile buffer, ring
 * slots, threads per CTA, dynamic shared memory bytes }.  TPT_EINVAL: nz outside 2..1056, no shape, or a null pointer. */
int tpt_debug_sweep_geometry(int nz, int blocked, int sharded, int *out12);

/* 1 if the plan is singular (all-Neumann Poisson), 0 if not, < 0 on error. */
int tpt_plan_is_singular(const tpt_plan *plan);

/* Bytes of device memory owned by the plan (matrices + vectors + workspace [+ staging]). */
int tpt_plan_device_bytes(const tpt_plan *plan, size_t *bytes_out);

/* Run ONE kernel slot (TPT_K_*) of the pipeline: in_dev -> out_dev (the Thomas slot works in place on
 * out_dev after copying in_dev to it if they differ; it uses the plan workspace as scratch).
 * For stage-by-stage comparison with the oracle.  DEVICE pointers, asynchronous on cuda_stream. */
int tpt_stage(tpt_plan *plan, int slot, const double *in_dev, double *out_dev, void *cuda_stream);

/* Per-kernel timing: while enabled, every tpt_solve brackets each kernel slot with CUDA events on the
 * launching stream (no host synchronisation is added to the solve).  tpt_plan_get_kernel_times
 * synchronises on the last profiled solve, returns the MEAN duration of each slot in milliseconds
 * over the profiled solves since the previous read-out (ms_host[TPT_K_COUNT], HOST), the total
 * number of kernel launches those solves made and how many solves they were, then resets the
 * accumulation.  At most 4096 solves may accumulate between read-outs (TPT_EINVAL beyond). */
int tpt_plan_set_profiling(tpt_plan *plan, int enabled);
int tpt_plan_get_kernel_times(tpt_plan *plan, float *ms_host, int *launches_out, int *solves_out);

/* Select the GEMM kernel for the transforms: 2 = persistent warp-specialised DMMA kernel fed by TMA through an
 * mbarrier ring (default; any grid with even nx and ny — "non-uniform grids in any direction", any N_x, N_y, PAPER.md:187:
 * edge tiles through TMA's out-of-bounds zero fill), 1 = cp.async-pipelined DMMA kernel (M, N multiples of 64),
 * 0 = generic FP64-FMA tile kernel (any shape, odd sizes included).  A variant falls back to the next lower one
 * for shapes it does not take.  For A/B measurement and tests; all are this library's own sm_100a kernels. */
int tpt_plan_set_gemm_variant(tpt_plan *plan, int variant);

/* Which kernel tpt_solve runs in each slot of this plan with its current variant settings (one code
 * per step 2.1-2.5): paths_out[TPT_K_COUNT], HOST.  For tests and the bench record — e.g. that a 1000 x 200 grid really
 * runs on the tensor-path GEMM. */
enum {
    TPT_PATH_NONE = 0,            /* slot inactive (direction not diagonalised, tpt_plan_create_dirs) */
    TPT_PATH_GEMM_GENERIC = 1,    /* DFMA tile kernel */
    TPT_PATH_GEMM_CPASYNC = 2,    /* cp.async-pipelined DMMA kernel */
    TPT_PATH_GEMM_TMA = 3,        /* persistent TMA / mbarrier DMMA kernel */
    TPT_PATH_FFT = 4,             /* fast transform of a uniform direction */
    TPT_PATH_THOMAS_STREAM = 5,   /* one thread per column, c' spilled to the workspace */
    TPT_PATH_THOMAS_ONCHIP = 6,   /* on-chip partitioned sweep, natural layout */
    TPT_PATH_THOMAS_BLOCKED = 7,  /* on-chip partitioned sweep on the tile-blocked mode-space layout */
    TPT_PATH_FUSED_SMALL = 8      /* all five steps in one cluster launch (grids that fit on chip) */
};
int tpt_plan_get_paths(const tpt_plan *plan, int *paths_out);

/* L2-resident slab pipeline of steps 2.2 -> 2.3 -> 2.4 (BASELINE north_star "Fusion"): the forward-y
 * transform, the z sweep and the inverse-y transform run x-slab by x-slab (G 16-column groups x ny x nz) through two
 * plan-owned slab buffers that stay in the 126 MB L2, so the mode-space field never travels to HBM (4 of a solve's 10
 * field-sized HBM passes).  groups: -1 = automatic (default: one-group slabs where the y transform is a fast transform,
 * the field is at least 256 MiB and a slab at most 40 MiB), 0 = off, G > 0 = force slabs of G groups (the slab buffers,
 * 2 * G * 16 * ny * nz doubles, are allocated at the next solve).  Needs the tile-blocked layout (nx % 16 == 0, default
 * kernel variants); ignored otherwise.  Results equal the unslabbed solve's bit for bit. */
int tpt_plan_set_slab_groups(tpt_plan *plan, int groups);

/* Kernel launches the last tpt_solve / tpt_solve_batch / tpt_solve_host[_async] / tpt_project on this plan enqueued
 * (>= 0), < 0 on error. */
int tpt_plan_launches(const tpt_plan *plan);

/* Small-grid execution path (BASELINE.json configs[0]): with the default kernel variants, a grid of at most 16384 points
 * whose z-plane slabs fit the shared memory of a thread-block cluster of 8 runs steps 2.1-2.5 and the
 * gauge as ONE launch — the planes stay on chip through both transforms of each side, the sweep's change of ownership
 * goes through the workspace in L2 between two cluster barriers.  GEMM transforms only.  enabled = 0 forces the five
 * separate kernels (default 1).  tpt_stage and the host-buffer solves always use the separate kernels. */
int tpt_plan_set_fused_small(tpt_plan *plan, int enabled);

/* Select the z-sweep kernel: 1 = on-chip partitioned Thomas kernel (column tiles resident in shared memory,
 * 16 B/pt of HBM traffic; used where nx*ny % 16 == 0 and nz <= 1056, default), 0 = streaming one-thread-per-column
 * kernel that spills c' to the plan workspace (any shape).  Both solve step 2.3 exactly. */
int tpt_plan_set_thomas_variant(tpt_plan *plan, int variant);

/* Synthetic input generator on the device ("white-noise" fields; recipe in DESIGN.md §4): out_dev[t] =
 * 2u - 1, u = top 53 bits of the splitmix64 finaliser of (offset + t + (seed + 1) * 0x9E3779B97F4A7C15 mod 2^64) * 2^-53 —
 * bit-identical to the host generator the tests and the oracle use, so large right-hand sides need not cross the bus.
 * Holds none of the method's arithmetic.  out_dev: DEVICE, count doubles, 8-byte aligned.  Asynchronous on cuda_stream. */
int tpt_fill_uniform(double *out_dev, size_t count, unsigned long long seed, unsigned long long offset, void *cuda_stream);

/* FP64 arithmetic-pipe microbenchmarks used as roofline denominators: kind 0 = register-resident
 * DFMA loop, kind 1 = register-resident DMMA (m8n8k4) loop.  Runs on the current device, returns
 * achieved TFLOP/s (2 flop per FMA) in *tflops_out.  Synchronous. */
int tpt_fp64_peak(int kind, double *tflops_out);

const char *tpt_strerror(int status);
const char *tpt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TPT_H */
