/*
 * oci.h — C ABI of the B200 (sm_100a) one-cell-inversion library.
 *
 * Method: transient, mono-energetic, isotropic-scattering slab S_N transport
 * (eq. 1), multiple balance in time (eqs. 2,3) and
 * simple corner balance in space (eqs. 4-11), iterated within each
 * time step by one-cell inversion (OCI, eqs. 19-28: every cell
 * solves its dense 4N x 4N system with incident fluxes lagged one iterate,
 * parallel block Jacobi) or, for comparison, by source iteration (SI,
 * eqs. 12-18).  "P:nnn" = line nnn of /root/reference/PAPER.md.
 *
 * All arithmetic is fp64 and runs in hand-written CUDA kernels; there is no
 * CPU fallback.  No torch / C++ types cross this boundary: plain pointers
 * (each documented as HOST or DEVICE) and sizes.
 *
 * Layout conventions (all arrays C-contiguous, double unless noted)
 *   angle index m = 0..N-1 ascending in mu_m (Gauss-Legendre, sum w = 2);
 *   the mirror image of direction m is N-1-m.
 *   slot s: 0 = (k,L)  1 = (k,R)  2 = (k+1/2,L)  3 = (k+1/2,R)
 *           k = time-average unknown, k+1/2 = time-edge unknown (eqs. 2,3),
 *           L/R = left/right half-cell (corner) average (eqs. 4-7).
 *   per-cell unknown vector Psi_j[4m+s]  (eqs. 23,24).
 *
 * Ownership: the caller owns every array passed in or out; inputs are copied
 * during the call.  The context is library-owned (oci_destroy).  Device
 * memory is supplied by the caller as one workspace (oci_workspace_bytes /
 * oci_setup) that must outlive the context; the library never allocates
 * device memory.  One context is not thread-safe; distinct contexts are.
 *
 * Return codes: 0 OK; 1 OCI_NOT_CONVERGED (max_iters reached; the state is
 * still committed); negative = failure, no state change:
 *   -1 invalid argument   -2 call order   -3 CUDA error
 *   -4 singular block     -5 workspace too small
 *   -6 OCI_E_NONFINITE: the scalar flux became NaN or Inf inside a step (a
 *      non-finite psi_edge or Q, or overflow); the iteration loop stops at
 *      once on the device, the state is undefined, restart with oci_set_flux.
 * Devices: the context belongs to the device its workspace lives on
 * (oci_setup); every entry point makes that device current for the duration
 * of the call and restores the caller's, so contexts on several devices can
 * live in one process.
 * No exception crosses the ABI.  oci_last_error() describes the last failure.
 */
#ifndef OCI_B200_H
#define OCI_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct oci_ctx oci_ctx;

enum { OCI_OK = 0, OCI_NOT_CONVERGED = 1, OCI_E_INVALID = -1, OCI_E_ORDER = -2, OCI_E_CUDA = -3,
       OCI_E_SINGULAR = -4, OCI_E_WORKSPACE = -5, OCI_E_NONFINITE = -6 };

/* Boundary conditions (vacuum and reflecting P:31).
 * INCIDENT_ISOTROPIC: `value` is the incident ANGULAR flux psi_m for every
 * incoming direction, constant in time, used for both the k and k+1/2
 * balance equations.  REFLECTING: incident psi_m = outgoing psi_{N-1-m} of the
 * previous iterate (lagged in both OCI and SI).
 * HALO (row f4, sharded slab): the face is a cut between two shards of one slab; the incident flux is the
 * neighbour shard's outgoing flux of the previous iterate, delivered by oci_shard_attach's mailboxes. */
enum { OCI_BC_VACUUM = 0, OCI_BC_INCIDENT_ISOTROPIC = 1, OCI_BC_REFLECTING = 2, OCI_BC_HALO = 3 };
typedef struct { int32_t kind; double value; } oci_bc;

/* Which kernel family oci_setup selected for the OCI apply (eq. 19):
 * SHARED   - all cells share one (dx, Sigma, Sigma_s): one inverse, applied
 *            as a dense [4N x 4N].[4N x cells] contraction on the fp64 tensor pipe;
 * PER_CELL - one inverse per distinct triple, applied as a batched GEMV that
 *            streams the inverses from HBM. */
enum { OCI_PATH_SHARED = 0, OCI_PATH_PER_CELL = 1 };

/* Which apply kernel serves that path for this block size (informational; valid after oci_setup):
 * GENERIC  - any n, shared block, simple shared-memory tiles;
 * RESIDENT - shared block, n in {64,128}: B^{-1} resident in registers, cells streamed by TMA;
 * KTILED   - shared block, n a multiple of 32 up to 1024: both operands streamed in K chunks by
 *            tensor-map TMA from L2 (config 4, n = 512);
 * PER_CELL - batched GEMV streaming one inverse per cell from HBM. */
enum { OCI_KERNEL_GENERIC = 0, OCI_KERNEL_RESIDENT = 1, OCI_KERNEL_KTILED = 2, OCI_KERNEL_PER_CELL = 3 };

/* Form of the OCI iteration inside oci_step (oci_set_iteration).  Both produce the iterates of
 * eq. (19), up to rounding order:
 * FULL    - every iteration applies the whole inverse, Psi^(l+1) = B^{-1} c^(l) (the paper's statement);
 * REDUCED - only the 2N RHS rows fed by incident fluxes change within a step (the (l) terms of
 *           eqs. 27,28), so a step is three kinds of pass over packed state (O = the 2N rows
 *           of Psi a neighbour reads, I = the other 2N, inc = the gathered neighbour values):
 *             FIX   once:    [Psi_fix; W Psi_fix] = X [psi_{k-1/2}; Q]         (4N+4) x (2N+4)
 *             ITER  L times: y^(l+1) = yfix + G inc^(l), phi^(l+1) = phifix + H inc^(l),
 *                            G = B^{-1}[O,I] diag|mu| (2N x 2N), H = W B^{-1}[:,I] diag|mu| (4 x 2N)
 *             FINAL once:    Psi^(L)[I] = ifix + F inc^(L-1), F = B^{-1}[I,I] diag|mu| (2N x 2N)
 *           Every unknown of every cell is still computed every step; the state is kept in the packed
 *           (O, I) order between steps and interleaved on demand (oci_get_angular_flux, si_step). */
enum { OCI_ITERATION_FULL = 0, OCI_ITERATION_REDUCED = 1, OCI_ITERATION_AUTO = 2 };
/* AUTO (the default) = REDUCED wherever a kernel of the reduced form is the faster one for this
 * problem: always on the PER_CELL path, on the SHARED path when a tensor-core kernel of the reduced
 * form serves the block size (or the block is small); FULL otherwise.  oci_get_info reports the
 * resolved form after oci_setup. */

/* Kernel family serving the REDUCED form (all three passes): GEMV - batched GEMV, one operator per
 * distinct block (any n; HBM-bound on the PER_CELL path);
 * RESIDENT - shared block, n in {64,128}: operators resident in shared memory, fp64 tensor pipe;
 * KTILED - shared block, or 2..16 distinct blocks (a multi-region slab), N a multiple of 16: operands
 *          streamed in K chunks by tensor-map TMA, fp64 tensor pipe; a block is a row offset into the
 *          stacked operators, a tile of cells that straddles an interface is done once per block;
 * OPREG - ONE shared block, N in {32, 64, 128} (config 4; N = 32 only when forced): each CTA keeps 64 operator rows as DMMA fragments in
 *          registers for the whole launch and only the cell rows stream (tensor-map TMA); fp64 tensor pipe.
 * WOODBURY - any problem: B^{-1} is never applied as a dense matrix.  The scattering matrix of eq. (22), has
 *          rank 4 (isotropic, one group), so B^{-1} c = t + kappa A^{-1} (1 (x) phi), t = A^{-1} c a 4x4 apply per angle,
 *          phi = (I_4 - kappa sum_m w_m A_m^{-1})^{-1} sum_m w_m t_m: O(N) work and bytes per cell instead of O(N^2);
 *          HBM-bound.  Same iterates up to rounding order.  Selected only on request.
 * oci_setup picks RESIDENT, else OPREG, else KTILED, else GEMV; oci_set_reduced_kernel overrides. */
enum { OCI_RKERNEL_AUTO = -1, OCI_RKERNEL_GEMV = 0, OCI_RKERNEL_RESIDENT = 1, OCI_RKERNEL_KTILED = 2, OCI_RKERNEL_OPREG = 3,
       OCI_RKERNEL_WOODBURY = 4 };

typedef struct {
    int64_t cells;        /* J */
    int32_t n_angles;     /* N */
    int32_t block_dim;    /* n = 4N */
    int64_t n_blocks;     /* distinct (dx, Sigma, Sigma_s) triples */
    int32_t path;         /* OCI_PATH_* */
    int32_t apply_kernel; /* OCI_KERNEL_* */
    int32_t iteration;    /* OCI_ITERATION_* */
    int32_t reduced_kernel; /* OCI_RKERNEL_* */
    int32_t small_step_cluster; /* CTAs of the one-launch step's cluster, 0 = the three-pass kernels (oci_set_small_step) */
    int32_t si_small_step_cluster; /* the same for si_step: CTAs of its one-launch step, 0 = three kernels per iteration */
} oci_info;

/* Problem statement (per-cell dx_j, Sigma_j, Sigma_s,j P:74-82).
 * dx, sigma_t, sigma_s: HOST [cells].  v = particle speed, dt = time step.
 * n_angles = N (even, 2 <= N <= 512: the setup and per-cell kernels stage O(4N)
 * doubles per CTA in shared memory).  Computes the Gauss-Legendre set on the host.
 * Errors: -1 if cells<1, N odd, <2 or >512, any dx<=0, Sigma<0, Sigma_s<0, v<=0,
 * dt<=0, a NULL pointer or an unknown BC kind.  A context with an OCI_BC_HALO face must be attached to
 * its slab (oci_shard_attach) before it can step. */
int oci_create(oci_ctx** out, int64_t cells, const double* dx, const double* sigma_t,
               const double* sigma_s, double v, double dt, int32_t n_angles, oci_bc left,
               oci_bc right);

/* DEVICE bytes the caller must supply to oci_setup. */
int64_t oci_workspace_bytes(const oci_ctx* ctx);

/* Form B = A - S (eqs. 13,16,20-22) for every distinct
 * (dx, Sigma, Sigma_s) triple (bitwise-equal classification), invert each
 * with partial pivoting on the device (the paper's `gesv`, hoisted out
 * of the loops), form the 4x4 inverses SI needs, zero the state.
 * d_workspace: DEVICE, 256-byte aligned, `bytes` >= oci_workspace_bytes().
 * cuda_stream: a cudaStream_t (as void*) used for every later call, or NULL.
 * Errors: -3, -4 (a block is singular), -5. */
int oci_setup(oci_ctx* ctx, void* d_workspace, int64_t bytes, void* cuda_stream);

/* Initial / restart condition psi_{m,0}(x): HOST [cells][N][2] = (L,R)
 * corner values at the previous time edge t_{k-1/2}.  Also seeds the iterate
 * (slots 0,2 <- L, slots 1,3 <- R).  A complete checkpoint together with
 * oci_get_angular_flux()[..][2:4].  _dev: same layout, DEVICE pointer. */
int oci_set_flux(oci_ctx* ctx, const double* psi_edge);
int oci_set_flux_dev(oci_ctx* ctx, const double* d_psi_edge);

/* Isotropic source Q: HOST [cells][4] in slot order; NULL = 0; sticky
 * until the next call.  _dev: DEVICE pointer.  With a HOST pointer the call
 * returns when the copy is done (the buffer may be reused at once); NULL and
 * the _dev variant are asynchronous on the context's stream. */
int oci_set_source(oci_ctx* ctx, const double* q);
int oci_set_source_dev(oci_ctx* ctx, const double* d_q);

/* Advance one time step by OCI (oci_step) or SI (si_step): iterate until
 *     max_{j,s} |phi^(l+1) - phi^(l)| <= tol * max_{j,s} |phi^(l+1)|
 * over all four scalar-flux slots ("ceases changing"), tested on
 * the device after every iteration; then commit psi_{k+1/2} as the next
 * step's psi_{k-1/2}.  tol < 0 never converges: exactly max_iters iterations.
 * iters (HOST, may be NULL): iterations done.  resid (HOST, may be NULL):
 * last d/r (d if r == 0).  One host read-back per call (per launch chunk).
 * Stream order: everything is queued on the context's stream.  In the REDUCED
 * form oci_step returns as soon as the iteration count is known, which is
 * BEFORE its last kernel (the FINAL pass, which writes the I rows of Psi) has
 * finished; every later call on this context is ordered behind it, but a
 * caller that reads the workspace from ANOTHER stream must synchronise with
 * the context's stream first.
 * Returns 0, 1 (OCI_NOT_CONVERGED), -1, -2, -3, -6. */
int oci_step(oci_ctx* ctx, double tol, int32_t max_iters, int32_t* iters, double* resid);
int si_step(oci_ctx* ctx, double tol, int32_t max_iters, int32_t* iters, double* resid);

/* Select the form of the OCI iteration (default OCI_ITERATION_AUTO).  May be called at any time
 * after oci_create; takes effect at the next oci_step.  Errors: -1. */
int oci_set_iteration(oci_ctx* ctx, int32_t iteration);

/* ---- Row f4: one slab sharded over several GPUs by contiguous cell ranges ----------------------
 * Shard r of W is an ordinary context over its own cells (one process per GPU, or several contexts in one process)
 * whose cut faces have kind OCI_BC_HALO: left face for r > 0, right face for r < W-1.  Within an iteration a
 * shard owes each neighbour the N outgoing values of its edge cell and every rank needs the maximum over ranks of the
 * two norms of the stopping rule; both travel as plain stores into peer memory (NVLink), issued by stream-ordered
 * kernels behind every iteration launch, with no host involvement per iteration and no collective library.  Because
 * the maximum is exact, every rank takes the same stopping decision and the iterates and iteration counts are those
 * of the unsharded problem, bit for bit.  REDUCED form of oci_step only (si_step and the FULL form return -1).
 *
 * oci_shard_mailbox_bytes: DEVICE bytes of one rank's mailbox.  The caller allocates one mailbox per rank in memory
 * every rank can address (peer-mapped / symmetric memory; 16-byte aligned) and passes all W device addresses, in rank
 * order, to oci_shard_attach on every rank (HOST array of W DEVICE pointers; after oci_setup, before oci_set_flux).
 * oci_shard_attach zeroes the rank's own mailbox on the context's stream: all ranks must have completed it (a
 * barrier across ranks after a stream synchronise) before any rank steps.  Errors: -1 (rank / world out of range,
 * W > 64, a cut face that is not HALO or a HALO face that is not a cut), -2.
 *
 * oci_shard_step advances n shards that live in THIS process by one time step, interleaving their launches
 * (iteration, push, pull) so that on a single device and stream every pull is ordered behind all pushes; n = 1 is the
 * one-process-per-GPU case, and oci_step on a sharded context is oci_shard_step with n = 1.  All shards of the slab,
 * in this process or not, must be stepped with the same tol and max_iters.  iters / resid as oci_step (identical on
 * every shard).  With n > 1 all contexts must share one device and one stream. */
int64_t oci_shard_mailbox_bytes(int32_t n_angles, int32_t world);
int oci_shard_attach(oci_ctx* ctx, int32_t rank, int32_t world, void* const* d_mailboxes);
int oci_shard_step(oci_ctx* const* ctxs, int32_t n, double tol, int32_t max_iters, int32_t* iters, double* resid);

/* Force the kernel family of the REDUCED form (default OCI_RKERNEL_AUTO).  Call BEFORE oci_setup; oci_setup
 * returns -1 if the forced family does not serve this problem (block size, number of blocks).  For tests and
 * for comparing families on shapes more than one serves.  Errors: -1 (unknown family). */
int oci_set_reduced_kernel(oci_ctx* ctx, int32_t kernel);

/* One-launch step for small shared-block problems (the launch-latency-bound end of S4..S128): FIX, every ITER iteration
 * with the stopping rule and FINAL inside ONE kernel on one thread-block cluster, the state resident in distributed
 * shared memory, a hardware cluster barrier per iteration instead of a grid-wide one.  Same operators, same iterates up to
 * rounding order.  mode -1 (default): used by itself when the problem is small enough to fit and to win and no kernel
 * family has been forced; 0: never; 1: required (oci_setup returns -1 if the problem does not fit: per-cell blocks, HALO
 * faces, N > 32, or a state larger than a cluster's shared memory).  Call BEFORE oci_setup.  oci_get_info reports the
 * cluster size in use.  A step that does not converge within the 64 iterations of one launch continues on the three-pass
 * kernels.  The same switch governs si_step, whose comparator gets the same treatment at the same sizes (every SI
 * iteration and the final sweep in one launch; modes -1 and 1 take it where it fits, and mode 1 never fails because of
 * si_step: where it does not fit, si_step runs its three kernels per iteration).  Errors: -1. */
int oci_set_small_step(oci_ctx* ctx, int32_t mode);

/* Results of the current state.  phi: [cells][4] (eq. 18);
 * psi: [cells][N][4].  HOST pointers; _dev variants take DEVICE pointers and
 * are asynchronous on the context's stream. */
int oci_get_scalar_flux(const oci_ctx* ctx, double* phi);
int oci_get_angular_flux(const oci_ctx* ctx, double* psi);
int oci_get_scalar_flux_dev(const oci_ctx* ctx, double* d_phi);
int oci_get_angular_flux_dev(const oci_ctx* ctx, double* d_psi);

/* Streaming read-back for time-stepping loops: oci_get_scalar_flux_async snapshots phi of the current state on the
 * context's stream (a device-to-device copy into a staging array, so the next step may overwrite phi) and copies the
 * snapshot to `phi_pinned` (HOST, page-locked, [cells][4]) on a side stream, concurrently with whatever is queued
 * next; it returns at once.  The data is valid after oci_synchronize (or the next oci_get_scalar_flux_async /
 * oci_synchronize, which wait for the previous snapshot's copy).  oci_synchronize waits for everything this context
 * has queued on its stream and its side stream.  Errors: -1, -2, -3. */
int oci_get_scalar_flux_async(oci_ctx* ctx, double* phi_pinned);
int oci_synchronize(oci_ctx* ctx);

/* Quadrature in use: HOST mu[N], w[N], ascending mu. */
int oci_get_quadrature(const oci_ctx* ctx, double* mu, double* w);

/* Problem / path description (valid after oci_create; n_blocks and path after oci_setup). */
int oci_get_info(const oci_ctx* ctx, oci_info* info);

/* Inverse of block `blk` as computed by oci_setup: HOST [4N][4N] row major
 * (B^{-1}[i][k]).  For verification of the setup kernel. */
int oci_get_block_inverse(const oci_ctx* ctx, int64_t blk, double* binv);

/* Kernel timing for roofline reports.  When enabled, every launch of the
 * OCI apply kernel (eq. 19) is bracketed by CUDA events on the context's
 * stream; oci_get_kernel_time returns the accumulated milliseconds and launch
 * count since the last enable and resets them. */
int oci_enable_kernel_timing(oci_ctx* ctx, int32_t on);
int oci_get_kernel_time(oci_ctx* ctx, double* ms, int64_t* launches);
/* REDUCED form only: the per-step FIX pass and FINAL pass, accumulated like oci_get_kernel_time
 * (which then counts the ITER kernel).  Any pointer may be NULL. */
int oci_get_aux_kernel_time(oci_ctx* ctx, double* fix_ms, int64_t* fix_launches, double* final_ms,
                            int64_t* final_launches);

/* Device time of the last oci_setup on this context (forming and inverting the blocks, packing the
 * operators of the reduced step): milliseconds between CUDA events on the context's stream.  Reported
 * once, separately from the per-step times.  Errors: -1, -2 (before oci_setup). */
int oci_get_setup_time(const oci_ctx* ctx, double* ms);

/* Number of kernels this library launched on this context so far. */
int64_t oci_launch_count(const oci_ctx* ctx);

const char* oci_last_error(const oci_ctx* ctx);
void oci_destroy(oci_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* OCI_B200_H */
