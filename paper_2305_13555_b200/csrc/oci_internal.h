// Internal declarations shared by the host driver (oci_api.cu) and the kernels.
// Not part of the C ABI (include/oci.h is).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "oci.h"

namespace oci {

constexpr int kNormSlots = 64;  // iterations launched between two host read-backs, at most
constexpr int kScratchSlot = kNormSlots;
constexpr int kMaxGroupedBlocks = 16;      // "a handful of materials": operators stay L2-resident, tensor-core path (row f2)   // norm slot nobody reads (the Psi_fix pass of the reduced iteration)

// Device-side view of one problem.  Passed to kernels by value.
// Psi buffers have one ghost row before row 0 and one after row J-1: psi[b]
// points at row 0, rows -1 and J hold the boundary data in the slots a
// neighbour cell would occupy, so the iteration kernels need no boundary
// branches.
struct DevView {
    int64_t J;
    int32_t N;
    int32_t n;                  // 4N
    int64_t nblk;
    double* binv;               // [nblk][n][n]  B^{-1}, row major
    double* psi[2];             // ping-pong iterates, [(J+2)][n] each
    double* cfix;               // [J][n]   iteration-invariant part of the RHS (a2)
    double* phi;                // [J][4]
    double* Q;                  // [J][4]
    double* qs;                 // [J][4]   SI scattering source (d1)
    double* dx;                 // [J]
    double* sig;                // [J]
    double* sigs;               // [J]
    int32_t* blk;               // [J] -> block id
    int64_t* rep;               // [nblk] -> a representative cell
    double* mu;                 // [N]
    double* w;                  // [N]
    double* coef;               // [n]  |mu_m| on the rows that take an incident flux, else 0
    double* ainv4;              // [nblk][N][16]  (A_m)^{-1} for SI
    double* si_scan;            // [chunks][N][8]  SI scan: chunk maps (P, z) and chunk inflows (si_sweep.cu)
    double* si_prev;            // [J][N][2]  psi_{k-1/2}, compact (si_sweep_fast.cu; aliases c_fix, which SI then does not use)
    double* si_part;            // [max(2, N/32)][J][4]  scalar-flux partials per lane group (si_sweep_fast.cu)
    double* si_src1;            // [J][4]  second buffer of the SI scattering source (the first is qs), by iteration parity
    double* si_inflow;          // [2][N][2]  boundary inflow of every angle, by iteration parity (si_sweep_fast.cu)
    double* si_agg;             // [N][segments][8]  carry scan: composition through a segment, [7] = the launch tag (si_sweep_fast.cu)
    double* phi_part;           // [ceil(n/128)][J][4]  per-item scalar-flux partials (K-tiled kernel)
    int32_t* tickets;           // [ceil(J/64)]  arrival counters of the K-tiled kernel's cell tiles (0 between launches)
    unsigned long long* norms;  // [kNormSlots][2]  bit patterns of (d, r), atomicMax targets
    int32_t* flags;             // [0] = 1 + index of a singular block, 0 if none; [8] grid-barrier counter of the fused loops; [12] their work-ticket counter; [16..17] u64 ticket counter of the SI carry scan (never reset)
    int32_t* perm;              // [nblk][n]  pivot rows of the blocked inversion (setup)
    int32_t* team_bar;          // [min(nblk, SMs)]  team-barrier counters of the blocked inversion (setup)
    // ---- interface-reduced step (oci_reduced.cu), K2 = 2N
    double* xop;                // [nblk][2*K2+8][K2+16]  FIX operator X (rows: O, I, scalar flux; zero padded)
    double* rop;                // [nblk][K2+8][K2]  rows 0..K2-1: G = B^{-1}[O,I] diag|mu|; K2..K2+3: H = W B^{-1}[:,I] diag|mu|; rest 0
    double* fop;                // [nblk][K2][K2]  F = B^{-1}[I,I] diag|mu|
    double* y[2];               // ping-pong interface iterates (O rows of Psi, packed), [(J+2)][K2], ghost rows as psi
    double* z;                  // [J][K2]  I rows of Psi, packed (written by the FINAL pass)
    double* yfix;               // [J][K2]  O rows of Psi_fix = B^{-1} c_fix
    double* ifix;               // [J][K2]  I rows of Psi_fix
    double* phifix;             // [J][4]   W Psi_fix
    double* q16;                // [J][16]  Q padded to one 128-byte row (K-tiled FIX pass only; else unused)
    // ---- O(N) apply through the rank-4 scattering matrix (oci_reduced_woodbury.cu)
    double* wba;                // [nblk][16][N]  (A_m)^{-1}, element-major (coalesced over the angles)
    double* wbd;                // [nblk][16][N]  kappa (A_m)^{-1} M, element-major
    double* wbm;                // [nblk][32]     M = (I_4 - kappa sum_m w_m A_m^{-1})^{-1} (16), kappa = dx Sigma_s / 4, padding
    int32_t* gitems;            // [ngroups][4] = (cell tile, block, mask lo, mask hi): a handful of materials on the K-tiled
                                // kernels (row f2); nullptr when all cells share one block (or have one each)
    int64_t ngroups;
    double v, dt;
    int32_t bcL, bcR;
    double bcLv, bcRv;
    int32_t sm_count;           // SMs of the device the workspace lives on (queried once in oci_setup)
    // ---- a7 without a copy: a fused iteration loop reports (iterations run, d, r) of its last iteration straight into
    // mapped, page-locked HOST memory and then the sequence number of the launch; the host polls the number
    unsigned long long* host_pub;   // [4] = seq, iterations, bits(d), bits(r); nullptr = do not publish
    unsigned long long pub_seq;
    // ---- row f4: this context is shard `rank` of `world` (shard_exchange.cu); world = 1 when not sharded
    int32_t rank, world;
    unsigned long long* peers;  // [world] device addresses of every rank's mailbox (peer mapped), in the workspace
};

// Tensor maps of the K-tiled shared-block kernel (oci_iter_shared_ktiled.cu), encoded once in oci_setup.
struct KtiledMaps {
    CUtensorMap cfix, psi[2], binv;
};

// Tensor maps of the K-tiled kernels of the reduced step (oci_reduced_ktiled.cu), encoded once in oci_setup.
struct RedKtiledMaps {
    CUtensorMap y[2], z, q16, xop, xop8, rop, rop8, fop;
};

// Tensor maps of the operator-in-registers kernels of the reduced step (oci_reduced_opreg.cu): boxes of 64 rows x 16 columns
struct RedOpregMaps {
    CUtensorMap y[2], z, q16, yfix, ifix;
};

// Tensor maps of the resident kernels of the reduced step (oci_reduced_resident.cu)
struct RedResidentMaps {
    CUtensorMap y_rows[2];   // box (K2+4) x 18: whole rows j0-1 .. j0+16 of y, padded pitch (ITER, FINAL)
    CUtensorMap y_half[2];   // box (N+4) x 16 at column N/2: the k+1/2 run of y (FIX)
    CUtensorMap z_half;      // same of z
    CUtensorMap q;           // box 4 x 16 of Q
    CUtensorMap rop, fop;    // the ITER / FINAL operator as one box of rows padded to K2+4
    CUtensorMap xop_rows;    // K2 rows of X (the O rows, the I rows), columns 0 .. K2+3
    CUtensorMap xop_phi;     // the 8-row scalar-flux block of X
};

// The stopping rule (reading S2), evaluated identically on host and device.
__host__ __device__ inline bool converged(double tol, double d, double r) { return tol >= 0.0 && d <= tol * r; }
// A NaN or Inf scalar flux (non-finite input, overflow) also ends the iteration loop, on the device as on the
// host: the step then returns OCI_E_NONFINITE instead of running to max_iters on garbage.
__host__ __device__ inline bool finite_norms(double d, double r) { return d <= 1.7976931348623157e308 && r <= 1.7976931348623157e308; }
__host__ __device__ inline bool stop_now(double tol, double d, double r) { return converged(tol, d, r) || !finite_norms(d, r); }

// Cells per chunk of the SI scan (si_sweep.cu): one chunk for tiny slabs (launch-latency bound), else
// the largest of 64, 32, 16, 8 that still gives every SM about 8 warps of (chunk, angle) threads.
inline int si_chunk_cells(int64_t J, int32_t N, int sm_count = 148)
{
    if (J <= 32) return (int)J;
    const int64_t lanes = N >= 32 ? (N + 31) / 32 * 32 : N;
    for (int S = 64; S > 8; S >>= 1)
        if (((J + S - 1) / S) * lanes >= (int64_t)sm_count * 8 * 32) return S;
    return 8;
}

// ---- launchers: each returns the number of kernels it launched, or -1 when a launch was refused (the CUDA
// error stays readable through cudaGetLastError)
inline int launched(int k) { return cudaPeekAtLastError() == cudaSuccess ? k : -1; }
// Opt-in to more than 48 KB of dynamic shared memory for every kernel of a file that needs it.  The attribute is
// per device, so oci_setup calls these with the context's device current (no per-process caching).
cudaError_t oci_setup_opt_in();
cudaError_t oci_shared_fast_opt_in();
cudaError_t oci_ktiled_opt_in();
cudaError_t oci_red_gemv_opt_in();
cudaError_t oci_red_ktiled_opt_in();
cudaError_t oci_red_resident_opt_in();
cudaError_t oci_red_opreg_opt_in();
cudaError_t oci_red_woodbury_opt_in();
cudaError_t oci_red_small_opt_in();
int launch_form_and_invert(const DevView& V, cudaStream_t s);
int launch_set_flux(const DevView& V, const double* d_psi_edge, int buf, cudaStream_t s);
int launch_cfix(const DevView& V, int buf, cudaStream_t s);
int launch_phi_norm(const DevView& V, int buf, int slot, int prev_slot, double tol, bool with_norms,
                    cudaStream_t s);
int launch_oci_iteration(const DevView& V, int path, int src, int slot, int prev_slot, double tol,
                         cudaStream_t s);
int launch_si_iteration(const DevView& V, int buf, int slot, int prev_slot, double tol, cudaStream_t s);
// fast form (si_sweep_fast.cu): N/2 a power of two
bool si_fast_supported(const DevView& V);
cudaError_t si_fast_opt_in();
int si_carry_segments(int64_t chunks);                 // segments per angle of the SI carry scan (sizes si_agg)
int launch_si_fast_begin(const DevView& V, int buf, cudaStream_t s);
int launch_si_fast_iteration(const DevView& V, int buf, int it, int slot, int prev_slot, double tol, cudaStream_t s);
int launch_si_fast_final(const DevView& V, int buf, int it0, double tol, int cnt, int force, cudaStream_t s);
// interface-reduced step (oci_reduced.cu, oci_reduced_resident.cu, oci_reduced_ktiled.cu)
enum { PASS_FIX = 0, PASS_ITER = 1, PASS_FINAL = 2 };
int launch_pack_operators(const DevView& V, cudaStream_t s);
int launch_pack_yz(const DevView& V, int buf, int ybuf, cudaStream_t s);
int launch_unpack_yz(const DevView& V, int buf, int ybuf, cudaStream_t s);
// ybase: FIX - the y buffer of the current iterate; ITER - the source buffer; FINAL - the source buffer
// of the first of the `cnt` queued iterations
int launch_red_gemv(const DevView& V, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force,
                    cudaStream_t s);
// row-major fp64 matrix [rows][cols] -> 2-D tensor map, box = box_rows x box_cols, zero fill outside; swizzle128
// needs box_cols = 16
bool oci_encode_2d(CUtensorMap* m, const double* base, uint64_t rows, uint64_t cols, uint32_t box_rows, uint32_t box_cols,
                   bool swizzle128);
bool oci_red_ktiled_supported(const DevView& V);
bool oci_red_ktiled_prepare(const DevView& V, RedKtiledMaps* M);
bool oci_red_ktiled_fuses_loop(const DevView& V);
int launch_red_ktiled(const DevView& V, const RedKtiledMaps& M, int pass, int ybase, int slot, int prev_slot, double tol,
                      int cnt, int force, cudaStream_t s);
int launch_shard_push(const DevView& V, int ybuf, int slot, int prev_slot, double tol, unsigned long long tag, cudaStream_t s);
int launch_shard_pull(const DevView& V, int ybuf, int slot, int prev_slot, double tol, unsigned long long tag, cudaStream_t s);
bool oci_red_opreg_supported(const DevView& V);
bool oci_red_opreg_prepare(const DevView& V, RedOpregMaps* M);
int launch_red_opreg(const DevView& V, const RedOpregMaps& M, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force,
                     cudaStream_t s);
// one-launch step of small shared-block problems (oci_reduced_small.cu): cluster size that serves V, 0 if none
int oci_red_small_cluster(const DevView& V);
int launch_red_small(const DevView& V, int C, int ybase, double tol, int cnt, int force, cudaStream_t s);
// one-launch SI step of small shared-block problems (si_small.cu; runs after launch_si_fast_begin): cluster size, 0 if none
int si_small_cluster(const DevView& V);
cudaError_t si_small_opt_in();
int launch_si_small(const DevView& V, int C, int buf, double tol, int cnt, int force, cudaStream_t s);
int launch_woodbury_setup(const DevView& V, cudaStream_t s);
int launch_red_woodbury(const DevView& V, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s);
bool oci_red_resident_supported(const DevView& V);
bool oci_red_resident_prepare(const DevView& V, RedResidentMaps* M);
int launch_red_resident(const DevView& V, const RedResidentMaps& M, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force,
                        cudaStream_t s);

}  // namespace oci
