// Interface-reduced OCI step: the same iterates as eq. (19), with every
// piece of work that does not change inside a time step hoisted out of the iteration, and the state
// between steps kept in the packed form the iteration reads.
//
// Within a step only the 2N RHS rows that take an incident flux change from one iterate to the next
// (the superscript-(l) terms of eqs. 27,28); the rest of c_j is c_fix (row a2).  With
//     I = rows that receive an incident flux  ((m,1),(m,3) for mu_m<0; (m,0),(m,2) for mu_m>0)
//     O = rows a neighbour reads               (the other two slots of each angle; O(q) = I(q) ^ 1)
// and inc^(l)[j] = the 2N neighbour values cell j gathers (row a3), eq. (19) reads
//     Psi^(l+1)[j] = B^{-1} c_fix[j]  +  B^{-1}[:, I] diag|mu| inc^(l)[j]  =  Psi_fix[j] + ...
// The next iterate needs only the O rows of Psi^(l+1) and the stopping rule only phi^(l+1) = W Psi^(l+1)
// (eq. 18), so a time step is three kinds of pass, each a small dense operator applied to every cell:
//
//   FIX   (once)   [yfix | ifix | phifix][j] = X [ psi_{k-1/2}[j] ; Q[j] ]            (4N+4) x (2N+4)
//                  X = [B^{-1}; W B^{-1}] . [alpha E_prev | (h/4) E_Q]: c_fix of eqs. (27),(28) has only 2N
//                  entries that carry psi_{k-1/2} (rows (m,0),(m,1), factor alpha = h/(2 v dt)) and an
//                  isotropic source that is the same for every angle (4 numbers per cell), so Psi_fix needs
//                  neither the c_fix array nor the full 4N x 4N apply;
//   ITER  (L x)    y^(l+1)[j]   = yfix[j]   + G inc^(l)[j],   G = B^{-1}[O, I] diag|mu|     2N x 2N
//                  phi^(l+1)[j] = phifix[j] + H inc^(l)[j],   H = W B^{-1}[:, I] diag|mu|    4 x 2N
//   FINAL (once)   z[j] = Psi^(L)[j][I] = ifix[j] + F inc^(L-1)[j],  F = B^{-1}[I, I] diag|mu|   2N x 2N
//
// about (6 + 4L)/16L of the flops (shared block) or bytes (per-cell blocks) of L full applies.  Up to
// rounding order the iterates are those of the plain method, so iteration counts and fluxes are held to
// the same parity tolerances as the full form.
//
// Packed state.  Angle m = half*(N/2) + mm, h = 0 for the k slot and 1 for the k+1/2 slot:
//     q = h*(N/2) + mm            (half = 0, mu<0)        q = N + (1-h)*(N/2) + mm     (half = 1, mu>0)
// O(q) = 4m + (half ? 2h+1 : 2h);  y[j][q] = Psi[j][O(q)],  z[j][q] = Psi[j][O(q)^1].  With ascending mu the
// first N entries of y[j] leave through the left face and feed cell j-1, the last N feed cell j+1:
// inc[j][q] = y[j+1][q] (q < N), y[j-1][q] (q >= N); |mu| is folded into G, H, F.  The y buffers carry ghost
// rows -1 and J like the Psi buffers do.  psi_{k-1/2}[j] (the commit, row a8) is the h = 1 entries of y[j]
// and z[j]: with this order ONE contiguous run [N/2, 3N/2) of each row, which is what lets a TMA unit
// fetch it as a box.  The full-layout Psi is produced from (y, z) only when somebody asks for it
// (oci_get_angular_flux, si_step, a FULL-form step): a change of layout, no arithmetic.
//
// This file: the operator packing (setup), the Psi <-> (y, z) layout kernels, and the generic kernels
// of the three passes (a batched GEMV with one operator per distinct block: HBM-bound when every cell
// has its own block, the fallback for shared blocks of sizes the tensor-core kernels do not take).
#include "device_utils.cuh"

namespace oci {

namespace {

// RHS row (full index) that column u < 2N of the FIX operator feeds: u < N walks y[j][N/2 + u], u >= N walks
// z[j][N/2 + (u - N)] (the k+1/2 runs)
__device__ __forceinline__ int fix_col_row(int u, int N)
{
    const int N2 = N >> 1;
    if (u < N2) return 4 * u + 0;            // y, mu<0: psi_{k+1/2,L} of angle u        -> row (m,0)
    if (u < N) return 4 * u + 1;             // y, mu>0: psi_{k+1/2,R} of angle u        -> row (m,1)
    if (u < N + N2) return 4 * (u - N) + 1;  // z, mu<0: psi_{k+1/2,R} of angle u - N    -> row (m,1)
    return 4 * (u - N) + 0;                  // z, mu>0: psi_{k+1/2,L} of angle u - N    -> row (m,0)
}

__device__ __forceinline__ double2 ldg_stream2(const double* p)
{
    double2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}

}  // namespace

// ---- setup: X, G, H, F of every distinct block from its inverse (one CTA per block)
__global__ void __launch_bounds__(256) pack_operators_kernel(DevView V)
{
    const int n = V.n, N = V.N, K2 = n >> 1, MO = K2 + 8, MF = 2 * K2 + 8, KF = K2 + 16;
    const int64_t b = blockIdx.x;
    const double* __restrict__ Bi = V.binv + (size_t)b * n * n;
    double* __restrict__ R = V.rop + (size_t)b * MO * K2;
    double* __restrict__ F = V.fop + (size_t)b * K2 * K2;
    double* __restrict__ X = V.xop + (size_t)b * MF * KF;
    const double h = V.dx[V.rep[b]];
    const double al = h / (2.0 * V.v * V.dt), q4 = 0.25 * h;
    for (int e = threadIdx.x; e < MO * K2; e += blockDim.x) {
        const int r = e / K2, p = e - r * K2;
        const int ip = o_row(p, N) ^ 1;
        const double cf = V.coef[ip];
        double val = 0.0;
        if (r < K2) {
            val = Bi[(size_t)o_row(r, N) * n + ip] * cf;
            F[(size_t)r * K2 + p] = Bi[(size_t)(o_row(r, N) ^ 1) * n + ip] * cf;
        } else if (r < K2 + 4) {
            const int s = r - K2;
            double a = 0.0;
            for (int m = 0; m < N; ++m) a = fma(V.w[m], Bi[(size_t)(4 * m + s) * n + ip], a);
            val = a * cf;
        }
        R[e] = val;
    }
    // X: rows [0,K2) = O rows, [K2,2K2) = I rows, [2K2,2K2+4) = the scalar-flux rows W B^{-1}, rest 0;
    // columns [0,K2) = alpha * B^{-1}[.][fix_col_row(u)], [K2,K2+4) = (h/4) sum_m B^{-1}[.][4m+s], rest 0
    for (int e = threadIdx.x; e < MF * KF; e += blockDim.x) {
        const int r = e / KF, u = e - r * KF;
        double val = 0.0;
        if (r < 2 * K2 + 4 && u < K2 + 4) {
            if (r < 2 * K2) {
                const int row = r < K2 ? o_row(r, N) : (o_row(r - K2, N) ^ 1);
                if (u < K2) {
                    val = al * Bi[(size_t)row * n + fix_col_row(u, N)];
                } else {
                    double a = 0.0;
                    for (int m = 0; m < N; ++m) a += Bi[(size_t)row * n + 4 * m + (u - K2)];
                    val = q4 * a;
                }
            } else {
                const int s = r - 2 * K2;
                double a = 0.0;
                if (u < K2) {
                    const int col = fix_col_row(u, N);
                    for (int m = 0; m < N; ++m) a = fma(V.w[m], Bi[(size_t)(4 * m + s) * n + col], a);
                    val = al * a;
                } else {
                    for (int m = 0; m < N; ++m) {
                        double c = 0.0;
                        for (int mp = 0; mp < N; ++mp) c += Bi[(size_t)(4 * m + s) * n + 4 * mp + (u - K2)];
                        a = fma(V.w[m], c, a);
                    }
                    val = q4 * a;
                }
            }
        }
        X[e] = val;
    }
}

int launch_pack_operators(const DevView& V, cudaStream_t s)
{
    pack_operators_kernel<<<(unsigned)V.nblk, 256, 0, s>>>(V);
    return 1;
}

// ---- (y[ybuf], z) <- Psi[buf], ghost rows of y included (after set_flux / si_step / a FULL-form step)
__global__ void __launch_bounds__(256) pack_yz_kernel(DevView V, int buf, int ybuf)
{
    const int n = V.n, N = V.N, K2 = n >> 1;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (V.J + 2) * K2) return;
    const int64_t row = t / K2 - 1;                       // -1 .. J
    const int q = (int)(t % K2);
    const int o = o_row(q, N);
    const double v = V.psi[buf][row * n + o];
    V.y[ybuf][row * K2 + q] = v;
    // vacuum / incident ghost rows are constant: both buffers hold them (reflecting ones are rewritten
    // by every iteration)
    if (row < 0 || row >= V.J) V.y[ybuf ^ 1][row * K2 + q] = v;
    else V.z[row * K2 + q] = V.psi[buf][row * n + (o ^ 1)];
}

int launch_pack_yz(const DevView& V, int buf, int ybuf, cudaStream_t s)
{
    const int64_t tot = (V.J + 2) * (V.n >> 1);
    pack_yz_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(V, buf, ybuf);
    return 1;
}

// ---- Psi[buf] <- (y[ybuf], z): the full layout on demand; the ghost rows of Psi take the O entries
// of the ghost rows of y (the only ones a neighbour reads)
__global__ void __launch_bounds__(256) unpack_yz_kernel(DevView V, int buf, int ybuf)
{
    const int n = V.n, N = V.N, K2 = n >> 1;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (V.J + 2) * K2) return;
    const int64_t row = t / K2 - 1;
    const int q = (int)(t % K2);
    const int o = o_row(q, N);
    const bool ghost = row < 0 || row >= V.J;
    // of a ghost row only the half that feeds the domain is meaningful (left ghost: q >= N)
    if (!ghost || (row < 0) == (q >= N)) V.psi[buf][row * n + o] = V.y[ybuf][row * K2 + q];
    if (!ghost) V.psi[buf][row * n + (o ^ 1)] = V.z[row * K2 + q];
}

int launch_unpack_yz(const DevView& V, int buf, int ybuf, cudaStream_t s)
{
    const int64_t tot = (V.J + 2) * (V.n >> 1);
    unpack_yz_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(V, buf, ybuf);
    return 1;
}

// ---- the three passes as a batched GEMV, one CTA per cell (PASS_* of oci_internal.h).
// FIX  :  [yfix | ifix | phifix][j] = X_b [psi_{k-1/2}[j]; Q[j]],  psi_{k-1/2} from y[ybase][j], z[j]
// ITER :  y^(l+1)[j] = yfix[j] + G_b inc,  phi^(l+1)[j] = phifix[j] + H_b inc, norms, ghost rows of y
// FINAL:  z[j] = ifix[j] + F_b inc^(L-1); L is found on the device from the norm slots of the `cnt`
//         queued iterations (`force`: this chunk ends at max_iters, finalise after cnt iterations if
//         none converged); y^(L) is already in place.
template <int PASS, int ROWS>
__global__ void __launch_bounds__(256) oci_red_gemv_kernel(DevView V, int ybase, int slot, int prev_slot, double tol,
                                                           int cnt, int force)
{
    int ysrc = ybase;
    if (PASS == PASS_ITER) {
        if (step_done(V.norms, prev_slot, tol)) return;
    } else if (PASS == PASS_FINAL) {
        int L = first_converged(V.norms, cnt, tol);
        if (L == 0) {
            if (!force) return;
            L = cnt;
        }
        ysrc = (ybase + L - 1) & 1;
    }
    extern __shared__ double sm[];
    const int n = V.n, N = V.N, K2 = n >> 1, N2 = N >> 1;
    const int K = PASS == PASS_FIX ? K2 + 4 : K2;                       // operator columns used
    const int ld = PASS == PASS_FIX ? K2 + 16 : K2;                     // operator row stride
    const int rows = PASS == PASS_FIX ? 2 * K2 + 4 : PASS == PASS_ITER ? K2 + 4 : K2;
    double* in = sm;             // [K]
    double* out = sm + K2 + 4;   // [rows]
    const int64_t j = blockIdx.x, J = V.J;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double* __restrict__ Ys = V.y[ysrc];
    double* __restrict__ Yd = V.y[ysrc ^ 1];

    if (PASS == PASS_FIX) {
        for (int u = tid; u < K; u += 256) {
            double v;
            if (u < N) v = Ys[j * K2 + N2 + u];
            else if (u < K2) v = V.z[j * K2 + N2 + (u - N)];
            else v = V.Q[j * 4 + (u - K2)];
            in[u] = v;
        }
    } else {
        for (int q = tid; q < K2; q += 256) in[q] = Ys[(q < N ? j + 1 : j - 1) * K2 + q];
    }
    __syncthreads();

    const int64_t b = V.blk[j];
    const double* __restrict__ M = PASS == PASS_FIX    ? V.xop + (size_t)b * (2 * K2 + 8) * ld
                                   : PASS == PASS_ITER ? V.rop + (size_t)b * (K2 + 8) * ld
                                                       : V.fop + (size_t)b * K2 * ld;
    for (int i0 = warp * ROWS; i0 < rows; i0 += 8 * ROWS) {
        double acc[ROWS];
#pragma unroll
        for (int r = 0; r < ROWS; ++r) acc[r] = 0.0;
        for (int k = 2 * lane; k < K; k += 64) {
            const double c0 = in[k], c1 = in[k + 1];
            double2 mrow[ROWS];
#pragma unroll
            for (int r = 0; r < ROWS; ++r)
                mrow[r] = (i0 + r < rows) ? ldg_stream2(M + (size_t)(i0 + r) * ld + k) : make_double2(0.0, 0.0);
#pragma unroll
            for (int r = 0; r < ROWS; ++r) acc[r] = fma(mrow[r].y, c1, fma(mrow[r].x, c0, acc[r]));
        }
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc[r] += __shfl_xor_sync(0xffffffffu, acc[r], o);
            if (lane == 0 && i0 + r < rows) out[i0 + r] = acc[r];
        }
    }
    __syncthreads();

    if (PASS == PASS_FIX) {
        for (int i = tid; i < K2; i += 256) {
            V.yfix[j * K2 + i] = out[i];
            V.ifix[j * K2 + i] = out[K2 + i];
        }
        if (tid < 4) V.phifix[j * 4 + tid] = out[2 * K2 + tid];
    } else if (PASS == PASS_ITER) {
        for (int i = tid; i < K2; i += 256) {
            const double v = V.yfix[j * K2 + i] + out[i];
            out[i] = v;
            Yd[j * K2 + i] = v;
        }
        if (warp == 0) {
            double d = 0.0, r = 0.0;
            if (lane < 4) {
                const double a = V.phifix[j * 4 + lane] + out[K2 + lane];
                const double old = V.phi[j * 4 + lane];
                V.phi[j * 4 + lane] = a;
                d = fabs(a - old);
                r = fabs(a);
            }
            d = warp_max(d);
            r = warp_max(r);
            if (lane == 0) {
                atomic_max_nonneg(&V.norms[2 * slot + 0], d);
                atomic_max_nonneg(&V.norms[2 * slot + 1], r);
            }
        }
        // reflecting ghost rows (reading S4): the mirror image of the edge cell's outgoing flux
        const bool gl = j == 0 && V.bcL == OCI_BC_REFLECTING, gr = j == J - 1 && V.bcR == OCI_BC_REFLECTING;
        if (gl || gr) {
            __syncthreads();
            for (int q = tid; q < K2; q += 256) {
                if (gl && q >= N) Yd[-(int64_t)K2 + q] = out[mirror_q(q, N)];
                if (gr && q < N) Yd[J * K2 + q] = out[mirror_q(q, N)];
            }
        }
    } else {
        for (int i = tid; i < K2; i += 256) V.z[j * K2 + i] = V.ifix[j * K2 + i] + out[i];
    }
}

int launch_red_gemv(const DevView& V, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force,
                    cudaStream_t s)
{
    const size_t smem = sizeof(double) * (V.n / 2 + 4 + V.n + 4);
    const unsigned grid = (unsigned)V.J;
    if (pass == PASS_FIX) oci_red_gemv_kernel<PASS_FIX, 4><<<grid, 256, smem, s>>>(V, ybase, 0, -1, tol, 0, 0);
    else if (pass == PASS_ITER) oci_red_gemv_kernel<PASS_ITER, 4><<<grid, 256, smem, s>>>(V, ybase, slot, prev_slot, tol, 0, 0);
    else oci_red_gemv_kernel<PASS_FINAL, 4><<<grid, 256, smem, s>>>(V, ybase, 0, -1, tol, cnt, force);
    return 1;
}

}  // namespace oci
