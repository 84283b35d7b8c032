// Interface-reduced OCI iteration: the same iterates as eq. (19), with the
// work that does not change inside a time step hoisted out of the iteration.
//
// Within a step only the 2N RHS rows that take an incident flux change from one iterate to the next
// (the superscript-(l) terms of eqs. 27,28); everything else of c_j is c_fix (row a2).  With
//     I = rows that receive an incident flux  ((m,1),(m,3) for mu_m<0; (m,0),(m,2) for mu_m>0)
//     O = rows a neighbour reads               (the other two slots of each angle; O(p) = I(p) ^ 1)
// and inc^(l)[j] = the 2N neighbour values cell j gathers (row a3), eq. (19) reads
//     Psi^(l+1)[j] = B^{-1} c_fix[j]  +  B^{-1}[:, I] diag|mu| inc^(l)[j]  =  Psi_fix[j] + ...
// The next iterate needs only the O rows of Psi^(l+1) (the neighbours' incident fluxes) and the
// stopping rule only phi^(l+1) = W Psi^(l+1) (eq. 18), so until the step has converged an iteration is
//     y^(l+1)[j]   = yfix[j]   + G inc^(l)[j],   G = B^{-1}[O, I] diag|mu|      (2N x 2N)
//     phi^(l+1)[j] = phifix[j] + H inc^(l)[j],   H = W B^{-1}[:, I] diag|mu|    (4 x 2N)
// a quarter of the flops (shared block) or bytes (per-cell blocks) of the full apply.  Once the last
// iteration L is known, the remaining rows follow from the same inc^(L-1):
//     Psi^(L)[j][I] = ifix[j] + F inc^(L-1)[j],  F = B^{-1}[I, I] diag|mu|      (2N x 2N)
// Per step: one full apply (Psi_fix, by the ordinary apply kernels with a zero gather coefficient), L
// reduced iterations, one finalisation.  Up to rounding order the iterates are those of the plain
// method, so iteration counts and fluxes are held to the same parity tolerances as the full form.
//
// Packing.  p = 2m + h, h = 0 for the k slot and 1 for the k+1/2 slot: O(p) = 4m + (mu_m<0 ? 2h : 2h+1).
// With ascending mu the first N entries of y[j] leave through the left face and feed cell j-1, the last N
// feed cell j+1:  inc[j][p] = y[j+1][p] (p < N),  y[j-1][p] (p >= N), and row I(p) is multiplied by
// |mu_m| = coef[I(p)].  The y buffers carry ghost rows -1 and J like the Psi buffers do.
//
// This file: the operator packing (setup), the Psi <-> y data movement, and the generic kernels of the
// reduced iteration (a batched GEMV with one operator per distinct block: HBM-bound when every cell
// has its own block, the fallback for shared blocks of sizes the tensor-core kernels do not take).
#include "device_utils.cuh"

namespace oci {

namespace {

__device__ __forceinline__ int o_row(int p, int N)   // full index of packed outgoing row p
{
    const int m = p >> 1, h = p & 1;
    return 4 * m + ((m < N / 2) ? 2 * h : 2 * h + 1);
}

__device__ __forceinline__ double2 ldg_stream2(const double* p)
{
    double2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}

}  // namespace

// First iteration index (1-based) whose norms satisfy the stopping rule, 0 if none of the `cnt` queued
// iterations did.  Slots past the last executed iteration are still zero from the memset, and
// converged(tol, 0, 0) holds for tol >= 0, so the scan must stop at the first hit.
__device__ __forceinline__ int first_converged(const unsigned long long* __restrict__ norms, int cnt, double tol)
{
    for (int i = 0; i < cnt; ++i) {
        const double d = __longlong_as_double((long long)__ldcg(norms + 2 * i + 0));
        const double r = __longlong_as_double((long long)__ldcg(norms + 2 * i + 1));
        if (converged(tol, d, r)) return i + 1;
    }
    return 0;
}

// ---- setup: G, H, F of every distinct block from its inverse (one CTA per block)
__global__ void __launch_bounds__(256) pack_operators_kernel(DevView V)
{
    const int n = V.n, N = V.N, K2 = n >> 1, MO = K2 + 8;
    const int64_t b = blockIdx.x;
    const double* __restrict__ Bi = V.binv + (size_t)b * n * n;
    double* __restrict__ R = V.rop + (size_t)b * MO * K2;
    double* __restrict__ F = V.fop + (size_t)b * K2 * K2;
    for (int e = threadIdx.x; e < MO * K2; e += blockDim.x) {
        const int q = e / K2, p = e - q * K2;
        const int ip = o_row(p, N) ^ 1;
        const double cf = V.coef[ip];
        double val = 0.0;
        if (q < K2) {
            val = Bi[(size_t)o_row(q, N) * n + ip] * cf;
            F[(size_t)q * K2 + p] = Bi[(size_t)(o_row(q, N) ^ 1) * n + ip] * cf;
        } else if (q < K2 + 4) {
            const int s = q - K2;
            double a = 0.0;
            for (int m = 0; m < N; ++m) a = fma(V.w[m], Bi[(size_t)(4 * m + s) * n + ip], a);
            val = a * cf;
        }
        R[e] = val;
    }
}

int launch_pack_operators(const DevView& V, cudaStream_t s)
{
    pack_operators_kernel<<<(unsigned)V.nblk, 256, 0, s>>>(V);
    return 1;
}

// ---- y[ybuf] <- outgoing rows of Psi[buf], ghost rows included (after set_flux / si_step)
__global__ void __launch_bounds__(256) pack_y_kernel(DevView V, int buf, int ybuf)
{
    const int n = V.n, N = V.N, K2 = n >> 1;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (V.J + 2) * K2) return;
    const int64_t row = t / K2 - 1;                       // -1 .. J
    const int p = (int)(t % K2);
    const double v = V.psi[buf][row * n + o_row(p, N)];
    V.y[ybuf][row * K2 + p] = v;
    // vacuum / incident ghost rows are constant: both buffers hold them (reflecting ones are rewritten
    // by every iteration)
    if (row < 0 || row >= V.J) V.y[ybuf ^ 1][row * K2 + p] = v;
}

int launch_pack_y(const DevView& V, int buf, int ybuf, cudaStream_t s)
{
    const int64_t tot = (V.J + 2) * (V.n >> 1);
    pack_y_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(V, buf, ybuf);
    return 1;
}

// ---- Psi_fix (full layout, Psi[buf]) -> yfix (O rows), ifix (I rows), both packed
__global__ void __launch_bounds__(256) split_fix_kernel(DevView V, int buf)
{
    // thread = (cell, angle): one 32-byte row segment in, two 16-byte packed pairs out
    const int N = V.N;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= V.J * N) return;
    const int m = (int)(t % N);
    const double2 a = *reinterpret_cast<const double2*>(V.psi[buf] + t * 4);
    const double2 b = *reinterpret_cast<const double2*>(V.psi[buf] + t * 4 + 2);
    const double2 even = make_double2(a.x, b.x), odd = make_double2(a.y, b.y);   // slots (0,2), (1,3)
    const bool neg = m < N / 2;                                                  // mu_m < 0: O = slots 0,2
    *reinterpret_cast<double2*>(V.yfix + t * 2) = neg ? even : odd;
    *reinterpret_cast<double2*>(V.ifix + t * 2) = neg ? odd : even;
}

int launch_split_fix(const DevView& V, int buf, cudaStream_t s)
{
    const int64_t tot = V.J * V.N;
    split_fix_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(V, buf);
    return 1;
}

// ---- reduced iteration / finalisation as a batched GEMV, one CTA per cell.
// FINAL = false:  y^(l+1)[j] = yfix[j] + G_b inc,  phi^(l+1)[j] = phifix[j] + H_b inc, norms, ghost rows of y.
// FINAL = true :  Psi^(L)[j][I] = ifix[j] + F_b inc^(L-1),  Psi^(L)[j][O] = y^(L)[j], ghost rows of Psi;
//                 L is found on the device from the norm slots of the `cnt` queued iterations
//                 (`force`: this chunk ends at max_iters, finalise after cnt iterations if none converged).
template <bool FINAL, int ROWS>
__global__ void __launch_bounds__(256) oci_red_percell_kernel(DevView V, int ybase, int slot, int prev_slot, double tol,
                                                              int pdst, int cnt, int force)
{
    int ysrc = ybase;
    if (!FINAL) {
        if (step_done(V.norms, prev_slot, tol)) return;
    } else {
        int L = first_converged(V.norms, cnt, tol);
        if (L == 0) {
            if (!force) return;
            L = cnt;
        }
        ysrc = (ybase + L - 1) & 1;
    }
    extern __shared__ double sm[];
    const int n = V.n, N = V.N, K2 = n >> 1;
    double* inc = sm;            // [K2]
    double* out = sm + K2;       // [K2 + 4]
    const int64_t j = blockIdx.x, J = V.J;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double* __restrict__ Ys = V.y[ysrc];
    double* __restrict__ Yd = V.y[ysrc ^ 1];

    for (int p = tid; p < K2; p += 256) inc[p] = Ys[(p < N ? j + 1 : j - 1) * K2 + p];
    __syncthreads();

    const int64_t b = V.blk[j];
    const double* __restrict__ M = FINAL ? V.fop + (size_t)b * K2 * K2 : V.rop + (size_t)b * (K2 + 8) * K2;
    const int rows = FINAL ? K2 : K2 + 4;
    for (int i0 = warp * ROWS; i0 < rows; i0 += 8 * ROWS) {
        double acc[ROWS];
#pragma unroll
        for (int r = 0; r < ROWS; ++r) acc[r] = 0.0;
        for (int k = 2 * lane; k < K2; k += 64) {
            const double c0 = inc[k], c1 = inc[k + 1];
            double2 mrow[ROWS];
#pragma unroll
            for (int r = 0; r < ROWS; ++r)
                mrow[r] = (i0 + r < rows) ? ldg_stream2(M + (size_t)(i0 + r) * K2 + k) : make_double2(0.0, 0.0);
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

    if (!FINAL) {
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
            for (int p = tid; p < K2; p += 256) {
                const int mir = 2 * (N - 1 - (p >> 1)) + (p & 1);
                if (gl && p >= N) Yd[-(int64_t)K2 + p] = out[mir];
                if (gr && p < N) Yd[J * K2 + p] = out[mir];
            }
        }
    } else {
        double* __restrict__ P = V.psi[pdst];
        for (int i = tid; i < K2; i += 256) {
            const int o = o_row(i, N);
            P[j * n + (o ^ 1)] = V.ifix[j * K2 + i] + out[i];
            P[j * n + o] = Yd[j * K2 + i];
        }
        const bool gl = j == 0 && V.bcL == OCI_BC_REFLECTING, gr = j == J - 1 && V.bcR == OCI_BC_REFLECTING;
        if (gl || gr) {
            for (int p = tid; p < K2; p += 256) {
                const int mir = 2 * (N - 1 - (p >> 1)) + (p & 1);
                if (gl && p >= N) P[-(int64_t)n + o_row(p, N)] = Yd[mir];
                if (gr && p < N) P[J * n + o_row(p, N)] = Yd[(J - 1) * K2 + mir];
            }
        }
    }
}

int launch_red_percell(const DevView& V, int ysrc, int slot, int prev_slot, double tol, cudaStream_t s)
{
    const size_t smem = sizeof(double) * (V.n + 4);
    oci_red_percell_kernel<false, 4><<<(unsigned)V.J, 256, smem, s>>>(V, ysrc, slot, prev_slot, tol, 0, 0, 0);
    return 1;
}

int launch_red_percell_final(const DevView& V, int ybase, int pdst, int cnt, int force, double tol, cudaStream_t s)
{
    const size_t smem = sizeof(double) * (V.n + 4);
    oci_red_percell_kernel<true, 4><<<(unsigned)V.J, 256, smem, s>>>(V, ybase, 0, -1, tol, pdst, cnt, force);
    return 1;
}

}  // namespace oci
