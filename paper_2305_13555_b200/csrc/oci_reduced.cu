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

// ---- setup: X, G, H, F of every distinct block from its inverse (gridDim.x = blocks, gridDim.y CTAs share a block)
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
    const int tid = blockIdx.y * blockDim.x + threadIdx.x, nth = gridDim.y * blockDim.x;
    for (int e = tid; e < MO * K2; e += nth) {
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
    for (int e = tid; e < MF * KF; e += nth) {
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
    const unsigned fy = V.nblk >= V.sm_count ? 1u : (unsigned)((2 * V.sm_count + V.nblk - 1) / V.nblk);
    pack_operators_kernel<<<dim3((unsigned)V.nblk, fy), 256, 0, s>>>(V);
    return launched(1);
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
    return launched(1);
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
    return launched(1);
}

// ---- the three passes as a batched GEMV (PASS_* of oci_internal.h), HBM-bound when every cell has its own
// operator.  EVERY WARP IS AN INDEPENDENT WORKER: the (cell, group of GR operator rows) pairs of the whole
// problem form one long stream that is cut into equal contiguous pieces, one per warp; a warp keeps the
// input vector of its current cell in a private strip of shared memory, streams its GR rows with 16-byte
// non-allocating loads (all GR x 16 B per lane in flight together), reduces them by shuffle, and lane r
// finishes row r.  No CTA barrier anywhere, so the 32 resident warps of an SM drift apart and HBM always
// sees requests; equal pieces of a fine-grained stream leave no tail wave (config 5 is only 3.5 waves of
// one-CTA-per-cell).
// FIX  :  [yfix | ifix | phifix][j] = X_b [psi_{k-1/2}[j]; Q[j]],  psi_{k-1/2} from y[ybase][j], z[j]
// ITER :  y^(l+1)[j] = yfix[j] + G_b inc,  phi^(l+1)[j] = phifix[j] + H_b inc, norms, ghost rows of y
// FINAL:  z[j] = ifix[j] + F_b inc^(L-1); L is found on the device from the norm slots of the `cnt`
//         queued iterations (`force`: this chunk ends at max_iters, finalise after cnt iterations if
//         none converged); y^(L) is already in place.
template <int PASS, int GR>
__global__ void __launch_bounds__(256, 2) oci_red_gemv_kernel(DevView V, int ybase, int slot, int prev_slot, double tol,
                                                           int cnt, int force)
{
    extern __shared__ double sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    int ysrc = ybase;
    if (PASS == PASS_ITER) {
        if (step_done(V.norms, prev_slot, tol)) return;
    } else if (PASS == PASS_FINAL) {
        // the last iteration of this chunk of launches, with all loads of the scan in flight at once
        int L = 0;
        for (int i0 = 0; i0 < cnt && L == 0; i0 += 32) {
            const int i = i0 + lane;
            bool hit = false;
            if (i < cnt) {
                const double d = __longlong_as_double((long long)__ldcg(V.norms + 2 * i + 0));
                const double r = __longlong_as_double((long long)__ldcg(V.norms + 2 * i + 1));
                hit = stop_now(tol, d, r);
            }
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            if (m) L = i0 + __ffs(m);
        }
        if (L == 0) {
            if (!force) return;
            L = cnt;
        }
        ysrc = (ybase + L - 1) & 1;
    }
    if (PASS == PASS_FIX) clear_step_state(V);
    const int n = V.n, N = V.N, K2 = n >> 1, N2 = N >> 1;
    const int K = PASS == PASS_FIX ? K2 + 4 : K2;                       // operator columns used
    const int ld = PASS == PASS_FIX ? K2 + 16 : K2;                     // operator row stride
    const int rows = PASS == PASS_FIX ? 2 * K2 + 4 : PASS == PASS_ITER ? K2 + 4 : K2;
    const int gpc = (rows + GR - 1) / GR;                               // row groups per cell
    const int64_t J = V.J, G = J * gpc;
    const int64_t wid = (int64_t)blockIdx.x * nwarp + warp, nw = (int64_t)gridDim.x * nwarp;
    const int64_t g_begin = G * wid / nw, g_end = G * (wid + 1) / nw;
    double* in = sm + (size_t)warp * (K2 + 8);                          // this warp's input vector [K] (+ zero pad)
    // ITER: `cnt` > 1 iterations run inside this one (cooperative) launch, separated by a grid-wide barrier;
    // iteration l reads y[(ybase + l) & 1] (through L2: other SMs wrote it) and reports its norms in slot + l
    const int nloop = PASS == PASS_ITER ? (cnt > 1 ? cnt : 1) : 1;
    const double* Ys = V.y[ysrc];
    double* Yd = V.y[ysrc ^ 1];

    // The (row group, 64-column slice) steps of this warp form one flat sequence; the 16-byte loads of step
    // s+1 are issued before step s is consumed, so a warp always has GR x 512 B of its stream in flight.
    // FIX: the four Q columns are not worth a slice of their own: the lane that finishes a row adds them
    const int KS_ = PASS == PASS_FIX ? K2 : K;                          // columns streamed in slices
    const int KI = (KS_ + 63) / 64;                                     // column slices per row
    const int64_t S = (g_end - g_begin) * KI;
    auto op_base = [&](int64_t g) -> const double* {
        const int64_t j = g / gpc;
        const int i0 = (int)(g - j * gpc) * GR;
        const int64_t b = V.blk[j];
        return (PASS == PASS_FIX    ? V.xop + (size_t)b * (2 * K2 + 8) * ld
                : PASS == PASS_ITER ? V.rop + (size_t)b * (K2 + 8) * ld
                                    : V.fop + (size_t)b * K2 * ld) + (size_t)i0 * ld;
    };
    auto load_step = [&](double2 (&dst)[GR], int64_t g, int ki) {
        const int64_t j = g / gpc;
        const int i0 = (int)(g - j * gpc) * GR;
        const double* __restrict__ M = op_base(g);
        const int k = 2 * lane + 64 * ki;
#pragma unroll
        for (int r = 0; r < GR; ++r)
            dst[r] = (i0 + r < rows && k < KS_) ? ldg_stream2(M + (size_t)r * ld + k) : make_double2(0.0, 0.0);
    };
    double2 cur[GR], nxt[GR];
    double acc[GR];
    double add = 0.0, old = 0.0;
    double2 qc0 = make_double2(0.0, 0.0), qc1 = make_double2(0.0, 0.0);
    if (S > 0) load_step(nxt, g_begin, 0);
  for (int l = 0; l < nloop; ++l) {
    if (PASS == PASS_ITER) {
        Ys = V.y[(ybase + l) & 1];
        Yd = V.y[(ybase + l + 1) & 1];
    }
    double dmax = 0.0, rmax = 0.0;
    int64_t jcur = -1;
    int64_t g = g_begin;
    int ki = 0;
    for (int64_t st = 0; st < S; ++st) {
#pragma unroll
        for (int r = 0; r < GR; ++r) cur[r] = nxt[r];
        {
            int kin = ki + 1;
            int64_t gn = g;
            if (kin == KI) { kin = 0; ++gn; }
            if (st + 1 < S) load_step(nxt, gn, kin);
        }
        const int64_t j = g / gpc;
        const int i0 = (int)(g - j * gpc) * GR;
        const int i = i0 + lane;
        const bool mine = lane < GR && i < rows;       // lane r < GR finishes row i0 + r
        if (ki == 0) {
            if (j != jcur) {
                __syncwarp();
                if (PASS == PASS_FIX) {
                    for (int u = lane; u < K; u += 32)
                        in[u] = u < N ? __ldcg(Ys + j * K2 + N2 + u) : u < K2 ? V.z[j * K2 + N2 + (u - N)] : V.Q[j * 4 + (u - K2)];
                } else {
                    for (int q = lane; q < K2; q += 32) in[q] = __ldcg(Ys + (q < N ? j + 1 : j - 1) * K2 + q);
                }
                if (lane < 4) in[K + lane] = 0.0;       // columns past K read as zero (the operator loads are zero there)
                __syncwarp();
                jcur = j;
            }
#pragma unroll
            for (int r = 0; r < GR; ++r) acc[r] = 0.0;
            // the additive operand of this lane's row, requested now, consumed after the last slice
            add = 0.0;
            if (mine) {
                if (PASS == PASS_FIX) {
                    const double* __restrict__ qrow = op_base(g) + (size_t)lane * ld + K2;
                    qc0 = ldg_stream2(qrow);
                    qc1 = ldg_stream2(qrow + 2);
                }
                if (PASS == PASS_FINAL) add = V.ifix[j * K2 + i];
                if (PASS == PASS_ITER) {
                    if (i < K2) add = V.yfix[j * K2 + i];
                    else { add = V.phifix[j * 4 + (i - K2)]; old = __ldcg(V.phi + j * 4 + (i - K2)); }
                }
            }
        }
        {
            const int k = 2 * lane + 64 * ki;
            const double2 c = k < KS_ ? *reinterpret_cast<const double2*>(in + k) : make_double2(0.0, 0.0);
#pragma unroll
            for (int r = 0; r < GR; ++r) acc[r] = fma(cur[r].y, c.y, fma(cur[r].x, c.x, acc[r]));
        }
        if (ki == KI - 1) {
            double o = 0.0;
#pragma unroll
            for (int r = 0; r < GR; ++r) {
#pragma unroll
                for (int sh = 16; sh > 0; sh >>= 1) acc[r] += __shfl_xor_sync(0xffffffffu, acc[r], sh);
                if (lane == r) o = acc[r];
            }
            if (mine) {
                if (PASS == PASS_FIX) {
                    o = fma(qc1.y, in[K2 + 3], fma(qc1.x, in[K2 + 2], fma(qc0.y, in[K2 + 1], fma(qc0.x, in[K2], o))));
                    if (i < K2) V.yfix[j * K2 + i] = o;
                    else if (i < 2 * K2) V.ifix[j * K2 + (i - K2)] = o;
                    else V.phifix[j * 4 + (i - 2 * K2)] = o;
                } else if (PASS == PASS_FINAL) {
                    V.z[j * K2 + i] = add + o;
                } else if (i < K2) {
                    const double v = add + o;
                    Yd[j * K2 + i] = v;
                    // reflecting ghost rows (reading S4): the mirror image of the edge cell's outgoing flux
                    if (j == 0 && i < N && V.bcL == OCI_BC_REFLECTING) Yd[-(int64_t)K2 + mirror_q(i, N)] = v;
                    if (j == J - 1 && i >= N && V.bcR == OCI_BC_REFLECTING) Yd[J * K2 + mirror_q(i, N)] = v;
                } else {
                    const double a = add + o;
                    V.phi[j * 4 + (i - K2)] = a;
                    dmax = nanmax(dmax, fabs(a - old));
                    rmax = nanmax(rmax, fabs(a));
                }
            }
            ki = 0;
            ++g;
        } else {
            ++ki;
        }
    }
    if (PASS == PASS_ITER) {
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0 && g_end > g_begin) {
            atomic_max_nonneg(&V.norms[2 * (slot + l) + 0], dmax);
            atomic_max_nonneg(&V.norms[2 * (slot + l) + 1], rmax);
        }
        if (nloop > 1) {
            // the operator does not depend on the iterate: the first step of the next iteration is requested
            // before the grid-wide barrier, so HBM stays busy across it
            if (l + 1 < nloop && S > 0) load_step(nxt, g_begin, 0);
            __threadfence();
            __syncthreads();
            if (threadIdx.x == 0) {
                unsigned int* bar = reinterpret_cast<unsigned int*>(V.flags) + 8;
                atomicAdd(bar, 1u);
                const unsigned int target = (unsigned int)(l + 1) * gridDim.x;
                unsigned int seen;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory");
                } while (seen < target);
            }
            __syncthreads();
            const bool stop = step_done(V.norms, slot + l, tol) || l + 1 == nloop;   // a7: every CTA takes the same decision
            if (stop && blockIdx.x == 0 && threadIdx.x == 0) publish_step(V, l + 1, slot + l);
            if (stop) break;
        }
    }
  }
}

int launch_red_gemv(const DevView& V, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force,
                    cudaStream_t s)
{
    constexpr int GR = 8;
    const int K2 = V.n / 2;
    const int rows = pass == PASS_FIX ? 2 * K2 + 4 : pass == PASS_ITER ? K2 + 4 : K2;
    const int64_t G = V.J * ((rows + GR - 1) / GR);
    // warps per CTA: 8 unless the private input vectors would not fit in shared memory (huge N)
    int nwarp = 8;
    while (nwarp > 1 && (size_t)nwarp * (K2 + 8) * 8 > 100 * 1024) nwarp >>= 1;
    const size_t smem = sizeof(double) * (size_t)nwarp * (K2 + 8);
    const int sm_count = V.sm_count;
    // one wave: every CTA resident, the stream cut into equal pieces
    int per_sm = 1;
    if (pass == PASS_FIX) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, oci_red_gemv_kernel<PASS_FIX, GR>, nwarp * 32, smem);
    else if (pass == PASS_ITER) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, oci_red_gemv_kernel<PASS_ITER, GR>, nwarp * 32, smem);
    else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, oci_red_gemv_kernel<PASS_FINAL, GR>, nwarp * 32, smem);
    if (per_sm < 1) per_sm = 1;
    int64_t ctas = (G + nwarp - 1) / nwarp;                 // at least one row group per warp
    if (ctas > (int64_t)sm_count * per_sm) ctas = (int64_t)sm_count * per_sm;
    const unsigned grid = (unsigned)ctas, block = (unsigned)nwarp * 32;
    if (pass == PASS_FIX) oci_red_gemv_kernel<PASS_FIX, GR><<<grid, block, smem, s>>>(V, ybase, 0, -1, tol, 0, 0);
    else if (pass == PASS_ITER && cnt > 1) {
        // `cnt` iterations in one launch with a grid-wide barrier between them: the grid is one resident wave
        DevView Vv = V;
        int zero = 0;
        void* args[] = {&Vv, &ybase, &slot, &prev_slot, &tol, &cnt, &zero};
        cudaLaunchCooperativeKernel((const void*)oci_red_gemv_kernel<PASS_ITER, GR>, dim3(grid), dim3(block), args, smem, s);
    } else if (pass == PASS_ITER) oci_red_gemv_kernel<PASS_ITER, GR><<<grid, block, smem, s>>>(V, ybase, slot, prev_slot, tol, 0, 0);
    else oci_red_gemv_kernel<PASS_FINAL, GR><<<grid, block, smem, s>>>(V, ybase, 0, -1, tol, cnt, force);
    return launched(1);
}

cudaError_t oci_red_gemv_opt_in()
{
    constexpr int GR = 8;
    cudaError_t e = cudaSuccess;
    const auto at = cudaFuncAttributeMaxDynamicSharedMemorySize;
    if ((e = cudaFuncSetAttribute(oci_red_gemv_kernel<PASS_FIX, GR>, at, 100 * 1024)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(oci_red_gemv_kernel<PASS_ITER, GR>, at, 100 * 1024)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(oci_red_gemv_kernel<PASS_FINAL, GR>, at, 100 * 1024)) != cudaSuccess)
        return e;
    return e;
}

}  // namespace oci
