// Kernel (a): form B = A - S per distinct (dx, Sigma, Sigma_s) and invert it with partial pivoting
// (eqs. 13,16,20-22 P:114-159; `gesv` P:208), the SI 4x4 inverses,
// and the small per-step / per-call data-movement kernels (a2 fixed RHS, set_flux, pack).
#include "device_utils.cuh"

namespace oci {

// The local 4x4 of eqs. (13)/(16) with rows 3,4 repaired (readings G1-G3):
// diagonal (|mu| + h Sigma)/2, off-diagonals with the signed mu, alpha = h/(2 v dt).
__device__ __forceinline__ void local4x4(double mu, double h, double sig, double v, double dt, double A[16])
{
    const double d = (fabs(mu) + h * sig) * 0.5;
    const double al = h / (2.0 * v * dt);
    const double al2 = h / (v * dt);
    A[0] = d;         A[1] = 0.5 * mu;  A[2] = al;        A[3] = 0.0;
    A[4] = -0.5 * mu; A[5] = d;         A[6] = 0.0;       A[7] = al;
    A[8] = -al2;      A[9] = 0.0;       A[10] = al2 + d;  A[11] = 0.5 * mu;
    A[12] = 0.0;      A[13] = -al2;     A[14] = -0.5 * mu; A[15] = al2 + d;
}

// a0: element (i,k) of B; gridDim.x = blocks, gridDim.y CTAs share a block.
__global__ void form_blocks_kernel(DevView V)
{
    const int64_t b = blockIdx.x;
    const int64_t r = V.rep[b];
    const int n = V.n;
    const double h = V.dx[r], sig = V.sig[r], sigs = V.sigs[r];
    double* B = V.binv + (size_t)b * n * n;
    for (int e = blockIdx.y * blockDim.x + threadIdx.x; e < n * n; e += gridDim.y * blockDim.x) {
        const int i = e / n, k = e - i * n;
        const int m = i >> 2, s = i & 3, mk = k >> 2, sk = k & 3;
        double val = 0.0;
        if (m == mk) {
            double A[16];
            local4x4(V.mu[m], h, sig, V.v, V.dt, A);
            val = A[4 * s + sk];
        }
        if (s == sk) val -= h * sigs * 0.25 * V.w[mk];   // eq. (22): S couples equal slots
        B[e] = val;
    }
}

// a1: in-place BLOCKED Gauss-Jordan inversion with partial (row) pivoting (the paper's `gesv`, hoisted out of
// both loops).  The unblocked algorithm (pivot = largest entry of column k among rows >= k, row interchange, the
// pivot row scaled, every other row eliminated, column k overwritten by the inverse's column; the interchanges
// undone at the end as column interchanges in reverse order) touches the whole matrix once per column.  Blocked:
// columns are taken NB at a time ("panel").
//   1. the panel (n x NB) is factored by the unblocked algorithm restricted to its own columns, one or a few rows per
//      thread held in registers, pivot row broadcast through shared memory: the pivots are those of the unblocked
//      algorithm because every earlier panel's update has already been applied to these columns;
//   2. what the NB steps do to any column x outside the panel is linear and the same for all of them:
//      x <- x + (W - E_K) (P x)_K, with P the panel's row interchanges, K its row range and W = the panel after step 1
//      (the steps applied to the unit vectors e_K: exactly what the in-place algorithm leaves in the panel columns).
//      So the rest of the matrix is updated by ONE rank-NB product per panel, C <- C + W R with R = rows K of P C and
//      rows K of C replaced by W_K R: an [n x NB].[NB x n] contraction on the fp64 tensor pipe (DMMA), operands in
//      shared memory, C streamed through L2.
// 2 n^3 flop per matrix as before, but n / NB passes over the matrix instead of n.
// A "team" of T CTAs shares one matrix (T = SMs / blocks when there are fewer blocks than SMs: config 4 has ONE block):
// rank 0 factors the panel, all ranks split the outside columns in chunks, a team-wide barrier (counter in global
// memory, cooperative launch) after each half.  With T = 1 (config 5: 4096 blocks) a team is a CTA.
template <int NB, int RPT>
__global__ void __launch_bounds__(256, 1) invert_blocked_kernel(DevView V, int T, int chunk)
{
    extern __shared__ unsigned char inv_smem[];
    const int n = V.n;
    constexpr int WLD = NB + 4;                       // pitch of W: 4 (mod 16) -> conflict-free DMMA A fragments
    const int RLD = chunk + 4;                        // pitch of R / D: 4 (mod 16) (chunk is a multiple of 16)
    double* Ws = reinterpret_cast<double*>(inv_smem);                 // [n][WLD]
    double* Rs = Ws + (size_t)n * WLD;                                // [NB][RLD]  rows K of the (interchanged) outside columns
    double* Ds = Rs + (size_t)NB * RLD;                               // [NB][RLD]  rows displaced out of K by the interchanges
    double* pivbuf = Ds + (size_t)NB * RLD;                           // [2][2][NB] pivot row / row k, double buffered
    double* red_val = pivbuf + 4 * NB;                                // [2][8]
    int* red_idx = reinterpret_cast<int*>(red_val + 16);              // [2][8]
    int* rowmap = red_idx + 16;                                       // [n]
    int* perm_s = rowmap + n;                                         // [NB] pivot rows of the current panel
    __shared__ int dead_s;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int b = blockIdx.x / T, tr = blockIdx.x % T;
    double* __restrict__ A = V.binv + (size_t)b * n * n;
    int* __restrict__ perm = V.perm + (size_t)b * n;
    unsigned int* tbar = reinterpret_cast<unsigned int*>(V.team_bar) + b;
    unsigned int phase = 0;
    auto team_barrier = [&]() {
        __syncthreads();
        if (T > 1) {
            ++phase;
            if (tid == 0) {
                __threadfence();
                atomicAdd(tbar, 1u);
                unsigned int seen;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(tbar) : "memory");
                } while (seen < phase * (unsigned)T);
            }
            __syncthreads();
        }
    };
    if (tid == 0) dead_s = 0;
    for (int i = tid; i < n; i += 256) rowmap[i] = i;
    __syncthreads();

    for (int k0 = 0; k0 < n; k0 += NB) {
        const int nbe = n - k0 < NB ? n - k0 : NB;                    // width of this panel (a multiple of 8)
        // ---------------------------------------------------------------- 1. panel factorisation (team rank 0)
        if (tr == 0 && !dead_s) {
            double prow[RPT][NB];
#pragma unroll
            for (int q = 0; q < RPT; ++q) {
                const int r = tid + 256 * q;
#pragma unroll
                for (int c = 0; c < NB; ++c) prow[q][c] = (r < n && c < nbe) ? A[(size_t)r * n + k0 + c] : 0.0;
            }
#pragma unroll
            for (int j = 0; j < NB; ++j) {
                if (j < nbe) {                                        // uniform over the CTA
                    const int k = k0 + j, pb = j & 1;
                    // pivot: largest |entry| of column k among rows >= k, ties -> lowest row (deterministic)
                    double best = -1.0;
                    int bi = n;
#pragma unroll
                    for (int q = 0; q < RPT; ++q) {
                        const int r = tid + 256 * q;
                        const double a = fabs(prow[q][j]);
                        if (r >= k && r < n && (a > best || (a == best && r < bi))) { best = a; bi = r; }
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        const double ob = __shfl_xor_sync(0xffffffffu, best, o);
                        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                        if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
                    }
                    if (lane == 0) { red_val[pb * 8 + warp] = best; red_idx[pb * 8 + warp] = bi; }
                    __syncthreads();
                    best = red_val[pb * 8];
                    int p = red_idx[pb * 8];
#pragma unroll
                    for (int w8 = 1; w8 < 8; ++w8) {
                        const double ob = red_val[pb * 8 + w8];
                        const int oi = red_idx[pb * 8 + w8];
                        if (ob > best || (ob == best && oi < p)) { best = ob; p = oi; }
                    }
                    if (!(best > 0.0)) {                              // singular (or NaN): report, stop the arithmetic
                        if (tid == 0) { atomicMax(V.flags, b + 1); dead_s = 1; }
                        p = k;
                    }
                    if (tid == 0) perm_s[j] = p;
                    // rows k and p change places: their owners publish them
                    double* pv = pivbuf + pb * 2 * NB;                // [0][.] = old row p (the pivot row), [1][.] = old row k
#pragma unroll
                    for (int q = 0; q < RPT; ++q) {
                        const int r = tid + 256 * q;
                        if (r == p) {
#pragma unroll
                            for (int c = 0; c < NB; ++c) pv[c] = prow[q][c];
                        }
                        if (r == k) {
#pragma unroll
                            for (int c = 0; c < NB; ++c) pv[NB + c] = prow[q][c];
                        }
                    }
                    __syncthreads();
                    const double pivinv = 1.0 / pv[j];
#pragma unroll
                    for (int q = 0; q < RPT; ++q) {
                        const int r = tid + 256 * q;
                        if (r == k) {                                  // the scaled pivot row; column k becomes the inverse's column
#pragma unroll
                            for (int c = 0; c < NB; ++c) prow[q][c] = (c == j) ? pivinv : pv[c] * pivinv;
                        } else {
                            if (r == p) {                              // the old row k has moved here
#pragma unroll
                                for (int c = 0; c < NB; ++c) prow[q][c] = pv[NB + c];
                            }
                            const double f = prow[q][j];
#pragma unroll
                            for (int c = 0; c < NB; ++c) prow[q][c] = (c == j) ? -f * pivinv : prow[q][c] - f * (pv[c] * pivinv);
                        }
                    }
                }
            }
            // W -> the panel columns (global: the other ranks read it there) and this CTA's shared memory
#pragma unroll
            for (int q = 0; q < RPT; ++q) {
                const int r = tid + 256 * q;
                if (r < n) {
#pragma unroll
                    for (int c = 0; c < NB; ++c) {
                        if (c < nbe) A[(size_t)r * n + k0 + c] = prow[q][c];
                        Ws[(size_t)r * WLD + c] = prow[q][c];
                    }
                }
            }
            __syncthreads();
            if (tid < nbe) perm[k0 + tid] = perm_s[tid];
        }
        team_barrier();
        const bool dead = *reinterpret_cast<volatile int*>(V.flags) != 0;
        // ---------------------------------------------------------------- 2. rank-NB update of the outside columns
        if (!dead) {
            if (tr != 0) {
                for (int e = tid; e < n * NB; e += 256) {
                    const int r = e / NB, c = e - r * NB;
                    Ws[(size_t)r * WLD + c] = c < nbe ? __ldcg(A + (size_t)r * n + k0 + c) : 0.0;
                }
                if (tid < nbe) perm_s[tid] = __ldcg(perm + k0 + tid);
            }
            __syncthreads();
            // where every affected row comes from after the panel's interchanges, applied in order
            if (tid == 0) {
                for (int jj = 0; jj < nbe; ++jj) {
                    const int k = k0 + jj, p = perm_s[jj];
                    const int t = rowmap[k]; rowmap[k] = rowmap[p]; rowmap[p] = t;
                }
            }
            __syncthreads();
            const int nchunks = (n + chunk - 1) / chunk;
            for (int cc = tr; cc < nchunks; cc += T) {
                const int c0 = cc * chunk;
                const int cw = n - c0 < chunk ? n - c0 : chunk;        // columns in this chunk (a multiple of 8)
                // rows K of the interchanged matrix -> Rs; rows pushed out of K -> Ds (panel columns: dead, never used)
                for (int e = tid; e < nbe * cw; e += 256) {
                    const int jj = e / cw, c = e - jj * cw;
                    Rs[jj * RLD + c] = __ldcg(A + (size_t)rowmap[k0 + jj] * n + c0 + c);
                    const int p = perm_s[jj];
                    Ds[jj * RLD + c] = __ldcg(A + (size_t)rowmap[p] * n + c0 + c);
                }
                __syncthreads();
                for (int e = tid; e < nbe * cw; e += 256) {
                    const int jj = e / cw, c = e - jj * cw;
                    const int p = perm_s[jj];
                    const int col = c0 + c;
                    if ((p < k0 || p >= k0 + nbe) && (col < k0 || col >= k0 + nbe)) A[(size_t)p * n + col] = Ds[jj * RLD + c];
                }
                __syncthreads();
                // C[:, chunk] <- C + W R (rows K: W_K R), 32 x 32 tiles per warp, DMMA.8x8x4
                const int g4 = lane >> 2, t4 = lane & 3;
                const int ntr = (n + 31) / 32, ntc = (cw + 31) / 32;
                for (int tile = warp; tile < ntr * ntc; tile += 8) {
                    const int tr0 = (tile / ntc) * 32, tc0 = (tile % ntc) * 32;
                    double acc[4][4][2];
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        const int r = tr0 + 8 * g + g4;
                        const bool inK = r >= k0 && r < k0 + nbe;
#pragma unroll
                        for (int t = 0; t < 4; ++t) {
                            const int c = tc0 + 8 * t + 2 * t4;
                            double2 v = make_double2(0.0, 0.0);
                            if (r < n && c < cw && !inK) v = __ldcg(reinterpret_cast<const double2*>(A + (size_t)r * n + c0 + c));
                            acc[g][t][0] = v.x;
                            acc[g][t][1] = v.y;
                        }
                    }
                    for (int ks = 0; ks < nbe / 4; ++ks) {
                        double a[4], bq[4];
#pragma unroll
                        for (int g = 0; g < 4; ++g) {
                            const int r = tr0 + 8 * g + g4;
                            a[g] = r < n ? Ws[(size_t)r * WLD + 4 * ks + t4] : 0.0;
                        }
#pragma unroll
                        for (int t = 0; t < 4; ++t) {
                            const int c = tc0 + 8 * t + g4;
                            bq[t] = c < cw ? Rs[(4 * ks + t4) * RLD + c] : 0.0;
                        }
#pragma unroll
                        for (int g = 0; g < 4; ++g)
#pragma unroll
                            for (int t = 0; t < 4; ++t) dmma(acc[g][t][0], acc[g][t][1], a[g], bq[t]);
                    }
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        const int r = tr0 + 8 * g + g4;
#pragma unroll
                        for (int t = 0; t < 4; ++t) {
                            const int c = tc0 + 8 * t + 2 * t4, col = c0 + c;
                            if (r < n && c < cw && (col < k0 || col >= k0 + nbe))
                                *reinterpret_cast<double2*>(A + (size_t)r * n + col) = make_double2(acc[g][t][0], acc[g][t][1]);
                        }
                    }
                }
                __syncthreads();
            }
            // the row map is the identity again for the next panel
            if (tid == 0) {
                for (int jj = nbe - 1; jj >= 0; --jj) {
                    const int k = k0 + jj, p = perm_s[jj];
                    const int t = rowmap[k]; rowmap[k] = rowmap[p]; rowmap[p] = t;
                }
            }
        }
        team_barrier();
    }
    if (*reinterpret_cast<volatile int*>(V.flags) != 0) return;
    // ---------------------------------------------------------------- 3. undo the row interchanges as column interchanges
    // applying "swap columns k, perm[k]" for k = n-1 .. 0 to a row is a gather: final[c] = row[src[c]]
    int* src = rowmap;                                               // identity at this point
    if (tid == 0) {
        for (int k = n - 1; k >= 0; --k) {
            const int p = __ldcg(perm + k);
            const int t = src[k]; src[k] = src[p]; src[p] = t;
        }
    }
    __syncthreads();
    double* rowbuf = Ws + (size_t)warp * n;                          // one row per warp (n <= n * WLD / 8 always)
    for (int r = tr * 8 + warp; r < n; r += 8 * T) {
        for (int c = lane; c < n; c += 32) rowbuf[c] = __ldcg(A + (size_t)r * n + c);
        __syncwarp();
        for (int c = lane; c < n; c += 32) A[(size_t)r * n + c] = rowbuf[src[c]];
        __syncwarp();
    }
}

// (A_m)^{-1}, 4x4, per (block, angle): Gauss-Jordan with partial pivoting on [A | I].
__global__ void ainv4_kernel(DevView V)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= V.nblk * V.N) return;
    const int64_t b = t / V.N;
    const int m = (int)(t - b * V.N);
    const int64_t r = V.rep[b];
    double A[16], I[16];
    local4x4(V.mu[m], V.dx[r], V.sig[r], V.v, V.dt, A);
#pragma unroll
    for (int i = 0; i < 16; ++i) I[i] = (i % 5 == 0) ? 1.0 : 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        int p = k;
        double best = fabs(A[4 * k + k]);
#pragma unroll
        for (int i = k + 1; i < 4; ++i) {
            double a = fabs(A[4 * i + k]);
            if (a > best) { best = a; p = i; }
        }
#pragma unroll
        for (int i = k + 1; i < 4; ++i) {
            if (i == p) {
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    double t1 = A[4 * k + c]; A[4 * k + c] = A[4 * i + c]; A[4 * i + c] = t1;
                    double t2 = I[4 * k + c]; I[4 * k + c] = I[4 * i + c]; I[4 * i + c] = t2;
                }
            }
        }
        const double pinv = 1.0 / A[4 * k + k];
#pragma unroll
        for (int c = 0; c < 4; ++c) { A[4 * k + c] *= pinv; I[4 * k + c] *= pinv; }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            if (i != k) {
                const double f = A[4 * i + k];
#pragma unroll
                for (int c = 0; c < 4; ++c) { A[4 * i + c] -= f * A[4 * k + c]; I[4 * i + c] -= f * I[4 * k + c]; }
            }
        }
    }
    double* out = V.ainv4 + (size_t)t * 16;
#pragma unroll
    for (int i = 0; i < 16; ++i) out[i] = I[i];
}

namespace {
struct InvCfg { int nb, chunk, T; size_t smem; };
// panel width by block size (rows per thread x panel width = 64 doubles in registers), team size, column chunk
InvCfg inv_config(const DevView& V)
{
    InvCfg c{};
    c.nb = V.n <= 512 ? 32 : V.n <= 1024 ? 16 : 8;
    c.T = 1;
    c.chunk = 128;
    if (V.nblk < V.sm_count) {
        // fewer blocks than SMs: several CTAs per block, narrower column chunks so that there is something to share
        c.chunk = 64;
        const int nchunks = (V.n + c.chunk - 1) / c.chunk;
        int T = V.sm_count / (int)V.nblk;
        if (T > nchunks) T = nchunks;
        c.T = T < 1 ? 1 : T;
    }
    c.smem = sizeof(double) * ((size_t)V.n * (c.nb + 4) + 2 * (size_t)c.nb * (c.chunk + 4) + 4 * c.nb + 16) + sizeof(int) * (16 + V.n + c.nb) + 64;
    return c;
}
template <int NB, int RPT>
int launch_invert(const DevView& V, const InvCfg& c, cudaStream_t s)
{
    const unsigned grid = (unsigned)(V.nblk * c.T);
    if (c.T > 1) {
        DevView Vv = V;
        int T = c.T, chunk = c.chunk;
        void* args[] = {&Vv, &T, &chunk};
        cudaLaunchCooperativeKernel((const void*)invert_blocked_kernel<NB, RPT>, dim3(grid), dim3(256), args, c.smem, s);
    } else {
        invert_blocked_kernel<NB, RPT><<<grid, 256, c.smem, s>>>(V, 1, c.chunk);
    }
    return launched(1);
}
}  // namespace

cudaError_t oci_setup_opt_in()
{
    const auto at = cudaFuncAttributeMaxDynamicSharedMemorySize;
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(invert_blocked_kernel<32, 1>, at, 226 * 1024)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(invert_blocked_kernel<32, 2>, at, 226 * 1024)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(invert_blocked_kernel<16, 4>, at, 226 * 1024)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(invert_blocked_kernel<8, 8>, at, 226 * 1024)) != cudaSuccess)
        return e;
    return cudaSuccess;
}

int launch_form_and_invert(const DevView& V, cudaStream_t s)
{
    // a0: element (i,k) of every B; a few CTAs per block when there are few blocks
    const unsigned fy = V.nblk >= V.sm_count ? 1u : (unsigned)((V.sm_count + V.nblk - 1) / V.nblk);
    form_blocks_kernel<<<dim3((unsigned)V.nblk, fy), 256, 0, s>>>(V);
    const InvCfg c = inv_config(V);
    if (c.T > 1) cudaMemsetAsync(V.team_bar, 0, sizeof(int) * (size_t)V.nblk, s);
    int k = 0;
    if (V.n <= 256) k = launch_invert<32, 1>(V, c, s);
    else if (V.n <= 512) k = launch_invert<32, 2>(V, c, s);
    else if (V.n <= 1024) k = launch_invert<16, 4>(V, c, s);
    else k = launch_invert<8, 8>(V, c, s);
    if (k < 0) return k;
    int64_t tot = V.nblk * V.N;
    ainv4_kernel<<<(unsigned)((tot + 127) / 128), 128, 0, s>>>(V);
    return launched(3);
}

// set_flux: seed the iterate from the corner values at the previous time edge (reading S3):
// slots (k,L),(k+1/2,L) <- L and (k,R),(k+1/2,R) <- R; constant ghost rows (vacuum / incident).
__global__ void set_flux_kernel(DevView V, const double* __restrict__ edge, int buf)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int n = V.n;
    if (t < V.J * n) {
        const int64_t j = t / n;
        const int idx = (int)(t - j * n);
        const int m = idx >> 2, s = idx & 3;
        const double val = edge[(j * V.N + m) * 2 + (s & 1)];
        V.psi[0][t] = val;
        V.psi[1][t] = val;
    }
    if (t < n) {   // ghost rows: incident value in every slot, or 0 (reflecting is refreshed by kernel c)
        const double gl = (V.bcL == OCI_BC_INCIDENT_ISOTROPIC) ? V.bcLv : 0.0;
        const double gr = (V.bcR == OCI_BC_INCIDENT_ISOTROPIC) ? V.bcRv : 0.0;
        for (int b = 0; b < 2; ++b) {
            V.psi[b][-(int64_t)n + t] = gl;
            V.psi[b][V.J * n + t] = gr;
        }
    }
}

int launch_set_flux(const DevView& V, const double* d_psi_edge, int buf, cudaStream_t s)
{
    int64_t tot = V.J * V.n;
    set_flux_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(V, d_psi_edge, buf);
    return launched(1);
}

// a2: c_fix[j][4m+s] = (h/4) Q[j][s] + (s<2 ? alpha * psi_{k-1/2}[j][m][s] : 0), where psi_{k-1/2} is the
// time-edge half (slots 2,3) of the iterate the previous step ended on: this read IS the commit (a8).
__global__ void __launch_bounds__(256) cfix_kernel(DevView V, int buf)
{
    // thread = (cell j, angle m): one 16-byte load of the time-edge pair, two 16-byte stores
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int N = V.N;
    if (t >= V.J * N) return;
    const int64_t j = t / N;
    const double h = V.dx[j];
    const double q4 = h * 0.25, al = h / (2.0 * V.v * V.dt);
    const double2 q01 = *reinterpret_cast<const double2*>(V.Q + j * 4);
    const double2 q23 = *reinterpret_cast<const double2*>(V.Q + j * 4 + 2);
    const double2 e = *reinterpret_cast<const double2*>(V.psi[buf] + t * 4 + 2);
    // same operation order as one thread per element: val = h/4 Q; val += alpha psi (s < 2)
    *reinterpret_cast<double2*>(V.cfix + t * 4) = make_double2(q4 * q01.x + al * e.x, q4 * q01.y + al * e.y);
    *reinterpret_cast<double2*>(V.cfix + t * 4 + 2) = make_double2(q4 * q23.x, q4 * q23.y);
}

int launch_cfix(const DevView& V, int buf, cudaStream_t s)
{
    int64_t tot = V.J * V.N;
    cfix_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(V, buf);
    return launched(1);
}

}  // namespace oci
