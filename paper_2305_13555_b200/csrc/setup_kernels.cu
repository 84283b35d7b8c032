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

// a0: one CTA per block; element (i,k) of B.
__global__ void form_blocks_kernel(DevView V)
{
    const int64_t b = blockIdx.x;
    const int64_t r = V.rep[b];
    const int n = V.n;
    const double h = V.dx[r], sig = V.sig[r], sigs = V.sigs[r];
    double* B = V.binv + (size_t)b * n * n;
    for (int e = threadIdx.x; e < n * n; e += blockDim.x) {
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

// a1: in-place Gauss-Jordan inversion with partial (row) pivoting, one CTA per matrix.
// The matrix stays where the inverse will live (global memory / L2); the pivot row and the
// multiplier column of the current step are staged in shared memory.
template <int THREADS>
__global__ void __launch_bounds__(THREADS) invert_blocks_kernel(DevView V)
{
    extern __shared__ double sm[];
    const int n = V.n;
    double* rowk = sm;                 // [n] scaled pivot row
    double* colk = sm + n;             // [n] multipliers
    int* perm = (int*)(sm + 2 * n);    // [n]
    __shared__ double red_val[THREADS / 32];
    __shared__ int red_idx[THREADS / 32];
    __shared__ int piv_row;

    double* A = V.binv + (size_t)blockIdx.x * n * n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = THREADS / 32;

    for (int k = 0; k < n; ++k) {
        // --- pivot search over rows k..n-1 of column k (ties -> lowest row, deterministic)
        double best = -1.0;
        int bi = n;
        for (int i = k + tid; i < n; i += THREADS) {
            double a = fabs(A[(size_t)i * n + k]);
            if (a > best) { best = a; bi = i; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            double ob = __shfl_xor_sync(0xffffffffu, best, o);
            int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
        }
        if (lane == 0) { red_val[warp] = best; red_idx[warp] = bi; }
        __syncthreads();
        if (tid == 0) {
            double bb = red_val[0];
            int ii = red_idx[0];
            for (int q = 1; q < NW; ++q)
                if (red_val[q] > bb || (red_val[q] == bb && red_idx[q] < ii)) { bb = red_val[q]; ii = red_idx[q]; }
            piv_row = ii;
            perm[k] = ii;
            if (!(bb > 0.0)) {                                           // singular: report, stop
                atomicMax(V.flags, (int)blockIdx.x + 1);
                piv_row = n;
            }
        }
        __syncthreads();
        const int p = piv_row;
        if (p >= n) return;            // singular (uniform across the CTA)
        // --- swap rows k and p; stage the (unscaled) pivot row
        for (int c = tid; c < n; c += THREADS) {
            double top = A[(size_t)k * n + c];
            double pr = A[(size_t)p * n + c];
            rowk[c] = pr;
            if (p != k) A[(size_t)p * n + c] = top;
        }
        __syncthreads();
        const double pivinv = 1.0 / rowk[k];
        __syncthreads();
        // --- multipliers (column k, after the swap); scale the pivot row
        for (int i = tid; i < n; i += THREADS) {
            colk[i] = (i == k) ? 0.0 : A[(size_t)i * n + k];
            rowk[i] = (i == k) ? pivinv : rowk[i] * pivinv;
        }
        __syncthreads();
        // --- rank-1 update of every row; column k becomes the inverse's column
        for (int i = warp; i < n; i += NW) {
            double* Ai = A + (size_t)i * n;
            if (i == k) {
                for (int c = lane; c < n; c += 32) Ai[c] = rowk[c];
            } else {
                const double f = colk[i];
                for (int c = lane; c < n; c += 32) {
                    double a = (c == k) ? 0.0 : Ai[c];
                    Ai[c] = a - f * rowk[c];
                }
            }
        }
        __syncthreads();
    }
    // --- undo the row interchanges as column interchanges, in reverse order
    for (int k = n - 1; k >= 0; --k) {
        const int p = perm[k];
        if (p != k) {
            for (int i = tid; i < n; i += THREADS) {
                double t = A[(size_t)i * n + k];
                A[(size_t)i * n + k] = A[(size_t)i * n + p];
                A[(size_t)i * n + p] = t;
            }
        }
        __syncthreads();
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

int launch_form_and_invert(const DevView& V, cudaStream_t s)
{
    form_blocks_kernel<<<(unsigned)V.nblk, 256, 0, s>>>(V);
    constexpr int T = 512;
    size_t smem = sizeof(double) * 2 * V.n + sizeof(int) * V.n;
    invert_blocks_kernel<T><<<(unsigned)V.nblk, T, smem, s>>>(V);
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
