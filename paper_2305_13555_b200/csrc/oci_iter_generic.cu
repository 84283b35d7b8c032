// Kernel (b), generic shared-block form: Psi^(l+1) = B^{-1} c for all cells at once as the dense
// contraction [cells x n] = [cells x n] . [n x n]^T on the fp64 tensor pipe (DMMA), with the RHS
// assembly fused into the producer:
//     c[j][k] = c_fix[j][k] + coef[k] * Psi^(l)[j + dir(k)][k ^ 1]
// (eqs. 27,28: rows (m,0),(m,2) of mu_m>0 take mu_m * psi_{m,.,j-1,R}; rows (m,1),(m,3) of
// mu_m<0 take |mu_m| * psi_{m,.,j+1,L}; with ascending mu, k < n/2 looks right (dir=+1), k >= n/2 looks
// left (dir=-1); the partner slot is k^1; ghost rows -1 and J carry the boundary data).
//
// This version works for any n = 4N: simple single-buffered shared-memory tiles.  The specialised
// kernels in oci_iter_shared_*.cu are the fast paths for the benchmark block sizes.
#include "device_utils.cuh"

namespace oci {

namespace {
constexpr int TM = 32;    // cells per CTA
constexpr int TN = 128;   // outputs per CTA (8 warps x 16)
constexpr int KC = 32;    // k per shared-memory chunk
constexpr int LD = KC + 4;   // padded row: stride = 4 (mod 16) doubles -> conflict-free fragment loads
}

__global__ void __launch_bounds__(256) oci_iter_generic_kernel(DevView V, int src, int prev_slot, double tol)
{
    if (step_done(V.norms, prev_slot, tol)) return;
    __shared__ double As[TM][LD];
    __shared__ double Bs[TN][LD];
    const int n = V.n, half = n >> 1;
    const double* __restrict__ Pold = V.psi[src];
    double* __restrict__ Pnew = V.psi[src ^ 1];
    const int64_t j0 = (int64_t)blockIdx.x * TM;
    const int i0 = blockIdx.y * TN;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g4 = lane >> 2, t4 = lane & 3;

    double acc[4][2][2];
#pragma unroll
    for (int g = 0; g < 4; ++g)
#pragma unroll
        for (int t = 0; t < 2; ++t) acc[g][t][0] = acc[g][t][1] = 0.0;

    for (int kc = 0; kc < n; kc += KC) {
        // ---- producer: assemble the RHS chunk (a3 + a4) straight from global memory
#pragma unroll
        for (int q = 0; q < TM * KC / 256; ++q) {
            const int e = tid + 256 * q;
            const int r = e / KC, kk = e % KC;
            const int k = kc + kk;
            const int64_t j = j0 + r;
            double val = 0.0;
            if (j < V.J && k < n) {
                const int64_t jn = (k < half) ? j + 1 : j - 1;
                val = fma(V.coef[k], Pold[jn * n + (k ^ 1)], V.cfix[j * n + k]);
            }
            As[r][kk] = val;
        }
#pragma unroll
        for (int q = 0; q < TN * KC / 256; ++q) {
            const int e = tid + 256 * q;
            const int r = e / KC, kk = e % KC;
            const int i = i0 + r, k = kc + kk;
            Bs[r][kk] = (i < n && k < n) ? V.binv[(size_t)i * n + k] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int ks = 0; ks < KC / 4; ++ks) {
            double a[4], b[2];
#pragma unroll
            for (int g = 0; g < 4; ++g) a[g] = As[8 * g + g4][4 * ks + t4];
#pragma unroll
            for (int t = 0; t < 2; ++t) b[t] = Bs[16 * warp + 8 * t + g4][4 * ks + t4];
#pragma unroll
            for (int g = 0; g < 4; ++g)
#pragma unroll
                for (int t = 0; t < 2; ++t) dmma(acc[g][t][0], acc[g][t][1], a[g], b[t]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        const int64_t j = j0 + 8 * g + g4;
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            const int i = i0 + 16 * warp + 8 * t + 2 * t4;
            if (j < V.J && i < n)
                *reinterpret_cast<double2*>(Pnew + j * n + i) = make_double2(acc[g][t][0], acc[g][t][1]);
        }
    }
}

int launch_oci_generic(const DevView& V, int src, int prev_slot, double tol, cudaStream_t s)
{
    dim3 grid((unsigned)((V.J + TM - 1) / TM), (unsigned)((V.n + TN - 1) / TN));
    oci_iter_generic_kernel<<<grid, 256, 0, s>>>(V, src, prev_slot, tol);
    return launched(1);
}

}  // namespace oci
