// Kernel (b), per-cell form: every cell has its own inverse (heterogeneous slab), so the apply is a
// batched GEMV  Psi^(l+1)[j] = B_j^{-1} c[j]  and the inverses (n*n*8 bytes per cell) are streamed from
// HBM once per iteration: bandwidth-bound.  One CTA per cell; the RHS is assembled into shared
// memory (rows a3, a4), the matrix is read with 128-bit loads, rows are reduced with warp shuffles;
// the scalar flux and the convergence norms (row a6, kernel c) are fused into the epilogue.
#include "device_utils.cuh"

namespace oci {

__device__ __forceinline__ double2 ldg_stream(const double* p)
{
    double2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}

template <int ROWS>   // rows per warp pass
__global__ void __launch_bounds__(256) oci_iter_percell_kernel(DevView V, int src, int slot, int prev_slot,
                                                               double tol)
{
    if (step_done(V.norms, prev_slot, tol)) return;
    extern __shared__ double sm[];
    const int n = V.n, half = n >> 1;
    double* cs = sm;          // [n]  RHS
    double* out = sm + n;     // [n]  result
    const int64_t j = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double* __restrict__ Pold = V.psi[src];
    double* __restrict__ Pnew = V.psi[src ^ 1];

    for (int k = tid; k < n; k += 256) {
        const int64_t jn = (k < half) ? j + 1 : j - 1;
        cs[k] = fma(V.coef[k], Pold[jn * n + (k ^ 1)], V.cfix[j * n + k]);
    }
    __syncthreads();

    const double* __restrict__ M = V.binv + (size_t)V.blk[j] * n * n;
    for (int i0 = warp * ROWS; i0 < n; i0 += 8 * ROWS) {
        double acc[ROWS];
#pragma unroll
        for (int r = 0; r < ROWS; ++r) acc[r] = 0.0;
        for (int k = 2 * lane; k < n; k += 64) {
            const double c0 = cs[k], c1 = cs[k + 1];
            double2 mrow[ROWS];
#pragma unroll
            for (int r = 0; r < ROWS; ++r)
                mrow[r] = (i0 + r < n) ? ldg_stream(M + (size_t)(i0 + r) * n + k) : make_double2(0.0, 0.0);
#pragma unroll
            for (int r = 0; r < ROWS; ++r) acc[r] = fma(mrow[r].y, c1, fma(mrow[r].x, c0, acc[r]));
        }
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc[r] += __shfl_xor_sync(0xffffffffu, acc[r], o);
            if (lane == 0 && i0 + r < n) out[i0 + r] = acc[r];
        }
    }
    __syncthreads();
    for (int i = tid; i < n; i += 256) Pnew[j * n + i] = out[i];

    // ---- fused kernel (c): phi, norms (warp 0), reading the result from shared memory
    if (warp == 0) {
        double a = 0.0;
        for (int idx = lane; idx < n; idx += 32) a = fma(V.w[idx >> 2], out[idx], a);
        a += __shfl_xor_sync(0xffffffffu, a, 4);
        a += __shfl_xor_sync(0xffffffffu, a, 8);
        a += __shfl_xor_sync(0xffffffffu, a, 16);
        double d = 0.0, r = 0.0;
        if (lane < 4) {
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
    // ---- reflecting ghost rows (reading S4), from the freshly written rows
    if ((j == 0 && V.bcL == OCI_BC_REFLECTING) || (j == V.J - 1 && V.bcR == OCI_BC_REFLECTING)) {
        const int N = V.N;
        for (int idx = tid; idx < n; idx += 256) {
            const int m = idx >> 2, s = idx & 3;
            if (j == 0 && V.bcL == OCI_BC_REFLECTING && m >= N / 2 && (s & 1))
                Pnew[-(int64_t)n + idx] = out[4 * (N - 1 - m) + (s - 1)];
            if (j == V.J - 1 && V.bcR == OCI_BC_REFLECTING && m < N / 2 && !(s & 1))
                Pnew[V.J * n + idx] = out[4 * (N - 1 - m) + (s + 1)];
        }
    }
}

int launch_oci_percell(const DevView& V, int src, int slot, int prev_slot, double tol, cudaStream_t s)
{
    size_t smem = sizeof(double) * 2 * V.n;
    oci_iter_percell_kernel<4><<<(unsigned)V.J, 256, smem, s>>>(V, src, slot, prev_slot, tol);
    return launched(1);
}

}  // namespace oci
