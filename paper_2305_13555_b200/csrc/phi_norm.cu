// Kernel (c): scalar flux phi = sum_m w_m psi_m per slot (eq. 18) and the two max-norms of
// the stopping rule (reading S2), with no host round trip: the norms are atomicMax'ed
// into a device slot that the NEXT launch reads (step_done).  Also refreshes the ghost rows of a
// reflecting boundary from the iterate it has just reduced (reading S4: lagged reflection).
//
// This stand-alone form serves SI, set_flux and the generic OCI path; the specialised OCI kernels
// fuse the same reduction into their epilogue.
#include "device_utils.cuh"

namespace oci {

__device__ __forceinline__ void refresh_ghost_rows(const DevView& V, double* P, int64_t j, int lane)
{
    const int n = V.n, N = V.N;
    if (j == 0 && V.bcL == OCI_BC_REFLECTING) {
        // incident on the left face for mu_m > 0 = outgoing psi_{N-1-m,.,0,L}; stored where a cell
        // j = -1 would keep its (k,R),(k+1/2,R) values
        for (int idx = lane; idx < n; idx += 32) {
            const int m = idx >> 2, s = idx & 3;
            if (m >= N / 2 && (s & 1)) P[-(int64_t)n + idx] = P[4 * (N - 1 - m) + (s - 1)];
        }
    }
    if (j == V.J - 1 && V.bcR == OCI_BC_REFLECTING) {
        for (int idx = lane; idx < n; idx += 32) {
            const int m = idx >> 2, s = idx & 3;
            if (m < N / 2 && !(s & 1)) P[V.J * n + idx] = P[(V.J - 1) * n + 4 * (N - 1 - m) + (s + 1)];
        }
    }
}

template <bool NORMS>
__global__ void __launch_bounds__(256) phi_norm_kernel(DevView V, int buf, int slot, int prev_slot, double tol)
{
    if (NORMS && step_done(V.norms, prev_slot, tol)) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int n = V.n;
    double* P = V.psi[buf];
    double dmax = 0.0, rmax = 0.0;
    for (int64_t j = (int64_t)blockIdx.x * 8 + warp; j < V.J; j += (int64_t)gridDim.x * 8) {
        const double* row = P + j * n;
        double acc = 0.0;
        for (int idx = lane; idx < n; idx += 32) acc = fma(V.w[idx >> 2], row[idx], acc);
        acc += __shfl_xor_sync(0xffffffffu, acc, 4);
        acc += __shfl_xor_sync(0xffffffffu, acc, 8);
        acc += __shfl_xor_sync(0xffffffffu, acc, 16);
        if (lane < 4) {
            const double old = V.phi[j * 4 + lane];
            V.phi[j * 4 + lane] = acc;
            dmax = fmax(dmax, fabs(acc - old));
            rmax = fmax(rmax, fabs(acc));
        }
        if (j == 0 || j == V.J - 1) refresh_ghost_rows(V, P, j, lane);
    }
    if (NORMS) {
        __shared__ double sd[8], sr[8];
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0) { sd[warp] = dmax; sr[warp] = rmax; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int q = 1; q < 8; ++q) { dmax = fmax(dmax, sd[q]); rmax = fmax(rmax, sr[q]); }
            atomic_max_nonneg(&V.norms[2 * slot + 0], dmax);
            atomic_max_nonneg(&V.norms[2 * slot + 1], rmax);
        }
    }
}

int launch_phi_norm(const DevView& V, int buf, int slot, int prev_slot, double tol, bool with_norms,
                    cudaStream_t s)
{
    int64_t blocks = (V.J + 7) / 8;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (with_norms) phi_norm_kernel<true><<<(unsigned)blocks, 256, 0, s>>>(V, buf, slot, prev_slot, tol);
    else phi_norm_kernel<false><<<(unsigned)blocks, 256, 0, s>>>(V, buf, slot, prev_slot, tol);
    return 1;
}

}  // namespace oci
