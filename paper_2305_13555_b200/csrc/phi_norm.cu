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
__global__ void __launch_bounds__(256, 2) phi_norm_kernel(DevView V, int buf, int slot, int prev_slot, double tol)
{
    if (NORMS && step_done(V.norms, prev_slot, tol)) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int n = V.n;
    constexpr int CP = 8;
    double* P = V.psi[buf];
    const double* __restrict__ Pr = P;
    double dmax = 0.0, rmax = 0.0;
    // CP cells per warp pass; a lane owns the 16-byte units idx = 2*lane (+64 i) of each row, i.e. slots
    // (0,1) of an angle on even lanes and (2,3) on odd lanes.  Every load of a pass (rows and the old
    // phi) is unconditional (cell index clamped) so that all of them are in flight together: the
    // kernel is bound by memory latency x bytes in flight, not by arithmetic.
    for (int64_t j0 = ((int64_t)blockIdx.x * 8 + warp) * CP; j0 < V.J; j0 += (int64_t)gridDim.x * 8 * CP) {
        double a0[CP], a1[CP];
        double2 oldv[CP];
#pragma unroll
        for (int c = 0; c < CP; ++c) {
            a0[c] = a1[c] = 0.0;
            const int64_t j = (j0 + c < V.J) ? j0 + c : V.J - 1;
            oldv[c] = (NORMS && lane < 2) ? *reinterpret_cast<const double2*>(V.phi + j * 4 + 2 * lane) : make_double2(0.0, 0.0);
        }
#pragma unroll 2
        for (int idx = 2 * lane; idx < n; idx += 64) {
            const double wq = V.w[idx >> 2];
#pragma unroll
            for (int c = 0; c < CP; ++c) {
                const int64_t j = (j0 + c < V.J) ? j0 + c : V.J - 1;
                const double2 v = *reinterpret_cast<const double2*>(Pr + j * n + idx);
                a0[c] = fma(wq, v.x, a0[c]);
                a1[c] = fma(wq, v.y, a1[c]);
            }
        }
#pragma unroll
        for (int c = 0; c < CP; ++c) {
#pragma unroll
            for (int o = 2; o < 32; o <<= 1) {
                a0[c] += __shfl_xor_sync(0xffffffffu, a0[c], o);
                a1[c] += __shfl_xor_sync(0xffffffffu, a1[c], o);
            }
        }
#pragma unroll
        for (int c = 0; c < CP; ++c) {
            const int64_t j = j0 + c;
            if (j < V.J) {
                if (lane < 2) {
                    *reinterpret_cast<double2*>(V.phi + j * 4 + 2 * lane) = make_double2(a0[c], a1[c]);
                    dmax = nanmax(dmax, nanmax(fabs(a0[c] - oldv[c].x), fabs(a1[c] - oldv[c].y)));
                    rmax = nanmax(rmax, nanmax(fabs(a0[c]), fabs(a1[c])));
                }
                if (j == 0 || j == V.J - 1) refresh_ghost_rows(V, P, j, lane);
            }
        }
    }
    if (NORMS) {
        __shared__ double sd[8], sr[8];
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0) { sd[warp] = dmax; sr[warp] = rmax; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int q = 1; q < 8; ++q) { dmax = nanmax(dmax, sd[q]); rmax = nanmax(rmax, sr[q]); }
            atomic_max_nonneg(&V.norms[2 * slot + 0], dmax);
            atomic_max_nonneg(&V.norms[2 * slot + 1], rmax);
        }
    }
}

int launch_phi_norm(const DevView& V, int buf, int slot, int prev_slot, double tol, bool with_norms,
                    cudaStream_t s)
{
    int64_t blocks = (V.J + 63) / 64;
    if (blocks > (int64_t)V.sm_count * 16) blocks = (int64_t)V.sm_count * 16;
    if (with_norms) phi_norm_kernel<true><<<(unsigned)blocks, 256, 0, s>>>(V, buf, slot, prev_slot, tol);
    else phi_norm_kernel<false><<<(unsigned)blocks, 256, 0, s>>>(V, buf, slot, prev_slot, tol);
    return launched(1);
}

}  // namespace oci
