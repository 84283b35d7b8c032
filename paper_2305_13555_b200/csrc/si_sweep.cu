// Kernel (d): the source-iteration comparator (eqs. 12-18).  "SI sweeps ... are readily
// parallelized over the number of angles": one thread per angle walks the cells in its
// direction of travel; the scattering source comes from phi^(l) (row d1), the upstream edge values
// from THIS sweep's previous cell (row d2; no (l) on the neighbour term of eqs. 14,17), reflecting
// boundaries from the previous iterate (reading S4, via the ghost rows).
//
// The 4x4 systems are pre-inverted per (block, angle).  With x = Ainv (base + |mu| e_in) the two
// carried values obey a 2x2 affine recurrence, so only two dependent FMAs per cell sit on the
// sequential chain; everything else (loads, Ainv*base) is off the chain and batched for ILP.
#include "device_utils.cuh"

namespace oci {

// d1: qs[j][s] = (h/4) Sigma_s phi^(l)[j][s]
__global__ void si_scatter_source_kernel(DevView V, int prev_slot, double tol)
{
    if (step_done(V.norms, prev_slot, tol)) return;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= V.J * 4) return;
    const int64_t j = t >> 2;
    V.qs[t] = V.dx[j] * 0.25 * V.sigs[j] * V.phi[t];
}

template <int U, bool SHARED_BLOCK>
__global__ void __launch_bounds__(32) si_sweep_kernel(DevView V, int buf, int prev_slot, double tol)
{
    if (step_done(V.norms, prev_slot, tol)) return;
    const int m = blockIdx.x * 32 + threadIdx.x;
    if (m >= V.N) return;
    const int n = V.n;
    const int64_t J = V.J;
    double* __restrict__ P = V.psi[buf];
    const double mu = V.mu[m];
    const bool pos = mu > 0.0;
    const double amu = fabs(mu);
    // mu>0: rows 0,2 receive the incident flux (k, k+1/2) and rows 1,3 leave the cell; mu<0: mirrored
    double in_k = pos ? P[-(int64_t)n + 4 * m + 1] : P[J * n + 4 * m + 0];
    double in_h = pos ? P[-(int64_t)n + 4 * m + 3] : P[J * n + 4 * m + 2];

    double Ai[16];
    if (SHARED_BLOCK) {
#pragma unroll
        for (int i = 0; i < 16; ++i) Ai[i] = V.ainv4[(size_t)m * 16 + i];
    }

    for (int64_t t0 = 0; t0 < J; t0 += U) {
        double y[U][4], G[U][4][2];
        // ---- off-chain: loads and y = Ainv * base for U cells
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t t = t0 + u;
            if (t < J) {
                const int64_t j = pos ? t : J - 1 - t;
                const double2 c01 = *reinterpret_cast<const double2*>(V.cfix + j * n + 4 * m);
                const double2 c23 = *reinterpret_cast<const double2*>(V.cfix + j * n + 4 * m + 2);
                const double2 q01 = *reinterpret_cast<const double2*>(V.qs + j * 4);
                const double2 q23 = *reinterpret_cast<const double2*>(V.qs + j * 4 + 2);
                const double b[4] = {c01.x + q01.x, c01.y + q01.y, c23.x + q23.x, c23.y + q23.y};
                if (!SHARED_BLOCK) {
                    const double* a = V.ainv4 + ((size_t)V.blk[j] * V.N + m) * 16;
#pragma unroll
                    for (int i = 0; i < 16; i += 2) {
                        const double2 v2 = *reinterpret_cast<const double2*>(a + i);
                        Ai[i] = v2.x; Ai[i + 1] = v2.y;
                    }
                }
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    y[u][r] = Ai[4 * r + 0] * b[0] + Ai[4 * r + 1] * b[1] + Ai[4 * r + 2] * b[2] + Ai[4 * r + 3] * b[3];
                    G[u][r][0] = amu * (pos ? Ai[4 * r + 0] : Ai[4 * r + 1]);
                    G[u][r][1] = amu * (pos ? Ai[4 * r + 2] : Ai[4 * r + 3]);
                }
            }
        }
        // ---- the sequential chain: two dependent FMAs per cell
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t t = t0 + u;
            if (t < J) {
                const int64_t j = pos ? t : J - 1 - t;
                double x[4];
#pragma unroll
                for (int r = 0; r < 4; ++r) x[r] = fma(G[u][r][1], in_h, fma(G[u][r][0], in_k, y[u][r]));
                in_k = pos ? x[1] : x[0];
                in_h = pos ? x[3] : x[2];
                *reinterpret_cast<double2*>(P + j * n + 4 * m) = make_double2(x[0], x[1]);
                *reinterpret_cast<double2*>(P + j * n + 4 * m + 2) = make_double2(x[2], x[3]);
            }
        }
    }
}

int launch_si_iteration(const DevView& V, int buf, int slot, int prev_slot, double tol, cudaStream_t s)
{
    int64_t tot = V.J * 4;
    si_scatter_source_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(V, prev_slot, tol);
    unsigned blocks = (unsigned)((V.N + 31) / 32);
    if (V.nblk == 1) si_sweep_kernel<8, true><<<blocks, 32, 0, s>>>(V, buf, prev_slot, tol);
    else si_sweep_kernel<4, false><<<blocks, 32, 0, s>>>(V, buf, prev_slot, tol);
    launch_phi_norm(V, buf, slot, prev_slot, tol, true, s);
    return 3;
}

}  // namespace oci
