// One-launch time step for SMALL shared-block problems (configs 1 and 2: launch-latency bound): the whole reduced step
// of oci_reduced.cu - FIX, every ITER iteration with the stopping rule, FINAL - inside ONE kernel running on ONE
// thread-block cluster, the state resident in (distributed) shared memory for the whole step.
//
// The three-pass path costs a small problem three launches and, per iteration, a grid-wide barrier through global
// memory plus a round trip of the iterate through L2 (about 5 us per iteration at config 2 for 1.2 MFLOP of work).
// Here a cluster of C <= 8 CTAs splits the cells into contiguous ranges; each CTA keeps, in its shared memory, the three
// operators (X, [G; H], F, transposed), both buffers of its part of the iterate y with one ghost row on either side,
// yfix, ifix, phifix and phi.  Per iteration:
//   compute (thread = (cell, 4 operator rows), lanes = cells: the input row comes from shared memory conflict free
//   (odd pitch), the operator as broadcast 32-byte loads) -> publish this CTA's two max-norms into every CTA's shared
//   memory (DSMEM stores) -> ONE hardware cluster barrier -> ghost rows of the new iterate from the neighbour CTAs'
//   edge rows (DSMEM loads) or the boundary condition, and the stopping decision from the C published pairs, taken
//   identically by every thread of the cluster.
// No global-memory traffic inside the loop except the (d, r) pair of every iteration for the host (row a7: it still
// reads the norm slots once per step to learn the iteration count).  Sums run in a fixed order and the norms are exact
// maxima, so a step is reproducible bit for bit.  The arithmetic is the dense method's: the same operators as the other
// families of the reduced form, applied with DFMA (at these sizes a step is latency, not throughput).
//
// Not served: per-cell blocks, OCI_BC_HALO faces (sharded slabs), problems whose state does not fit a cluster's shared
// memory or that are large enough for the three-pass kernels to win; oci_step falls back to those by itself.  If a step
// does not converge within the 64 iterations one launch runs, the kernel leaves y, yfix, ifix, phifix and phi in
// global memory exactly as FIX + 64 ITER launches would have and the three-pass kernels continue from there.
#include <cooperative_groups.h>

#include "device_utils.cuh"

namespace cg = cooperative_groups;

namespace oci {

namespace {

constexpr int SM_MAX_THREADS = 1024;                       // CTA size is chosen at launch: 256 (tiny problems) or 1024
constexpr int SM_R = 4;                                    // operator rows per thread item

struct SmallLayout {                                       // offsets in doubles inside a CTA's dynamic shared memory
    int Jc, P, K2;
    int opx, opr, opf, y0, y1, yfix, ifix, zin, qin, phifix, phi, red, pub, total;
};

__host__ __device__ inline SmallLayout small_layout(int N, int Jc)
{
    SmallLayout L{};
    const int K2 = 2 * N;
    L.Jc = Jc;
    L.K2 = K2;
    L.P = K2 + 1;                                          // odd pitch: lanes = cells read a column without bank conflicts
    int o = 0;
    auto take = [&](int n) { const int at = o; o += (n + 3) & ~3; return at; };   // 32-byte aligned pieces
    L.opx = take((K2 + 4) * (2 * K2 + 4));                 // X^T  [K2+4 inputs][2K2+4 rows]
    L.opr = take(K2 * (K2 + 4));                           // [G; H]^T  [K2][K2+4]
    L.opf = take(K2 * K2);                                 // F^T  [K2][K2]
    L.y0 = take((Jc + 2) * L.P);                           // iterate, buffer 0, rows -1 .. Jc
    L.y1 = take((Jc + 2) * L.P);
    L.yfix = take(Jc * L.P);                               // also the staging area of z (FINAL)
    L.ifix = take(Jc * L.P);
    L.zin = take(Jc * (N + 1));                            // the k+1/2 run of z (FIX input)
    L.qin = take(Jc * 4);
    L.phifix = take(Jc * 4);
    L.phi = take(Jc * 4);
    L.red = take(2 * (SM_MAX_THREADS / 32));
    L.pub = take(2 * 8 * 2);                               // [parity][rank][d, r] published by every CTA of the cluster
    L.total = o;
    return L;
}

}  // namespace

__global__ void __launch_bounds__(SM_MAX_THREADS, 1) oci_red_small_kernel(DevView V, int ybase, double tol, int cnt, int force)
{
    extern __shared__ __align__(32) double ssm[];
    cg::cluster_group cluster = cg::this_cluster();
    const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    const int N = V.N, K2 = 2 * N, N2 = N >> 1;
    const int J = (int)V.J;
    const int Jc = (J + C - 1) / C;
    const SmallLayout L = small_layout(N, Jc);
    const int j0 = rank * Jc;
    const int nc = J - j0 < Jc ? (J - j0 > 0 ? J - j0 : 0) : Jc;          // cells of this CTA (the launcher keeps it > 0)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int SM_THREADS = (int)blockDim.x;
    const int P = L.P;
    double* opx = ssm + L.opx;
    double* opr = ssm + L.opr;
    double* opf = ssm + L.opf;
    double* ybuf[2] = {ssm + L.y0 + P, ssm + L.y1 + P};                   // row 0 of either buffer (ghost rows at -1, nc)
    double* yfix = ssm + L.yfix;
    double* ifix = ssm + L.ifix;
    double* zin = ssm + L.zin;
    double* qin = ssm + L.qin;
    double* phifix = ssm + L.phifix;
    double* phi = ssm + L.phi;
    double* red = ssm + L.red;
    double* pub = ssm + L.pub;
    const int MX = 2 * K2 + 4, KX = K2 + 4, MR = K2 + 4;

    // ---- load: operators (transposed), my cells of the committed state, Q, the old scalar flux
    if (rank == 0) {
        for (int i = tid; i < 2 * kNormSlots; i += SM_THREADS) V.norms[i] = 0ull;
        if (tid == 0) V.flags[8] = 0;
    }
    for (int e = tid; e < MX * KX; e += SM_THREADS) {
        const int r = e / KX, u = e - r * KX;
        opx[u * MX + r] = V.xop[(size_t)r * (K2 + 16) + u];
    }
    for (int e = tid; e < MR * K2; e += SM_THREADS) {
        const int r = e / K2, k = e - r * K2;
        opr[k * MR + r] = V.rop[(size_t)r * K2 + k];
    }
    for (int e = tid; e < K2 * K2; e += SM_THREADS) {
        const int r = e / K2, k = e - r * K2;
        opf[k * K2 + r] = V.fop[(size_t)r * K2 + k];
    }
    {
        const double* __restrict__ Yg = V.y[ybase];
        for (int e = tid; e < (nc + 2) * K2; e += SM_THREADS) {           // rows j0-1 .. j0+nc: the global ghost rows ride along
            const int r = e / K2, q = e - r * K2;
            ybuf[0][(r - 1) * P + q] = Yg[((int64_t)j0 + r - 1) * K2 + q];
        }
        for (int e = tid; e < nc * N; e += SM_THREADS) {
            const int c = e / N, u = e - c * N;
            zin[c * (N + 1) + u] = V.z[((int64_t)j0 + c) * K2 + N2 + u];
        }
        for (int e = tid; e < nc * 4; e += SM_THREADS) {
            qin[e] = V.Q[(int64_t)j0 * 4 + e];
            phi[e] = V.phi[(int64_t)j0 * 4 + e];
        }
    }
    __syncthreads();

    // ---- FIX: [yfix | ifix | phifix][c] = X [psi_{k-1/2}[c]; Q[c]]   (psi_{k-1/2} = the k+1/2 runs of y and z)
    {
        const int groups = MX / SM_R;
        for (int t = tid; t < groups * nc; t += SM_THREADS) {
            const int g = t / nc, c = t - g * nc, r0 = g * SM_R;
            double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
            const double* __restrict__ yr = ybuf[0] + c * P + N2;
            const double* __restrict__ zr = zin + c * (N + 1);
            const double* __restrict__ op = opx + r0;
#pragma unroll 4
            for (int u = 0; u < KX; ++u) {
                const double x = u < N ? yr[u] : u < K2 ? zr[u - N] : qin[c * 4 + (u - K2)];
                const double4 w = *reinterpret_cast<const double4*>(op + u * MX);
                a0 = fma(w.x, x, a0); a1 = fma(w.y, x, a1); a2 = fma(w.z, x, a2); a3 = fma(w.w, x, a3);
            }
            const double a[4] = {a0, a1, a2, a3};
#pragma unroll
            for (int i = 0; i < SM_R; ++i) {
                const int r = r0 + i;
                if (r < K2) yfix[c * P + r] = a[i];
                else if (r < 2 * K2) ifix[c * P + (r - K2)] = a[i];
                else phifix[c * 4 + (r - 2 * K2)] = a[i];
            }
        }
    }
    __syncthreads();

    // ghost rows of buffer `b` (the iterate the next iteration reads): the neighbour CTA's edge row, or the boundary
    auto fill_ghosts = [&](int b) {
        for (int q = tid; q < 2 * K2; q += SM_THREADS) {
            const bool left = q < K2;
            const int qq = left ? q : q - K2;
            double v;
            if (left) {
                if (rank > 0) {
                    const double* nb = cluster.map_shared_rank(ybuf[b], rank - 1);
                    v = nb[(Jc - 1) * P + qq];                            // every CTA but the last holds Jc cells
                } else if (V.bcL == OCI_BC_REFLECTING) v = qq >= N ? ybuf[b][mirror_q(qq, N)] : 0.0;
                else v = V.bcL == OCI_BC_INCIDENT_ISOTROPIC ? V.bcLv : 0.0;
                ybuf[b][-P + qq] = v;
            } else {
                if (j0 + nc < J) {
                    const double* nb = cluster.map_shared_rank(ybuf[b], rank + 1);
                    v = nb[qq];
                } else if (V.bcR == OCI_BC_REFLECTING) v = qq < N ? ybuf[b][(nc - 1) * P + mirror_q(qq, N)] : 0.0;
                else v = V.bcR == OCI_BC_INCIDENT_ISOTROPIC ? V.bcRv : 0.0;
                ybuf[b][nc * P + qq] = v;
            }
        }
    };
    // (buffer 0 came from global memory with its ghost rows: the neighbours' rows of the committed iterate, or the
    // boundary data exactly as the three-pass kernels keep them)

    // ---- ITER loop: y^(l+1) = yfix + G inc^(l), phi^(l+1) = phifix + H inc^(l), norms, stop
    int Lit = 0;                                                          // iterations done
    bool conv = false;
    for (int l = 0; l < cnt; ++l) {
        const double* __restrict__ src = ybuf[l & 1];
        double* __restrict__ dst = ybuf[(l + 1) & 1];
        double dmax = 0.0, rmax = 0.0;
        const int groups = MR / SM_R;
        for (int t = tid; t < groups * nc; t += SM_THREADS) {
            const int g = t / nc, c = t - g * nc, r0 = g * SM_R;
            double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
            const double* __restrict__ xr = src + (c + 1) * P;            // q < N: the right neighbour's outgoing flux
            const double* __restrict__ xl = src + (c - 1) * P;            // q >= N: the left neighbour's
            const double* __restrict__ op = opr + r0;
#pragma unroll 4
            for (int k = 0; k < N; ++k) {
                const double x = xr[k];
                const double4 w = *reinterpret_cast<const double4*>(op + k * MR);
                a0 = fma(w.x, x, a0); a1 = fma(w.y, x, a1); a2 = fma(w.z, x, a2); a3 = fma(w.w, x, a3);
            }
#pragma unroll 4
            for (int k = N; k < K2; ++k) {
                const double x = xl[k];
                const double4 w = *reinterpret_cast<const double4*>(op + k * MR);
                a0 = fma(w.x, x, a0); a1 = fma(w.y, x, a1); a2 = fma(w.z, x, a2); a3 = fma(w.w, x, a3);
            }
            const double a[4] = {a0, a1, a2, a3};
            if (r0 < K2) {
#pragma unroll
                for (int i = 0; i < SM_R; ++i) dst[c * P + r0 + i] = yfix[c * P + r0 + i] + a[i];
            } else {
#pragma unroll
                for (int i = 0; i < SM_R; ++i) {
                    const double nw = phifix[c * 4 + i] + a[i], old = phi[c * 4 + i];
                    phi[c * 4 + i] = nw;
                    dmax = nanmax(dmax, fabs(nw - old));
                    rmax = nanmax(rmax, fabs(nw));
                }
            }
        }
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0) { red[2 * warp] = dmax; red[2 * warp + 1] = rmax; }
        __syncthreads();
        if (tid == 0) {
            for (int w = 1; w < SM_THREADS / 32; ++w) { dmax = nanmax(dmax, red[2 * w]); rmax = nanmax(rmax, red[2 * w + 1]); }
            for (int r = 0; r < C; ++r) {
                double* pr = cluster.map_shared_rank(pub, r) + (l & 1) * 16 + 2 * rank;
                pr[0] = dmax;
                pr[1] = rmax;
            }
        }
        if (C > 1) cluster.sync();                                        // every CTA's y^(l+1) and norms are in place
        else __syncthreads();
        double d = 0.0, r = 0.0;
        for (int k = 0; k < C; ++k) { d = nanmax(d, pub[(l & 1) * 16 + 2 * k]); r = nanmax(r, pub[(l & 1) * 16 + 2 * k + 1]); }
        if (rank == 0 && tid == 0) {                                      // a7: the host reads the norm slots once per step
            V.norms[2 * l + 0] = (unsigned long long)__double_as_longlong(d);
            V.norms[2 * l + 1] = (unsigned long long)__double_as_longlong(r);
        }
        fill_ghosts((l + 1) & 1);
        __syncthreads();
        Lit = l + 1;
        if (stop_now(tol, d, r)) conv = true;
        if ((conv || l + 1 == cnt) && rank == 0 && tid == 0) publish_step(V, Lit, l);   // (this thread wrote slot l itself)
        if (conv) break;
    }
    const bool finalize = conv || force != 0;

    // ---- FINAL: z = ifix + F inc^(L-1), staged in shared memory (yfix is dead) for a coalesced store
    if (finalize) {
        const double* __restrict__ src = ybuf[(Lit + 1) & 1];             // y^(L-1) with the ghost rows iteration L-1 read
        const int groups = K2 / SM_R;
        for (int t = tid; t < groups * nc; t += SM_THREADS) {
            const int g = t / nc, c = t - g * nc, r0 = g * SM_R;
            double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
            const double* __restrict__ xr = src + (c + 1) * P;
            const double* __restrict__ xl = src + (c - 1) * P;
            const double* __restrict__ op = opf + r0;
#pragma unroll 4
            for (int k = 0; k < N; ++k) {
                const double x = xr[k];
                const double4 w = *reinterpret_cast<const double4*>(op + k * K2);
                a0 = fma(w.x, x, a0); a1 = fma(w.y, x, a1); a2 = fma(w.z, x, a2); a3 = fma(w.w, x, a3);
            }
#pragma unroll 4
            for (int k = N; k < K2; ++k) {
                const double x = xl[k];
                const double4 w = *reinterpret_cast<const double4*>(op + k * K2);
                a0 = fma(w.x, x, a0); a1 = fma(w.y, x, a1); a2 = fma(w.z, x, a2); a3 = fma(w.w, x, a3);
            }
            const double a[4] = {a0, a1, a2, a3};
#pragma unroll
            for (int i = 0; i < SM_R; ++i) yfix[c * P + r0 + i] = ifix[c * P + r0 + i] + a[i];   // z, in place of yfix
        }
        __syncthreads();
        for (int e = tid; e < nc * K2; e += SM_THREADS) {
            const int c = e / K2, q = e - c * K2;
            V.z[((int64_t)j0 + c) * K2 + q] = yfix[c * P + q];
        }
    } else {
        // not converged within this launch: the three-pass kernels continue from global memory
        for (int e = tid; e < nc * K2; e += SM_THREADS) {
            const int c = e / K2, q = e - c * K2;
            V.yfix[((int64_t)j0 + c) * K2 + q] = yfix[c * P + q];
            V.ifix[((int64_t)j0 + c) * K2 + q] = ifix[c * P + q];
        }
        for (int e = tid; e < nc * 4; e += SM_THREADS) V.phifix[(int64_t)j0 * 4 + e] = phifix[e];
    }
    // ---- the state: y^(L) (and y^(L-1), which a later FINAL launch reads) with the reflecting ghost rows, phi
    for (int b = 0; b < 2; ++b) {
        double* __restrict__ Yg = V.y[(ybase + Lit + b) & 1];
        const double* __restrict__ ys = ybuf[(Lit + b) & 1];
        for (int e = tid; e < nc * K2; e += SM_THREADS) {
            const int c = e / K2, q = e - c * K2;
            Yg[((int64_t)j0 + c) * K2 + q] = ys[c * P + q];
        }
        if (j0 == 0 && V.bcL == OCI_BC_REFLECTING)
            for (int q = N + tid; q < K2; q += SM_THREADS) Yg[-(int64_t)K2 + q] = ys[-P + q];
        if (j0 + nc == J && V.bcR == OCI_BC_REFLECTING)
            for (int q = tid; q < N; q += SM_THREADS) Yg[(int64_t)J * K2 + q] = ys[nc * P + q];
    }
    for (int e = tid; e < nc * 4; e += SM_THREADS) V.phi[(int64_t)j0 * 4 + e] = phi[e];
    if (C > 1) cluster.sync();                                            // nobody leaves while a neighbour may still read its rows
}

// Cluster size that serves this problem, 0 if the one-launch step does not (oci_step then uses the three-pass kernels)
int oci_red_small_cluster(const DevView& V)
{
    if (V.nblk != 1 || V.bcL == OCI_BC_HALO || V.bcR == OCI_BC_HALO) return 0;
    const int64_t K2 = 2 * (int64_t)V.N;
    if (V.N > 64) return 0;                                               // the operators alone would fill shared memory
    const int64_t work = V.J * (K2 + 4) * K2;                             // multiply-adds of one iteration
    if (work > 4000000) return 0;                                         // large enough for the grid-wide kernels to win
    for (int C = work <= 65536 ? 1 : 8; C >= 1; C >>= 1) {
        if (C > 1 && V.J < 8 * C) continue;                               // at least 8 cells per CTA
        const int Jc = (int)((V.J + C - 1) / C);
        if ((int64_t)(C - 1) * Jc >= V.J) continue;                       // the last CTA must own a cell
        if ((size_t)small_layout(V.N, Jc).total * 8 <= 220 * 1024) return C;
        if (C == 1) break;
    }
    return 0;
}

cudaError_t oci_red_small_opt_in()
{
    return cudaFuncSetAttribute(oci_red_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024);
}

int launch_red_small(const DevView& V, int C, int ybase, double tol, int cnt, int force, cudaStream_t s)
{
    const int Jc = (int)((V.J + C - 1) / C);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)C);
    // thread items of one iteration in the busiest CTA: as many threads as there are items (a warp at least, 1024 at
    // most), since for a tiny problem every barrier and every serial reduction over the warps is pure latency
    const int64_t items = (int64_t)Jc * ((2 * V.N + 4) / SM_R);
    int threads = (int)((items + 31) / 32) * 32;
    threads = threads < 32 ? 32 : threads > SM_MAX_THREADS ? SM_MAX_THREADS : threads;
    cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = (size_t)small_layout(V.N, Jc).total * 8;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)C;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, oci_red_small_kernel, V, ybase, tol, cnt, force);
    return launched(1);
}

}  // namespace oci
