// One-launch time step for SMALL shared-block problems (configs 1 and 2: launch-latency bound): the whole reduced step
// of oci_reduced.cu - FIX, every ITER iteration with the stopping rule, FINAL - inside ONE kernel running on ONE
// thread-block cluster, the state resident in (distributed) shared memory for the whole step.
//
// The three-pass path costs a small problem three launches and, per iteration, a grid-wide barrier through global
// memory plus a round trip of the iterate through L2 (about 5 us per iteration at config 2 for 1.2 MFLOP of work).
// Here a cluster of C <= 16 CTAs (8 portable; 16 where the device co-schedules one) splits the cells into contiguous ranges; each CTA keeps, in its shared memory, the three
// operators (X, [G; H], F, transposed), both buffers of its part of the iterate y with one ghost row on either side,
// yfix, ifix, phifix and phi.  Per iteration:
//   compute (a warp takes tiles of 16 cells x up to 40 operator rows: DMMA.8x8x4 with both operands as fragments
//   straight from shared memory, rows pitched 4 (mod 16) doubles) -> publish this CTA's two max-norms into every CTA's
//   shared memory (DSMEM stores) -> ONE hardware cluster barrier -> ghost rows of the new iterate from the neighbour
//   CTAs' edge rows (DSMEM loads) or the boundary condition, and the stopping decision from the C published pairs,
//   taken identically by every thread of the cluster.
// No global-memory traffic inside the loop except the (d, r) pair of every iteration for the host (row a7: it still
// reads the norm slots once per step to learn the iteration count).  Sums run in a fixed order and the norms are exact
// maxima, so a step is reproducible bit for bit.  The arithmetic is the dense method's: the same operators as the other
// families of the reduced form, on the same fp64 tensor pipe (at these sizes a step is latency, not throughput).
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

constexpr int SM_MAX_THREADS = 256;                        // CTA size is chosen at launch: one warp per work item, 8 at most
constexpr int SM_NBG = 5;                                  // n8 blocks of operator rows per work item (40 rows) at most
constexpr int SM_MAX_CLUSTER = 16;                         // 8 is the portable limit; 16 where the device schedules it

// smallest pitch >= k that is 4 (mod 16) doubles: fragment loads of 8 rows x 4 columns hit 32 distinct banks
__host__ __device__ inline int sm_pitch(int k) { return k + ((4 - k) % 16 + 16) % 16; }

struct SmallLayout {                                       // offsets in doubles inside a CTA's dynamic shared memory
    int Jc, P, K2, PX, PR;                                 // P: pitch of y / yfix / ifix rows; PX, PR: of the operator rows
    int mx, mr, mf;                                        // operator rows, padded to whole n8 blocks
    int opx, opr, opf, y0, y1, yfix, ifix, phifix, phi, red, pub, total;
};

__host__ __device__ inline SmallLayout small_layout(int N, int Jc)
{
    SmallLayout L{};
    const int K2 = 2 * N;
    L.Jc = Jc;
    L.K2 = K2;
    L.P = sm_pitch(K2 + 4);                                // a row of y, or the FIX input vector [K2 + 4] (which borrows buffer 1)
    L.PX = sm_pitch(K2 + 4);
    L.PR = sm_pitch(K2);
    L.mx = (2 * K2 + 4 + 7) / 8 * 8;
    L.mr = (K2 + 4 + 7) / 8 * 8;
    L.mf = (K2 + 7) / 8 * 8;
    int o = 0;
    auto take = [&](int n) { const int at = o; o += (n + 3) & ~3; return at; };   // 32-byte aligned pieces
    L.opx = take(L.mx * L.PX);                             // X      [2K2+4 rows][K2+4]
    L.opr = take(L.mr * L.PR);                             // [G; H] [K2+4 rows][K2]
    L.opf = take(L.mf * L.PR);                             // F      [K2 rows][K2]
    L.y0 = take((Jc + 2) * L.P);                           // iterate, buffer 0, rows -1 .. Jc
    L.y1 = take((Jc + 2) * L.P);                           // buffer 1; during FIX: the input vectors [psi_{k-1/2}; Q]
    L.yfix = take(Jc * L.P);                               // also the staging area of z (FINAL)
    L.ifix = take(Jc * L.P);
    L.phifix = take(Jc * 4);
    L.phi = take(Jc * 4);
    L.red = take(2 * (SM_MAX_THREADS / 32));
    L.pub = take(2 * SM_MAX_CLUSTER * 2);                  // [parity][rank][d, r] published by every CTA of the cluster
    L.total = o;
    return L;
}

// One work item of a "gathered GEMM" pass: out[cell][row] = sum_k Op[row][k] in(cell, k) for the 16 cells c0 .. c0+15 and
// NB n8 blocks of operator rows from block t0 on, as DMMA.8x8x4 (cells = the M dimension).  The input of the lane's two
// cells (c0 + g4, c0 + 8 + g4) is row lo[g] for k < split and row hi[g] from there on (ITER / FINAL: the right / left
// neighbour's row; FIX: one row); `out` receives (cell, row, v[row], v[row+1]) in accumulator layout.
template <int NB, typename Out>
__device__ __forceinline__ void small_item_nb(const double* __restrict__ op, int opp, int K, int split, const double* const (&lo)[2],
                                              const double* const (&hi)[2], int c0, int t0, Out out)
{
    const int lane = threadIdx.x & 31, g4 = lane >> 2, t4 = lane & 3;
    double acc[2][NB][2];
#pragma unroll
    for (int g = 0; g < 2; ++g)
#pragma unroll
        for (int t = 0; t < NB; ++t) acc[g][t][0] = acc[g][t][1] = 0.0;
    const double* __restrict__ bp = op + (size_t)(8 * t0 + g4) * opp + t4;
    // the fragments of k-step k + 4 are requested before the DMMAs of k-step k are issued
    double a0 = (t4 < split ? lo[0] : hi[0])[t4], a1 = (t4 < split ? lo[1] : hi[1])[t4], b[NB];
#pragma unroll
    for (int t = 0; t < NB; ++t) b[t] = bp[(size_t)(8 * t) * opp];
    for (int k = 0; k < K; k += 4) {
        const int kn = (k + 4 < K ? k + 4 : k) + t4;
        const double na0 = (kn < split ? lo[0] : hi[0])[kn], na1 = (kn < split ? lo[1] : hi[1])[kn];
        double nb_[NB];
#pragma unroll
        for (int t = 0; t < NB; ++t) nb_[t] = bp[(size_t)(8 * t) * opp + kn - t4];
#pragma unroll
        for (int t = 0; t < NB; ++t) {
            dmma(acc[0][t][0], acc[0][t][1], a0, b[t]);
            dmma(acc[1][t][0], acc[1][t][1], a1, b[t]);
        }
        a0 = na0;
        a1 = na1;
#pragma unroll
        for (int t = 0; t < NB; ++t) b[t] = nb_[t];
    }
#pragma unroll
    for (int g = 0; g < 2; ++g)
#pragma unroll
        for (int t = 0; t < NB; ++t) out(c0 + 8 * g + g4, 8 * (t0 + t) + 2 * t4, acc[g][t][0], acc[g][t][1]);
}

template <typename Out>
__device__ __forceinline__ void small_item(const double* __restrict__ op, int opp, int K, int split, const double* const (&lo)[2],
                                           const double* const (&hi)[2], int c0, int t0, int nb, Out out)
{
    switch (nb) {                                          // the block count as a template argument: no predicated DMMA
    case 5: small_item_nb<5>(op, opp, K, split, lo, hi, c0, t0, out); break;
    case 4: small_item_nb<4>(op, opp, K, split, lo, hi, c0, t0, out); break;
    case 3: small_item_nb<3>(op, opp, K, split, lo, hi, c0, t0, out); break;
    case 2: small_item_nb<2>(op, opp, K, split, lo, hi, c0, t0, out); break;
    default: small_item_nb<1>(op, opp, K, split, lo, hi, c0, t0, out); break;
    }
}

}  // namespace

// nbg: n8 blocks of operator rows per work item (<= SM_NBG), chosen by the launcher so that the warps of a CTA all get work
__global__ void __launch_bounds__(SM_MAX_THREADS, 1) oci_red_small_kernel(DevView V, int ybase, double tol, int cnt, int force, int nbg)
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
    double* xin = ybuf[1];                                                // FIX input vectors [psi_{k-1/2}; Q], pitch P
    double* yfix = ssm + L.yfix;
    double* ifix = ssm + L.ifix;
    double* phifix = ssm + L.phifix;
    double* phi = ssm + L.phi;
    double* red = ssm + L.red;
    double* pub = ssm + L.pub;
    const int PX = L.PX, PR = L.PR;
    const int nwarps = SM_THREADS >> 5;
    const int ntile = (nc + 15) / 16;                                     // tiles of 16 cells
    // A TINY problem (config 1: 20 cells x 12 rows) is a chain of latencies, not arithmetic: a DMMA work item is ~2000
    // cycles of dependent tensor-pipe and shared-memory round trips for 8 k-steps of 4.  There thread = (cell, operator row)
    // and a row is K2 (+4) dependent DFMAs on broadcast operands: a few hundred cycles per pass.
    const bool tiny = C == 1 && nc * (2 * K2 + 4) <= 4 * SM_MAX_THREADS && K2 <= 16;
    auto dot = [&](const double* __restrict__ orow, const double* __restrict__ lo, const double* __restrict__ hi, int K, int split) {
        double a = 0.0;
        for (int k = 0; k < K; ++k) a = fma(orow[k], (k < split ? lo : hi)[k], a);
        return a;
    };

    // ---- load: operators (rows pitched for conflict-free fragment loads, padding rows zero), my cells of the committed
    // state, the FIX input vectors [y(k+1/2 run) | z(k+1/2 run) | Q], the old scalar flux
    if (rank == 0) {
        for (int i = tid; i < 2 * kNormSlots; i += SM_THREADS) V.norms[i] = 0ull;
        if (tid == 0) { V.flags[8] = 0; V.flags[12] = 0; }
    }
    for (int e = tid; e < L.mx * (K2 + 4); e += SM_THREADS) {
        const int r = e / (K2 + 4), u = e - r * (K2 + 4);
        opx[r * PX + u] = r < 2 * K2 + 4 ? V.xop[(size_t)r * (K2 + 16) + u] : 0.0;
    }
    for (int e = tid; e < L.mr * K2; e += SM_THREADS) {
        const int r = e / K2, k = e - r * K2;
        opr[r * PR + k] = r < K2 + 4 ? V.rop[(size_t)r * K2 + k] : 0.0;
    }
    for (int e = tid; e < L.mf * K2; e += SM_THREADS) {
        const int r = e / K2, k = e - r * K2;
        opf[r * PR + k] = r < K2 ? V.fop[(size_t)r * K2 + k] : 0.0;
    }
    {
        const double* __restrict__ Yg = V.y[ybase];
        for (int e = tid; e < (nc + 2) * K2; e += SM_THREADS) {           // rows j0-1 .. j0+nc: the global ghost rows ride along
            const int r = e / K2, q = e - r * K2;
            const double v = Yg[((int64_t)j0 + r - 1) * K2 + q];
            ybuf[0][(r - 1) * P + q] = v;
            if (r >= 1 && r <= nc && q >= N2 && q < N2 + N) xin[(r - 1) * P + (q - N2)] = v;
        }
        for (int e = tid; e < nc * N; e += SM_THREADS) {
            const int c = e / N, u = e - c * N;
            xin[c * P + N + u] = V.z[((int64_t)j0 + c) * K2 + N2 + u];
        }
        for (int e = tid; e < nc * 4; e += SM_THREADS) {
            xin[(e >> 2) * P + K2 + (e & 3)] = V.Q[(int64_t)j0 * 4 + e];
            phi[e] = V.phi[(int64_t)j0 * 4 + e];
        }
    }
    if (C > 1) cluster.sync();                     // every CTA of the cluster is running before anybody touches its shared memory
    else __syncthreads();

    // ---- FIX: [yfix | ifix | phifix][c] = X [psi_{k-1/2}[c]; Q[c]]   (psi_{k-1/2} = the k+1/2 runs of y and z)
    if (tiny) {
        for (int e = tid; e < nc * (2 * K2 + 4); e += SM_THREADS) {
            const int c = e / (2 * K2 + 4), r = e - c * (2 * K2 + 4);
            const double v = dot(opx + r * PX, xin + c * P, xin + c * P, K2 + 4, K2 + 4);
            if (r < K2) yfix[c * P + r] = v;
            else if (r < 2 * K2) ifix[c * P + r - K2] = v;
            else phifix[c * 4 + r - 2 * K2] = v;
        }
    } else {
        const int nbt = L.mx / 8, ngr = (nbt + nbg - 1) / nbg;
        for (int it = warp; it < ntile * ngr; it += nwarps) {
            const int tile = it / ngr, gr = it - tile * ngr;
            const int t0 = gr * nbg, nb = nbt - t0 < nbg ? nbt - t0 : nbg;
            const int g4 = lane >> 2;
            const int ca = 16 * tile + g4 < nc ? 16 * tile + g4 : nc - 1, cb = 16 * tile + 8 + g4 < nc ? 16 * tile + 8 + g4 : nc - 1;
            const double* const rows[2] = {xin + ca * P, xin + cb * P};    // (a ragged tile's missing cells: clamped, dropped)
            small_item(opx, PX, K2 + 4, K2 + 4, rows, rows, 16 * tile, t0, nb,
                       [&](int c, int r, double v0, double v1) {
                           if (c >= nc) return;
                           if (r < K2) { yfix[c * P + r] = v0; yfix[c * P + r + 1] = v1; }
                           else if (r < 2 * K2) { ifix[c * P + r - K2] = v0; ifix[c * P + r - K2 + 1] = v1; }
                           else if (r < 2 * K2 + 4) { phifix[c * 4 + r - 2 * K2] = v0; phifix[c * 4 + r - 2 * K2 + 1] = v1; }
                       });
        }
    }
    __syncthreads();

    // ghost rows of buffer `b` (the iterate the next iteration reads), written BEFORE the cluster barrier: every CTA
    // pushes its two edge rows into its neighbours' ghost rows (DSMEM stores; a remote load after the barrier would add its
    // round trip to every iteration) and the CTAs at the ends of the slab apply the boundary condition to their own.
    // Nobody reads buffer b during the iteration that writes it, and the barrier orders the stores before the reads.
    auto push_ghosts = [&](int b) {
        for (int q = SM_THREADS - 1 - tid; q < 2 * K2; q += SM_THREADS) {   // from the last warp down: warp 0 publishes the norms
            const bool left = q < K2;
            const int qq = left ? q : q - K2;
            if (left) {
                if (rank > 0) cluster.map_shared_rank(ybuf[b], rank - 1)[Jc * P + qq] = ybuf[b][qq];   // every CTA but the last holds Jc cells
                else ybuf[b][-P + qq] = V.bcL == OCI_BC_REFLECTING ? (qq >= N ? ybuf[b][mirror_q(qq, N)] : 0.0)
                                                                    : (V.bcL == OCI_BC_INCIDENT_ISOTROPIC ? V.bcLv : 0.0);
            } else {
                if (j0 + nc < J) cluster.map_shared_rank(ybuf[b], rank + 1)[-P + qq] = ybuf[b][(nc - 1) * P + qq];
                else ybuf[b][nc * P + qq] = V.bcR == OCI_BC_REFLECTING ? (qq < N ? ybuf[b][(nc - 1) * P + mirror_q(qq, N)] : 0.0)
                                                                       : (V.bcR == OCI_BC_INCIDENT_ISOTROPIC ? V.bcRv : 0.0);
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
        if (tiny) {
            for (int e = tid; e < nc * (K2 + 4); e += SM_THREADS) {
                const int c = e / (K2 + 4), r = e - c * (K2 + 4);
                const double v = dot(opr + r * PR, src + (c + 1) * P, src + (c - 1) * P, K2, N);
                if (r < K2) {
                    dst[c * P + r] = yfix[c * P + r] + v;
                } else {
                    const int i = r - K2;
                    const double nv = phifix[c * 4 + i] + v, ov = phi[c * 4 + i];
                    phi[c * 4 + i] = nv;
                    dmax = nanmax(dmax, fabs(nv - ov));
                    rmax = nanmax(rmax, fabs(nv));
                }
            }
        } else {
            const int nbt = L.mr / 8, ngr = (nbt + nbg - 1) / nbg;
            for (int it = warp; it < ntile * ngr; it += nwarps) {
                const int tile = it / ngr, gr = it - tile * ngr;
                const int t0 = gr * nbg, nb = nbt - t0 < nbg ? nbt - t0 : nbg;
                // q < N: the right neighbour's outgoing flux, q >= N: the left neighbour's (a ragged tile's missing
                // cells: clamped, their results dropped)
                const int g4 = lane >> 2;
                const int ca = 16 * tile + g4 < nc ? 16 * tile + g4 : nc - 1, cb = 16 * tile + 8 + g4 < nc ? 16 * tile + 8 + g4 : nc - 1;
                const double* const rr[2] = {src + (ca + 1) * P, src + (cb + 1) * P};
                const double* const rl[2] = {src + (ca - 1) * P, src + (cb - 1) * P};
                small_item(opr, PR, K2, N, rr, rl, 16 * tile, t0, nb,
                           [&](int c, int r, double v0, double v1) {
                               if (c >= nc) return;
                               if (r < K2) {
                                   dst[c * P + r] = yfix[c * P + r] + v0;
                                   dst[c * P + r + 1] = yfix[c * P + r + 1] + v1;
                               } else if (r < K2 + 4) {
                                   const int i = r - K2;
                                   const double n0 = phifix[c * 4 + i] + v0, n1 = phifix[c * 4 + i + 1] + v1;
                                   const double o0 = phi[c * 4 + i], o1 = phi[c * 4 + i + 1];
                                   phi[c * 4 + i] = n0;
                                   phi[c * 4 + i + 1] = n1;
                                   dmax = nanmax(dmax, nanmax(fabs(n0 - o0), fabs(n1 - o1)));
                                   rmax = nanmax(rmax, nanmax(fabs(n0), fabs(n1)));
                               }
                           });
            }
        }
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0) { red[2 * warp] = dmax; red[2 * warp + 1] = rmax; }
        __syncthreads();
        if (warp == 0) {                                                  // lane w: warp w's pair; lane r publishes to rank r
            dmax = warp_max(lane < nwarps ? red[2 * lane] : 0.0);
            rmax = warp_max(lane < nwarps ? red[2 * lane + 1] : 0.0);
            if (lane < C) {
                double* pr = cluster.map_shared_rank(pub, lane) + (l & 1) * 2 * SM_MAX_CLUSTER + 2 * rank;
                pr[0] = dmax;
                pr[1] = rmax;
            }
        }
        push_ghosts((l + 1) & 1);
        if (C > 1) cluster.sync();                                        // every CTA's y^(l+1), ghost rows and norms are in place
        else __syncthreads();
        double d = 0.0, r = 0.0;
        for (int k = 0; k < C; ++k) {
            d = nanmax(d, pub[(l & 1) * 2 * SM_MAX_CLUSTER + 2 * k]);
            r = nanmax(r, pub[(l & 1) * 2 * SM_MAX_CLUSTER + 2 * k + 1]);
        }
        if (rank == 0 && tid == 0) {                                      // a7: the host reads the norm slots once per step
            V.norms[2 * l + 0] = (unsigned long long)__double_as_longlong(d);
            V.norms[2 * l + 1] = (unsigned long long)__double_as_longlong(r);
        }
        Lit = l + 1;
        if (stop_now(tol, d, r)) conv = true;
        if ((conv || l + 1 == cnt) && rank == 0 && tid == 0) publish_step(V, Lit, l);   // (this thread wrote slot l itself)
        if (conv) break;
    }
    const bool finalize = conv || force != 0;

    // ---- FINAL: z = ifix + F inc^(L-1), staged in shared memory (yfix is dead) for a coalesced store
    if (finalize) {
        const double* __restrict__ src = ybuf[(Lit + 1) & 1];             // y^(L-1) with the ghost rows iteration L-1 read
        const int nbt = L.mf / 8, ngr = (nbt + nbg - 1) / nbg;
        if (tiny) {
            for (int e = tid; e < nc * K2; e += SM_THREADS) {
                const int c = e / K2, r = e - c * K2;
                yfix[c * P + r] = ifix[c * P + r] + dot(opf + r * PR, src + (c + 1) * P, src + (c - 1) * P, K2, N);
            }
        }
        for (int it = tiny ? ntile * ngr : warp; it < ntile * ngr; it += nwarps) {
            const int tile = it / ngr, gr = it - tile * ngr;
            const int t0 = gr * nbg, nb = nbt - t0 < nbg ? nbt - t0 : nbg;
            const int g4 = lane >> 2;
            const int ca = 16 * tile + g4 < nc ? 16 * tile + g4 : nc - 1, cb = 16 * tile + 8 + g4 < nc ? 16 * tile + 8 + g4 : nc - 1;
            const double* const rr[2] = {src + (ca + 1) * P, src + (cb + 1) * P};
            const double* const rl[2] = {src + (ca - 1) * P, src + (cb - 1) * P};
            small_item(opf, PR, K2, N, rr, rl, 16 * tile, t0, nb,
                       [&](int c, int r, double v0, double v1) {
                           if (c >= nc || r >= K2) return;
                           yfix[c * P + r] = ifix[c * P + r] + v0;          // z, in place of yfix
                           yfix[c * P + r + 1] = ifix[c * P + r + 1] + v1;
                       });
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

namespace {
// blocks of operator rows per work item and CTA size: one warp per work item of an iteration in the busiest CTA, 8 warps at
// most (for a tiny problem every barrier and every serial reduction over the warps is pure latency); a tile's operator
// rows are split into as many equal groups as it takes to give every warp an item
void small_shape(const DevView& V, int C, int* nbg, int* threads)
{
    const int Jc = (int)((V.J + C - 1) / C), ntile = (Jc + 15) / 16, nbt = (2 * V.N + 4 + 7) / 8;
    int groups = (SM_MAX_THREADS / 32 + ntile - 1) / ntile;
    groups = groups > nbt ? nbt : groups;
    const int per = (nbt + groups - 1) / groups;
    *nbg = per > SM_NBG ? SM_NBG : per;
    const int items = ntile * ((nbt + *nbg - 1) / *nbg);
    *threads = items * 32 > SM_MAX_THREADS ? SM_MAX_THREADS : items * 32;
    // a tiny problem runs thread = (cell, operator row) (the kernel's `tiny` test): one thread per row of an ITER pass
    const int K2 = 2 * V.N;
    if (C == 1 && V.J * (2 * K2 + 4) <= 4 * SM_MAX_THREADS && K2 <= 16) {
        int t = ((int)V.J * (K2 + 4) + 31) / 32 * 32;
        *threads = t > SM_MAX_THREADS ? SM_MAX_THREADS : t < 32 ? 32 : t;
    }
}

void small_config(const DevView& V, int C, cudaLaunchConfig_t* cfg, cudaLaunchAttribute* at, int* nbg)
{
    int threads;
    small_shape(V, C, nbg, &threads);
    *cfg = cudaLaunchConfig_t{};
    cfg->gridDim = dim3((unsigned)C);
    cfg->blockDim = dim3((unsigned)threads);
    cfg->dynamicSmemBytes = (size_t)small_layout(V.N, (int)((V.J + C - 1) / C)).total * 8;
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)C;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg->attrs = at;
    cfg->numAttrs = 1;
}

// clusters of more than 8 CTAs are not portable: ask the device whether it can co-schedule one
bool small_cluster_fits(const DevView& V, int C)
{
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute at[1];
    int nbg, n = 0;
    small_config(V, C, &cfg, at, &nbg);
    if (cudaOccupancyMaxActiveClusters(&n, oci_red_small_kernel, &cfg) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return n >= 1;
}
}  // namespace

// Cluster size that serves this problem, 0 if the one-launch step does not (oci_step then uses the three-pass kernels)
int oci_red_small_cluster(const DevView& V)
{
    if (V.nblk != 1 || V.bcL == OCI_BC_HALO || V.bcR == OCI_BC_HALO) return 0;
    const int64_t K2 = 2 * (int64_t)V.N;
    if (V.N > 64) return 0;                                               // the operators alone would fill shared memory
    const int64_t work = V.J * (K2 + 4) * K2;                             // multiply-adds of one iteration
    if (work > 4000000) return 0;                                         // large enough for the grid-wide kernels to win
    for (int C = work <= 65536 ? 1 : SM_MAX_CLUSTER; C >= 1; C >>= 1) {
        if (C > 1 && V.J < 8 * C) continue;                               // at least 8 cells per CTA
        const int Jc = (int)((V.J + C - 1) / C);
        if ((int64_t)(C - 1) * Jc >= V.J) continue;                       // the last CTA must own a cell
        if ((size_t)small_layout(V.N, Jc).total * 8 > 220 * 1024) continue;
        if (C > 8 && !small_cluster_fits(V, C)) continue;
        return C;
    }
    return 0;
}

cudaError_t oci_red_small_opt_in()
{
    cudaError_t e = cudaFuncSetAttribute(oci_red_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(oci_red_small_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
}

int launch_red_small(const DevView& V, int C, int ybase, double tol, int cnt, int force, cudaStream_t s)
{
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute at[1];
    int nbg;
    small_config(V, C, &cfg, at, &nbg);
    cfg.stream = s;
    cudaLaunchKernelEx(&cfg, oci_red_small_kernel, V, ybase, tol, cnt, force, nbg);
    return launched(1);
}

}  // namespace oci
