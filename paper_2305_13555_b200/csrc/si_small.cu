// One-launch SI step for SMALL shared-block problems: the comparator's counterpart of oci_reduced_small.cu, so that at
// the launch-latency-bound sizes (configs 1 and 2) OCI and SI are compared kernel against kernel, not one launch against
// three launches per iteration.  Same method and scan formulation as si_sweep_fast.cu (eqs. 12-18): the pair
// an angle carries from cell to cell obeys e_out = P e_in + z, so a sweep is a scan of affine maps over cells.
//
// One thread-block cluster of C <= 16 CTAs splits the cells into contiguous ranges; a CTA keeps psi_{k-1/2}, both
// buffers of the scattering source, Q and phi of its cells in shared memory.  thread = (chunk of the CTA's cells, angle).
// Per iteration:
//   reduce  : every thread composes the map of its chunk; the maps of a CTA are scanned in the direction of travel and the
//             CTA's composition is published into every CTA's shared memory (DSMEM stores)           -> cluster barrier
//   apply   : a thread applies the maps of the CTAs and chunks before its own to the boundary inflow, sweeps its chunk
//             and leaves w_m psi in shared memory; the angle sums (fixed order), phi, the two max-norms and the next
//             scattering source follow; the norms and the outflow at a reflecting face (the mirror angle's inflow of
//             the NEXT iteration: reading S4) are published to every CTA                             -> cluster barrier
//   stop    : decided identically by every thread from the C published pairs.
// After the loop the last sweep is repeated from phi^(L-1) and the kept chunk inflows and writes Psi^(L) and its ghost
// rows (as si_sweep_fast.cu's FINAL pass).  If the step does not converge within the iterations of one launch the kernel
// leaves psi_{k-1/2}, phi, both source buffers and both inflow arrays in global memory exactly as that many launches of the
// three-kernel iteration would have, and those continue.  Sums run in a fixed order: bit-reproducible.
//
// It does si_prev_kernel's work itself (psi_{k-1/2}, the first source, the boundary inflow).  Not served: per-cell
// blocks, OCI_BC_HALO faces, N > 32 or N / 2 not a power of two (the continuation must be si_sweep_fast.cu's), states
// larger than a cluster's shared memory.
#include <cooperative_groups.h>

#include "device_utils.cuh"

namespace cg = cooperative_groups;

namespace oci {

namespace {

constexpr int SS_T = 256;
constexpr int SS_MAXC = 16;

struct Aff {      // e -> P e + z
    double p00, p01, p10, p11, z0, z1;
};
__device__ __forceinline__ Aff aff_identity() { return Aff{1.0, 0.0, 0.0, 1.0, 0.0, 0.0}; }
__device__ __forceinline__ Aff aff_compose(const Aff& b, const Aff& a)      // apply a first, then b
{
    Aff r;
    r.p00 = fma(b.p00, a.p00, b.p01 * a.p10);
    r.p01 = fma(b.p00, a.p01, b.p01 * a.p11);
    r.p10 = fma(b.p10, a.p00, b.p11 * a.p10);
    r.p11 = fma(b.p10, a.p01, b.p11 * a.p11);
    r.z0 = fma(b.p00, a.z0, fma(b.p01, a.z1, b.z0));
    r.z1 = fma(b.p10, a.z0, fma(b.p11, a.z1, b.z1));
    return r;
}
__device__ __forceinline__ void aff_apply(const Aff& a, double& e0, double& e1)
{
    const double n0 = fma(a.p00, e0, fma(a.p01, e1, a.z0));
    const double n1 = fma(a.p10, e0, fma(a.p11, e1, a.z1));
    e0 = n0;
    e1 = n1;
}

struct SsLayout {                                          // offsets in doubles inside a CTA's dynamic shared memory
    int prev, src0, src1, q, phi, part, maps, agg, aggl, infl, pub, red, total;
};
__host__ __device__ inline SsLayout ss_layout(int N, int Jc)
{
    SsLayout L{};
    int o = 0;
    auto take = [&](int n) { const int at = o; o += (n + 3) & ~3; return at; };
    const int K = SS_T / N;
    L.prev = take(Jc * N * 2);                             // psi_{k-1/2}  [cell][angle][L, R]
    L.src0 = take(Jc * 4);                                 // (h/4)(Sigma_s phi + Q), by iteration parity
    L.src1 = take(Jc * 4);
    L.q = take(Jc * 4);
    L.phi = take(Jc * 4);
    L.part = take(Jc * (N * 4 + 4));                       // A^-1 b, then w_m psi, of the current sweep  [cell][angle][4], cell
                                                           // rows 4 doubles apart from a multiple of 16: the angle sums read
                                                           // (cell, slot) across a warp without bank conflicts
    L.maps = take(K * N * 6);                              // chunk maps of this CTA
    L.agg = take(SS_MAXC * N * 6);                         // every CTA's composition, written by its owner
    L.aggl = take(N * 6);                                  // this CTA's, before it is pushed
    L.infl = take(2 * N * 2);                              // boundary inflow of every angle, by iteration parity
    L.pub = take(2 * SS_MAXC * 2);                         // [parity][rank][d, r]
    L.red = take(2 * (SS_T / 32));
    L.total = o;
    return L;
}

}  // namespace

__global__ void __launch_bounds__(SS_T, 1) si_small_kernel(DevView V, int buf, double tol, int cnt, int force)
{
    extern __shared__ __align__(32) double ssm[];
    cg::cluster_group cluster = cg::this_cluster();
    const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    const int N = V.N, n = V.n, J = (int)V.J;
    const int Jc = (J + C - 1) / C;
    const SsLayout L = ss_layout(N, Jc);
    const int j0 = rank * Jc;
    const int nc = J - j0 < Jc ? (J - j0 > 0 ? J - j0 : 0) : Jc;          // cells of this CTA (the launcher keeps it > 0)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double* prev = ssm + L.prev;
    double* src[2] = {ssm + L.src0, ssm + L.src1};
    double* qq = ssm + L.q;
    double* phi = ssm + L.phi;
    double* part = ssm + L.part;
    const int PP = N * 4 + 4;                                             // pitch of a cell's row of `part`
    double* maps = ssm + L.maps;
    double* agg = ssm + L.agg;
    double* aggl = ssm + L.aggl;
    double* infl = ssm + L.infl;
    double* pub = ssm + L.pub;
    double* red = ssm + L.red;

    // thread = (chunk k of this CTA's cells, angle m)
    // chunks per CTA: about sqrt(cells) of them - a thread walks its chunk's cells AND the maps of the chunks before it
    int K = 1;
    while ((K + 1) * (K + 1) <= nc && K + 1 <= SS_T / N) ++K;
    const int k = tid / N, m = tid - k * N;
    const bool worker = k < K;
    const int cpk = (nc + K - 1) / K;                                     // cells per chunk
    const int cb = min(k * cpk, nc), ce = min(cb + cpk, nc);             // this chunk: local cells [cb, ce)
    const int mw = worker ? m : 0;
    const double mu = V.mu[mw];
    const bool pos = mu > 0.0;
    const double amu = fabs(mu), wm = V.w[mw];
    const int mir = N - 1 - mw;
    const int out_bc = pos ? V.bcR : V.bcL;
    double Ai[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) Ai[i] = V.ainv4[(size_t)mw * 16 + i];
    double Gk[4], Gh[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        Gk[r] = amu * (pos ? Ai[4 * r + 0] : Ai[4 * r + 1]);
        Gh[r] = amu * (pos ? Ai[4 * r + 2] : Ai[4 * r + 3]);
    }
    const int rep0 = V.rep[0];
    const double dx0 = V.dx[rep0], sg0 = V.sigs[rep0];
    const double al0 = dx0 / (2.0 * V.v * V.dt), q4 = 0.25 * dx0;
    // is this thread's chunk the one its angle leaves the slab through?
    const bool exits = worker && ce > cb && (pos ? (j0 + nc == J && ce == nc) : (rank == 0 && cb == 0));

    // ---- load (si_prev_kernel's work, a8: this read of the time-edge half of the committed iterate IS the commit):
    // psi_{k-1/2}, Q, phi, the first source (row d1) and the boundary inflow of every angle from the ghost rows of Psi
    if (rank == 0) {
        for (int i = tid; i < 2 * kNormSlots; i += SS_T) V.norms[i] = 0ull;
    }
    {
        const double* __restrict__ Pc = V.psi[buf];
        for (int e = tid; e < nc * N; e += SS_T)
            *reinterpret_cast<double2*>(prev + 2 * e) = *reinterpret_cast<const double2*>(Pc + ((size_t)j0 * N + e) * 4 + 2);
        for (int e = tid; e < nc * 4; e += SS_T) {
            const double ph = V.phi[(size_t)j0 * 4 + e], qv = V.Q[(size_t)j0 * 4 + e];
            qq[e] = qv;
            phi[e] = ph;
            src[0][e] = q4 * fma(sg0, ph, qv);
        }
        for (int a = tid; a < N; a += SS_T) {
            const bool ap = V.mu[a] > 0.0;
            const double i0 = ap ? Pc[-(int64_t)n + 4 * a + 1] : Pc[(size_t)J * n + 4 * a + 0];
            const double i1 = ap ? Pc[-(int64_t)n + 4 * a + 3] : Pc[(size_t)J * n + 4 * a + 2];
            infl[2 * a] = infl[2 * N + 2 * a] = i0;
            infl[2 * a + 1] = infl[2 * N + 2 * a + 1] = i1;
        }
    }
    if (C > 1) cluster.sync();
    else __syncthreads();

    // one cell of the sweep: x = A^-1 b + |mu| A^-1[:, inflow columns] (in_k, in_h)
    auto cell = [&](int c, const double* __restrict__ s, double in_k, double in_h, double (&x)[4]) {
        const double2 e = *reinterpret_cast<const double2*>(prev + ((size_t)c * N + mw) * 2);
        const double b[4] = {fma(al0, e.x, s[c * 4 + 0]), fma(al0, e.y, s[c * 4 + 1]), s[c * 4 + 2], s[c * 4 + 3]};
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const double y = Ai[4 * r + 0] * b[0] + Ai[4 * r + 1] * b[1] + Ai[4 * r + 2] * b[2] + Ai[4 * r + 3] * b[3];
            x[r] = fma(Gh[r], in_h, fma(Gk[r], in_k, y));
        }
    };

    int Lit = 0;
    bool conv = false;
    double cin_k = 0.0, cin_h = 0.0;                                     // this chunk's inflow in the last executed iteration
    for (int l = 0; l < cnt; ++l) {
        const double* __restrict__ s_cur = src[l & 1];
        double* __restrict__ s_nxt = src[(l + 1) & 1];
        const double* inf_cur = infl + (l & 1) * 2 * N;
        // ---- reduce: the map of this chunk (walk it with a zero inflow: z; the linear part is P^len)
        if (worker) {
            Aff A = aff_identity();
            const Aff P1 = Aff{pos ? Gk[1] : Gk[0], pos ? Gh[1] : Gh[0], pos ? Gk[3] : Gk[2], pos ? Gh[3] : Gh[2], 0.0, 0.0};
#pragma unroll 2
            for (int t = cb; t < ce; ++t) {
                const int c = pos ? t : ce - 1 - (t - cb);
                double y[4];
                cell(c, s_cur, 0.0, 0.0, y);                              // A^-1 b: kept for the apply phase
                double* pp = part + (size_t)c * PP + m * 4;
                *reinterpret_cast<double2*>(pp) = make_double2(y[0], y[1]);
                *reinterpret_cast<double2*>(pp + 2) = make_double2(y[2], y[3]);
                Aff g = P1;
                g.z0 = pos ? y[1] : y[0];
                g.z1 = pos ? y[3] : y[2];
                A = aff_compose(g, A);
            }
            double* mp = maps + ((size_t)k * N + m) * 6;
            mp[0] = A.p00; mp[1] = A.p01; mp[2] = A.p10; mp[3] = A.p11; mp[4] = A.z0; mp[5] = A.z1;
        }
        __syncthreads();
        // ---- the chunks before this one inside the CTA, in the direction of travel; the CTA's composition to everybody
        Aff pre = aff_identity();
        if (worker) {
            for (int i = 0; i < K; ++i) {
                const int kk = pos ? i : K - 1 - i;
                if (kk == k) break;
                const double* mp = maps + ((size_t)kk * N + m) * 6;
                pre = aff_compose(Aff{mp[0], mp[1], mp[2], mp[3], mp[4], mp[5]}, pre);
            }
            if (C > 1 && k == (pos ? K - 1 : 0)) {
                const double* mp = maps + ((size_t)k * N + m) * 6;
                const Aff all = aff_compose(Aff{mp[0], mp[1], mp[2], mp[3], mp[4], mp[5]}, pre);
                double* ag = aggl + (size_t)m * 6;
                ag[0] = all.p00; ag[1] = all.p01; ag[2] = all.p10; ag[3] = all.p11; ag[4] = all.z0; ag[5] = all.z1;
            }
        }
        if (C > 1) {
            __syncthreads();
            // every thread pushes a few words: one thread per angle storing to 16 CTAs would serialise 96 remote stores
            for (int idx = tid; idx < C * N * 6; idx += SS_T) {
                const int r = idx / (N * 6), w = idx - r * (N * 6);
                cluster.map_shared_rank(agg, r)[(size_t)rank * N * 6 + w] = aggl[w];
            }
            cluster.sync();
        }
        // ---- apply: inflow of the slab -> of this CTA -> of this chunk, then the sweep
        double in_k = 0.0, in_h = 0.0;
        if (worker) {
            in_k = inf_cur[2 * m];
            in_h = inf_cur[2 * m + 1];
            for (int i = 0; i < C; ++i) {
                const int rr = pos ? i : C - 1 - i;
                if (rr == rank) break;
                const double* ag = agg + ((size_t)rr * N + m) * 6;
                aff_apply(Aff{ag[0], ag[1], ag[2], ag[3], ag[4], ag[5]}, in_k, in_h);
            }
            aff_apply(pre, in_k, in_h);
            cin_k = in_k;
            cin_h = in_h;
            for (int t = cb; t < ce; ++t) {
                const int c = pos ? t : ce - 1 - (t - cb);
                double* pp = part + (size_t)c * PP + m * 4;
                const double2 y01 = *reinterpret_cast<const double2*>(pp), y23 = *reinterpret_cast<const double2*>(pp + 2);
                const double x0 = fma(Gh[0], in_h, fma(Gk[0], in_k, y01.x)), x1 = fma(Gh[1], in_h, fma(Gk[1], in_k, y01.y));
                const double x2 = fma(Gh[2], in_h, fma(Gk[2], in_k, y23.x)), x3 = fma(Gh[3], in_h, fma(Gk[3], in_k, y23.y));
                in_k = pos ? x1 : x0;
                in_h = pos ? x3 : x2;
                *reinterpret_cast<double2*>(pp) = make_double2(wm * x0, wm * x1);
                *reinterpret_cast<double2*>(pp + 2) = make_double2(wm * x2, wm * x3);
            }
            // the outflow at a reflecting face is the mirror angle's inflow of the next iteration, in every CTA
            if (exits && out_bc == OCI_BC_REFLECTING) {
                for (int r = 0; r < C; ++r) {
                    double* in2 = (C > 1 ? cluster.map_shared_rank(infl, r) : infl) + ((l + 1) & 1) * 2 * N;
                    in2[2 * mir] = in_k;
                    in2[2 * mir + 1] = in_h;
                }
            }
        }
        __syncthreads();
        // ---- eq. (18): phi = sum over the angles (fixed order), norms, the next scattering source (row d1)
        double dmax = 0.0, rmax = 0.0;
        for (int e = tid; e < nc * 4; e += SS_T) {
            const int c = e >> 2, r = e & 3;
            double sum = 0.0;
            for (int a = 0; a < N; ++a) sum += part[(size_t)c * PP + a * 4 + r];
            const double o = phi[e];
            phi[e] = sum;
            s_nxt[e] = q4 * fma(sg0, sum, qq[e]);
            dmax = nanmax(dmax, fabs(sum - o));
            rmax = nanmax(rmax, fabs(sum));
        }
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0) { red[2 * warp] = dmax; red[2 * warp + 1] = rmax; }
        __syncthreads();
        if (warp == 0) {
            dmax = warp_max(lane < SS_T / 32 ? red[2 * lane] : 0.0);
            rmax = warp_max(lane < SS_T / 32 ? red[2 * lane + 1] : 0.0);
            if (lane < C) {
                double* pr = (C > 1 ? cluster.map_shared_rank(pub, lane) : pub) + (l & 1) * 2 * SS_MAXC + 2 * rank;
                pr[0] = dmax;
                pr[1] = rmax;
            }
        }
        if (C > 1) cluster.sync();
        else __syncthreads();
        double d = 0.0, r = 0.0;
        for (int i = 0; i < C; ++i) {
            d = nanmax(d, pub[(l & 1) * 2 * SS_MAXC + 2 * i]);
            r = nanmax(r, pub[(l & 1) * 2 * SS_MAXC + 2 * i + 1]);
        }
        if (rank == 0 && tid == 0) {                                      // a7: the host reads the norm slots once per step
            V.norms[2 * l + 0] = (unsigned long long)__double_as_longlong(d);
            V.norms[2 * l + 1] = (unsigned long long)__double_as_longlong(r);
        }
        Lit = l + 1;
        if (stop_now(tol, d, r)) conv = true;
        if ((conv || l + 1 == cnt) && rank == 0 && tid == 0) publish_step(V, Lit, l);
        if (conv) break;
    }

    if (conv || force != 0) {
        // ---- FINAL: the last sweep again, from phi^(L-1) and the kept chunk inflows; Psi^(L) and its ghost rows
        double* __restrict__ Pg = V.psi[buf];
        if (worker) {
            const double* __restrict__ s_cur = src[(Lit - 1) & 1];
            double in_k = cin_k, in_h = cin_h;
            for (int t = cb; t < ce; ++t) {
                const int c = pos ? t : ce - 1 - (t - cb);
                double x[4];
                cell(c, s_cur, in_k, in_h, x);
                in_k = pos ? x[1] : x[0];
                in_h = pos ? x[3] : x[2];
                double* o = Pg + ((size_t)(j0 + c)) * n + 4 * m;
                *reinterpret_cast<double2*>(o) = make_double2(x[0], x[1]);
                *reinterpret_cast<double2*>(o + 2) = make_double2(x[2], x[3]);
            }
            if (exits && out_bc == OCI_BC_REFLECTING) {
                if (pos) { Pg[(size_t)J * n + 4 * mir + 0] = in_k; Pg[(size_t)J * n + 4 * mir + 2] = in_h; }
                else { Pg[-(int64_t)n + 4 * mir + 1] = in_k; Pg[-(int64_t)n + 4 * mir + 3] = in_h; }
            }
        }
    } else {
        // not converged within this launch: the three-kernel iterations continue from global memory
        for (int e = tid; e < nc * N * 2; e += SS_T) V.si_prev[(size_t)j0 * N * 2 + e] = prev[e];
        for (int e = tid; e < nc * 4; e += SS_T) {
            V.qs[(size_t)j0 * 4 + e] = src[0][e];
            V.si_src1[(size_t)j0 * 4 + e] = src[1][e];
        }
        if (rank == 0)
            for (int e = tid; e < 4 * N; e += SS_T) V.si_inflow[e] = infl[e];
    }
    for (int e = tid; e < nc * 4; e += SS_T) V.phi[(size_t)j0 * 4 + e] = phi[e];
    if (C > 1) cluster.sync();                                            // nobody leaves while a neighbour may still write its memory
}

// Cluster size that serves this problem, 0 if the one-launch SI step does not
int si_small_cluster(const DevView& V)
{
    if (V.nblk != 1 || V.bcL == OCI_BC_HALO || V.bcR == OCI_BC_HALO) return 0;
    if (V.N > 32 || !si_fast_supported(V)) return 0;
    const int64_t work = V.J * V.N;
    if (work > 65536) return 0;                                           // large enough for the grid-wide kernels
    for (int C = work <= 2048 ? 1 : SS_MAXC; C >= 1; C >>= 1) {
        if (C > 1 && V.J < 4 * C) continue;
        const int Jc = (int)((V.J + C - 1) / C);
        if ((int64_t)(C - 1) * Jc >= V.J) continue;                       // the last CTA must own a cell
        if ((size_t)ss_layout(V.N, Jc).total * 8 > 200 * 1024) continue;
        if (C > 8) {
            cudaLaunchConfig_t cfg{};
            cudaLaunchAttribute at[1];
            cfg.gridDim = dim3((unsigned)C);
            cfg.blockDim = dim3(SS_T);
            cfg.dynamicSmemBytes = (size_t)ss_layout(V.N, Jc).total * 8;
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = (unsigned)C;
            at[0].val.clusterDim.y = at[0].val.clusterDim.z = 1;
            cfg.attrs = at;
            cfg.numAttrs = 1;
            int nact = 0;
            if (cudaOccupancyMaxActiveClusters(&nact, si_small_kernel, &cfg) != cudaSuccess || nact < 1) {
                cudaGetLastError();
                continue;
            }
        }
        return C;
    }
    return 0;
}

cudaError_t si_small_opt_in()
{
    cudaError_t e = cudaFuncSetAttribute(si_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 208 * 1024);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(si_small_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
}

int launch_si_small(const DevView& V, int C, int buf, double tol, int cnt, int force, cudaStream_t s)
{
    const int Jc = (int)((V.J + C - 1) / C);
    cudaLaunchConfig_t cfg{};
    cudaLaunchAttribute at[1];
    cfg.gridDim = dim3((unsigned)C);
    cfg.blockDim = dim3(SS_T);
    cfg.dynamicSmemBytes = (size_t)ss_layout(V.N, Jc).total * 8;
    cfg.stream = s;
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)C;
    at[0].val.clusterDim.y = at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, si_small_kernel, V, buf, tol, cnt, force);
    return launched(1);
}

}  // namespace oci
