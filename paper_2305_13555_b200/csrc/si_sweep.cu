// Kernel (d): the source-iteration comparator (eqs. 12-18).  "SI sweeps ... are readily
// parallelized over the number of angles"; the scattering source comes from phi^(l) (row d1),
// the upstream edge values from THIS sweep's previous cell (row d2; no (l) on the neighbour term of
// eqs. 14,17), reflecting boundaries from the previous iterate (reading S4, via the ghost rows).
//
// The 4x4 systems are pre-inverted per (block, angle).  With x = Ainv (b + |mu| e_in) the pair of
// values an angle carries from cell to cell (its outgoing edge flux at k and k+1/2) obeys the 2x2
// affine recurrence  e_out = G_j e_in + z_j,  so the sweep is a scan over cells of affine maps
// and is parallel over cells as well as angles:
//
//   phase 1  si_chunk_kernel<.,1>  thread = (chunk of S cells, angle): walk the chunk with zero inflow,
//            composing the chunk's map (P_c = prod G_j, z_c); nothing but 6 doubles is written;
//   phase 2  si_carry_kernel       one CTA per angle: scan of the chunk maps (thread-local compose,
//            warp shuffle scan, 8 warp totals through shared memory) -> the inflow of every chunk;
//   phase 3  si_chunk_kernel<.,3>  walk the chunk again from its true inflow and store Psi.
//
// A warp holds 32 consecutive angles of one cell, so every global access is a contiguous 1 KB line
// segment; reads c_fix twice and writes Psi once per iteration (HBM-bound at the large configs).
// Per-thread arithmetic on the sequential chain: two dependent FMAs per cell.
#include "device_utils.cuh"

namespace oci {

namespace {

struct Affine {      // e -> P e + z, P row major
    double p00, p01, p10, p11, z0, z1;
};
__device__ __forceinline__ Affine affine_identity() { return Affine{1.0, 0.0, 0.0, 1.0, 0.0, 0.0}; }
// (b o a): apply a first, then b
__device__ __forceinline__ Affine compose(const Affine& b, const Affine& a)
{
    Affine r;
    r.p00 = fma(b.p00, a.p00, b.p01 * a.p10);
    r.p01 = fma(b.p00, a.p01, b.p01 * a.p11);
    r.p10 = fma(b.p10, a.p00, b.p11 * a.p10);
    r.p11 = fma(b.p10, a.p01, b.p11 * a.p11);
    r.z0 = fma(b.p00, a.z0, fma(b.p01, a.z1, b.z0));
    r.z1 = fma(b.p10, a.z0, fma(b.p11, a.z1, b.z1));
    return r;
}
__device__ __forceinline__ Affine shfl_up_affine(const Affine& a, int o)
{
    Affine r;
    r.p00 = __shfl_up_sync(0xffffffffu, a.p00, o);
    r.p01 = __shfl_up_sync(0xffffffffu, a.p01, o);
    r.p10 = __shfl_up_sync(0xffffffffu, a.p10, o);
    r.p11 = __shfl_up_sync(0xffffffffu, a.p11, o);
    r.z0 = __shfl_up_sync(0xffffffffu, a.z0, o);
    r.z1 = __shfl_up_sync(0xffffffffu, a.z1, o);
    return r;
}

}  // namespace

// PHASE 1: reduce the chunk to its affine map.  PHASE 3: sweep the chunk from its inflow, store Psi.
// scan[(c*N + m)*8 + 0..5] = (P_c, z_c), [6..7] = inflow of chunk c (written by si_carry_kernel).
template <int U, bool SHARED_BLOCK, int PHASE>
__global__ void __launch_bounds__(128) si_chunk_kernel(DevView V, int buf, int prev_slot, double tol, int S, int C, int Nr)
{
    if (step_done(V.norms, prev_slot, tol)) return;
    const int64_t gid = (int64_t)blockIdx.x * 128 + threadIdx.x;
    const int m = (int)(gid % Nr);
    const int64_t c = gid / Nr;
    if (m >= V.N || c >= C) return;
    const int n = V.n;
    const int64_t J = V.J;
    double* __restrict__ P = V.psi[buf];
    const double mu = V.mu[m];
    const bool pos = mu > 0.0;
    const double amu = fabs(mu);
    double* sc = V.si_scan + ((size_t)c * V.N + m) * 8;
    // mu>0: rows 0,2 receive the incident flux (k, k+1/2) and rows 1,3 leave the cell; mu<0: mirrored
    double in_k = 0.0, in_h = 0.0;
    if (PHASE == 3) {
        if (C == 1) {
            in_k = pos ? P[-(int64_t)n + 4 * m + 1] : P[J * n + 4 * m + 0];
            in_h = pos ? P[-(int64_t)n + 4 * m + 3] : P[J * n + 4 * m + 2];
        } else {
            in_k = sc[6];
            in_h = sc[7];
        }
    }
    Affine A = affine_identity();

    double Ai[16];
    if (SHARED_BLOCK) {
#pragma unroll
        for (int i = 0; i < 16; ++i) Ai[i] = V.ainv4[(size_t)m * 16 + i];
    }
    const int64_t t_begin = c * S;
    const int64_t t_end = (t_begin + S < J) ? t_begin + S : J;

    for (int64_t t0 = t_begin; t0 < t_end; t0 += U) {
        double y[U][4], G[U][4][2];
        // ---- off-chain, step 1: every load of the U cells is issued before anything consumes one
        // (indices clamped into the chunk instead of branching, so the loads are unconditional)
        double2 c01[U], c23[U], f01[U], f23[U];
        double hs[U];
        const double* ap[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t t = (t0 + u < t_end) ? t0 + u : t_end - 1;
            const int64_t j = pos ? t : J - 1 - t;
            c01[u] = *reinterpret_cast<const double2*>(V.cfix + j * n + 4 * m);
            c23[u] = *reinterpret_cast<const double2*>(V.cfix + j * n + 4 * m + 2);
            f01[u] = *reinterpret_cast<const double2*>(V.phi + j * 4);
            f23[u] = *reinterpret_cast<const double2*>(V.phi + j * 4 + 2);
            hs[u] = V.dx[j] * 0.25 * V.sigs[j];                                  // (h/4) Sigma_s, eqs. 14,17
            if (!SHARED_BLOCK) ap[u] = V.ainv4 + ((size_t)V.blk[j] * V.N + m) * 16;
        }
        // ---- off-chain, step 2: d1 (scattering source from phi^(l)), y = Ainv * b
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const double b[4] = {fma(hs[u], f01[u].x, c01[u].x), fma(hs[u], f01[u].y, c01[u].y),
                                 fma(hs[u], f23[u].x, c23[u].x), fma(hs[u], f23[u].y, c23[u].y)};
            if (!SHARED_BLOCK) {
#pragma unroll
                for (int i = 0; i < 16; i += 2) {
                    const double2 v2 = *reinterpret_cast<const double2*>(ap[u] + i);
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
        // ---- the sequential chain: two dependent FMAs per cell
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t t = t0 + u;
            if (t < t_end) {
                if (PHASE == 1) {
                    Affine g;
                    g.p00 = pos ? G[u][1][0] : G[u][0][0];  g.p01 = pos ? G[u][1][1] : G[u][0][1];
                    g.p10 = pos ? G[u][3][0] : G[u][2][0];  g.p11 = pos ? G[u][3][1] : G[u][2][1];
                    g.z0 = pos ? y[u][1] : y[u][0];
                    g.z1 = pos ? y[u][3] : y[u][2];
                    A = compose(g, A);
                } else {
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
    if (PHASE == 1) {
        *reinterpret_cast<double2*>(sc + 0) = make_double2(A.p00, A.p01);
        *reinterpret_cast<double2*>(sc + 2) = make_double2(A.p10, A.p11);
        *reinterpret_cast<double2*>(sc + 4) = make_double2(A.z0, A.z1);
    }
}

// PHASE 2: exclusive scan of the chunk maps of one angle, applied to the boundary inflow.
__global__ void __launch_bounds__(256) si_carry_kernel(DevView V, int buf, int prev_slot, double tol, int C)
{
    if (step_done(V.norms, prev_slot, tol)) return;
    __shared__ Affine wtot[8];
    const int m = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = V.n;
    const double* __restrict__ P = V.psi[buf];
    const bool pos = V.mu[m] > 0.0;
    const int cpl = (C + 255) / 256;
    const int c0 = tid * cpl;
    const int c1 = (c0 + cpl < C) ? c0 + cpl : C;
    Affine loc = affine_identity();
    for (int c = c0; c < c1; ++c) {
        const double* sc = V.si_scan + ((size_t)c * V.N + m) * 8;
        const double2 a = *reinterpret_cast<const double2*>(sc), b = *reinterpret_cast<const double2*>(sc + 2),
                      z = *reinterpret_cast<const double2*>(sc + 4);
        loc = compose(Affine{a.x, a.y, b.x, b.y, z.x, z.y}, loc);
    }
    Affine inc = loc;   // inclusive scan over the lanes of the warp
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const Affine up = shfl_up_affine(inc, o);
        if (lane >= o) inc = compose(inc, up);
    }
    if (lane == 31) wtot[warp] = inc;
    Affine exc = shfl_up_affine(inc, 1);
    if (lane == 0) exc = affine_identity();
    __syncthreads();
    Affine pre = affine_identity();   // everything before this warp
    for (int w8 = 0; w8 < warp; ++w8) pre = compose(wtot[w8], pre);
    pre = compose(exc, pre);
    // boundary inflow (ghost rows: vacuum 0, incident value, or the lagged mirror image; reading S4)
    const double e0 = pos ? P[-(int64_t)n + 4 * m + 1] : P[V.J * n + 4 * m + 0];
    const double e1 = pos ? P[-(int64_t)n + 4 * m + 3] : P[V.J * n + 4 * m + 2];
    double in_k = fma(pre.p00, e0, fma(pre.p01, e1, pre.z0));
    double in_h = fma(pre.p10, e0, fma(pre.p11, e1, pre.z1));
    for (int c = c0; c < c1; ++c) {
        double* sc = V.si_scan + ((size_t)c * V.N + m) * 8;
        const double2 a = *reinterpret_cast<const double2*>(sc), b = *reinterpret_cast<const double2*>(sc + 2),
                      z = *reinterpret_cast<const double2*>(sc + 4);
        *reinterpret_cast<double2*>(sc + 6) = make_double2(in_k, in_h);
        const double nk = fma(a.x, in_k, fma(a.y, in_h, z.x));
        const double nh = fma(b.x, in_k, fma(b.y, in_h, z.y));
        in_k = nk;
        in_h = nh;
    }
}

int launch_si_iteration(const DevView& V, int buf, int slot, int prev_slot, double tol, cudaStream_t s)
{
    const int S = si_chunk_cells(V.J, V.N, V.sm_count);
    const int C = (int)((V.J + S - 1) / S);
    int Nr = 32;
    if (V.N >= 32) Nr = (V.N + 31) / 32 * 32;
    else while (Nr / 2 >= V.N) Nr /= 2;
    const int64_t threads = (int64_t)C * Nr;
    const unsigned blocks = (unsigned)((threads + 127) / 128);
    int nlaunch = 0;
    if (C > 1) {
        if (V.nblk == 1) si_chunk_kernel<8, true, 1><<<blocks, 128, 0, s>>>(V, buf, prev_slot, tol, S, C, Nr);
        else si_chunk_kernel<4, false, 1><<<blocks, 128, 0, s>>>(V, buf, prev_slot, tol, S, C, Nr);
        si_carry_kernel<<<(unsigned)V.N, 256, 0, s>>>(V, buf, prev_slot, tol, C);
        nlaunch += 2;
    }
    if (V.nblk == 1) si_chunk_kernel<8, true, 3><<<blocks, 128, 0, s>>>(V, buf, prev_slot, tol, S, C, Nr);
    else si_chunk_kernel<4, false, 3><<<blocks, 128, 0, s>>>(V, buf, prev_slot, tol, S, C, Nr);
    nlaunch += 1 + launch_phi_norm(V, buf, slot, prev_slot, tol, true, s);
    return launched(nlaunch);
}

}  // namespace oci
