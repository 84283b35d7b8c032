// O(N) apply of the one-cell inverse through the rank-4 structure of the scattering matrix (SURVEY §8(f) row f3,
// second half; eq. (22)): B = A - S with A = blockdiag(A_m) (eqs. 20,21) and
// S = U V,  U = kappa (1_N (x) I_4)  [4N x 4],  V = (w^T (x) I_4)  [4 x 4N],  kappa = dx Sigma_s / 4   (reading G5),
// so by the Sherman-Morrison-Woodbury identity
//     B^{-1} c = t + A^{-1} U (I_4 - V A^{-1} U)^{-1} V t,      t = A^{-1} c  (one 4x4 apply per angle)
// With s = V t = sum_m w_m t_m (a 4-vector per cell) and M = (I_4 - kappa sum_m w_m A_m^{-1})^{-1}:
//     phi = V B^{-1} c = M s            (the scalar flux of the result, eq. 18)
//     Psi_m = t_m + kappa A_m^{-1} phi  (every angle sees the same self-consistent scattering source)
// about 50 N multiply-adds and 16 N doubles of operator per cell instead of (4N)^2 of each.  It holds because the
// scattering of eq. (1) is isotropic and one-group; the dense kernels remain the general method (and the roofline
// target), this family is selected only on request (oci_set_reduced_kernel(OCI_RKERNEL_WOODBURY)).
//
// The family serves the interface-reduced step of oci_reduced.cu with the same packed state (y, z, yfix, ifix,
// phifix), the same three passes and the same loop control, so everything around the kernels (fused cooperative
// iteration loop, device-side stop, sharding, layout conversion) is shared with the dense families:
//   FIX  :  c = c_fix (eqs. 27,28 without the (l) terms)            -> yfix, ifix, phifix
//   ITER :  c = |mu| inc^(l) on the two incident rows of each angle -> y^(l+1) = yfix + Psi[O], phi^(l+1) = phifix + phi
//   FINAL:  the same from inc^(L-1)                                 -> z = ifix + Psi[I]
// Two kernels.  The direct one (any N, per-cell blocks, FIX, small problems): thread = (cell, angle), the 4-vector s
// summed over the angles of a cell by warp shuffles (N a power of two) and, across the warps of a cell or for other N,
// through shared memory in a fixed order.  The TMA-staged one (ITER / FINAL, one shared block, N in {16, 32, 64, 128}):
// s = P inc as DMMA straight from the staged rows.  Both deterministic.
// HBM-bound: per cell and iteration 6N doubles of state (+ 16N + 17 of operator when every cell has its own block).
#include <cuda.h>

#include "device_utils.cuh"

namespace oci {

namespace {

// inverse of a 4x4 by Gauss-Jordan with partial pivoting, in place on [A | I]; returns false on a zero pivot
__device__ bool invert4(double (&A)[16], double (&I)[16])
{
#pragma unroll
    for (int i = 0; i < 16; ++i) I[i] = (i % 5 == 0) ? 1.0 : 0.0;
    bool ok = true;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        int p = k;
        double best = fabs(A[4 * k + k]);
#pragma unroll
        for (int i = k + 1; i < 4; ++i) {
            const double a = fabs(A[4 * i + k]);
            if (a > best) { best = a; p = i; }
        }
#pragma unroll
        for (int i = k + 1; i < 4; ++i) {
            if (i == p) {
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const double t1 = A[4 * k + c]; A[4 * k + c] = A[4 * i + c]; A[4 * i + c] = t1;
                    const double t2 = I[4 * k + c]; I[4 * k + c] = I[4 * i + c]; I[4 * i + c] = t2;
                }
            }
        }
        if (!(best > 0.0)) ok = false;
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
    return ok;
}

}  // namespace

// ---- setup: one warp per distinct block.  Element-major copies (so that the threads of a cell read them coalesced)
// of the per-angle inverses of ainv4_kernel and of their product with the 4x4 that closes the scattering source:
//     wba[b][e][m] = A_m^{-1}[e/4][e%4],   wbd[b][e][m] = (kappa A_m^{-1} M)[e/4][e%4],
//     wbm[b] = [ M (16) | kappa ],   M = (I_4 - kappa sum_m w_m A_m^{-1})^{-1},
// so that Psi_m = t_m + D_m s and phi = M s with s = sum_m w_m t_m.
__global__ void __launch_bounds__(128) woodbury_setup_kernel(DevView V)
{
    const int lane = threadIdx.x & 31;
    const int64_t b = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (b >= V.nblk) return;
    const int N = V.N;
    const int64_t r = V.rep[b];
    const double kappa = 0.25 * V.dx[r] * V.sigs[r];
    double K[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) K[e] = 0.0;
    for (int m = lane; m < N; m += 32) {
        const double* __restrict__ a = V.ainv4 + ((size_t)b * N + m) * 16;
        const double wm = V.w[m];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const double v = a[e];
            V.wba[((size_t)b * 16 + e) * N + m] = v;
            K[e] = fma(wm, v, K[e]);
        }
    }
#pragma unroll
    for (int e = 0; e < 16; ++e)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) K[e] += __shfl_xor_sync(0xffffffffu, K[e], o);
    double T[16], M[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) T[e] = ((e % 5 == 0) ? 1.0 : 0.0) - kappa * K[e];
    const bool ok = invert4(T, M);                                        // every lane (all hold the same K)
    if (lane == 0) {
        if (!ok) atomicCAS(V.flags, 0, (int)b + 1);                      // singular exactly when B is (reported like a1)
        double* out = V.wbm + (size_t)b * 32;
#pragma unroll
        for (int e = 0; e < 16; ++e) out[e] = M[e];
        out[16] = kappa;
    }
    for (int m = lane; m < N; m += 32) {
        const double* __restrict__ a = V.ainv4 + ((size_t)b * N + m) * 16;
#pragma unroll
        for (int rr = 0; rr < 4; ++rr)
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
                double d = 0.0;
#pragma unroll
                for (int k = 0; k < 4; ++k) d = fma(a[4 * rr + k], M[4 * k + cc], d);
                V.wbd[((size_t)b * 16 + 4 * rr + cc) * N + m] = kappa * d;
            }
    }
}

int launch_woodbury_setup(const DevView& V, cudaStream_t s)
{
    const int64_t threads = V.nblk * 32;
    woodbury_setup_kernel<<<(unsigned)((threads + 127) / 128), 128, 0, s>>>(V);
    return launched(1);
}

namespace {

// Sum of p over the angles of this thread's cell, delivered to every thread of the cell.  The order of the additions is
// fixed by the geometry alone and the same for every lane, so a step is reproducible bit for bit and does not depend on
// where in a CTA a cell lands.  `sm` = this call's half of a double buffer (consecutive calls alternate halves, which
// makes one CTA barrier per call enough).
// W = 0: any N - every term goes through shared memory and is summed in angle order.
// W = 8, 16, 32 (N a power of two, W = min(N, 32)): a transposing butterfly - the first level exchanges two of the four
// values and keeps two, the second exchanges one and keeps one, the remaining levels reduce a single value: 6 shuffles
// instead of 20 for a full warp, after which the lane with bits (hi, hi2) holds the total of slot 2 hi + hi2.  N <= 32:
// the four totals are broadcast by four more shuffles; N > 32: the partials of the cell's N/32 warps meet in shared memory.
template <int W>
__device__ __forceinline__ void cell_sum(double (&p)[4], int N, int cell_slot, double* __restrict__ sm)
{
    if (W == 0) {
        *reinterpret_cast<double4*>(sm + threadIdx.x * 4) = make_double4(p[0], p[1], p[2], p[3]);
        __syncthreads();
        const double* __restrict__ q = sm + (size_t)cell_slot * N * 4;
        p[0] = p[1] = p[2] = p[3] = 0.0;
        for (int k = 0; k < N; ++k) {
            const double4 a = *reinterpret_cast<const double4*>(q + k * 4);
            p[0] += a.x; p[1] += a.y; p[2] += a.z; p[3] += a.w;
        }
        return;
    }
    const int lane = threadIdx.x & 31;
    constexpr int H = W > 0 ? W / 2 : 1, Q4 = W > 0 ? W / 4 : 1;
    const bool hi = (lane & H) != 0;
    double k0 = hi ? p[2] : p[0], k1 = hi ? p[3] : p[1];
    k0 += __shfl_xor_sync(0xffffffffu, hi ? p[0] : p[2], H);
    k1 += __shfl_xor_sync(0xffffffffu, hi ? p[1] : p[3], H);
    const bool hi2 = (lane & Q4) != 0;
    double keep = hi2 ? k1 : k0;
    keep += __shfl_xor_sync(0xffffffffu, hi2 ? k0 : k1, Q4);
#pragma unroll
    for (int o = Q4 / 2; o > 0; o >>= 1) keep += __shfl_xor_sync(0xffffffffu, keep, o);
    if (N <= 32) {
        const int base = lane & ~(W - 1);
#pragma unroll
        for (int i = 0; i < 4; ++i) p[i] = __shfl_sync(0xffffffffu, keep, base + (i >> 1) * H + (i & 1) * Q4);
        return;
    }
    const int warp = threadIdx.x >> 5, wpc = N >> 5;
    if ((lane & 7) == 0) sm[warp * 4 + (lane >> 3)] = keep;               // lanes 0, 8, 16, 24 hold slots 0..3
    __syncthreads();
    const double* __restrict__ q = sm + (warp / wpc) * wpc * 4;
    p[0] = p[1] = p[2] = p[3] = 0.0;
    for (int w = 0; w < wpc; ++w) {
        const double4 a = *reinterpret_cast<const double4*>(q + w * 4);
        p[0] += a.x; p[1] += a.y; p[2] += a.z; p[3] += a.w;
    }
}

// what a thread reads for one (cell, angle): FIX - the k+1/2 entries of y and z, and Q; ITER / FINAL - the two
// gathered neighbour values and the two entries of the additive operand; pf / po: phifix and the old scalar flux of
// slot m & 3 (threads of angles 0..3 only).  Everything an item consumes is requested one item ahead, so that no
// instruction of the current item waits on a scoreboard the loads of the next item are counted on.
struct WbRaw {
    double a, b, c, d, pf, po;
    double4 q;
};

// the 4x4 pieces a pass needs for one (block, angle), scaled once.  ITER / FINAL, with a, b the two gathered values:
//   w t_m = pk a + pe b        pk, pe = w |mu| (the two columns of A_m^{-1} that the incident rows feed)
//   stored rows = [g0 a + g1 b, g2 a + g3 b] + [dk; de] s      g = |mu| (those rows of the two columns), dk, de = rows of D_m
// FIX: t = A_m^{-1} c with all four columns (pk, pe, pk2, pe2 = columns 0..3, unscaled) and all of D_m
template <int PASS>
struct WbOps {
    double pk[4], pe[4], dk[4], de[4];
    double g[PASS == PASS_FIX ? 1 : 4];
    double pk2[PASS == PASS_FIX ? 4 : 1], pe2[PASS == PASS_FIX ? 4 : 1], dk2[PASS == PASS_FIX ? 4 : 1], de2[PASS == PASS_FIX ? 4 : 1];
};

template <int PASS>
__device__ __forceinline__ void load_ops(WbOps<PASS>& O, const double* __restrict__ a, const double* __restrict__ d, int N, int half,
                                         double amu, double wm)
{
    // a, d: wba / wbd of this block at this thread's angle; element e of the 4x4 is e * N doubles further
    if (PASS == PASS_FIX) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            O.pk[r] = a[(size_t)(4 * r + 0) * N];
            O.pe[r] = a[(size_t)(4 * r + 1) * N];
            O.pk2[r] = a[(size_t)(4 * r + 2) * N];
            O.pe2[r] = a[(size_t)(4 * r + 3) * N];
            O.dk[r] = d[(size_t)(0 + r) * N];
            O.de[r] = d[(size_t)(4 + r) * N];
            O.dk2[r] = d[(size_t)(8 + r) * N];
            O.de2[r] = d[(size_t)(12 + r) * N];
        }
    } else {
        // incident rows (eqs. 27,28): (m,1),(m,3) for mu < 0 (half 0), (m,0),(m,2) for mu > 0; the pass stores the O rows
        // (the other two, ITER) or the I rows themselves (FINAL)
        const int Ik = half ? 0 : 1;
        const int Rk = PASS == PASS_ITER ? (Ik ^ 1) : Ik;
        const double* __restrict__ ac = a + (size_t)Ik * N;
        const double* __restrict__ dr = d + (size_t)(4 * Rk) * N;
        double ck[4], ce[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            ck[r] = ac[(size_t)(4 * r) * N];
            ce[r] = ac[(size_t)(4 * r + 2) * N];
            O.dk[r] = dr[(size_t)r * N];
            O.de[r] = dr[(size_t)(8 + r) * N];
        }
        O.g[0] = amu * (Rk ? ck[1] : ck[0]);
        O.g[1] = amu * (Rk ? ce[1] : ce[0]);
        O.g[2] = amu * (Rk ? ck[3] : ck[2]);
        O.g[3] = amu * (Rk ? ce[3] : ce[2]);
        const double wa = wm * amu;
#pragma unroll
        for (int r = 0; r < 4; ++r) { O.pk[r] = wa * ck[r]; O.pe[r] = wa * ce[r]; }
    }
}

}  // namespace

// ---- the three passes.  SHARED: all cells share one block, whose 4x4 pieces for this thread's angle live in registers
// for the whole launch; otherwise they are streamed per cell (coalesced over the angles).  A CTA of TPB threads takes
// TPB / N whole cells at a time (thread = (cell slot, angle)), groups of cells strided over the grid.
// IDX: the type of cell and element indices (int32_t when (J + 2) * 2N fits, which keeps the address arithmetic of the
// six streams of an item to one instruction each).
template <int PASS, bool SHARED, int TPB, int W, typename IDX>
__global__ void __launch_bounds__(TPB, TPB == 256 ? 2 : 1)
oci_red_woodbury_kernel(DevView V, int ybase, int slot, int prev_slot, double tol, int cnt, int force)
{
    extern __shared__ __align__(32) double wsm[];
    const int lane = threadIdx.x & 31;
    int ysrc = ybase;
    if (PASS == PASS_ITER) {
        if (step_done(V.norms, prev_slot, tol)) return;
    } else if (PASS == PASS_FINAL) {
        // the last executed iteration of this chunk of launches (all loads of the scan in flight at once)
        int L = 0;
        for (int i0 = 0; i0 < cnt && L == 0; i0 += 32) {
            const int i = i0 + lane;
            bool hit = false;
            if (i < cnt) {
                const double d = __longlong_as_double((long long)__ldcg(V.norms + 2 * i + 0));
                const double r = __longlong_as_double((long long)__ldcg(V.norms + 2 * i + 1));
                hit = stop_now(tol, d, r);
            }
            const unsigned msk = __ballot_sync(0xffffffffu, hit);
            if (msk) L = i0 + __ffs(msk);
        }
        if (L == 0) {
            if (!force) return;
            L = cnt;
        }
        ysrc = (ybase + L - 1) & 1;
    }
    if (PASS == PASS_FIX) clear_step_state(V);

    const int N = V.N, K2 = 2 * N, N2 = N >> 1;
    const IDX J = (IDX)V.J;
    const int cpb = TPB / N;                                               // cells a CTA handles at a time
    const int cs = threadIdx.x / N;                                        // this thread's cell slot ...
    const bool active = W > 0 || cs < cpb;                                 // (idle threads when N does not divide TPB)
    const int m = active ? threadIdx.x - cs * N : 0;                       // ... and angle
    const int cslot = active ? cs : 0;
    constexpr int sm_half = W == 0 ? 4 * TPB : 4 * (TPB / 32);

    // packed positions of this angle's two outgoing entries (k slot, k+1/2 slot)
    const int half = m >= N2, mm = m - half * N2;
    const int qk = pack_q(half, 0, mm, N), qe = pack_q(half, 1, mm, N);
    const double amu = fabs(V.mu[m]), wm = V.w[m];
    const int nbr = half ? -K2 : K2;                 // row offset of the neighbour the inflow comes from
    const bool ghost_l = PASS == PASS_ITER && !half && V.bcL == OCI_BC_REFLECTING;
    const bool ghost_r = PASS == PASS_ITER && half && V.bcR == OCI_BC_REFLECTING;
    const int mqk = mirror_q(qk, N), mqe = mirror_q(qe, N);
    // the scalar flux phi = M s (eq. 18): slot m & 3 by the threads of angles 0..3 (N = 2: slots m and m + 2)
    const bool phi_lane = PASS != PASS_FINAL && active && m < 4;
    const int psl = m & 3;

    WbOps<PASS> O;
    double alpha = 0.0, q4 = 0.0, mrow[4] = {0.0, 0.0, 0.0, 0.0};
    if (SHARED) {
        load_ops<PASS>(O, V.wba + m, V.wbd + m, N, half, amu, wm);
        const double h = V.dx[V.rep[0]];
        alpha = h / (2.0 * V.v * V.dt);
        q4 = 0.25 * h;
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) mrow[cc] = V.wbm[4 * psl + cc];
    }

    const IDX ngroups = (J + cpb - 1) / cpb;
    const IDX jstep = (IDX)gridDim.x * cpb;
    const int nloop = PASS == PASS_ITER ? (cnt > 1 ? cnt : 1) : 1;
    int flip = 0;
  for (int l = 0; l < nloop; ++l) {
    const double* __restrict__ Ys = V.y[PASS == PASS_ITER ? (ybase + l) & 1 : ysrc];
    double* __restrict__ Yd = V.y[PASS == PASS_ITER ? (ybase + l + 1) & 1 : ysrc ^ 1];
    // per-thread column pointers; j * K2 walks the cells of this thread
    const double* __restrict__ in_k = PASS == PASS_FIX ? Ys + qe : Ys + nbr + qk;
    const double* __restrict__ in_e = PASS == PASS_FIX ? V.z + qe : Ys + nbr + qe;
    const double* __restrict__ fx_k = (PASS == PASS_ITER ? V.yfix : V.ifix) + qk;
    const double* __restrict__ fx_e = (PASS == PASS_ITER ? V.yfix : V.ifix) + qe;
    double* __restrict__ out_k = (PASS == PASS_ITER ? Yd : PASS == PASS_FINAL ? V.z : V.yfix) + qk;
    double* __restrict__ out_e = (PASS == PASS_ITER ? Yd : PASS == PASS_FINAL ? V.z : V.yfix) + qe;
    // (the loaded values are not touched before the item that consumes them: a select right behind a load would make
    // the prefetch wait for its own data)
    auto load_raw = [&](IDX jc, IDX o) {
        WbRaw R;
        // ITER / FINAL: inc^(l), the neighbour's outgoing flux of the previous iterate (ghost rows at the domain faces),
        // through L2: other SMs wrote it in the previous iteration of this launch
        R.a = __ldcg(in_k + o);
        R.b = PASS == PASS_FIX ? in_e[o] : __ldcg(in_e + o);
        R.c = R.d = R.pf = R.po = 0.0;
        R.q = make_double4(0.0, 0.0, 0.0, 0.0);
        if (PASS == PASS_FIX) {
            R.q = *reinterpret_cast<const double4*>(V.Q + jc * 4);
        } else {
            R.c = fx_k[o];
            R.d = fx_e[o];
            if (PASS == PASS_ITER && phi_lane) {
                R.pf = V.phifix[jc * 4 + psl];
                R.po = __ldcg(V.phi + jc * 4 + psl);
            }
        }
        return R;
    };
    double dmax = 0.0, rmax = 0.0;
    IDX j = (IDX)blockIdx.x * cpb + cs, off = j * K2;
    const IDX ostep = jstep * K2;
    WbRaw nxt = (active && j < J) ? load_raw(j, off) : load_raw(0, 0);     // clamped: unconditional loads
    for (IDX grp = blockIdx.x; grp < ngroups; grp += gridDim.x, j += jstep, off += ostep) {
        WbRaw R = nxt;
        const bool valid = active && j < J;
        if (grp + gridDim.x < ngroups) {
            const bool okn = active && j + jstep < J;
            nxt = load_raw(okn ? j + jstep : 0, okn ? off + ostep : 0);
        }
        if (!valid) R.a = R.b = 0.0;                                       // an idle thread adds nothing to the cell sums
        int64_t b = 0;
        if (!SHARED) {
            b = V.blk[valid ? j : 0];
            load_ops<PASS>(O, V.wba + (size_t)b * 16 * N + m, V.wbd + (size_t)b * 16 * N + m, N, half, amu, wm);
            if (PASS == PASS_FIX) {
                const double h = V.dx[valid ? j : 0];
                alpha = h / (2.0 * V.v * V.dt);
                q4 = 0.25 * h;
            }
            if (phi_lane) {
#pragma unroll
                for (int cc = 0; cc < 4; ++cc) mrow[cc] = __ldg(V.wbm + (size_t)b * 32 + 4 * psl + cc);
            }
        }
        // ---- s = sum_m w_m t_m (over the cell), t = A_m^{-1} c; what is stored = t + D_m s
        double t[4], p[4];
        if (PASS == PASS_FIX) {
            // c_fix of eqs. (27),(28): psi_{k-1/2} = the k+1/2 entries of the committed state (row a8) and Q
            const double pL = half ? R.b : R.a, pR = half ? R.a : R.b;     // slots (k+1/2,L), (k+1/2,R)
            const double c0 = fma(alpha, pL, q4 * R.q.x), c1 = fma(alpha, pR, q4 * R.q.y), c2 = q4 * R.q.z, c3 = q4 * R.q.w;
            const double wv = valid ? wm : 0.0;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                t[r] = fma(O.pe2[r], c3, fma(O.pk2[r], c2, fma(O.pe[r], c1, O.pk[r] * c0)));
                p[r] = wv * t[r];
            }
        } else {
#pragma unroll
            for (int r = 0; r < 4; ++r) p[r] = fma(O.pe[r], R.b, O.pk[r] * R.a);
        }
        cell_sum<W>(p, N, cslot, wsm + (flip ? sm_half : 0));
        flip ^= 1;
        if (!valid) continue;
        if (phi_lane) {
            const double ph = fma(mrow[3], p[3], fma(mrow[2], p[2], fma(mrow[1], p[1], mrow[0] * p[0])));
            if (PASS == PASS_FIX) V.phifix[j * 4 + psl] = ph;
            if (PASS == PASS_ITER) {
                // a6: phi^(l+1) = phifix + phi and the two max-norms of the stopping rule
                const double nw = R.pf + ph;
                V.phi[j * 4 + psl] = nw;
                dmax = nanmax(dmax, fabs(nw - R.po));
                rmax = nanmax(rmax, fabs(nw));
            }
            if (N == 2) {                                                  // two angles: slots 2, 3 as well
                const double* __restrict__ Mb = V.wbm + (size_t)b * 32 + 4 * (psl + 2);
                const double ph2 = fma(Mb[3], p[3], fma(Mb[2], p[2], fma(Mb[1], p[1], Mb[0] * p[0])));
                if (PASS == PASS_FIX) V.phifix[j * 4 + psl + 2] = ph2;
                if (PASS == PASS_ITER) {
                    const double nw = V.phifix[j * 4 + psl + 2] + ph2, old = __ldcg(V.phi + j * 4 + psl + 2);
                    V.phi[j * 4 + psl + 2] = nw;
                    dmax = nanmax(dmax, fabs(nw - old));
                    rmax = nanmax(rmax, fabs(nw));
                }
            }
        }
        if (PASS == PASS_FIX) {
            double psi[4];
            psi[0] = fma(O.dk[3], p[3], fma(O.dk[2], p[2], fma(O.dk[1], p[1], fma(O.dk[0], p[0], t[0]))));
            psi[1] = fma(O.de[3], p[3], fma(O.de[2], p[2], fma(O.de[1], p[1], fma(O.de[0], p[0], t[1]))));
            psi[2] = fma(O.dk2[3], p[3], fma(O.dk2[2], p[2], fma(O.dk2[1], p[1], fma(O.dk2[0], p[0], t[2]))));
            psi[3] = fma(O.de2[3], p[3], fma(O.de2[2], p[2], fma(O.de2[1], p[1], fma(O.de2[0], p[0], t[3]))));
            out_k[off] = half ? psi[1] : psi[0];                           // yfix: O rows (a neighbour reads them)
            out_e[off] = half ? psi[3] : psi[2];
            V.ifix[off + qk] = half ? psi[0] : psi[1];                     // I rows
            V.ifix[off + qe] = half ? psi[2] : psi[3];
        } else {
            // rows (Rk, Rk + 2) of Psi_m: the O rows for ITER, the I rows for FINAL
            const double tk = fma(O.g[1], R.b, O.g[0] * R.a), te = fma(O.g[3], R.b, O.g[2] * R.a);
            const double vk = R.c + fma(O.dk[3], p[3], fma(O.dk[2], p[2], fma(O.dk[1], p[1], fma(O.dk[0], p[0], tk))));
            const double ve = R.d + fma(O.de[3], p[3], fma(O.de[2], p[2], fma(O.de[1], p[1], fma(O.de[0], p[0], te))));
            out_k[off] = vk;
            out_e[off] = ve;
            // reflecting ghost rows (reading S4): the mirror image of the edge cell's outgoing flux
            if (ghost_l && j == 0) {
                Yd[mqk - K2] = vk;
                Yd[mqe - K2] = ve;
            }
            if (ghost_r && j == J - 1) {
                Yd[(int64_t)J * K2 + mqk] = vk;
                Yd[(int64_t)J * K2 + mqe] = ve;
            }
        }
    }
    if (PASS == PASS_ITER) {
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0) {
            atomic_max_nonneg(&V.norms[2 * (slot + l) + 0], dmax);
            atomic_max_nonneg(&V.norms[2 * (slot + l) + 1], rmax);
        }
        if (nloop > 1) {
            // grid-wide barrier (cooperative launch), then the stopping rule on the now final norms (a7)
            __threadfence();
            __syncthreads();
            if (threadIdx.x == 0) {
                unsigned int* bar = reinterpret_cast<unsigned int*>(V.flags) + 8;
                atomicAdd(bar, 1u);
                const unsigned int target = (unsigned int)(l + 1) * gridDim.x;
                unsigned int seen;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory");
                } while (seen < target);
            }
            __syncthreads();
            const bool stop = step_done(V.norms, slot + l, tol) || l + 1 == nloop;
            if (stop && blockIdx.x == 0 && threadIdx.x == 0) publish_step(V, l + 1, slot + l);
            if (stop) break;
        }
    }
  }
}

// ---- ITER / FINAL with a shared block and N in {16, 32, 64, 128}: the rows STAGED BY TMA, the sum over the angles ON
// THE TENSOR PIPE.  The direct kernel above keeps one item per thread in flight and pays a 48-instruction shuffle
// butterfly per cell for s = sum_m w_m t_m: latency- and issue-bound at 53-57 % of the HBM bandwidth.  But
//     s[cell] = P inc[cell],   P = [w |mu| A_m^{-1}[:, I]]  (4 x 2N)
// is a contraction of the gathered rows with a tiny operator - the scalar-flux block of the dense kernels with A^{-1}
// in place of B^{-1} - so it runs as DMMA.8x8x4 straight from the staged rows:
//   * a producer warp streams, per group of gc = 1024 / N cells, the two half rows every cell gathers (two tensor-map
//     boxes of gc rows x (N + 4) columns: columns [0, N) of rows j0+1 .. j0+gc and columns [N, 2N) of rows j0-1 ..
//     j0+gc-2; the 4 extra columns give the bank-conflict-free pitch, as in oci_reduced_resident.cu), the gc rows of the
//     additive operand and, for ITER, the phifix / old-phi rows (1-D bulk copies) into a 2-stage ring (two CTAs per SM);
//   * phase A: warp w takes k-steps [w KS/8, (w+1) KS/8) of the KS = N/2 k-steps for all gc/8 blocks of 8 cells
//     (A fragments from the boxes, its slice of P as B fragments in registers) and leaves partial sums in shared memory;
//     256 threads add the eight partials of (cell, slot) in warp order: s, deterministic;
//   * phase B: thread = (cell, angle), four cells per thread: Psi_m = t_m + D_m s from registers and shared memory.
// About 45 instructions per (cell, 32 angles) instead of 175.
constexpr int WT_STAGES = 2;                       // two CTAs per SM: four stages in flight per SM
constexpr int WT_CONS = 256;                       // consumer threads; + one producer warp
constexpr int WT_WARPS = WT_CONS / 32;

// (two CTAs of nine warps per SM put five warps on one SM partition: 16 K registers / 5 warps = 96 per thread)
template <int PASS, int NT, int CONS>
__global__ void __launch_bounds__(CONS + 32, CONS == 256 ? 2 : 4)
oci_red_woodbury_tma_kernel(DevView V, const __grid_constant__ CUtensorMap map_y0, const __grid_constant__ CUtensorMap map_y1, int ybase,
                            int slot, int prev_slot, double tol, int cnt, int force)
{
    extern __shared__ __align__(128) unsigned char wt_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int ysrc = ybase;
    if (PASS == PASS_ITER) {
        if (step_done(V.norms, prev_slot, tol)) return;
    } else {
        int L = 0;
        for (int i0 = 0; i0 < cnt && L == 0; i0 += 32) {
            const int i = i0 + lane;
            bool hit = false;
            if (i < cnt) {
                const double d = __longlong_as_double((long long)__ldcg(V.norms + 2 * i + 0));
                const double r = __longlong_as_double((long long)__ldcg(V.norms + 2 * i + 1));
                hit = stop_now(tol, d, r);
            }
            const unsigned msk = __ballot_sync(0xffffffffu, hit);
            if (msk) L = i0 + __ffs(msk);
        }
        if (L == 0) {
            if (!force) return;
            L = cnt;
        }
        ysrc = (ybase + L - 1) & 1;
    }
    constexpr int N = NT, K2 = 2 * N, N2 = N >> 1;                         // N is a template parameter: every offset is an immediate
    const int J = (int)V.J;                                                // the launcher guarantees 32-bit element offsets
    constexpr int WARPS = CONS / 32;                                       // consumer warps; + one producer warp
    constexpr int gc = 4 * CONS / N;                                       // cells per group (stage)
    constexpr int U = 4;                                                   // cells per thread and group: gc N / 256
    constexpr int LDH = N + 4;                                             // pitch of a half-row box: 4 (mod 16) doubles
    constexpr int KS = K2 / 4, KSW = KS / WARPS;                        // k-steps of P inc, per warp
    constexpr int NB = gc / 8;                                             // blocks of 8 cells
    static_assert(KSW >= 1 && NB >= 1 && gc * N == U * CONS && KSW * WARPS == KS, "shape");
    // stage: lo box [gc][LDH] | hi box [gc][LDH] | additive rows [gc][K2] | phifix [gc][4] | old phi [gc][4]
    constexpr int box_dbl = gc * LDH, fx_dbl = gc * K2;
    constexpr int stage_dbl = 2 * box_dbl + fx_dbl + (PASS == PASS_ITER ? 8 * gc : 0);
    static_assert((box_dbl * 8) % 128 == 0 && (stage_dbl * 8) % 128 == 0, "TMA destinations stay 128-byte aligned");
    double* ring = reinterpret_cast<double*>(wt_raw);
    double* part = ring + (size_t)WT_STAGES * stage_dbl;                   // [8 warps][gc][4] partial sums of phase A
    double* s_sm = part + WARPS * gc * 4;                               // [gc][4]
    uint64_t* full = reinterpret_cast<uint64_t*>(s_sm + gc * 4);
    uint64_t* empty = full + WT_STAGES;
    volatile int* grp_s = reinterpret_cast<volatile int*>(empty + WT_STAGES);   // first cell of the group in a stage, -1: no more
    if (threadIdx.x == 0) {
        for (int st = 0; st < WT_STAGES; ++st) { mbar_init(&full[st], 1); mbar_init(&empty[st], WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int ngroups = (J + gc - 1) / gc;
    // Which groups a CTA takes.  Inside the fused loop (grid-wide barrier per iteration) they are handed out by a global
    // ticket counter, so that a CTA that runs ahead takes more and all reach the barrier together; iteration l owns the
    // tickets [l (ngroups + grid), +ngroups), and every CTA draws exactly one ticket past the end per iteration.  A
    // single pass (FINAL, one iteration per launch) takes them strided.  The producer announces the group of a stage
    // in shared memory (-1: no more) before it arms the stage.
    const bool dynamic = PASS == PASS_ITER && cnt > 1;
    int* ticket = V.flags + 12;
    const int nloop = PASS == PASS_ITER ? (cnt > 1 ? cnt : 1) : 1;
    const double* __restrict__ fx = PASS == PASS_ITER ? V.yfix : V.ifix;
    int it0 = 0;                                                           // groups this CTA has streamed in earlier iterations

    // consumer-side constants
    const bool consumer = warp < WARPS;
    const int tid = consumer ? threadIdx.x : 0;
    const int m = tid % N, c0 = tid / N;                                   // angle; first cell slot (then c0 + 256/N, ...)
    constexpr int cstep = CONS / N;
    const int half = m >= N2, mm = m - half * N2;
    const int qk = pack_q(half, 0, mm, N), qe = pack_q(half, 1, mm, N);
    const double amu = fabs(V.mu[m]), wm = V.w[m];
    const bool ghost_l = PASS == PASS_ITER && !half && V.bcL == OCI_BC_REFLECTING;
    const bool ghost_r = PASS == PASS_ITER && half && V.bcR == OCI_BC_REFLECTING;
    const int mqk = mirror_q(qk, N), mqe = mirror_q(qe, N);
    const bool phi_lane = PASS == PASS_ITER && m < 4;
    const int psl = m & 3;
    // phase B offsets inside a stage: mu < 0 (half 0) gathers from the lo box (the right neighbours' columns [0, N)),
    // mu > 0 from the hi box (the left neighbours' columns [N, 2N))
    const int o_a = (half ? box_dbl : 0) + c0 * LDH + (qk - half * N), o_b = (half ? box_dbl : 0) + c0 * LDH + (qe - half * N);
    const int o_c = 2 * box_dbl + c0 * K2 + qk, o_d = 2 * box_dbl + c0 * K2 + qe;
    const int o_pf = 2 * box_dbl + fx_dbl + c0 * 4 + psl, o_po = o_pf + 4 * gc;
    WbOps<PASS> O;
    double mrow[4] = {0.0, 0.0, 0.0, 0.0};
    double bfr[KSW];                                                       // phase A: this warp's slice of P as DMMA B fragments
    const int g4 = lane >> 2, t4 = lane & 3;
    if (consumer) {
        load_ops<PASS>(O, V.wba + m, V.wbd + m, N, half, amu, wm);
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) mrow[cc] = V.wbm[4 * psl + cc];
        // B[k][n] = P[slot n][k], n = g4 < 4 (columns 4..7 of the n8 block are zero), k = 4 ks + t4 a packed entry q:
        // P[slot][q] = w |mu| A_m^{-1}[slot][incident row of q]
#pragma unroll
        for (int i = 0; i < KSW; ++i) {
            const int q = 4 * (warp * KSW + i) + t4;
            int hq, hh, mq;
            unpack_q(q, N, hq, hh, mq);
            const int ma = hq * N2 + mq;                                   // angle of packed entry q
            const int col = (hq ? 0 : 1) + 2 * hh;                         // its incident row: (m,1),(m,3) for mu < 0, (m,0),(m,2) for mu > 0
            bfr[i] = g4 < 4 ? V.w[ma] * fabs(V.mu[ma]) * V.wba[(size_t)(4 * g4 + col) * N + ma] : 0.0;
        }
    }

  for (int l = 0; l < nloop; ++l) {
    const int ys = PASS == PASS_ITER ? (ybase + l) & 1 : ysrc;
    const CUtensorMap* my = ys ? &map_y1 : &map_y0;
    double* __restrict__ Yd = PASS == PASS_ITER ? V.y[ys ^ 1] : V.z;
    if (!consumer) {
        // ---- producer: one elected lane streams this CTA's groups of this iteration
        if (lane == 0) {
            if (l > 0) asm volatile("fence.proxy.async;" ::: "memory");   // rows other SMs stored before the grid barrier
            for (int i = 0;; ++i) {
                const int u = it0 + i, st = u % WT_STAGES;
                int g = (int)blockIdx.x + i * (int)gridDim.x;
                if (dynamic) g = atomicAdd(ticket, 1) - l * (ngroups + (int)gridDim.x);
                if (u >= WT_STAGES) mbar_wait(&empty[st], ((u / WT_STAGES) - 1) & 1);
                if (g >= ngroups) {                                        // no more groups in this iteration
                    grp_s[st] = -1;
                    mbar_arrive(&full[st]);
                    it0 = u + 1;
                    break;
                }
                const int j0 = g * gc;
                grp_s[st] = j0;
                const int rows = J - j0 < gc ? J - j0 : gc;
                double* sg = ring + (size_t)st * stage_dbl;
                const uint32_t fb = (uint32_t)rows * K2 * 8, pb = (uint32_t)rows * 32;
                mbar_expect_tx(&full[st], 2 * box_dbl * 8 + fb + (PASS == PASS_ITER ? 2 * pb : 0));
                tma_load_2d(sg, my, 0, j0 + 2, &full[st]);                 // map row = cell + 1: the right neighbours j0+1 ..
                tma_load_2d(sg + box_dbl, my, N, j0, &full[st]);           // the left neighbours j0-1 ..
                tma_load_1d(sg + 2 * box_dbl, fx + (int64_t)j0 * K2, fb, &full[st]);
                if (PASS == PASS_ITER) {
                    tma_load_1d(sg + 2 * box_dbl + fx_dbl, V.phifix + (int64_t)j0 * 4, pb, &full[st]);
                    tma_load_1d(sg + 2 * box_dbl + fx_dbl + 4 * gc, V.phi + (int64_t)j0 * 4, pb, &full[st]);
                }
            }
        }
    } else {
        double dmax = 0.0, rmax = 0.0;
        for (int i = 0;; ++i) {
            const int u = it0 + i, st = u % WT_STAGES;
            const double* sg = ring + (size_t)st * stage_dbl;
            mbar_wait(&full[st], (u / WT_STAGES) & 1);
            const int j0 = grp_s[st];
            if (j0 < 0) {                                                  // (uniform over the CTA) the iteration's last stage
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[st]);
                it0 = u + 1;
                break;
            }
            // ---- phase A: partial s = P inc over this warp's k-steps, all blocks of 8 cells
            {
                double acc[NB][2];
#pragma unroll
                for (int bq = 0; bq < NB; ++bq) acc[bq][0] = acc[bq][1] = 0.0;
#pragma unroll
                for (int ii = 0; ii < KSW; ++ii) {
                    const int ks = warp * KSW + ii;                        // 4 ks < N: lo box, else hi box
                    const double* ap = sg + (4 * ks < N ? 4 * ks : box_dbl + 4 * ks - N) + g4 * LDH + t4;
#pragma unroll
                    for (int bq = 0; bq < NB; ++bq) dmma(acc[bq][0], acc[bq][1], ap[bq * 8 * LDH], bfr[ii]);
                }
                if (t4 < 2) {
#pragma unroll
                    for (int bq = 0; bq < NB; ++bq)
                        *reinterpret_cast<double2*>(part + ((size_t)warp * gc + bq * 8 + g4) * 4 + 2 * t4) = make_double2(acc[bq][0], acc[bq][1]);
                }
            }
            named_bar_sync(1, CONS);
            if (tid < gc * 4) {
                double sum = part[tid];
#pragma unroll
                for (int w = 1; w < WARPS; ++w) sum += part[w * gc * 4 + tid];
                s_sm[tid] = sum;
            }
            named_bar_sync(1, CONS);
            // ---- phase B: thread = (cell, angle), U cells per thread, two at a time
#pragma unroll
            for (int h2 = 0; h2 < U; h2 += 2) {
                double a[2], b[2], c[2], d[2], pf[2], po[2];
                double4 sv[2];
#pragma unroll
                for (int w = 0; w < 2; ++w) {
                    const int cs = (h2 + w) * cstep;                       // + c0: this item's cell slot
                    a[w] = sg[o_a + cs * LDH];
                    b[w] = sg[o_b + cs * LDH];
                    c[w] = sg[o_c + cs * K2];
                    d[w] = sg[o_d + cs * K2];
                    pf[w] = po[w] = 0.0;
                    if (phi_lane) { pf[w] = sg[o_pf + cs * 4]; po[w] = sg[o_po + cs * 4]; }
                    sv[w] = *reinterpret_cast<const double4*>(s_sm + (c0 + cs) * 4);
                }
                if (h2 + 2 == U) {
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[st]);                // the stage is free again: everything is in registers
                }
#pragma unroll
                for (int w = 0; w < 2; ++w) {
                    const int j = j0 + c0 + (h2 + w) * cstep;
                    if (j >= J) continue;
                    const double p0 = sv[w].x, p1 = sv[w].y, p2 = sv[w].z, p3 = sv[w].w;
                    if (phi_lane) {
                        // a6: phi^(l+1) = phifix + M s and the two max-norms of the stopping rule
                        const double nw = pf[w] + fma(mrow[3], p3, fma(mrow[2], p2, fma(mrow[1], p1, mrow[0] * p0)));
                        V.phi[j * 4 + psl] = nw;
                        dmax = nanmax(dmax, fabs(nw - po[w]));
                        rmax = nanmax(rmax, fabs(nw));
                    }
                    const double tk = fma(O.g[1], b[w], O.g[0] * a[w]), te = fma(O.g[3], b[w], O.g[2] * a[w]);
                    const double vk = c[w] + fma(O.dk[3], p3, fma(O.dk[2], p2, fma(O.dk[1], p1, fma(O.dk[0], p0, tk))));
                    const double ve = d[w] + fma(O.de[3], p3, fma(O.de[2], p2, fma(O.de[1], p1, fma(O.de[0], p0, te))));
                    double* __restrict__ out = Yd + j * K2;
                    out[qk] = vk;
                    out[qe] = ve;
                    if (ghost_l && j == 0) {
                        Yd[mqk - K2] = vk;
                        Yd[mqe - K2] = ve;
                    }
                    if (ghost_r && j == J - 1) {
                        Yd[(int64_t)J * K2 + mqk] = vk;
                        Yd[(int64_t)J * K2 + mqe] = ve;
                    }
                }
            }
        }
        if (PASS == PASS_ITER) {
            dmax = warp_max(dmax);
            rmax = warp_max(rmax);
            if (lane == 0) {
                atomic_max_nonneg(&V.norms[2 * (slot + l) + 0], dmax);
                atomic_max_nonneg(&V.norms[2 * (slot + l) + 1], rmax);
            }
        }
    }
    if (PASS == PASS_ITER && nloop > 1) {
        // grid-wide barrier (cooperative launch), then the stopping rule on the now final norms (a7)
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned int* bar = reinterpret_cast<unsigned int*>(V.flags) + 8;
            atomicAdd(bar, 1u);
            const unsigned int target = (unsigned int)(l + 1) * gridDim.x;
            unsigned int seen;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory");
            } while (seen < target);
        }
        __syncthreads();
        const bool stop = step_done(V.norms, slot + l, tol) || l + 1 == nloop;
        if (stop && blockIdx.x == 0 && threadIdx.x == 0) publish_step(V, l + 1, slot + l);
        if (stop) break;
    }
  }
}

// ---- FIX with a shared block and N in {16, 32, 64, 128}, the same way: s = P_fix [psi_{k-1/2}; Q] on the tensor pipe.
// c_fix (eqs. 27,28 without the (l) terms) has 2N entries that carry psi_{k-1/2} (rows (m,0), (m,1), factor alpha) and
// an isotropic Q, so s = sum_m w_m A_m^{-1} c_fix,m = P_fix x with x = [y(k+1/2 run) | z(k+1/2 run) | Q] (the input
// vector of the dense FIX operator) and P_fix 4 x (2N + 4).  Column m of either k+1/2 run belongs to angle m, so the two
// boxes (gc rows x N + 4 columns at column N/2 of y and z) serve phase A as A fragments and phase B as per-angle reads.
// One CTA per SM (phase B holds all of A_m^{-1} and D_m: 32 doubles), three stages.
constexpr int WF_STAGES = 3;

template <int NT>
__global__ void __launch_bounds__(WT_CONS + 32, 1)
oci_red_woodbury_fix_kernel(DevView V, const __grid_constant__ CUtensorMap map_y, const __grid_constant__ CUtensorMap map_z, int ybase)
{
    extern __shared__ __align__(128) unsigned char wt_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    clear_step_state(V);
    constexpr int N = NT, K2 = 2 * N, N2 = N >> 1;
    const int J = (int)V.J;
    constexpr int gc = 1024 / N, U = 4, LDH = N + 4, KS = K2 / 4, KSW = KS / WT_WARPS, NB = gc / 8;
    constexpr int box_dbl = gc * LDH;
    constexpr int stage_dbl = 2 * box_dbl + 4 * gc;                        // y box | z box | Q rows
    static_assert((box_dbl * 8) % 128 == 0 && (stage_dbl * 8) % 128 == 0, "TMA destinations stay 128-byte aligned");
    double* ring = reinterpret_cast<double*>(wt_raw);
    double* part = ring + (size_t)WF_STAGES * stage_dbl;                   // [8 warps][gc][4]
    double* s_sm = part + WT_WARPS * gc * 4;                               // [gc][4]
    uint64_t* full = reinterpret_cast<uint64_t*>(s_sm + gc * 4);
    uint64_t* empty = full + WF_STAGES;
    if (threadIdx.x == 0) {
        for (int st = 0; st < WF_STAGES; ++st) { mbar_init(&full[st], 1); mbar_init(&empty[st], WT_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int ngroups = (J + gc - 1) / gc;
    const int my_groups = (int)blockIdx.x < ngroups ? (ngroups - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;

    if (warp >= WT_WARPS) {
        // ---- producer
        if (lane == 0) {
            for (int i = 0; i < my_groups; ++i) {
                const int st = i % WF_STAGES;
                if (i >= WF_STAGES) mbar_wait(&empty[st], ((i / WF_STAGES) - 1) & 1);
                const int j0 = ((int)blockIdx.x + i * (int)gridDim.x) * gc;
                const int rows = J - j0 < gc ? J - j0 : gc;
                double* sg = ring + (size_t)st * stage_dbl;
                mbar_expect_tx(&full[st], 2 * box_dbl * 8 + (uint32_t)rows * 32);
                tma_load_2d(sg, &map_y, N2, j0 + 1, &full[st]);            // y map row = cell + 1
                tma_load_2d(sg + box_dbl, &map_z, N2, j0, &full[st]);
                tma_load_1d(sg + 2 * box_dbl, V.Q + (int64_t)j0 * 4, (uint32_t)rows * 32, &full[st]);
            }
        }
        return;
    }
    // ---- consumers
    const int tid = threadIdx.x;
    const int m = tid % N, c0 = tid / N;                                   // angle; first cell slot (then c0 + 256/N, ...)
    constexpr int cstep = WT_CONS / N;
    const int half = m >= N2, mm = m - half * N2;
    const int qk = pack_q(half, 0, mm, N), qe = pack_q(half, 1, mm, N);
    const double wm = V.w[m];
    const bool phi_lane = m < 4;
    const int psl = m & 3;
    const double h = V.dx[V.rep[0]];
    const double alpha = h / (2.0 * V.v * V.dt), q4 = 0.25 * h;
    WbOps<PASS_FIX> O;                                                     // all of A_m^{-1} (columns 0..3) and D_m (rows 0..3)
    load_ops<PASS_FIX>(O, V.wba + m, V.wbd + m, N, half, 0.0, wm);
    double mrow[4];
#pragma unroll
    for (int cc = 0; cc < 4; ++cc) mrow[cc] = V.wbm[4 * psl + cc];
    // phase A: this warp's slice of P_fix as DMMA B fragments.  B[k][n] = P_fix[slot n][k], n = g4 < 4.  Input column u < N
    // is angle u's entry of the y run: psi_{k-1/2,L} (row (m,0)) for mu < 0, psi_{k-1/2,R} (row (m,1)) for mu > 0; column
    // N + u its entry of the z run: the other corner.  The last k-step is Q: P_fix[slot][2N + s'] = (h/4) sum_m w_m A_m^{-1}[slot][s'].
    const int g4 = lane >> 2, t4 = lane & 3;
    double bfr[KSW], bq = 0.0;
#pragma unroll
    for (int i = 0; i < KSW; ++i) {
        const int u = 4 * (warp * KSW + i) + t4;
        const int ma = u < N ? u : u - N;
        const int col = (u < N) == (ma < N2) ? 0 : 1;
        bfr[i] = g4 < 4 ? V.w[ma] * alpha * V.wba[(size_t)(4 * g4 + col) * N + ma] : 0.0;
    }
    if (warp == 0 && g4 < 4) {
        for (int ma = 0; ma < N; ++ma) bq = fma(V.w[ma], V.wba[(size_t)(4 * g4 + t4) * N + ma], bq);
        bq *= q4;
    }

    for (int i = 0; i < my_groups; ++i) {
        const int st = i % WF_STAGES;
        const int j0 = ((int)blockIdx.x + i * (int)gridDim.x) * gc;
        const double* sg = ring + (size_t)st * stage_dbl;
        mbar_wait(&full[st], (i / WF_STAGES) & 1);
        // ---- phase A: partial s over this warp's k-steps (warp 0: + the Q k-step), all blocks of 8 cells
        {
            double acc[NB][2];
#pragma unroll
            for (int bb = 0; bb < NB; ++bb) acc[bb][0] = acc[bb][1] = 0.0;
#pragma unroll
            for (int ii = 0; ii < KSW; ++ii) {
                const int ks = warp * KSW + ii;                            // 4 ks < N: the y run, else the z run
                const double* ap = sg + (4 * ks < N ? 4 * ks : box_dbl + 4 * ks - N) + g4 * LDH + t4;
#pragma unroll
                for (int bb = 0; bb < NB; ++bb) dmma(acc[bb][0], acc[bb][1], ap[bb * 8 * LDH], bfr[ii]);
            }
            if (warp == 0) {
                const double* ap = sg + 2 * box_dbl + g4 * 4 + t4;
#pragma unroll
                for (int bb = 0; bb < NB; ++bb) dmma(acc[bb][0], acc[bb][1], ap[bb * 32], bq);
            }
            if (t4 < 2) {
#pragma unroll
                for (int bb = 0; bb < NB; ++bb)
                    *reinterpret_cast<double2*>(part + ((size_t)warp * gc + bb * 8 + g4) * 4 + 2 * t4) = make_double2(acc[bb][0], acc[bb][1]);
            }
        }
        named_bar_sync(1, WT_CONS);
        if (tid < gc * 4) {
            double sum = part[tid];
#pragma unroll
            for (int w = 1; w < WT_WARPS; ++w) sum += part[w * gc * 4 + tid];
            s_sm[tid] = sum;
        }
        named_bar_sync(1, WT_CONS);
        // ---- phase B: thread = (cell, angle): c = c_fix,m, t = A_m^{-1} c, Psi_fix,m = t + D_m s
#pragma unroll
        for (int u4 = 0; u4 < U; ++u4) {
            const int cs = c0 + u4 * cstep;
            const double a = sg[cs * LDH + m], b = sg[box_dbl + cs * LDH + m];
            const double4 Q = *reinterpret_cast<const double4*>(sg + 2 * box_dbl + cs * 4);
            const double4 sv = *reinterpret_cast<const double4*>(s_sm + cs * 4);
            if (u4 + 1 == U) {
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[st]);                    // the stage is free again
            }
            const int j = j0 + cs;
            if (j >= J) continue;
            const double pL = half ? b : a, pR = half ? a : b;             // slots (k+1/2,L), (k+1/2,R) of the committed state (a8)
            const double c0v = fma(alpha, pL, q4 * Q.x), c1v = fma(alpha, pR, q4 * Q.y), c2v = q4 * Q.z, c3v = q4 * Q.w;
            double psi[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) psi[r] = fma(O.pe2[r], c3v, fma(O.pk2[r], c2v, fma(O.pe[r], c1v, O.pk[r] * c0v)));
            psi[0] = fma(O.dk[3], sv.w, fma(O.dk[2], sv.z, fma(O.dk[1], sv.y, fma(O.dk[0], sv.x, psi[0]))));
            psi[1] = fma(O.de[3], sv.w, fma(O.de[2], sv.z, fma(O.de[1], sv.y, fma(O.de[0], sv.x, psi[1]))));
            psi[2] = fma(O.dk2[3], sv.w, fma(O.dk2[2], sv.z, fma(O.dk2[1], sv.y, fma(O.dk2[0], sv.x, psi[2]))));
            psi[3] = fma(O.de2[3], sv.w, fma(O.de2[2], sv.z, fma(O.de2[1], sv.y, fma(O.de2[0], sv.x, psi[3]))));
            double* __restrict__ yf = V.yfix + j * K2;
            double* __restrict__ jf = V.ifix + j * K2;
            yf[qk] = half ? psi[1] : psi[0];                               // O rows (a neighbour reads them)
            yf[qe] = half ? psi[3] : psi[2];
            jf[qk] = half ? psi[0] : psi[1];                               // I rows
            jf[qe] = half ? psi[2] : psi[3];
            if (phi_lane) V.phifix[j * 4 + psl] = fma(mrow[3], sv.w, fma(mrow[2], sv.z, fma(mrow[1], sv.y, mrow[0] * sv.x)));
        }
    }
}

namespace {
struct WbLaunch { unsigned grid; size_t smem; };

template <int PASS, bool SHARED, int TPB, int W, typename IDX>
WbLaunch wb_config(const DevView& V)
{
    WbLaunch c{};
    c.smem = 2 * sizeof(double) * 4 * (W == 0 ? TPB : TPB / 32);
    const int cpb = TPB / V.N;
    const int64_t groups = (V.J + cpb - 1) / cpb;
    int per_sm = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, oci_red_woodbury_kernel<PASS, SHARED, TPB, W, IDX>, TPB, c.smem);
    if (per_sm < 1) per_sm = 1;
    const int64_t cap = (int64_t)V.sm_count * per_sm;                     // one resident wave (the fused loop needs it)
    c.grid = (unsigned)(groups < cap ? groups : cap);
    return c;
}

template <int PASS, bool SHARED, int TPB, int W, typename IDX>
void launch_wb_i(const DevView& V, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    const WbLaunch c = wb_config<PASS, SHARED, TPB, W, IDX>(V);
    if (PASS == PASS_ITER && cnt > 1) {
        DevView Vv = V;
        void* args[] = {&Vv, &ybase, &slot, &prev_slot, &tol, &cnt, &force};
        cudaLaunchCooperativeKernel((const void*)oci_red_woodbury_kernel<PASS, SHARED, TPB, W, IDX>, dim3(c.grid), dim3(TPB), args, c.smem, s);
        return;
    }
    oci_red_woodbury_kernel<PASS, SHARED, TPB, W, IDX><<<c.grid, TPB, c.smem, s>>>(V, ybase, slot, prev_slot, tol, cnt, force);
}

template <int PASS, bool SHARED, int TPB, int W>
void launch_wb_w(const DevView& V, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    // 32-bit indices when every element offset (ghost rows and one grid stride past the end included) fits
    const int64_t lim = (V.J + 2 + (int64_t)V.sm_count * 8 * (TPB / V.N + 1)) * 2 * V.N;
    if (lim < ((int64_t)1 << 31)) launch_wb_i<PASS, SHARED, TPB, W, int32_t>(V, ybase, slot, prev_slot, tol, cnt, force, s);
    else launch_wb_i<PASS, SHARED, TPB, W, int64_t>(V, ybase, slot, prev_slot, tol, cnt, force, s);
}

// consumer threads of a CTA: 128 (four CTAs per SM: the CTA barriers of one group overlap another CTA's work) where a
// group of 4 * 128 / N cells still has a whole block of 8 cells, else 256
int wt_cons(int N) { return N <= 64 ? 128 : 256; }

size_t wt_smem(const DevView& V, int pass)
{
    const int N = V.N, cons = wt_cons(N), gc = 4 * cons / N;
    const size_t stage = ((size_t)2 * gc * (N + 4) + (size_t)gc * 2 * N + (pass == PASS_ITER ? 8 * gc : 0)) * 8;
    return WT_STAGES * stage + (size_t)(cons / 32 + 1) * gc * 4 * 8 + 2 * WT_STAGES * 8 + WT_STAGES * 4 + 128;
}

// the TMA / tensor-pipe kernel: ITER / FINAL, one shared block, N in {16, 32, 64, 128}, 32-bit element offsets, and enough
// cell groups to give every SM a few (below that the problem is launch-latency bound and the direct kernel serves it)
bool wt_serves(const DevView& V, int pass)
{
    const int N = V.N;
    (void)pass;
    return V.nblk == 1 && (N == 16 || N == 32 || N == 64 || N == 128) && (V.J + 2) * 2 * (int64_t)N < ((int64_t)1 << 31) &&
           V.J * (int64_t)N >= (int64_t)V.sm_count * 4 * WT_CONS;
}

// tensor maps of the two y buffers (rows -1 .. J, boxes of 1024/N rows x N+4 columns), encoded per launch: a handful
// of host instructions, and no state to keep in the context
template <int PASS, int NT>
void launch_wt_w(const DevView& V, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    constexpr int CONS = NT <= 64 ? 128 : 256;
    const size_t smem = wt_smem(V, PASS);
    const int gc = 4 * CONS / NT, K2 = 2 * NT;
    CUtensorMap m0, m1;
    if (!oci_encode_2d(&m0, V.y[0] - K2, (uint64_t)V.J + 2, K2, gc, NT + 4, false) ||
        !oci_encode_2d(&m1, V.y[1] - K2, (uint64_t)V.J + 2, K2, gc, NT + 4, false)) {
        cudaMemsetAsync(nullptr, 0, 1, s);                                  // leaves an error for launched() to pick up
        return;
    }
    const int64_t groups = (V.J + gc - 1) / gc;
    int per_sm = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, oci_red_woodbury_tma_kernel<PASS, NT, CONS>, CONS + 32, smem);
    if (per_sm < 1) per_sm = 1;
    const int64_t cap = (int64_t)V.sm_count * per_sm;
    const unsigned grid = (unsigned)(groups < cap ? groups : cap);
    if (PASS == PASS_ITER && cnt > 1) {
        DevView Vv = V;
        void* args[] = {&Vv, &m0, &m1, &ybase, &slot, &prev_slot, &tol, &cnt, &force};
        cudaLaunchCooperativeKernel((const void*)oci_red_woodbury_tma_kernel<PASS, NT, CONS>, dim3(grid), dim3(CONS + 32), args, smem, s);
        return;
    }
    oci_red_woodbury_tma_kernel<PASS, NT, CONS><<<grid, CONS + 32, smem, s>>>(V, m0, m1, ybase, slot, prev_slot, tol, cnt, force);
}

size_t wf_smem(int N)
{
    const int gc = 1024 / N;
    return WF_STAGES * ((size_t)2 * gc * (N + 4) + 4 * gc) * 8 + (size_t)(WT_WARPS + 1) * gc * 4 * 8 + 2 * WF_STAGES * 8 + 128;
}

template <int NT>
void launch_wf_w(const DevView& V, int ybase, cudaStream_t s)
{
    const int gc = 1024 / NT, K2 = 2 * NT;
    CUtensorMap my, mz;
    if (!oci_encode_2d(&my, V.y[ybase & 1] - K2, (uint64_t)V.J + 2, K2, gc, NT + 4, false) ||
        !oci_encode_2d(&mz, V.z, (uint64_t)V.J, K2, gc, NT + 4, false)) {
        cudaMemsetAsync(nullptr, 0, 1, s);                                  // leaves an error for launched() to pick up
        return;
    }
    const int64_t groups = (V.J + gc - 1) / gc;
    const unsigned grid = (unsigned)(groups < V.sm_count ? groups : V.sm_count);   // (two CTAs per SM: 96 registers, spills, 82 vs 49 us)
    oci_red_woodbury_fix_kernel<NT><<<grid, WT_CONS + 32, wf_smem(NT), s>>>(V, my, mz, ybase);
}

void launch_wf(const DevView& V, int ybase, cudaStream_t s)
{
    switch (V.N) {
    case 16: launch_wf_w<16>(V, ybase, s); break;
    case 32: launch_wf_w<32>(V, ybase, s); break;
    case 64: launch_wf_w<64>(V, ybase, s); break;
    default: launch_wf_w<128>(V, ybase, s); break;
    }
}

template <int PASS>
void launch_wt(const DevView& V, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    switch (V.N) {
    case 16: launch_wt_w<PASS, 16>(V, ybase, slot, prev_slot, tol, cnt, force, s); break;
    case 32: launch_wt_w<PASS, 32>(V, ybase, slot, prev_slot, tol, cnt, force, s); break;
    case 64: launch_wt_w<PASS, 64>(V, ybase, slot, prev_slot, tol, cnt, force, s); break;
    default: launch_wt_w<PASS, 128>(V, ybase, slot, prev_slot, tol, cnt, force, s); break;
    }
}

// CTAs of 256 threads (one or more whole cells each) unless a cell has more angles than that; the butterfly for
// power-of-two N >= 8, the shared-memory sum otherwise
template <int PASS, bool SHARED>
void launch_wb(const DevView& V, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    const int N = V.N;
    if (SHARED && wt_serves(V, PASS)) {
        if (PASS == PASS_FIX) launch_wf(V, ybase, s);
        else launch_wt<PASS == PASS_FIX ? PASS_ITER : PASS>(V, ybase, slot, prev_slot, tol, cnt, force, s);
        return;
    }
    const bool pow2 = (N & (N - 1)) == 0 && N >= 8;
    if (N > 256) {
        if (pow2) launch_wb_w<PASS, SHARED, 512, 32>(V, ybase, slot, prev_slot, tol, cnt, force, s);
        else launch_wb_w<PASS, SHARED, 512, 0>(V, ybase, slot, prev_slot, tol, cnt, force, s);
    } else if (!pow2) launch_wb_w<PASS, SHARED, 256, 0>(V, ybase, slot, prev_slot, tol, cnt, force, s);
    else if (N == 8) launch_wb_w<PASS, SHARED, 256, 8>(V, ybase, slot, prev_slot, tol, cnt, force, s);
    else if (N == 16) launch_wb_w<PASS, SHARED, 256, 16>(V, ybase, slot, prev_slot, tol, cnt, force, s);
    else launch_wb_w<PASS, SHARED, 256, 32>(V, ybase, slot, prev_slot, tol, cnt, force, s);
}

template <bool SHARED>
void launch_wb_pass(const DevView& V, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    if (pass == PASS_FIX) launch_wb<PASS_FIX, SHARED>(V, ybase, 0, -1, tol, 0, 0, s);
    else if (pass == PASS_ITER) launch_wb<PASS_ITER, SHARED>(V, ybase, slot, prev_slot, tol, cnt, 0, s);
    else launch_wb<PASS_FINAL, SHARED>(V, ybase, 0, -1, tol, cnt, force, s);
}
}  // namespace

namespace {
template <int NT>
cudaError_t wt_opt_in()
{
    const auto at = cudaFuncAttributeMaxDynamicSharedMemorySize;
    const int bytes = 160 * 1024;
    constexpr int CONS = NT <= 64 ? 128 : 256;
    cudaError_t e = cudaFuncSetAttribute(oci_red_woodbury_tma_kernel<PASS_ITER, NT, CONS>, at, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(oci_red_woodbury_tma_kernel<PASS_FINAL, NT, CONS>, at, bytes);
    return e != cudaSuccess ? e : cudaFuncSetAttribute(oci_red_woodbury_fix_kernel<NT>, at, bytes);
}
}  // namespace

cudaError_t oci_red_woodbury_opt_in()
{
    cudaError_t e;
    if ((e = wt_opt_in<16>()) != cudaSuccess || (e = wt_opt_in<32>()) != cudaSuccess || (e = wt_opt_in<64>()) != cudaSuccess ||
        (e = wt_opt_in<128>()) != cudaSuccess)
        return e;
    return cudaSuccess;
}

int launch_red_woodbury(const DevView& V, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    if (V.nblk == 1) launch_wb_pass<true>(V, pass, ybase, slot, prev_slot, tol, cnt, force, s);
    else launch_wb_pass<false>(V, pass, ybase, slot, prev_slot, tol, cnt, force, s);
    return launched(1);
}

}  // namespace oci
