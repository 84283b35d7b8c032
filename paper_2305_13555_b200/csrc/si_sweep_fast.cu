// Kernel (d), fast form: the source-iteration comparator (eqs. 12-18) given the same treatment the OCI step
// got (si_sweep.cu has the method and the scan formulation; this file serves N/2 a power of two, i.e. every BASELINE
// config).  Within the iterations of a time step SI needs only the scalar flux phi^(l) and, per angle, the pair of edge
// values it carries from cell to cell - the angular flux Psi is needed ONCE, after convergence.  So an iteration
//   * never writes Psi and never re-reads it for phi: the weighted angle sum of eq. (18) is formed in the sweep itself,
//     in registers, by a butterfly reduction over the lanes of a warp that hold the angles of one direction
//     (31 shuffles for 8 cells x 4 slots x 32 angles), one partial array per group of lanes;
//   * reads psi_{k-1/2} from a compact [J][N][2] copy made once per step (half the bytes of c_fix) and the
//     angle-independent part of the right-hand side of eqs. (14),(17), (h/4)(Sigma_s phi^(l) + Q) (row d1), from a
//     [J][4] array, two buffers by iteration parity;
//   * the partials are added in a fixed order (deterministic), phi overwritten, the two max-norms of the stopping rule
//     taken and the next iteration's scattering source formed by the threads of the tile that produced them (staged
//     chunk kernels: the partials never leave shared memory) or by a tiny combine kernel (the unstaged shapes);
//   * the reflecting-boundary inflow (reading S4: lagged) travels through a per-angle inflow array instead of the
//     ghost rows of Psi.
// After the device-side stop a FINAL pass repeats the last sweep from phi^(L-1) and the stored chunk inflows and writes
// Psi^(L) and its ghost rows.  Per iteration at config 3: 2 x 68 MB read instead of 0.5 GB of traffic.
//
// A chunk c always covers cells [cS, cS+S); angles with mu < 0 walk the cells of a chunk, and the chunks, downwards.
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

// Lanes of one group (2^loggs consecutive lanes, all angles of one direction) hold NV values each.  Each step a lane
// keeps one half of its values and hands the other half to its partner (lane ^ o), adding what it receives: the
// group sum of all NV values costs NV - 1 shuffles per lane instead of NV log2(group).  Afterwards the lane with
// group index lg holds, in v[0 .. R), the sums of values [(lg >> sh) R, +R), R = max(NV >> loggs, 1); when the group
// has more lanes than there are values (sh = loggs - log2 NV > 0) the lanes with equal lg >> sh hold copies.
template <int NV, int loggs>
__device__ __forceinline__ void butterfly_reduce(double (&v)[NV], int lane)
{
    int cnt = NV / 2;
#pragma unroll
    for (int step = 0; step < 5; ++step) {
        const int o = (1 << loggs) >> (step + 1);                  // uniform over the kernel
        if (o >= 1) {
            if (cnt >= 1) {
                const bool upper = (lane & o) != 0;
#pragma unroll
                for (int i = 0; i < NV / 2; ++i) {
                    if (i < cnt) {
                        const double send = upper ? v[i] : v[i + cnt];
                        const double keep = upper ? v[i + cnt] : v[i];
                        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, o);
                    }
                }
                cnt >>= 1;
            } else {
                v[0] += __shfl_xor_sync(0xffffffffu, v[0], o);
            }
        }
    }
}

}  // namespace

// psi_{k-1/2}[j][m][L,R] <- the time-edge half (slots 2,3) of the committed iterate: this read IS the commit (a8);
// also the boundary inflow of every angle for the first iteration, from the ghost rows of Psi
__global__ void __launch_bounds__(256) si_prev_kernel(DevView V, int buf)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int N = V.N, n = V.n;
    if (t < V.J * N) *reinterpret_cast<double2*>(V.si_prev + t * 2) = *reinterpret_cast<const double2*>(V.psi[buf] + t * 4 + 2);
    if (t < V.J * 4) {                                   // d1 for the first iteration: (h/4)(Sigma_s phi^(0) + Q)
        const int64_t j = t >> 2;
        V.qs[t] = 0.25 * V.dx[j] * fma(V.sigs[j], V.phi[t], V.Q[t]);
    }
    if (t < N) {
        const int m = (int)t;
        const double* P = V.psi[buf];
        const bool pos = V.mu[m] > 0.0;
        V.si_inflow[2 * m + 0] = pos ? P[-(int64_t)n + 4 * m + 1] : P[V.J * n + 4 * m + 0];
        V.si_inflow[2 * m + 1] = pos ? P[-(int64_t)n + 4 * m + 3] : P[V.J * n + 4 * m + 2];
    }
}

// MODE 1: reduce the chunk to its affine map.  MODE 3: sweep the chunk from its inflow, accumulate the phi partials.
// MODE 4 (final): sweep the chunk and store Psi.  `it` = iteration index within the step (phi buffer parity).
// scan[(m*C + c)*8 + 0..5] = (P_c, z_c), [6..7] = inflow of chunk c (written by si_carry3_kernel).
// STAGED: the CTA's chunks are consecutive, so everything they read - the psi_{k-1/2} rows of their cells (all angles:
// one contiguous run of [J][N][2]) and the source rows - arrives as TWO bulk copies (UBLKCP) requested by one thread at
// the start of the CTA and the sweep reads shared memory: the kernel was bound by the latency of 16-byte loads issued
// from registers (1.7 TB/s at config 3), the copies of the other resident CTAs now overlap a CTA's arithmetic.
template <int U, bool SHARED_BLOCK, int MODE, int LOGGS, bool STAGED>
__global__ void __launch_bounds__(128, STAGED && SHARED_BLOCK ? 4 : 3) si_chunk2_kernel(DevView V, int buf, int it, int prev_slot, double tol, int S, int C, int Nr, int cnt, int force)
{
    extern __shared__ __align__(128) unsigned char si_smem[];
    if (MODE == 4) {
        // the last executed iteration of this chunk of launches; its phi^(L-1) and chunk inflows are still in place
        int L = first_converged(V.norms, cnt, tol);
        if (L == 0) {
            if (!force) return;
            L = cnt;
        }
        it += L - 1;
    } else if (step_done(V.norms, prev_slot, tol)) {
        return;
    }
    const int lane = threadIdx.x & 31;
    const int n = V.n, N = V.N;
    const int64_t J = V.J;
    const double* __restrict__ src_cur = (it & 1) ? V.si_src1 : V.qs;       // (h/4)(Sigma_s phi^(l) + Q), row d1
    const double* inflow_cur = V.si_inflow + (size_t)(it & 1) * 2 * N;
    double* inflow_nxt = V.si_inflow + (size_t)((it + 1) & 1) * 2 * N;
    const uint64_t pol_keep = l2_policy_evict_last();
    const double gam2 = 1.0 / (2.0 * V.v * V.dt);
    const double al0 = V.dx[V.rep[0]] * gam2;            // alpha = h / (2 v dt) of the shared block
    constexpr int loggs = LOGGS;
    const int gs = 1 << loggs;
    // STAGED: persistent CTAs walk the tiles (128 threads = 128 / Nr consecutive chunks x all angles) with a two-stage ring
    const int ntiles = (int)(((int64_t)C * Nr + 127) / 128);
    const int cpb = STAGED ? 128 / Nr : 1;               // chunks per tile
    const size_t stage_doubles = (size_t)cpb * S * (N * 2 + 4);
    uint64_t* bars = reinterpret_cast<uint64_t*>(si_smem);
    double* ring = reinterpret_cast<double*>(si_smem + 128);
    // MODE 3, staged: the scalar-flux partials of a tile stay in shared memory ([lane group][cell][4]) and the
    // tile's threads finish phi, the norms and the next scattering source themselves (the combine kernel's work, in its order)
    constexpr bool FUSED = STAGED && MODE == 3;
    const int nparts = N / 2 >= 32 ? N / 32 : 2;
    const int tile_cells = cpb * S;
    double* sphi = ring + 2 * stage_doubles;
    double dmax = 0.0, rmax = 0.0;
    const int slot = cnt;                                // MODE 3: the norm slot of this iteration rides in `cnt`
    auto request = [&](int tile, int stage) {            // one thread: the two bulk copies of a tile
        const int64_t c0 = (int64_t)tile * cpb * S;
        const int64_t c1 = (c0 + (int64_t)cpb * S < J) ? c0 + (int64_t)cpb * S : J;
        const uint32_t ncell = (uint32_t)(c1 - c0);
        double* sp = ring + stage * stage_doubles;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(&bars[stage], ncell * (uint32_t)N * 16u + ncell * 32u);
        tma_load_1d_hint(sp, V.si_prev + c0 * N * 2, ncell * (uint32_t)N * 16u, &bars[stage], pol_keep);   // re-read by the next phase: L2
        tma_load_1d(sp + (size_t)cpb * S * N * 2, src_cur + c0 * 4, ncell * 32u, &bars[stage]);
    };
    if (STAGED) {
        if (threadIdx.x == 0) {
            mbar_init(&bars[0], 1);
            mbar_init(&bars[1], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            request(blockIdx.x, 0);
            if ((int)(blockIdx.x + gridDim.x) < ntiles) request(blockIdx.x + gridDim.x, 1);
        }
        __syncthreads();
    }
    // the angle of a thread is the same in every tile (Nr divides 128)
    const int m_t = (int)(((int64_t)blockIdx.x * 128 + threadIdx.x) % Nr);
    const int m0 = m_t < N ? m_t : 0;
    double Ai[16];
    if (SHARED_BLOCK) {
#pragma unroll
        for (int i = 0; i < 16; ++i) Ai[i] = V.ainv4[(size_t)m0 * 16 + i];
    }

  int seq = 0;                                           // tiles this CTA has taken
  for (int tile = blockIdx.x; tile < (STAGED ? ntiles : (int)blockIdx.x + 1); tile += gridDim.x, ++seq) {
    const int64_t gid = (int64_t)tile * 128 + threadIdx.x;
    int m = (int)(gid % Nr);
    int64_t c = gid / Nr;
    const bool live = m < N && c < C;                    // (shuffles below need every lane of the warp)
    if (!live) { m = 0; c = STAGED ? (int64_t)tile * cpb : 0; }   // (a cell this tile has staged)
    const double mu = V.mu[m];
    const bool pos = mu > 0.0;
    const double amu = fabs(mu);
    const int stage = seq & 1;
    const double* sprev = ring + stage * stage_doubles;  // STAGED: the tile in shared memory, cells from cell0 on
    const double* ssrc = sprev + (size_t)cpb * S * N * 2;
    const int64_t cell0 = (int64_t)tile * cpb * S;
    double* sc = V.si_scan + ((size_t)m * C + c) * 8;            // angle major: the carry kernel streams one angle's maps
    // mu>0: rows 0,2 receive the incident flux (k, k+1/2) and rows 1,3 leave the cell; mu<0: mirrored
    double in_k = 0.0, in_h = 0.0;
    if (MODE != 1) {
        if (C == 1) { in_k = inflow_cur[2 * m]; in_h = inflow_cur[2 * m + 1]; }
        else { in_k = sc[6]; in_h = sc[7]; }
    }
    Affine A = affine_identity();
    const int64_t c_begin = c * S;
    const int64_t c_end = (c_begin + S < J) ? c_begin + S : J;
    const int len = (int)(c_end - c_begin);
    const double wm = V.w[m];
    // phi partials: one array per group of 2^loggs lanes
    const int part = m >> loggs;
    double* __restrict__ Pp = V.si_part + (size_t)part * J * 4;
    if (STAGED) mbar_wait(&bars[stage], (seq >> 1) & 1);

    for (int t0 = 0; t0 < S; t0 += U) {                  // uniform trip count: every lane of the warp shuffles
        double y[U][4], G[U][4][2];
        double2 e[U], s01[U], s23[U];
        double al[U];
        const double* ap[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int t = (t0 + u < len) ? t0 + u : len - 1;              // clamped: unconditional loads
            const int64_t j = pos ? c_begin + t : c_end - 1 - t;
            if (STAGED) {
                e[u] = *reinterpret_cast<const double2*>(sprev + ((j - cell0) * N + m) * 2);
                s01[u] = *reinterpret_cast<const double2*>(ssrc + (j - cell0) * 4);
                s23[u] = *reinterpret_cast<const double2*>(ssrc + (j - cell0) * 4 + 2);
            } else {
                e[u] = ldg2_hint(V.si_prev + (j * N + m) * 2, pol_keep);      // re-read twice per iteration: asked to stay in L2
                s01[u] = __ldcg(reinterpret_cast<const double2*>(src_cur + j * 4));
                s23[u] = __ldcg(reinterpret_cast<const double2*>(src_cur + j * 4 + 2));
            }
            al[u] = SHARED_BLOCK ? al0 : V.dx[j] * gam2;
            if (!SHARED_BLOCK) ap[u] = V.ainv4 + ((size_t)V.blk[j] * N + m) * 16;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            // eqs. (14),(17): b = (h/4)(Sigma_s phi^(l) + Q) + alpha psi_{k-1/2} on the k rows
            const double b[4] = {fma(al[u], e[u].x, s01[u].x), fma(al[u], e[u].y, s01[u].y), s23[u].x, s23[u].y};
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
        double v[4 * U];
        // ---- the sequential chain: two dependent FMAs per cell
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const bool in = t0 + u < len;
            if (MODE == 1) {
                if (in) {
                    Affine g;
                    g.p00 = pos ? G[u][1][0] : G[u][0][0];  g.p01 = pos ? G[u][1][1] : G[u][0][1];
                    g.p10 = pos ? G[u][3][0] : G[u][2][0];  g.p11 = pos ? G[u][3][1] : G[u][2][1];
                    g.z0 = pos ? y[u][1] : y[u][0];
                    g.z1 = pos ? y[u][3] : y[u][2];
                    A = compose(g, A);
                }
            } else {
                double x[4];
#pragma unroll
                for (int r = 0; r < 4; ++r) x[r] = fma(G[u][r][1], in_h, fma(G[u][r][0], in_k, y[u][r]));
                if (in) {
                    in_k = pos ? x[1] : x[0];
                    in_h = pos ? x[3] : x[2];
                }
                if (MODE == 4) {
                    if (in && live) {
                        const int64_t j = pos ? c_begin + t0 + u : c_end - 1 - (t0 + u);
                        double* P = V.psi[buf];
                        *reinterpret_cast<double2*>(P + j * n + 4 * m) = make_double2(x[0], x[1]);
                        *reinterpret_cast<double2*>(P + j * n + 4 * m + 2) = make_double2(x[2], x[3]);
                    }
                } else {
                    // eq. (18): this angle's share of phi of the u-th cell of the block (0 outside the chunk)
                    const double ww = (in && live) ? wm : 0.0;
#pragma unroll
                    for (int r = 0; r < 4; ++r) v[4 * u + r] = ww * x[r];
                }
            }
        }
        if (MODE == 3) {
            butterfly_reduce<4 * U, LOGGS>(v, lane);
            constexpr int lognv = U == 8 ? 5 : 4;
            constexpr int sh = loggs > lognv ? loggs - lognv : 0;
            constexpr int R = loggs >= lognv ? 1 : (4 * U) >> loggs;
            const int lg = lane & (gs - 1);
            if ((lg & ((1 << sh) - 1)) == 0) {
#pragma unroll
                for (int i = 0; i < 4 * U; ++i) {
                    if (i < R) {
                        const int idx = (lg >> sh) * R + i, u = idx >> 2, r = idx & 3;
                        if (t0 + u < len && live) {
                            const int64_t j = pos ? c_begin + t0 + u : c_end - 1 - (t0 + u);
                            if (FUSED) sphi[((size_t)part * tile_cells + (j - cell0)) * 4 + r] = v[i];
                            else Pp[j * 4 + r] = v[i];
                        }
                    }
                }
            }
        }
    }
    if (live) {
    if (MODE == 1) {
        *reinterpret_cast<double2*>(sc + 0) = make_double2(A.p00, A.p01);
        *reinterpret_cast<double2*>(sc + 2) = make_double2(A.p10, A.p11);
        *reinterpret_cast<double2*>(sc + 4) = make_double2(A.z0, A.z1);
    } else {
        // the chunk an angle leaves the slab through: its outflow is the mirror angle's inflow at a reflecting face
        // (reading S4: used by the NEXT iteration); an angle whose own inflow face is not reflecting keeps its constant
        const bool last = pos ? c == C - 1 : c == 0, first = pos ? c == 0 : c == C - 1;
        const int out_bc = pos ? V.bcR : V.bcL, in_bc = pos ? V.bcL : V.bcR;
        const int mir = N - 1 - m;
        if (MODE == 3) {
            if (last && out_bc == OCI_BC_REFLECTING) { inflow_nxt[2 * mir] = in_k; inflow_nxt[2 * mir + 1] = in_h; }
            if (first && in_bc != OCI_BC_REFLECTING) { inflow_nxt[2 * m] = inflow_cur[2 * m]; inflow_nxt[2 * m + 1] = inflow_cur[2 * m + 1]; }
        } else if (last && out_bc == OCI_BC_REFLECTING) {
            // ghost rows of Psi^(L), where a cell beyond the face would keep the values the edge cell gathers
            double* P = V.psi[buf];
            if (pos) { P[J * n + 4 * mir + 0] = in_k; P[J * n + 4 * mir + 2] = in_h; }
            else { P[-(int64_t)n + 4 * mir + 1] = in_k; P[-(int64_t)n + 4 * mir + 3] = in_h; }
        }
    }
    }
    if (FUSED || (STAGED && tile + 2 * (int)gridDim.x < ntiles)) {   // the stage is free once every thread has left it: refill it
        __syncthreads();
        if (threadIdx.x == 0 && tile + 2 * (int)gridDim.x < ntiles) request(tile + 2 * gridDim.x, stage);
    }
    if (FUSED) {
        double* __restrict__ src_nxt = (it & 1) ? V.qs : V.si_src1;
        const int64_t cell1 = (cell0 + tile_cells < J) ? cell0 + tile_cells : J;
        const int units = (int)(cell1 - cell0) * 2;          // 16-byte units of phi
        for (int e = threadIdx.x; e < units; e += 128) {
            const int64_t ge = cell0 * 2 + e;
            const double2 o = reinterpret_cast<const double2*>(V.phi)[ge];
            const double2 q = reinterpret_cast<const double2*>(V.Q)[ge];
            const int64_t j = ge >> 1;
            const double q4 = 0.25 * V.dx[j], sg = V.sigs[j];
            double2 sum = make_double2(0.0, 0.0);
            for (int pp = 0; pp < nparts; ++pp) {
                const double2 v2 = *reinterpret_cast<const double2*>(sphi + ((size_t)pp * tile_cells) * 4 + 2 * e);
                sum.x += v2.x;
                sum.y += v2.y;
            }
            reinterpret_cast<double2*>(V.phi)[ge] = sum;
            reinterpret_cast<double2*>(src_nxt)[ge] = make_double2(q4 * fma(sg, sum.x, q.x), q4 * fma(sg, sum.y, q.y));
            dmax = nanmax(dmax, nanmax(fabs(sum.x - o.x), fabs(sum.y - o.y)));
            rmax = nanmax(rmax, nanmax(fabs(sum.x), fabs(sum.y)));
        }
        __syncthreads();                                     // the next tile's partials go to the same place
    }
  }
  if (FUSED) {
      __shared__ double sd[4], sr[4];
      dmax = warp_max(dmax);
      rmax = warp_max(rmax);
      if (lane == 0) { sd[threadIdx.x >> 5] = dmax; sr[threadIdx.x >> 5] = rmax; }
      __syncthreads();
      if (threadIdx.x == 0) {
          for (int q = 1; q < 4; ++q) { dmax = nanmax(dmax, sd[q]); rmax = nanmax(rmax, sr[q]); }
          atomic_max_nonneg(&V.norms[2 * slot + 0], dmax);
          atomic_max_nonneg(&V.norms[2 * slot + 1], rmax);
      }
  }
}

// Exclusive scan of the chunk maps of one angle in its direction of travel, applied to the boundary inflow.  An angle's
// C chunks are cut into G segments of CARRY_T * CARRY_K chunks; a CTA takes one (segment, angle) - handed out by a
// ticket counter in segment-major order, so a CTA only ever waits for CTAs that are already running - loads the
// CARRY_K maps of each thread up front (ONE DRAM round trip instead of one per map), scans them (thread, warp shuffle,
// CTA), publishes the composition of its segment in si_agg and composes the segments before its own from there (they
// are all published at about the same time: one L2 round trip; released by a tag that is unique to the launch: the
// ticket counter never goes back, ticket / (N G) + 1 = the launch's epoch).  Config 3 (8192 chunks per angle): 37 us -> see DESIGN.md 6.6.
constexpr int CARRY_T = 512, CARRY_K = 4;

__global__ void __launch_bounds__(CARRY_T) si_carry3_kernel(DevView V, int it, int prev_slot, double tol, int C, int G)
{
    if (step_done(V.norms, prev_slot, tol)) return;      // (every CTA of the launch takes this branch or none does)
    __shared__ Affine wtot[CARRY_T / 32];
    __shared__ Affine s_before;
    __shared__ unsigned long long s_ticket;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, N = V.N;
    if (tid == 0) s_ticket = atomicAdd(reinterpret_cast<unsigned long long*>(V.flags + 16), 1ull);
    __syncthreads();
    const unsigned long long per = (unsigned long long)N * G;
    const unsigned long long tag = s_ticket / per + 1;
    const int local = (int)(s_ticket % per), g = local / N, m = local - g * N;
    const bool pos = V.mu[m] > 0.0;
    auto chunk_of = [&](int tau) { return pos ? tau : C - 1 - tau; };
    const int c0 = g * (CARRY_T * CARRY_K) + tid * CARRY_K;       // positions in travel order
    double2 a[CARRY_K], b[CARRY_K], z[CARRY_K];
#pragma unroll
    for (int k = 0; k < CARRY_K; ++k) {
        const int tau = c0 + k < C ? c0 + k : C - 1;
        const double* sc = V.si_scan + ((size_t)m * C + chunk_of(tau)) * 8;
        a[k] = __ldcg(reinterpret_cast<const double2*>(sc));
        b[k] = __ldcg(reinterpret_cast<const double2*>(sc + 2));
        z[k] = __ldcg(reinterpret_cast<const double2*>(sc + 4));
    }
    Affine loc = affine_identity();
#pragma unroll
    for (int k = 0; k < CARRY_K; ++k)
        if (c0 + k < C) loc = compose(Affine{a[k].x, a[k].y, b[k].x, b[k].y, z[k].x, z[k].y}, loc);
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
    if (warp == 0) {
        // every CTA publishes the composition of ITS segment as soon as it has it (nobody waits to publish), then lane q
        // of warp 0 fetches segment q's and the lanes compose them in order: one L2 round trip, not a chain of G - 1
        if (lane == 0 && g + 1 < G) {
            Affine own = affine_identity();
            for (int w = 0; w < CARRY_T / 32; ++w) own = compose(wtot[w], own);
            double* rec = V.si_agg + ((size_t)m * G + g) * 8;
            rec[0] = own.p00; rec[1] = own.p01; rec[2] = own.p10; rec[3] = own.p11;
            rec[4] = own.z0;  rec[5] = own.z1;
            asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(rec + 7), "l"(tag) : "memory");
        }
        Affine before = affine_identity();
        for (int q0 = 0; q0 < g; q0 += 32) {             // (G <= 32 for every slab up to 2^21 cells: one pass)
            Affine mine = affine_identity();
            if (q0 + lane < g) {
                const double* rec = V.si_agg + ((size_t)m * G + q0 + lane) * 8;
                unsigned long long seen;
                do {
                    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(rec + 7) : "memory");
                } while (seen != tag);
                mine = Affine{__ldcg(rec + 0), __ldcg(rec + 1), __ldcg(rec + 2), __ldcg(rec + 3), __ldcg(rec + 4), __ldcg(rec + 5)};
            }
            // inclusive scan over the lanes (identity beyond g), the last lane holds the composition of this pass
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const Affine up = shfl_up_affine(mine, o);
                if (lane >= o) mine = compose(mine, up);
            }
            const Affine all = Affine{__shfl_sync(0xffffffffu, mine.p00, 31), __shfl_sync(0xffffffffu, mine.p01, 31),
                                      __shfl_sync(0xffffffffu, mine.p10, 31), __shfl_sync(0xffffffffu, mine.p11, 31),
                                      __shfl_sync(0xffffffffu, mine.z0, 31),  __shfl_sync(0xffffffffu, mine.z1, 31)};
            before = compose(all, before);
        }
        if (lane == 0) s_before = before;
    }
    __syncthreads();
    Affine pre = s_before;            // everything before this warp
    for (int w = 0; w < warp; ++w) pre = compose(wtot[w], pre);
    pre = compose(exc, pre);
    const double* inflow_cur = V.si_inflow + (size_t)(it & 1) * 2 * N;
    const double e0 = inflow_cur[2 * m], e1 = inflow_cur[2 * m + 1];
    double in_k = fma(pre.p00, e0, fma(pre.p01, e1, pre.z0));
    double in_h = fma(pre.p10, e0, fma(pre.p11, e1, pre.z1));
#pragma unroll
    for (int k = 0; k < CARRY_K; ++k) {
        if (c0 + k < C) {
            double* sc = V.si_scan + ((size_t)m * C + chunk_of(c0 + k)) * 8;
            *reinterpret_cast<double2*>(sc + 6) = make_double2(in_k, in_h);
            const double nk = fma(a[k].x, in_k, fma(a[k].y, in_h, z[k].x));
            const double nh = fma(b[k].x, in_k, fma(b[k].y, in_h, z[k].y));
            in_k = nk;
            in_h = nh;
        }
    }
}

// phi^(l+1) = sum of the partials (fixed order), the two max-norms against phi^(l), and the next iteration's
// scattering source (h/4)(Sigma_s phi^(l+1) + Q) into the other source buffer (the FINAL pass re-reads this one).
// One 16-byte unit per thread and every load of the unit requested before the first one is used: the kernel is a handful
// of dependent DRAM round trips otherwise (38 us at config 3 with a grid-stride loop over 296 CTAs, 5 us like this).
template <int PARTS>
__global__ void __launch_bounds__(256) si_combine_kernel(DevView V, int it, int slot, int prev_slot, double tol)
{
    if (step_done(V.norms, prev_slot, tol)) return;
    double* __restrict__ src_nxt = (it & 1) ? V.qs : V.si_src1;
    const int64_t tot = V.J * 2;                         // 16-byte units
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double dmax = 0.0, rmax = 0.0;
    if (e < tot) {
        double2 v[PARTS];
#pragma unroll
        for (int p = 0; p < PARTS; ++p) v[p] = __ldcg(reinterpret_cast<const double2*>(V.si_part + (size_t)p * V.J * 4) + e);
        const double2 o = reinterpret_cast<const double2*>(V.phi)[e];
        const double2 q = reinterpret_cast<const double2*>(V.Q)[e];
        const int64_t j = e >> 1;
        const double q4 = 0.25 * V.dx[j], sg = V.sigs[j];
        double2 s = make_double2(0.0, 0.0);
#pragma unroll
        for (int p = 0; p < PARTS; ++p) {
            s.x += v[p].x;
            s.y += v[p].y;
        }
        reinterpret_cast<double2*>(V.phi)[e] = s;
        reinterpret_cast<double2*>(src_nxt)[e] = make_double2(q4 * fma(sg, s.x, q.x), q4 * fma(sg, s.y, q.y));
        dmax = nanmax(fabs(s.x - o.x), fabs(s.y - o.y));
        rmax = nanmax(fabs(s.x), fabs(s.y));
    }
    __shared__ double sd[8], sr[8];
    dmax = warp_max(dmax);
    rmax = warp_max(rmax);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { sd[warp] = dmax; sr[warp] = rmax; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q) { dmax = nanmax(dmax, sd[q]); rmax = nanmax(rmax, sr[q]); }
        atomic_max_nonneg(&V.norms[2 * slot + 0], dmax);
        atomic_max_nonneg(&V.norms[2 * slot + 1], rmax);
    }
}

// N/2 a power of two: the lanes of a direction form groups of 2^k (k <= 5) for the butterfly
bool si_fast_supported(const DevView& V)
{
    const int h = V.N / 2;
    return h >= 1 && (h & (h - 1)) == 0;
}

// segments of the carry scan per angle for C chunks (si_agg holds [N][segments][8] doubles)
int si_carry_segments(int64_t C) { return (int)((C + CARRY_T * CARRY_K - 1) / (CARRY_T * CARRY_K)); }

int si_fast_parts(const DevView& V)
{
    const int h = V.N / 2;
    return h >= 32 ? V.N / 32 : 2;
}

namespace {
struct SiGeom { int S, C, Nr, loggs; unsigned blocks; };
SiGeom si_geom(const DevView& V)
{
    SiGeom g{};
    // short chunks: the sweeps are latency bound, so parallelism over cells matters more than the length of the scan
    g.S = si_chunk_cells(V.J, V.N, V.sm_count);
    if (g.S > 16) g.S = V.J <= 32 ? g.S : 16;
    g.C = (int)((V.J + g.S - 1) / g.S);
    g.Nr = 32;
    if (V.N >= 32) g.Nr = (V.N + 31) / 32 * 32;
    else while (g.Nr / 2 >= V.N) g.Nr /= 2;
    const int h = V.N / 2;
    g.loggs = 0;
    while ((1 << (g.loggs + 1)) <= (h < 32 ? h : 32)) ++g.loggs;
    g.blocks = (unsigned)(((int64_t)g.C * g.Nr + 127) / 128);
    return g;
}
}  // namespace

int launch_si_fast_begin(const DevView& V, int buf, cudaStream_t s)
{
    const int64_t tot = V.J * (V.N > 4 ? V.N : 4);
    si_prev_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(V, buf);
    return launched(1);
}

namespace {
// returns true when the staged form ran (MODE 3: it has then done the combine kernel's work as well)
template <int MODE, int LG>
bool launch_chunk2(const DevView& V, const SiGeom& g, int buf, int it, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    // staged form: a tile covers whole chunks (Nr <= 128); persistent CTAs, as many as are resident (about three per SM), two tiles of shared
    // memory each (at most 2 x 34 KB + the barriers: opted in by si_fast_opt_in)
    const size_t stage_bytes = g.Nr <= 128 ? (size_t)(128 / g.Nr) * g.S * ((size_t)V.N * 16 + 32) : 0;
    const size_t smem = stage_bytes == 0 ? 0 : 128 + 2 * stage_bytes + (MODE == 3 ? (size_t)si_fast_parts(V) * (128 / g.Nr) * g.S * 32 : 0);
    if (stage_bytes > 0 && stage_bytes <= 36 * 1024 && smem <= 80 * 1024) {
        const unsigned per_sm = (unsigned)(227 * 1024 / (smem + 1024));     // resident CTAs: one wave
        const unsigned grid = g.blocks < per_sm * (unsigned)V.sm_count ? g.blocks : per_sm * (unsigned)V.sm_count;
        if (V.nblk == 1) si_chunk2_kernel<4, true, MODE, LG, true><<<grid, 128, smem, s>>>(V, buf, it, prev_slot, tol, g.S, g.C, g.Nr, cnt, force);
        else si_chunk2_kernel<4, false, MODE, LG, true><<<grid, 128, smem, s>>>(V, buf, it, prev_slot, tol, g.S, g.C, g.Nr, cnt, force);
        return true;
    }
    if (V.nblk == 1) si_chunk2_kernel<4, true, MODE, LG, false><<<g.blocks, 128, 0, s>>>(V, buf, it, prev_slot, tol, g.S, g.C, g.Nr, cnt, force);
    else si_chunk2_kernel<4, false, MODE, LG, false><<<g.blocks, 128, 0, s>>>(V, buf, it, prev_slot, tol, g.S, g.C, g.Nr, cnt, force);
    return false;
}
}  // namespace

namespace {
template <int MODE, int LG>
cudaError_t opt_in_chunk2()
{
    cudaError_t e = cudaFuncSetAttribute(si_chunk2_kernel<4, true, MODE, LG, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 80 * 1024);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(si_chunk2_kernel<4, false, MODE, LG, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 80 * 1024);
}
}  // namespace

// the staged chunk kernels keep two tiles in shared memory (per device: called by oci_setup)
cudaError_t si_fast_opt_in()
{
    cudaError_t e;
    if ((e = opt_in_chunk2<1, 0>()) != cudaSuccess || (e = opt_in_chunk2<4, 0>()) != cudaSuccess ||
        (e = opt_in_chunk2<3, 0>()) != cudaSuccess || (e = opt_in_chunk2<3, 1>()) != cudaSuccess ||
        (e = opt_in_chunk2<3, 2>()) != cudaSuccess || (e = opt_in_chunk2<3, 3>()) != cudaSuccess ||
        (e = opt_in_chunk2<3, 4>()) != cudaSuccess || (e = opt_in_chunk2<3, 5>()) != cudaSuccess)
        return e;
    return cudaSuccess;
}

// `it`: iteration index within the step (source buffer parity); slot / prev_slot: norm slots within the launch chunk
int launch_si_fast_iteration(const DevView& V, int buf, int it, int slot, int prev_slot, double tol, cudaStream_t s)
{
    const SiGeom g = si_geom(V);
    int k = 0;
    if (g.C > 1) {
        launch_chunk2<1, 0>(V, g, buf, it, prev_slot, tol, 0, 0, s);
        const int G = si_carry_segments(g.C);
        si_carry3_kernel<<<(unsigned)(V.N * G), CARRY_T, 0, s>>>(V, it, prev_slot, tol, g.C, G);
        k += 2;
    }
    bool fused = false;                                  // (MODE 3 takes the norm slot in place of `cnt`)
    switch (g.loggs) {                                   // lanes per direction group of the butterfly: 2^loggs
    case 0: fused = launch_chunk2<3, 0>(V, g, buf, it, prev_slot, tol, slot, 0, s); break;
    case 1: fused = launch_chunk2<3, 1>(V, g, buf, it, prev_slot, tol, slot, 0, s); break;
    case 2: fused = launch_chunk2<3, 2>(V, g, buf, it, prev_slot, tol, slot, 0, s); break;
    case 3: fused = launch_chunk2<3, 3>(V, g, buf, it, prev_slot, tol, slot, 0, s); break;
    case 4: fused = launch_chunk2<3, 4>(V, g, buf, it, prev_slot, tol, slot, 0, s); break;
    default: fused = launch_chunk2<3, 5>(V, g, buf, it, prev_slot, tol, slot, 0, s); break;
    }
    if (fused) return launched(k + 1);
    const unsigned cb = (unsigned)((V.J * 2 + 255) / 256);
    switch (si_fast_parts(V)) {
    case 2: si_combine_kernel<2><<<cb, 256, 0, s>>>(V, it, slot, prev_slot, tol); break;
    case 4: si_combine_kernel<4><<<cb, 256, 0, s>>>(V, it, slot, prev_slot, tol); break;
    case 8: si_combine_kernel<8><<<cb, 256, 0, s>>>(V, it, slot, prev_slot, tol); break;
    default: si_combine_kernel<16><<<cb, 256, 0, s>>>(V, it, slot, prev_slot, tol); break;
    }
    return launched(k + 2);
}

// it0: iteration index of the first of the `cnt` queued iterations
int launch_si_fast_final(const DevView& V, int buf, int it0, double tol, int cnt, int force, cudaStream_t s)
{
    const SiGeom g = si_geom(V);
    launch_chunk2<4, 0>(V, g, buf, it0, -1, tol, cnt, force, s);
    return launched(1);
}

}  // namespace oci
