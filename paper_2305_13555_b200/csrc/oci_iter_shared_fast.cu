// Kernel (b)+(c), shared-block fast path for block sizes n = 4N in {64, 128} ("resident" form).
//
// Psi^(l+1)[j] = B^{-1} c[j] for all cells is the dense contraction [J x n] = [J x n].[n x n]^T
// (eq. 19, one inverse for the whole slab).  On sm_100a the fp64 tensor pipe is reached only
// by mma.sync DMMA.8x8x4 (tcgen05 has no f64 kind), one instruction per 16 clk per SM sub-partition,
// so the issue slots are nearly free and the design goal is to keep that pipe fed:
//
//   * one persistent CTA per SM, 8 MMA warps + 4 auxiliary warps; MMA warp w owns output rows [n/8*w, n/8*(w+1)) and keeps its
//     slice of B^{-1} as DMMA B-fragments IN REGISTERS for the whole kernel (n=128: 64 doubles per
//     thread) - the inverse is read from L2 once per CTA per launch and never touches shared memory;
//   * cell tiles of 32 stream through shared-memory rings filled by 1-D bulk TMA
//     (cp.async.bulk + mbarrier complete_tx): per cell the c_fix row and the two neighbour half-rows
//     the RHS needs (rows a3: first half of Psi^(l)[j+1], second half of Psi^(l)[j-1]; ghost rows make
//     the domain edges look like neighbours);
//   * the RHS (row a4) is assembled in place in shared memory, c = c_fix + coef * psi_nbr[k^1], only on
//     the 2N rows that take an incident flux; rows are padded to stride = 4 (mod 16) doubles so the
//     A-fragment loads are bank-conflict free;
//   * epilogue: accumulators -> global Psi^(l+1) (16-byte stores), the scalar flux (eq. 18) reduced
//     across lanes by shuffle and across warps through shared memory, the two max-norms by atomicMax
//     (row a6), and the reflecting ghost rows (reading S4) - no second pass over Psi.
#include "device_utils.cuh"

namespace oci {

namespace {

constexpr int TM = 32;        // cells per tile
constexpr int CSLOTS = 4;    // RHS tiles in flight (loaded / assembled / in the DMMAs)
constexpr int PSLOTS = 2;    // neighbour half-row tiles in flight (dead once the RHS is assembled)

#ifdef OCI_DBG_TRACE
#define TRACE(slotidx)                                                                        \
    do {                                                                                      \
        if (lane == 0 && blockIdx.x == 5 && it < 32) {                                        \
            unsigned long long t_;                                                            \
            asm volatile("mov.u64 %0, %%clock64;" : "=l"(t_)::"memory");                      \
            reinterpret_cast<unsigned long long*>(V.qs)[(warp * 32 + it) * 8 + (slotidx)] = t_; \
        }                                                                                     \
    } while (0)
#else
#define TRACE(slotidx) do {} while (0)
#endif

template <int NT>
struct Cfg {
    static constexpr int LD = NT + 4;                 // padded row (doubles): LD = 4 (mod 16)
    static constexpr int KS = NT / 4;                 // k-steps of 4
    static constexpr int NB = NT / 64;                // n8 blocks per warp (8 warps)
    static constexpr int TILE_DOUBLES = TM * LD;
    static constexpr size_t SMEM = sizeof(double) * ((CSLOTS + PSLOTS) * TILE_DOUBLES + 3 * 8 * TM * 4) + (3 * CSLOTS + 3) * 8 + 64;
};

}  // namespace

// Warp roles: warps 0..7 = MMA warps (two warpgroups, 224 registers each after setmaxnreg); warps 8..10
// of the auxiliary warpgroup (56 registers) issue TMA.
//
// The fp64 pipe is shared by DMMA and DFMA/DADD, and a saturating DMMA stream starves the fp64
// instructions of other warps, so ALL fp64 work lives in the MMA warps, as side work that is
// independent of the current tile's DMMAs and interleaved with them by the instruction scheduler:
// while the DMMAs of tile t run, each thread assembles 8 RHS values of tile t+1 and (warps 0..3)
// reduces the scalar flux of tile t-2.  No wait in the steady state blocks (every barrier a warp
// waits on was completed about a tile earlier), so the warps drift apart and cover each other's
// epilogues.  Hand-offs (mbarriers):
//   full[s]   TMA bytes of RHS slot s (and its neighbour slot) have landed (3 arrivals + tx bytes)
//   cdone[s]  RHS of stage s assembled                    (256 arrivals, mid-way through the previous tile)
//   freeb[s]  MMA warps are done with stage s             (8 arrivals)   the issuer waits
//   pw[b]     phi partials of buffer b written            (8 arrivals)   reduced two tiles later
constexpr int PBUF = 3;
template <int NT>
__global__ void __launch_bounds__(384, 1)
oci_iter_resident_kernel(DevView V, int src, int slot, int prev_slot, double tol)
{
    using C = Cfg<NT>;
    if (step_done(V.norms, prev_slot, tol)) return;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* cbuf = reinterpret_cast<double*>(smem_raw);                          // [CSLOTS][TM][LD]  c_fix -> RHS
    double* pbuf = cbuf + CSLOTS * C::TILE_DOUBLES;                              // [PSLOTS][TM][LD]  neighbour half-rows
    double* phi_part = pbuf + PSLOTS * C::TILE_DOUBLES;                          // [PBUF][8 warps][TM][4]
    uint64_t* full = reinterpret_cast<uint64_t*>(phi_part + PBUF * 8 * TM * 4);  // [CSLOTS]
    uint64_t* cdone = full + CSLOTS;
    uint64_t* freeb = cdone + CSLOTS;
    uint64_t* pw = freeb + CSLOTS;                                               // [PBUF]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int N = NT / 4, HALF = NT / 2;
    const int64_t J = V.J;
    const double* __restrict__ Pold = V.psi[src];
    double* __restrict__ Pnew = V.psi[src ^ 1];
    const int64_t ntiles = (J + TM - 1) / TM;
    const int my_tiles = (int)((ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x);   // >= 1
    auto tile_j0 = [&](int it) { return ((int64_t)blockIdx.x + (int64_t)it * gridDim.x) * TM; };
    auto tile_rows = [&](int it) {
        const int64_t j0 = tile_j0(it);
        return (int)((J - j0 < TM) ? (J - j0) : TM);
    };

    if (tid == 0) {
        for (int s = 0; s < CSLOTS; ++s) {
            mbar_init(&full[s], 3);
            mbar_init(&cdone[s], 256);
            mbar_init(&freeb[s], 8);
        }
        for (int b = 0; b < PBUF; ++b) mbar_init(&pw[b], 8);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= 8) {
        // =========================== loader warps ===========================
        // 1-D bulk TMA, one cell row per lane: warp 8 copies the c_fix rows, warp 9 the first half of
        // Psi^(l)[j+1] (k < n/2), warp 10 the second half of Psi^(l)[j-1] (k >= n/2) (rows a3).  A tile is
        // requested as soon as its RHS slot (ring of CSLOTS, freed when the DMMAs of tile it-CSLOTS end) and
        // its neighbour slot (ring of PSLOTS, freed when tile it-PSLOTS has been assembled) are free:
        // two tile-times before it is needed.
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        if (warp < 11) {
            const double* __restrict__ cfix = V.cfix;
            for (int it = 0; it < my_tiles; ++it) {
                const int cslot = it % CSLOTS, pslot = it % PSLOTS;
                TRACE(0);
                if (it >= CSLOTS) mbar_wait(&freeb[cslot], ((it - CSLOTS) / CSLOTS) & 1);
                TRACE(1);
                if (it >= PSLOTS) mbar_wait(&cdone[(it - PSLOTS) % CSLOTS], ((it - PSLOTS) / CSLOTS) & 1);
                TRACE(2);
                fence_proxy_async();
                const int64_t j0 = tile_j0(it);
                const int rows = tile_rows(it);
                double* cs = cbuf + cslot * C::TILE_DOUBLES;
                double* ps = pbuf + pslot * C::TILE_DOUBLES;
                const uint32_t bytes = (warp == 8) ? NT * 8 : HALF * 8;
                if (lane == 0) mbar_expect_tx(&full[cslot], (uint32_t)rows * bytes);
                __syncwarp();
                if (lane < rows) {
                    const int64_t j = j0 + lane;
                    if (warp == 8) tma_load_1d(cs + lane * C::LD, cfix + j * NT, NT * 8, &full[cslot]);
                    else if (warp == 9) tma_load_1d(ps + lane * C::LD, Pold + (j + 1) * NT, HALF * 8, &full[cslot]);
                    else tma_load_1d(ps + lane * C::LD + HALF, Pold + (j - 1) * NT + HALF, HALF * 8, &full[cslot]);
                }
                TRACE(3);
            }
        }
    } else {
        // =========================== MMA warps ===========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
        const int g4 = lane >> 2, t4 = lane & 3;
        // this warp's slice of B^{-1} as B-fragments: b[ks][t] = Binv[warp*8*NB + 8t + g4][4ks + t4]
        double bfr[C::KS][C::NB];
        {
            const double* __restrict__ Bw = V.binv + (size_t)(warp * 8 * C::NB + g4) * NT + t4;
#pragma unroll
            for (int ks = 0; ks < C::KS; ++ks)
#pragma unroll
                for (int t = 0; t < C::NB; ++t) bfr[ks][t] = __ldg(Bw + (size_t)(8 * t) * NT + 4 * ks);
        }
        double wq[C::NB];   // quadrature weights of the angles this lane's accumulators belong to
#pragma unroll
        for (int t = 0; t < C::NB; ++t) wq[t] = V.w[(warp * 8 * C::NB + 8 * t + 2 * t4) >> 2];
        // RHS assembly (row a4): this thread always patches the same row k_a, one of the 2N rows that take
        // an incident flux: c[k_a] = c_fix[k_a] + |mu| * psi_nbr[k_a ^ 1]
        const int a_idx = tid & (HALF - 1);
        const int a_m = a_idx >> 1;
        const int k_a = 4 * a_m + ((a_m < N / 2) ? 1 + 2 * (a_idx & 1) : 2 * (a_idx & 1));
        const double coef_a = V.coef[k_a];
        constexpr int ROWS_PER_PASS = 256 / HALF;
        const int r_a = tid / HALF;
        // Both pieces of side work below are written branch-free (predicated stores only) so that they sit
        // in the same basic block as the tile's DMMAs and the scheduler can interleave them.
        // (rows past a ragged tile's end, or a slot past the last tile, hold stale finite-or-not data that
        // is patched too: harmless, those rows are never stored and every slot written here is idle)
        auto assemble = [&](int it) {
            double* cs = cbuf + (it % CSLOTS) * C::TILE_DOUBLES + k_a;
            const double* ps = pbuf + (it % PSLOTS) * C::TILE_DOUBLES + (k_a ^ 1);
#pragma unroll
            for (int q = 0; q < TM / ROWS_PER_PASS; ++q) {
                const int r = r_a + q * ROWS_PER_PASS;
                cs[r * C::LD] = fma(coef_a, ps[r * C::LD], cs[r * C::LD]);
            }
            mbar_arrive(&cdone[it % CSLOTS]);
        };
        // scalar flux (eq. 18) and max-norms of one finished tile: thread tid < 128 owns (cell tid/4, slot tid%4)
        double dmax = 0.0, rmax = 0.0;
        const int ptid = tid & (TM * 4 - 1);
        auto reduce_phi = [&](int it, double old, bool valid) {
            const double* pp = phi_part + (size_t)(it % PBUF) * 8 * TM * 4 + ptid;
            double s = 0.0;
#pragma unroll
            for (int w8 = 0; w8 < 8; ++w8) s += pp[w8 * TM * 4];
            const bool ok = valid && tid < TM * 4 && (tid >> 2) < tile_rows(it);
            if (ok) V.phi[tile_j0(it) * 4 + tid] = s;
            dmax = ok ? nanmax(dmax, fabs(s - old)) : dmax;
            rmax = ok ? nanmax(rmax, fabs(s)) : rmax;
        };
        auto load_phi_old = [&](int it) {
            return (it < my_tiles && tid < TM * 4 && (tid >> 2) < tile_rows(it)) ? V.phi[tile_j0(it) * 4 + tid] : 0.0;
        };

        mbar_wait(&full[0], 0);
        assemble(0);
        // warps w and w+4 share an SM sub-partition and would otherwise stay in lockstep (same work,
        // same barriers), idling the fp64 pipe together at every tile boundary: start the second
        // warpgroup a fraction of a tile late so each covers the other's epilogue
        if (warp >= 4) __nanosleep(1000);
        double q0 = 0.0, q1 = 0.0;   // phi^(l) of tiles it-2 and it-1, fetched two tiles before they are needed

        for (int it = 0; it < my_tiles; ++it) {
            const int st = it % CSLOTS;
            const int64_t j0 = tile_j0(it);
            const int rows = tile_rows(it);
            const double* cs = cbuf + st * C::TILE_DOUBLES;
            double* pp = phi_part + (size_t)(it % PBUF) * 8 * TM * 4;
            const double cur = load_phi_old(it);
            const int itp = it >= 2 ? it - 2 : 0;

            TRACE(0);
            mbar_wait(&cdone[st], (it / CSLOTS) & 1);                      // RHS of this tile complete
            TRACE(1);
            if (it + 1 < my_tiles) mbar_wait(&full[(it + 1) % CSLOTS], ((it + 1) / CSLOTS) & 1);
            if (it >= 2) mbar_wait(&pw[itp % PBUF], (itp / PBUF) & 1);
            TRACE(2);
            // ---- side work, independent of this tile's DMMAs
            assemble(it + 1);
            reduce_phi(itp, q0, it >= 2);
            q0 = q1;
            q1 = cur;

            TRACE(3);
            // ---- a5: D[cell][i] += c[cell][k] * Binv[i][k]
            double acc[4][C::NB][2];
#pragma unroll
            for (int g = 0; g < 4; ++g)
#pragma unroll
                for (int t = 0; t < C::NB; ++t) acc[g][t][0] = acc[g][t][1] = 0.0;
            const double* arow = cs + g4 * C::LD + t4;
#ifdef OCI_DBG_REPEAT
            for (int rep = 0; rep < OCI_DBG_REPEAT; ++rep)
#endif
#pragma unroll
            for (int ks = 0; ks < C::KS; ++ks) {
                double a[4];
#pragma unroll
                for (int g = 0; g < 4; ++g) a[g] = arow[(8 * g) * C::LD + 4 * ks];
#pragma unroll
                for (int g = 0; g < 4; ++g)
#pragma unroll
                    for (int t = 0; t < C::NB; ++t) dmma(acc[g][t][0], acc[g][t][1], a[g], bfr[ks][t]);
            }
            TRACE(4);
            // ---- epilogue: Psi^(l+1) and this warp's partial scalar flux
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                const int r = 8 * g + g4;
                double p0 = 0.0, p1 = 0.0;
#pragma unroll
                for (int t = 0; t < C::NB; ++t) {
                    if (r < rows)
                        *reinterpret_cast<double2*>(Pnew + (j0 + r) * NT + warp * 8 * C::NB + 8 * t + 2 * t4) =
                            make_double2(acc[g][t][0], acc[g][t][1]);
                    p0 = fma(wq[t], acc[g][t][0], p0);
                    p1 = fma(wq[t], acc[g][t][1], p1);
                }
                // lanes t4 and t4^2 hold the same slots (s = 2*(t4&1) + {0,1}) of neighbouring angles
                p0 += __shfl_xor_sync(0xffffffffu, p0, 2);
                p1 += __shfl_xor_sync(0xffffffffu, p1, 2);
                if (t4 < 2) {
                    pp[(warp * TM + r) * 4 + 2 * t4 + 0] = p0;
                    pp[(warp * TM + r) * 4 + 2 * t4 + 1] = p1;
                }
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&freeb[st]);
                mbar_arrive(&pw[it % PBUF]);
            }
            TRACE(5);
        }
        // ---- drain: the last two tiles' scalar flux
        if (my_tiles >= 2) {
            mbar_wait(&pw[(my_tiles - 2) % PBUF], ((my_tiles - 2) / PBUF) & 1);
            reduce_phi(my_tiles - 2, q0, true);
        }
        mbar_wait(&pw[(my_tiles - 1) % PBUF], ((my_tiles - 1) / PBUF) & 1);
        reduce_phi(my_tiles - 1, q1, true);
        if (warp < 4) {
            dmax = warp_max(dmax);
            rmax = warp_max(rmax);
            if (lane == 0) {
                atomic_max_nonneg(&V.norms[2 * slot + 0], dmax);
                atomic_max_nonneg(&V.norms[2 * slot + 1], rmax);
            }
        }
        // ---- reflecting ghost rows (reading S4) from the rows this CTA wrote (pw waits above order them)
        if (blockIdx.x == 0 && V.bcL == OCI_BC_REFLECTING) {
            for (int idx = tid; idx < NT; idx += 256) {
                const int m = idx >> 2, s = idx & 3;
                if (m >= N / 2 && (s & 1)) Pnew[-(int64_t)NT + idx] = __ldcg(Pnew + 4 * (N - 1 - m) + (s - 1));
            }
        }
        if ((ntiles - 1) % gridDim.x == blockIdx.x && V.bcR == OCI_BC_REFLECTING) {
            for (int idx = tid; idx < NT; idx += 256) {
                const int m = idx >> 2, s = idx & 3;
                if (m < N / 2 && !(s & 1)) Pnew[J * NT + idx] = __ldcg(Pnew + (J - 1) * NT + 4 * (N - 1 - m) + (s + 1));
            }
        }
    }
}

bool oci_shared_fast_supported(const DevView& V) { return V.nblk == 1 && (V.n == 128 || V.n == 64); }

int launch_oci_shared_fast(const DevView& V, int src, int slot, int prev_slot, double tol, cudaStream_t s)
{
    const int sm_count = V.sm_count;
    const int64_t ntiles = (V.J + TM - 1) / TM;
    const unsigned grid = (unsigned)(ntiles < sm_count ? ntiles : sm_count);
    if (V.n == 128) {
        oci_iter_resident_kernel<128><<<grid, 384, Cfg<128>::SMEM, s>>>(V, src, slot, prev_slot, tol);
    } else {
        oci_iter_resident_kernel<64><<<grid, 384, Cfg<64>::SMEM, s>>>(V, src, slot, prev_slot, tol);
    }
    return launched(1);
}

cudaError_t oci_shared_fast_opt_in()
{
    cudaError_t e = cudaFuncSetAttribute(oci_iter_resident_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg<128>::SMEM);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(oci_iter_resident_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg<64>::SMEM);
}

}  // namespace oci
