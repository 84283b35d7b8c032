// Kernel (b)+(c), shared-block path for large blocks (n = 4N a multiple of 32; config 4: n = 512):
// the "K-tiled" form.  Psi^(l+1)[j] = B^{-1} c[j] for all cells is the dense contraction
// [J x n] = [J x n].[n x n]^T (eq. 19).  At n = 512 the inverse is 2 MiB: it lives in L2, not in
// an SM, so both operands stream through shared memory in K chunks:
//
//   * persistent CTAs, one per SM; work item = 64 cells x 128 outputs, full K; items are numbered so
//     that the n/128 items of one cell tile run on neighbouring SMs at the same time (the RHS tile is
//     then read from HBM once and from L2 by the others);
//   * 8 MMA warps (2 x 4, each 32 cells x 32 outputs, 16 DMMA.8x8x4 accumulators) + 1 TMA warp;
//   * operands arrive by 2-D tensor-map TMA (cp.async.bulk.tensor, SASS UTMALDG) in chunks of 16 k:
//     c_fix[64 x 16], the neighbour rows Psi^(l)[j +- 1][64 x 16] (ghost rows make the domain edges look
//     like neighbours; rows past the last cell are zero-filled by the TMA unit), B^{-1}[128 x 16];
//     6-stage ring, full / assembled / empty mbarriers;
//   * shared memory is dense with the hardware 128-byte swizzle; one DMMA consumes the k-set
//     {2s, 2s+1, 2s+8, 2s+9} of the chunk (any k order is legal as long as both operands agree), which
//     makes every fragment load bank-conflict free under that swizzle;
//   * RHS assembly (rows a3, a4) in place in shared memory, c[k] = c_fix[k] + coef[k] * psi_nbr[k^1]:
//     k and k^1 share a 16-byte unit, so one 16-byte load of each operand and one 8-byte store; done
//     by the MMA warps for chunk q+1 while chunk q's DMMAs run;
//   * epilogue: accumulators -> Psi^(l+1) (16-byte stores) and the reflecting ghost rows straight from
//     registers; scalar flux (eq. 18) partial over the item's 32 angles by shuffle + shared memory,
//     written to a partial buffer; the last of the n/128 items of a cell tile to finish (ticket
//     counter) adds the partials in fixed order, so phi is deterministic, and takes the two max-norms.
#include <cuda.h>

#include "device_utils.cuh"

namespace oci {

namespace {

constexpr int KT_M = 64;      // cells per work item
constexpr int KT_N = 128;     // outputs per work item
constexpr int KT_K = 16;      // k per chunk = one 128-byte swizzle row
constexpr int KT_STAGES = 6;
constexpr int KT_A_BYTES = KT_M * KT_K * 8;   // 8 KB
constexpr int KT_B_BYTES = KT_N * KT_K * 8;   // 16 KB
constexpr int KT_STAGE_BYTES = 2 * KT_A_BYTES + KT_B_BYTES;
constexpr int KT_MAX_N = 1024;
constexpr size_t KT_SMEM = 1024 /*alignment slack*/ + (size_t)KT_STAGES * KT_STAGE_BYTES + 4 * KT_M * 4 * 8 /*phi_s*/ +
                           KT_MAX_N * 8 /*coef*/ + 3 * KT_STAGES * 8 + 64;


}  // namespace

__global__ void __launch_bounds__(288, 1)
oci_iter_ktiled_kernel(DevView V, const __grid_constant__ CUtensorMap map_cfix, const __grid_constant__ CUtensorMap map_psi,
                       const __grid_constant__ CUtensorMap map_binv, int src, int slot, int prev_slot, double tol)
{
    if (step_done(V.norms, prev_slot, tol)) return;
    extern __shared__ unsigned char smem_raw[];
    // aligned up inside the shared window (pointer arithmetic on the array keeps the LDS/STS address space)
    unsigned char* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    unsigned char* stages = base;                                                    // [S][cfix 8K | nbr 8K | binv 16K]
    double* phi_s = reinterpret_cast<double*>(base + (size_t)KT_STAGES * KT_STAGE_BYTES);   // [4 wn][64][4]
    double* coef_s = phi_s + 4 * KT_M * 4;                                            // [n]
    uint64_t* full = reinterpret_cast<uint64_t*>(coef_s + KT_MAX_N);
    uint64_t* asmd = full + KT_STAGES;
    uint64_t* empty = asmd + KT_STAGES;
    int* ticket_s = reinterpret_cast<int*>(empty + KT_STAGES);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = V.n, N = V.N, half = n >> 1;
    const int64_t J = V.J;
    const int kch = n / KT_K;                             // chunks per item
    const int ntn = (n + KT_N - 1) / KT_N;                // items per cell tile
    const int64_t nct = (J + KT_M - 1) / KT_M;
    const int64_t nitems = nct * ntn;
    const int my_items = (int)((nitems - blockIdx.x + gridDim.x - 1) / gridDim.x);

    if (tid == 0) {
        for (int s = 0; s < KT_STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&asmd[s], 256);
            mbar_init(&empty[s], 8);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int k = tid; k < n; k += blockDim.x) coef_s[k] = V.coef[k];
    __syncthreads();

    if (warp == 8) {
        // =========================== TMA producer (one thread) ===========================
        if (lane == 0) {
            asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_cfix)) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_psi)) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_binv)) : "memory");
            int q = 0;
            for (int it = 0; it < my_items; ++it) {
                const int64_t item = (int64_t)blockIdx.x + (int64_t)it * gridDim.x;
                const int j0 = (int)(item / ntn) * KT_M;
                const int i0 = (int)(item % ntn) * KT_N;
                for (int kc = 0; kc < kch; ++kc, ++q) {
                    const int s = q % KT_STAGES;
                    if (q >= KT_STAGES) mbar_wait(&empty[s], ((q / KT_STAGES) - 1) & 1);
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    unsigned char* st = stages + (size_t)s * KT_STAGE_BYTES;
                    const int k0 = kc * KT_K;
                    mbar_expect_tx(&full[s], KT_STAGE_BYTES);
                    tma_load_2d(st, &map_cfix, k0, j0, &full[s]);
                    // psi map row = cell + 1 (ghost row first); k < n/2 (mu<0) looks right, else left (rows a3)
                    tma_load_2d(st + KT_A_BYTES, &map_psi, k0, j0 + 1 + (k0 < half ? 1 : -1), &full[s]);
                    tma_load_2d(st + 2 * KT_A_BYTES, &map_binv, k0, i0, &full[s]);
                }
            }
        }
        return;
    }

    // =========================== MMA warps ===========================
    const int g4 = lane >> 2, t4 = lane & 3;
    const int wm = warp >> 2, wn = warp & 3;
    // byte offset of this lane's fragment element inside a 128-byte swizzled row, per k-step:
    // logical 16-byte unit ks + 4*(t4>>1), XOR row&7 (= g4), element t4&1
    int foff[4];
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) foff[ks] = (((ks + 4 * (t4 >> 1)) ^ g4) << 4) + ((t4 & 1) << 3);
    const int a_row = (wm * 32 + g4) * 128;              // + g*1024
    const int b_row = (wn * 32 + g4) * 128;              // + t*1024
    // assembly: this thread patches 16-byte units (row tid/8 + {0,32}, physical unit tid&7)
    const int as_row = tid >> 3;
    const int as_unit = (tid & 7) ^ (as_row & 7);        // logical unit -> k = k0 + 2*unit
    const int as_off = as_row * 128 + ((tid & 7) << 4);

    double* __restrict__ Pnew = V.psi[src ^ 1];
    double dmax = 0.0, rmax = 0.0;

    auto assemble = [&](int q, int kc) {
        unsigned char* st = stages + (size_t)(q % KT_STAGES) * KT_STAGE_BYTES;
        const int k = kc * KT_K + 2 * as_unit;
        const bool upper = k >= half;                      // mu > 0: even rows (s = 0,2) take coef * partner (odd)
        const double cf = coef_s[k + (upper ? 0 : 1)];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            double2* cs = reinterpret_cast<double2*>(st + as_off + h * 32 * 128);
            const double2 ps = *reinterpret_cast<const double2*>(st + KT_A_BYTES + as_off + h * 32 * 128);
            double2 c = *cs;
            if (upper) c.x = fma(cf, ps.y, c.x);
            else c.y = fma(cf, ps.x, c.y);
            *cs = c;
        }
        mbar_arrive(&asmd[q % KT_STAGES]);
    };

    int q = 0;
    mbar_wait(&full[0], 0);
    assemble(0, 0);
    const int total_chunks = my_items * kch;

    for (int it = 0; it < my_items; ++it) {
        const int64_t item = (int64_t)blockIdx.x + (int64_t)it * gridDim.x;
        const int64_t ct = item / ntn;
        const int nt = (int)(item % ntn);
        const int64_t j0 = ct * KT_M;
        const int i0 = nt * KT_N;

        double acc[4][4][2];
#pragma unroll
        for (int g = 0; g < 4; ++g)
#pragma unroll
            for (int t = 0; t < 4; ++t) acc[g][t][0] = acc[g][t][1] = 0.0;

        for (int kc = 0; kc < kch; ++kc, ++q) {
            const int s = q % KT_STAGES;
            mbar_wait(&asmd[s], (q / KT_STAGES) & 1);          // RHS of this chunk assembled by everyone
            if (q + 1 < total_chunks) {
                mbar_wait(&full[(q + 1) % KT_STAGES], ((q + 1) / KT_STAGES) & 1);
                assemble(q + 1, (kc + 1 == kch) ? 0 : kc + 1);
            }
            const unsigned char* st = stages + (size_t)s * KT_STAGE_BYTES;
            const unsigned char* As = st + a_row;
            const unsigned char* Bs = st + 2 * KT_A_BYTES + b_row;
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
                double a[4], b[4];
#pragma unroll
                for (int g = 0; g < 4; ++g) a[g] = *reinterpret_cast<const double*>(As + g * 1024 + foff[ks]);
#pragma unroll
                for (int t = 0; t < 4; ++t) b[t] = *reinterpret_cast<const double*>(Bs + t * 1024 + foff[ks]);
#pragma unroll
                for (int g = 0; g < 4; ++g)
#pragma unroll
                    for (int t = 0; t < 4; ++t) dmma(acc[g][t][0], acc[g][t][1], a[g], b[t]);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
        }

        // ---- epilogue: Psi^(l+1), reflecting ghost rows, scalar-flux partial of this item
        const bool refl_l = V.bcL == OCI_BC_REFLECTING, refl_r = V.bcR == OCI_BC_REFLECTING;
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            const int r = wm * 32 + 8 * g + g4;
            const int64_t j = j0 + r;
            double p0 = 0.0, p1 = 0.0;
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int i = i0 + wn * 32 + 8 * t + 2 * t4;       // even; slots (i&3, i&3 + 1)
                if (j < J && i < n) {
                    *reinterpret_cast<double2*>(Pnew + j * n + i) = make_double2(acc[g][t][0], acc[g][t][1]);
                    const int m = i >> 2;
                    // reading S4: the mirror image of the edge cell's outgoing flux becomes the ghost row
                    if (j == 0 && refl_l && m < N / 2) Pnew[-(int64_t)n + 4 * (N - 1 - m) + (i & 3) + 1] = acc[g][t][0];
                    if (j == J - 1 && refl_r && m >= N / 2) Pnew[J * n + 4 * (N - 1 - m) + (i & 3)] = acc[g][t][1];
                    const double wq = V.w[m];
                    p0 = fma(wq, acc[g][t][0], p0);
                    p1 = fma(wq, acc[g][t][1], p1);
                }
            }
            // lanes t4 and t4^2 hold the same slots (2*(t4&1) + {0,1}) of neighbouring angles
            p0 += __shfl_xor_sync(0xffffffffu, p0, 2);
            p1 += __shfl_xor_sync(0xffffffffu, p1, 2);
            if (t4 < 2) {
                phi_s[(wn * KT_M + r) * 4 + 2 * t4 + 0] = p0;
                phi_s[(wn * KT_M + r) * 4 + 2 * t4 + 1] = p1;
            }
        }
        named_bar_sync(1, 256);
        {
            // thread tid owns (cell tid/4, slot tid%4) of the item
            const int64_t j = j0 + (tid >> 2);
            double ssum = phi_s[0 * KT_M * 4 + tid] + phi_s[1 * KT_M * 4 + tid] + phi_s[2 * KT_M * 4 + tid] + phi_s[3 * KT_M * 4 + tid];
            bool last = true;
            if (ntn > 1) {
                if (j < J) V.phi_part[((int64_t)nt * J + j) * 4 + (tid & 3)] = ssum;
                __threadfence();
                named_bar_sync(1, 256);
                if (tid == 0) {
                    const int old = atomicAdd(&V.tickets[ct], 1);
                    *ticket_s = old;
                    if (old == ntn - 1) V.tickets[ct] = 0;          // re-arm for the next launch
                }
                named_bar_sync(1, 256);
                last = (*ticket_s == ntn - 1);
                if (last) {
                    __threadfence();
                    ssum = 0.0;
                    if (j < J)
                        for (int p = 0; p < ntn; ++p) ssum += __ldcg(&V.phi_part[((int64_t)p * J + j) * 4 + (tid & 3)]);
                }
            }
            if (last && j < J) {
                const double old = V.phi[j * 4 + (tid & 3)];
                V.phi[j * 4 + (tid & 3)] = ssum;
                dmax = nanmax(dmax, fabs(ssum - old));
                rmax = nanmax(rmax, fabs(ssum));
            }
            named_bar_sync(1, 256);                                  // phi_s / ticket_s reusable
        }
    }
    dmax = warp_max(dmax);
    rmax = warp_max(rmax);
    if (lane == 0) {
        atomic_max_nonneg(&V.norms[2 * slot + 0], dmax);
        atomic_max_nonneg(&V.norms[2 * slot + 1], rmax);
    }
}

// ---- host side: tensor maps (driver entry point fetched through the runtime: no link dependency on libcuda)
namespace {
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

}  // namespace

// row-major fp64 matrix [rows][cols] -> 2-D tensor map with a box of box_rows x box_cols, zero fill outside;
// swizzle128: box_cols must be 16 (one 128-byte row per box row), else the box lands dense in shared memory
bool oci_encode_2d(CUtensorMap* m, const double* base, uint64_t rows, uint64_t cols, uint32_t box_rows, uint32_t box_cols,
                   bool swizzle128)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {cols * 8};
    cuuint32_t box[2] = {box_cols, box_rows};
    cuuint32_t estr[2] = {1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base), dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
              CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool oci_ktiled_supported(const DevView& V)
{
    return V.nblk == 1 && V.n % 32 == 0 && V.n <= KT_MAX_N && V.J + 2 < (int64_t)1 << 31;
}

bool oci_ktiled_prepare(const DevView& V, KtiledMaps* M)
{
    const uint64_t n = (uint64_t)V.n;
    return oci_encode_2d(&M->cfix, V.cfix, (uint64_t)V.J, n, KT_M, KT_K, true) &&
           oci_encode_2d(&M->psi[0], V.psi[0] - n, (uint64_t)V.J + 2, n, KT_M, KT_K, true) &&
           oci_encode_2d(&M->psi[1], V.psi[1] - n, (uint64_t)V.J + 2, n, KT_M, KT_K, true) &&
           oci_encode_2d(&M->binv, V.binv, n, n, KT_N, KT_K, true);
}

int launch_oci_ktiled(const DevView& V, const KtiledMaps& M, int src, int slot, int prev_slot, double tol, cudaStream_t s)
{
    const int sm_count = V.sm_count;
    const int64_t nitems = ((V.J + KT_M - 1) / KT_M) * ((V.n + KT_N - 1) / KT_N);
    const unsigned grid = (unsigned)(nitems < sm_count ? nitems : sm_count);
    oci_iter_ktiled_kernel<<<grid, 288, KT_SMEM, s>>>(V, M.cfix, M.psi[src], M.binv, src, slot, prev_slot, tol);
    return launched(1);
}

cudaError_t oci_ktiled_opt_in()
{
    return cudaFuncSetAttribute(oci_iter_ktiled_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)KT_SMEM);
}

}  // namespace oci
