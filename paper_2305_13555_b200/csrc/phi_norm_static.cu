// The library's ONE entry point that allocates nothing (include/oci_static.h): scalar flux and the two max-norms of the
// stopping rule (kernel (c), eq. 18) of an angular-flux array, with the kernel's scratch memory in a
// file-scope device array instead of the caller's workspace.  A variant of phi_norm.cu's kernel: same accumulation order
// per (cell, slot) - a lane adds its angles in ascending order, then the butterfly over lanes 2, 4, 8, 16 - so phi is bit
// for bit what the workspace path produces; the norms go through per-CTA pairs in the scratch array and the last CTA to
// arrive reduces them (a max: order-independent), instead of atomicMax into the workspace's norm slots.
//
// Scratch layout (bytes): [0, 4) arrival counter, [256, 256 + 16 * ctas) one (d, r) pair per CTA of 64 cells.  The array is
// shared by every call on the device and keeps the last call's contents: the entry point zeroes the counter on the stream
// before the launch (the last CTA also resets it), every pair that is read has been written by the same launch.  Calls
// that overlap on the GPU race.
//
// In host code the array's NAME is a host-side stand-in, not a device address: the device address comes from
// cudaGetSymbolAddress, once per device with that device current (oci_static_prepare), and is what the kernel is given.
#include <cuda_runtime.h>

#include <atomic>
#include <mutex>

#include "device_utils.cuh"
#include "oci_static.h"

namespace {

constexpr int ST_THREADS = 256;                            // 8 warps
constexpr int ST_CP = 8;                                   // cells per warp
constexpr int ST_CELLS_PER_CTA = 8 * ST_CP;                // 64
constexpr int ST_MAX_CTAS = OCI_STATIC_MAX_CELLS / ST_CELLS_PER_CTA;
constexpr int ST_MAX_DEVICES = 64;

static __device__ __align__(256) unsigned char g_static_scratch[OCI_STATIC_SCRATCH_BYTES];

static_assert(OCI_STATIC_SCRATCH_BYTES == 256 + ST_MAX_CTAS * 16, "scratch = counter block + one pair per CTA");

std::mutex g_mu;
std::atomic<void*> g_scratch_ptr[ST_MAX_DEVICES];         // device address of g_static_scratch, per device (zero-initialised)
thread_local const char* g_err = "";

int fail_static(int code, const char* msg)
{
    g_err = msg;
    return code;
}

__global__ void __launch_bounds__(ST_THREADS) phi_norm_static_kernel(const double* __restrict__ psi, const double* __restrict__ w,
                                                                     const double* __restrict__ phi_old, double* __restrict__ phi,
                                                                     double* __restrict__ norms, unsigned char* scratch, int64_t J, int N)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int n = 4 * N;
    unsigned int* counter = reinterpret_cast<unsigned int*>(scratch);
    double* pairs = reinterpret_cast<double*>(scratch + 256);
    double dmax = 0.0, rmax = 0.0;
    // a lane owns the 16-byte units idx = 2 * lane (+ 64 i) of each row: slots (0,1) of an angle on even lanes, (2,3) on
    // odd lanes; every load of the pass is unconditional (cell index clamped) so that all of them are in flight together
    const int64_t j0 = ((int64_t)blockIdx.x * 8 + warp) * ST_CP;
    if (j0 < J) {
        double a0[ST_CP], a1[ST_CP];
        double2 oldv[ST_CP];
#pragma unroll
        for (int c = 0; c < ST_CP; ++c) {
            a0[c] = a1[c] = 0.0;
            const int64_t j = (j0 + c < J) ? j0 + c : J - 1;
            oldv[c] = (phi_old != nullptr && lane < 2) ? *reinterpret_cast<const double2*>(phi_old + j * 4 + 2 * lane) : make_double2(0.0, 0.0);
        }
#pragma unroll 2
        for (int idx = 2 * lane; idx < n; idx += 64) {
            const double wq = w[idx >> 2];
#pragma unroll
            for (int c = 0; c < ST_CP; ++c) {
                const int64_t j = (j0 + c < J) ? j0 + c : J - 1;
                const double2 v = *reinterpret_cast<const double2*>(psi + j * n + idx);
                a0[c] = fma(wq, v.x, a0[c]);
                a1[c] = fma(wq, v.y, a1[c]);
            }
        }
#pragma unroll
        for (int c = 0; c < ST_CP; ++c) {
#pragma unroll
            for (int o = 2; o < 32; o <<= 1) {
                a0[c] += __shfl_xor_sync(0xffffffffu, a0[c], o);
                a1[c] += __shfl_xor_sync(0xffffffffu, a1[c], o);
            }
        }
#pragma unroll
        for (int c = 0; c < ST_CP; ++c) {
            const int64_t j = j0 + c;
            if (j < J && lane < 2) {
                *reinterpret_cast<double2*>(phi + j * 4 + 2 * lane) = make_double2(a0[c], a1[c]);
                if (phi_old != nullptr) dmax = oci::nanmax(dmax, oci::nanmax(fabs(a0[c] - oldv[c].x), fabs(a1[c] - oldv[c].y)));
                rmax = oci::nanmax(rmax, oci::nanmax(fabs(a0[c]), fabs(a1[c])));
            }
        }
    }
    // ---- this CTA's pair into the scratch array, then the last CTA to arrive reduces all of them
    __shared__ double sd[8], sr[8];
    __shared__ bool last;
    dmax = oci::warp_max(dmax);
    rmax = oci::warp_max(rmax);
    if (lane == 0) { sd[warp] = dmax; sr[warp] = rmax; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q) { dmax = oci::nanmax(dmax, sd[q]); rmax = oci::nanmax(rmax, sr[q]); }
        pairs[2 * (size_t)blockIdx.x + 0] = dmax;
        pairs[2 * (size_t)blockIdx.x + 1] = rmax;
        __threadfence();
        last = atomicAdd(counter, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    dmax = rmax = 0.0;
    for (unsigned int b = threadIdx.x; b < gridDim.x; b += ST_THREADS) {
        dmax = oci::nanmax(dmax, __ldcg(pairs + 2 * (size_t)b + 0));
        rmax = oci::nanmax(rmax, __ldcg(pairs + 2 * (size_t)b + 1));
    }
    dmax = oci::warp_max(dmax);
    rmax = oci::warp_max(rmax);
    __syncthreads();
    if (lane == 0) { sd[warp] = dmax; sr[warp] = rmax; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q) { dmax = oci::nanmax(dmax, sd[q]); rmax = oci::nanmax(rmax, sr[q]); }
        norms[0] = dmax;
        norms[1] = rmax;
        *counter = 0u;                                     // ready for the next call
    }
}

}  // namespace

extern "C" {

int oci_static_prepare(void)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_static(-3, cudaGetErrorString(e));
    if (dev < 0 || dev >= ST_MAX_DEVICES) return fail_static(-1, "oci_static_prepare: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_scratch_ptr[dev].load() != nullptr) return 0;
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);        // the device address on the CURRENT device
    if (e != cudaSuccess || p == nullptr) {
        cudaGetLastError();
        return fail_static(-3, e != cudaSuccess ? cudaGetErrorString(e) : "cudaGetSymbolAddress returned NULL");
    }
    g_scratch_ptr[dev].store(p);
    return 0;
}

int oci_static_scalar_flux_norms(const double* d_psi, const double* d_w, const double* d_phi_old, double* d_phi, double* d_norms,
                                 int64_t cells, int32_t n_angles, void* stream)
{
    if (!d_psi || !d_w || !d_phi || !d_norms) return fail_static(-1, "oci_static_scalar_flux_norms: NULL pointer");
    if (cells < 1 || cells > OCI_STATIC_MAX_CELLS)
        return fail_static(-1, "oci_static_scalar_flux_norms: cells outside [1, 1048576] (OCI_STATIC_MAX_CELLS: the static scratch array "
                               "holds one pair per 64 cells); use the workspace path of oci.h for larger slabs");
    if (n_angles < 2 || (n_angles & 1) || n_angles > 512)
        return fail_static(-1, "oci_static_scalar_flux_norms: n_angles must be even and in [2, 512]");
    if (d_phi_old == d_phi) return fail_static(-1, "oci_static_scalar_flux_norms: d_phi_old must not alias d_phi");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_static(-3, cudaGetErrorString(e));
    if (dev < 0 || dev >= ST_MAX_DEVICES) return fail_static(-1, "oci_static_scalar_flux_norms: device ordinal beyond 63");
    if (g_scratch_ptr[dev].load() == nullptr) {
        if (int rc = oci_static_prepare()) return rc;
    }
    unsigned char* scratch = static_cast<unsigned char*>(g_scratch_ptr[dev].load());
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const unsigned ctas = (unsigned)((cells + ST_CELLS_PER_CTA - 1) / ST_CELLS_PER_CTA);
    // the arrival counter must start at zero (the array keeps whatever the last call - possibly an aborted one - left)
    e = cudaMemsetAsync(scratch, 0, 4, s);
    if (e != cudaSuccess) return fail_static(-3, cudaGetErrorString(e));
    phi_norm_static_kernel<<<ctas, ST_THREADS, 0, s>>>(d_psi, d_w, d_phi_old, d_phi, d_norms, scratch, cells, (int)n_angles);
    e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail_static(-3, cudaGetErrorString(e));
    }
    return 0;
}

const char* oci_static_last_error(void) { return g_err; }

}  // extern "C"
