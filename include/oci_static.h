/* oci_static.h - ONE entry point of liboci_b200.so that allocates nothing.
 *
 * Why: some callers cannot call cudaMalloc - code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it.  Everything else in this library works inside a workspace the caller allocates (oci.h); this call needs no
 * workspace and no context at all.  Its scratch memory is a file-scope `static __device__ __align__(256)` array of
 * OCI_STATIC_SCRATCH_BYTES (260 KiB) inside the library: every GPU that loads the library holds it until the process exits.
 *
 * What it computes (the stand-alone kernel (c) of the method, csrc/phi_norm.cu):
 *     phi[j][s]  = sum_m w[m] psi[j][m][s]                        scalar flux, eq. (18), s = (k,L), (k,R), (k+1/2,L), (k+1/2,R)
 *     norms[0]   = max_{j,s} |phi[j][s] - phi_old[j][s]|          (0 if phi_old is NULL)
 *     norms[1]   = max_{j,s} |phi[j][s]|                           the two max-norms of the stopping rule d <= tol * r
 * The scratch holds one (d, r) pair per CTA of 64 cells and an arrival counter; the last CTA to arrive reduces the pairs.
 *
 * Limits: 1 <= cells <= OCI_STATIC_MAX_CELLS (1 048 576), 2 <= n_angles <= 512 and even.  Anything else is rejected with
 * OCI_E_INVALID (-1) and a message (oci_static_last_error); nothing is launched.
 *
 * The call makes no cudaMalloc / cudaFree / cudaHostAlloc and calls no allocating library routine; it launches one kernel
 * and one 4-byte cudaMemsetAsync (the arrival counter) on `stream`.  ALL CALLS ON A DEVICE SHARE THE ONE ARRAY, which keeps
 * the last call's contents: the call clears what must start at zero itself, and two calls that overlap on the GPU (different
 * streams, or a captured graph replayed concurrently with another call) RACE - order them on one stream or with events.
 * Host threads may call concurrently only if their streams are so ordered.
 */
#ifndef OCI_STATIC_H
#define OCI_STATIC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OCI_STATIC_MAX_CELLS 1048576
#define OCI_STATIC_SCRATCH_BYTES (256 + (OCI_STATIC_MAX_CELLS / 64) * 16)

/* Once per device, with that device current (cudaSetDevice), before the first oci_static_scalar_flux_norms on it - and
 * before any stream capture begins: resolves the device address of the scratch array (cudaGetSymbolAddress; this is also
 * where the CUDA runtime loads the kernel).  oci_static_scalar_flux_norms calls it by itself if it has not been called
 * for the current device.  Returns 0, or -3 (OCI_E_CUDA) with a message. */
int oci_static_prepare(void);

/* DEVICE pointers, on the current device:
 *   d_psi      in   [cells][n_angles][4] doubles, the angular flux in the layout of oci_get_angular_flux_dev
 *   d_w        in   [n_angles] doubles, the quadrature weights (oci_get_quadrature gives them on the host)
 *   d_phi_old  in   [cells][4] doubles or NULL (then norms[0] = 0); may NOT alias d_phi
 *   d_phi      out  [cells][4] doubles
 *   d_norms    out  [2] doubles (d, r); a NaN or Inf in phi yields a NaN / Inf norm (never silently dropped)
 * stream: a cudaStream_t (NULL = the default stream).  The caller owns every buffer; results are valid once the stream
 * has passed the call.  Returns 0; -1 (OCI_E_INVALID: NULL pointer, size beyond the limits above); -3 (OCI_E_CUDA). */
int oci_static_scalar_flux_norms(const double* d_psi, const double* d_w, const double* d_phi_old, double* d_phi, double* d_norms,
                                 int64_t cells, int32_t n_angles, void* stream);

/* Message of the calling thread's last failed oci_static_* call ("" if none). */
const char* oci_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
