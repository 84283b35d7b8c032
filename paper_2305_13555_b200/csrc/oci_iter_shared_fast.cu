// Specialised shared-block OCI kernels (placeholder until the fast paths land).
#include "device_utils.cuh"

namespace oci {

bool oci_shared_fast_supported(const DevView&) { return false; }

int launch_oci_shared_fast(const DevView&, int, int, int, double, cudaStream_t) { return 0; }

}  // namespace oci
