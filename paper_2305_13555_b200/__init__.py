"""B200-native one-cell-inversion (OCI) transient slab S_N transport: thin Python binding over the
C-ABI library `liboci_b200.so` (include/oci.h).  Argument marshalling only: every step of the path
runs in the CUDA kernels under csrc/.  PyTorch supplies device memory and the stream, nothing else.
There is no CPU fallback: importing works without a GPU (so the symbol table can be checked), any
compute call without the CUDA library or a device raises."""
from .binding import (OCI, OCIError, BC_VACUUM, BC_INCIDENT_ISOTROPIC, BC_REFLECTING, BC_HALO, PATH_SHARED,  # noqa: F401
                      PATH_PER_CELL, KERNEL_GENERIC, KERNEL_RESIDENT, KERNEL_KTILED, KERNEL_PER_CELL, ITERATION_FULL, ITERATION_REDUCED, ITERATION_AUTO, RKERNEL_AUTO, RKERNEL_GEMV, RKERNEL_RESIDENT, RKERNEL_KTILED, RKERNEL_OPREG, RKERNEL_WOODBURY, load_library, library_path, EXPORTED_SYMBOLS, probe_fp64_tensor_tflops, shard_mailbox_bytes, shard_step)
