"""paper_1912_06636_b200 -- B200-native (sm_100a) real-space grid operations of arXiv:1912.06636.

The product is the C-ABI library libaims_gpu.so (include/aims_gpu.h, csrc/); this package is the thin Python
binding over it (argument marshalling only).  There is no CPU fallback: a missing library raises.
"""
from .binding import (AimsError, Context, aims_gpu_add_tau_matrix, aims_gpu_batch_points, aims_gpu_bloch_fold, aims_gpu_create,  # noqa: F401
                      aims_gpu_density_hessian, aims_gpu_destroy, aims_gpu_eval_basis, aims_gpu_integrate_hamiltonian,
                      aims_gpu_integrate_hamiltonian_ks, aims_gpu_partition_weights, aims_gpu_partition_weights_noalloc, aims_gpu_periodic_images, aims_gpu_pulay_forces,
                      aims_gpu_pulay_forces_ks, aims_gpu_pulay_forces_stress, aims_gpu_set_deterministic, aims_gpu_update_density, aims_gpu_wrap_points, exported_symbols, load_library)
