"""B200-native batched differentiable rod step (DLO-Lab hot path): thin Python binding over the C-ABI library.

The product is `libdlo_b200.so` (include/dlo.h); this package only marshals arguments.  There is no CPU path:
importing works anywhere (so the build check can run without a GPU) but every compute call needs a CUDA device.
"""
from .binding import (DloConfig, DloMaterial, DloSim, DloError, lib, dlo_create, dlo_destroy, dlo_set_pins, dlo_set_cuts,  # noqa: F401
                      dlo_set_primitives, dlo_set_grippers, dlo_set_state, dlo_restore_state, dlo_set_actions,
                      dlo_rollout_forward, dlo_get_state, dlo_get_position_residual, dlo_backward, dlo_get_state_adjoint, dlo_rollout_forward_host, dlo_backward_host, dlo_check_numerics,
                      dlo_set_kernel_timing, dlo_get_kernel_timing, dlo_measure_fp32_peak, dlo_scratch_bytes, dlo_static_scratch_bytes, dlo_rollout_forward_static, make_config, STATIC_SCRATCH_BYTES, dlo_launch_count, dlo_last_error, dlo_version, EXPORTS)
