"""paper_1910_01070_b200 -- B200-native (sm_100a CUDA) batched Helios-r2 emission
forward model + likelihood (Kitzmann et al. 2020, arXiv:1910.01070, Sect. 2.8).

The product is the C-ABI library declared in include/helios.h
(csrc/ -> libhelios_b200.so); this package is its thin ctypes binding.
"""
from .binding import (  # noqa: F401
    Helios, HeliosError, lib,
    helios_create, helios_destroy, helios_set_stream, helios_set_option, helios_load_opacity,
    helios_set_atmosphere, helios_set_observation, helios_reserve, helios_forward_batch,
    helios_loglike_batch, helios_forward_highres, helios_forward_batch_host, helios_get_stats,
    helios_get_angles, helios_get_stage_ms, helios_set_tp_elements, helios_set_extras, helios_get_n_params,
    helios_teff_batch, helios_teff_batch_host, helios_measure_peaks, helios_observe_noalloc, HELIOS_EXTRA_DISTANCE, HELIOS_EXTRA_ERROR_INFLATION, HELIOS_EXTRA_GREY_CLOUD,
    HELIOS_OK, HELIOS_EINVAL, HELIOS_ENOMEM, HELIOS_ECUDA, HELIOS_ESTATE,
    HELIOS_OPT_KERNEL, HELIOS_OPT_MODELS_PER_CTA, HELIOS_OPT_TIMING, HELIOS_OPT_NU_ORDER, HELIOS_OPT_FUSED_OBS, HELIOS_OPT_GRAPHS, NU_ORDER_GRID, NU_ORDER_OPACITY,
    KERNEL_AUTO, KERNEL_DIRECT, KERNEL_SLAB, KERNEL_LEVEL_PARALLEL,
)
from .build import build_library, LIB_PATH  # noqa: F401
