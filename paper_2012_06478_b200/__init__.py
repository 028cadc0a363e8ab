"""B200-native hot path of the Realistic Microstructure Simulator (arXiv 2012.06478).

The product is librms_b200.so (C ABI in include/rms.h, CUDA kernels for sm_100a in csrc/); this
package is its thin Python binding.  Nothing here computes on the CPU and nothing imports oracle/.
"""
from .binding import (  # noqa: F401
    RMS_ADOPT_DEVICE_PTR,
    RMS_LABELS_ON_DEVICE,
    RMS_NO_BRICKS,
    RMS_RUN_LABEL_GATHER,
    RmsError,
    Substrate,
    Walkers,
    load_library,
    rms_run,
    rms_substrate_create,
    rms_walkers_init,
    rms_walkers_init_weighted,
    rms_substrate_label_volumes,
    rms_substrate_label_volumes_static,
    rms_volume_weighted_signal,
)
from .api import simulate, shard_range  # noqa: F401
