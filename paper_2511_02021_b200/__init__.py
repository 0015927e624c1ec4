"""paper_2511_02021_b200 -- B200-native (sm_100a) velocity-tendency / divergence / vorticity sweep of
ICON's dynamical core (arxiv/paper_2511_02021). The product is the C-ABI library
``libicon_dycore.so`` (include/icon_dycore.h); this package is its thin Python binding."""
from .binding import (ICON_F32, ICON_F64, ICON_HOST_ONLY, ICON_LOCALITY_WORKLIST, ICON_NO_WORKLIST,  # noqa: F401
                      ICON_OPT_CC_TILE, ICON_OPT_CC_PACE, ICON_OPT_TENDENCY_KERNEL, ICON_PERMUTE, TABLES, IconError, IconGrid, dycore_div_vort,
                      dycore_step, dycore_step_host, dycore_step_w, dycore_velocity_tendencies, dycore_velocity_tendencies_noalloc, dycore_metric_from_zhalf, dycore_velocity_tendencies_metric, dycore_w_tendency, dycore_halo_pack, icon_grid_create, load_library)
