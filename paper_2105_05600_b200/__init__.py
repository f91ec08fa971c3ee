"""B200-native ROSEFusion hot path (arxiv 2105.05600): particle-swarm fitness evaluation, on-device swarm
update and projective TSDF integration behind a small C ABI (include/rosefusion_b200.h)."""
from .api import (RF_F16_W8, RF_F32_W8, RF_TRACK_MODE_F1, RF_TRACK_NO_EARLY_STOP, RF_TRACK_NO_GRAPH, RF_TRACK_NO_PDL, RF_TRACK_NO_POINTS, RF_TRACK_NO_OVERLAP, RF_TRACK_RESCALE_ISO,
                  RF_TRACK_RESCALE_ANISO, RF_TRACK_MODE_EQ14, RF_TRACK_THRESH_EQ21,
                  RF_TRACK_STOP_EMPTY, RF_TRACK_STOP_SMALL, EXPORTS, RFError, Volume, gn_noalloc_scratch_bytes, launch_count, lib, microbench_l2)

__all__ = ["Volume", "RFError", "lib", "microbench_l2", "gn_noalloc_scratch_bytes", "launch_count", "EXPORTS", "RF_F32_W8", "RF_F16_W8",
           "RF_TRACK_NO_EARLY_STOP", "RF_TRACK_NO_GRAPH", "RF_TRACK_NO_PDL", "RF_TRACK_NO_OVERLAP", "RF_TRACK_RESCALE_ISO", "RF_TRACK_RESCALE_ANISO", "RF_TRACK_MODE_EQ14", "RF_TRACK_THRESH_EQ21", "RF_TRACK_MODE_F1", "RF_TRACK_NO_POINTS", "RF_TRACK_STOP_EMPTY",
           "RF_TRACK_STOP_SMALL"]
