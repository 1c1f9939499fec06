"""Seeded synthetic inputs shared by the oracle tests and the CUDA path (no method arithmetic)."""
from .gen import (Workload, Cfg3Sequence, cell_centres, cfg0, cfg1, cfg2, cfg3, cfg4a, cfg4a_member,
                  cfg4b, wd_half_plane, random_smooth, lane_emden, wd_scale_length, u01, uniform,
                  KM, M_WD_CODE, levelset_front, hydro_state, shock_tube, hydro_blobs)
