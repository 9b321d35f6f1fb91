"""Seeded synthetic inputs (parameters and parking scenes) handed identically to the CPU oracle
and to the CUDA library.  This module holds DATA RECIPES ONLY -- none of the method's arithmetic
(no kinematics, no barrier, no costs, no random-number mapping used by the solver).  It imports
neither `oracle/` nor `paper_2508_05773_b200/`."""
from .params import Params, default_params
from .parking import (Scene, scene_cfg0, scene_cfg1, scene_cfg2, scene_cfg2_superellipse, scene_cfg3, scene_static,
                      scene_batch, vehicle_disc_centres)
from . import parking
from .mpcc import PathScene, scene_mpcc, spline_table

__all__ = ["Params", "default_params", "Scene", "scene_cfg0", "scene_cfg1", "scene_cfg2",
           "scene_cfg2_superellipse", "scene_cfg3", "scene_static", "scene_batch", "vehicle_disc_centres",
           "PathScene", "scene_mpcc", "spline_table", "parking"]
