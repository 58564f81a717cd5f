"""Seeded synthetic inputs for the batched-ADMM radiosurgery path.

This module is the ONLY code shared by the fp64 CPU oracle (`oracle/`) and the CUDA
path (`paper_2509_08602_b200/`).  It holds none of the method's arithmetic: it only
produces the *inputs* of `admm_setup` / `admm_solve_batch` -- the dense dose-rate
matrix Phi, the point classes, the objective weightings and the per-plan row masks --
with the shapes BASELINE.json `configs` names.  The inputs stand in for the paper's 20
clinical Gamma Knife cases (Table 1 :187-211), which are not public.

The recipe is stated in DESIGN.md section "Synthetic inputs".
"""
from .generate import (  # noqa: F401
    CONFIGS,
    ClassSpec,
    Workload,
    default_rho,
    scaled_rho,
    make_workload,
    make_tiny_workload,
    make_candidates,
    pick_from_union,
    pack_mask,
    splitmix64,
    uniform01,
    weight_grid,
    with_plans_of,
    with_sector_coupling,
)
