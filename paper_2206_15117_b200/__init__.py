"""B200-native gridding / degridding hot path of the GPU imager of arxiv/paper_2206_15117.

The product is `libimager.so` (CUDA, sm_100a; C-ABI in include/imager.h).  This package is its thin Python
binding: the four hot-path calls keep their C names.  Nothing here computes anything on the CPU.
"""
from .binding import (ImagerError, Plan, load_library, hogbom as imager_hogbom, hogbom_static as imager_hogbom_static, reproject as imager_reproject, MODE_DELTA, MODE_PSWF, MODE_WPROJ, MODE_AWPROJ_ADJOINT,
                      MODE_AWPROJ_PAPER, MODE_MOSAIC_PB, MODE_USER, REUSE_INDEX, PATH_REFERENCE, DEGRID_RESIDUAL, EXPORTS)


def imager_plan_create(params: dict, max_nvis: int, user_tables=None, user_tables_degrid=None, stream=None) -> Plan:
    return Plan(params, max_nvis, user_tables, user_tables_degrid, stream)


def imager_index(plan: Plan, uvw, a_index=None, stream=None):
    plan.index(uvw, a_index, stream)


def imager_grid(plan: Plan, uvw, vis, weights, grid, a_index=None, sum_weights=None, flags: int = 0, stream=None):
    plan.grid(uvw, vis, weights, grid, a_index, sum_weights, flags, stream)


def imager_degrid(plan: Plan, uvw, grid, vis_out, a_index=None, flags: int = 0, stream=None):
    plan.degrid(uvw, grid, vis_out, a_index, flags, stream)


def imager_plan_destroy(plan: Plan):
    plan.close()
