import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


# The tests compute-sanitizer is run on (profiles/r02_sanitizers.md): small problems that between them launch every kernel
# of the library, every tcgen05 variant included (pixel contraction as CTA pairs and single CTA, every stage X / stage YZ
# form of the separable route, NUFFT, render, fit, the CUDA-core variants).
SANITIZE = (
    "test_gpu_parity.py::test_qmap_matches_oracle", "test_gpu_parity.py::test_orient_matches_oracle",
    "test_gpu_parity.py::test_effective_strength_matches_oracle", "test_gpu_parity.py::test_cfg1_sphere_full_pattern",
    "test_gpu_parity.py::test_ragged_random_batch_with_orientations", "test_gpu_parity.py::test_sparse_blobs_exercise_block_skipping",
    "test_gpu_parity.py::test_empty_and_single_voxel", "test_gpu_parity.py::test_forward_pixel_and_explicit_q",
    "test_gpu_parity.py::test_issuers_stay_in_step_on_mixed_odd_even_kstep_units",
    "test_gpu_parity.py::test_create_destroy_create_runs_every_route",
    "test_gpu_qgrid.py::test_ragged_batch_with_orientations", "test_gpu_qgrid.py::test_batch_with_a_vacuum_item_and_a_single_voxel",
    "test_gpu_qgrid.py::test_wide_grids_use_narrower_stage_x_tiles", "test_gpu_qgrid.py::test_cfg1_sphere_on_a_uniform_q_grid",
    "test_gpu_qgrid.py::test_tile_parities_select_the_stage_yz_variants",
    "test_gpu_nufft.py::test_cfg1_sphere_full_pattern", "test_gpu_nufft.py::test_ragged_random_batch_with_orientations",
    "test_gpu_nufft.py::test_empty_and_single_voxel", "test_gpu_nufft.py::test_fused_prefix_pass_on_an_oriented_batch",
    "test_gpu_qgrid.py::test_fused_prefix_pass_on_an_oriented_batch",
    "test_gpu_render.py::test_shape_batches_large_enough_for_the_sparse_render_and_fused_prefix_pass",
    "test_gpu_render.py::test_ellipsoids_ragged_dims_random_orientations", "test_gpu_render.py::test_spherical_harmonics_droplets",
    "test_gpu_render.py::test_radial_maps", "test_gpu_render.py::test_volume_maps",
    "test_gpu_fitting.py::test_discrepancy_matches_oracle_over_several_chunks_and_a_ragged_tail",
    "test_gpu_fitting.py::test_ideal_detector_counts_equal_the_oracles",
    "test_gpu_fitting.py::test_discrepancy_with_16_byte_loads_and_without",
    "test_gpu_parity.py::test_effective_strength_on_both_column_walks",
    "test_gpu_parity.py::test_orient_single_grid_whose_slices_are_shared_by_several_blocks",
)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "san: the subset compute-sanitizer is run on (-m 'gpu and san')")


def pytest_collection_modifyitems(config, items):
    for it in items:
        if any(it.nodeid.split("[")[0].endswith(name) for name in SANITIZE):
            it.add_marker(pytest.mark.san)
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)
