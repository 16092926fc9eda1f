"""Seeded synthetic inputs and the BASELINE.json workload table.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_1009_1380_b200/``).  It holds none of the method's arithmetic: no
Fourier transforms, no gridding kernel, no Radon geometry -- only phantom
rasterisation and random draws (``numpy.random.default_rng(seed)``).

The paper's workload is experimental phase-contrast scans of two 60 um glass
spheres at ALS beamline 8.3.2 (Fig. 1).  That data is
not available; the phantoms below take its shapes (piecewise-constant discs,
an edge-enhanced "Laplacian" two-sphere slice) and stand in
for it.  The recipe is restated in DESIGN.md section 5.
"""
from .configs import CONFIGS, RadonConfig, get_config
from .phantoms import (
    additive_disks,
    painted_disks,
    two_sphere_slice,
    make_image,
    make_batch_slice,
    gaussian_blob,
    single_disk,
    white_noise,
    delta_image,
    random_complex,
)

__all__ = [
    "CONFIGS", "RadonConfig", "get_config",
    "additive_disks", "painted_disks", "two_sphere_slice", "make_image",
    "make_batch_slice", "gaussian_blob", "single_disk", "white_noise",
    "delta_image", "random_complex",
]
