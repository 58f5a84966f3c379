"""B200-native (sm_100a) field evaluation for the coupled-wave method of arXiv 2404.07293.

The product is libscw.so (include/scwatter.h); this package is its thin Python binding.
Build the library in-tree with `python -m paper_2404_07293_b200.build`.
"""
from .binding import (SCW_C64, SCW_C128, SCW_PATH_AUTO, SCW_PATH_SIMT, SCW_PATH_TENSOR, SCW_SIDE_ABOVE, SCW_SIDE_BELOW,
                      Context, Exterior, Layer, PlaneWaves, ScwError, lib, scw_assemble_spectra, scw_eval_points,
                      scw_eval_points_noalloc, SCW_POINTS_NOALLOC_MAX_J,
                      scw_calibrate, scw_exterior_grid, scw_exterior_points, scw_exterior_spectra, scw_absorbance, scw_build_V, scw_propagate_alpha, scw_synthesize_grid, scw_sweep_detector, scw_sweep_intensity,
                      scw_sweep_wavelengths, scw_sweep_wavelengths_host)

__all__ = ["SCW_C64", "SCW_C128", "SCW_PATH_AUTO", "SCW_PATH_SIMT", "SCW_PATH_TENSOR", "SCW_SIDE_ABOVE", "SCW_SIDE_BELOW",
           "Context", "Exterior", "Layer", "PlaneWaves", "ScwError", "lib", "scw_assemble_spectra", "scw_eval_points",
           "scw_eval_points_noalloc", "SCW_POINTS_NOALLOC_MAX_J",
           "scw_calibrate", "scw_exterior_grid", "scw_exterior_points", "scw_exterior_spectra", "scw_absorbance", "scw_build_V", "scw_propagate_alpha", "scw_synthesize_grid", "scw_sweep_detector", "scw_sweep_intensity", "scw_sweep_wavelengths",
           "scw_sweep_wavelengths_host"]
