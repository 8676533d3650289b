"""Seeded synthetic inputs shared by the CPU oracle and the CUDA path (no method arithmetic)."""
from . import rng  # noqa: F401
from .workloads import (  # noqa: F401
    CONFIGS, Config, Scene, build_scene, scaled, focused, elements, guide_elements, focus_mask,
    exposure_times, observer_ecliptic, tangent_points, variance_scalars, noise_plane_np,
    noise_plane_t, noise_values_np, variance_plane_np, injected_index, injected_amplitudes,
    GAUSS_K, GM_SUN, C_AU_PER_DAY, OBLIQUITY, PIXEL_SCALE, DEG,
)
