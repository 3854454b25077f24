"""Seeded synthetic input generators (scenes, cameras, ray batches).

Shared by the oracle tests and by the CUDA path's tests/bench.  This package
holds NONE of the method's arithmetic (no RNG of the method, no partition, no
sampling, no intersection): it only produces triangles, materials, cameras and
plain random ray batches from `numpy.random.default_rng(seed)`.
"""
from .scenes import (  # noqa: F401
    MAT_DIFFUSE, MAT_GLOSSY, MAT_SPECULAR, MAT_EMISSIVE, MATERIAL_DTYPE,
    Scene, make_camera, cornell, interior, landscape, furnace_sphere,
    emissive_box, floor_plane, checker_floor, random_rays, by_name,
)
