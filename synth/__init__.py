"""Seeded synthetic inputs for the fem_assemble path.

This package is shared by the CPU oracle tests and the CUDA path.  It holds NO
arithmetic of the method (no shape functions, no constitutive law, no CSR
logic): only meshes, displacement / history fields and material *descriptions*
built from a counter-based RNG.  Neither `oracle/` nor
`paper_2606_17390_b200/` is imported here.
"""
from .rng import uniform, normal, permutation  # noqa: F401
from .mesh import structured_hex_mesh, void_mask_mesh  # noqa: F401
from .configs import make_config, CONFIG_NAMES  # noqa: F401
