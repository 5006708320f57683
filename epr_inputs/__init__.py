"""Seeded synthetic inputs for the EPR hot path (numpy only).

This package is the ONE thing the fp64 oracle's tests and the CUDA path's tests / bench share.
It holds none of the method's arithmetic (no closure stencil, no ray map, no splat / gather, no
Paganin filter, no projection): it builds random-ellipsoid phantoms, the per-config physical
scalars, and detector images by an independent *wave-optics* simulation (paraxial Fresnel
propagation of the exit wave, PAPER.md:333-343 Eq. (S5)-(S7) — the physics the method inverts,
which the method itself never evaluates) plus Poisson noise.

The recipe is stated in DESIGN.md §"Synthetic inputs".
"""
from .configs import CONFIGS, Workload, make_workload, shard_range  # noqa: F401
from .phantom import ellipsoid_phantom  # noqa: F401
from .simulate import fresnel_detector, poisson_noise  # noqa: F401
