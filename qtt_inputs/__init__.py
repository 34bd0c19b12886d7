"""Seeded synthetic input generators shared by the oracle tests, the GPU parity
tests and bench.py.

This module holds NONE of the method's arithmetic (no MPS/MPO algebra, no
encoding, no stencils): it only produces dense N x N velocity fields, laid out
``F[x][y]`` on the grid x_j = y_j = j/N, and raw random site tensors, with
``numpy.random.default_rng(seed)``.  Both the CPU oracle and the CUDA path are
fed the SAME host arrays produced here, so parity never depends on reproducing
an RNG on the device.

The recipes are the ones BASELINE.json ``configs`` states (stand-ins for the
paper's decaying-jet / decaying-turbulence workloads, Sec. III
and PAPER.md:689-726 App. C); DESIGN.md section "Input recipe" restates them.
"""
from .fields import (  # noqa: F401
    CONFIGS,
    grid,
    config1_field,
    shear_layer,
    decaying_jet,
    decaying_turbulence,
    random_cores,
    bond_profile,
    config_fields,
    taylor_green_3d,
)
