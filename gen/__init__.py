"""Seeded synthetic PLIC workloads (inputs only -- none of the method's arithmetic).

This module serves both the fp64 oracle (``oracle/``) and the CUDA path
(``paper_2006_12838_b200``); it imports neither.  Every workload is a set of
fp32 SoA arrays ``V0, nx, ny, nz`` generated on the host with numpy's
counter-based Philox generator in fixed chunks of ``CHUNK`` cells: cell ``i``
depends only on ``(seed, stream, i // CHUNK)`` and its position in the chunk,
never on N, the thread count or the machine.  Gaussians and uniforms are drawn
in fp64, normals are normalised in fp64 and rounded to fp32 once.

The paper uses no public dataset; its own benchmark set is synthetic (random 3D
normals, a share of 2D normals, one axis normal, one face diagonal, V0 equally
spaced including 0 and 1 -- PAPER.md:250, 262).  The workloads below take that
shape with the sizes BASELINE.json's ``configs`` name; the recipe is restated
in DESIGN.md.
"""
from .workloads import (CHUNK, random_sphere, edge_cells, config1, snapped_beta,
                        paper_benchmark_set, paper_normals, roundtrip_volumes, sphere_lattice,
                        sphere_fill_lattice,
                        shard_range)

__all__ = ["CHUNK", "random_sphere", "edge_cells", "config1", "snapped_beta",
           "paper_benchmark_set", "paper_normals", "roundtrip_volumes", "sphere_lattice", "sphere_fill_lattice",
           "shard_range"]
