"""CPU FP64 oracle of the D3Q19 LBM-LES step — TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2607_04516_b200``.  See ``oracle/lbm_oracle.c`` for what it follows.
"""
from .lbm_oracle import Oracle, build, lattice, feq, collide_cell, collide_cell_vec, collide_cell_damped, vk_spectrum, round_half  # noqa: F401
from . import mesh_voxel  # noqa: F401,E402
