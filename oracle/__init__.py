"""CPU oracle for the SHO projection hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs of
``bench.py`` may import this package.  It never imports ``paper_1905_00480_b200`` (the CUDA path)
and shares no code with it.  See ``oracle/sho_oracle.c`` for the arithmetic and its citations.
"""
from .sho_oracle import (  # noqa: F401
    build,
    nsho,
    index,
    hermite_phys,
    phi,
    box,
    project,
    project_pairs,
    add,
    add_points,
    add_points_bands,
    dmul,
    num_threads,
)
from .sho_umatrix import rlm_index, umatrix  # noqa: F401,E402
