"""fp64 CPU oracle for the 3D R2C / C2R path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares nothing with
``paper_2202_12756_b200`` (no code, tables, headers or helpers) and neither imports
the other.  See ``oracle/fft3d_oracle.c`` for what is computed and the citations.
"""
from .fft3d_oracle import (  # noqa: F401
    build_oracle,
    dft3d_direct,
    idft3d_direct,
    fft1d,
    r2c,
    c2r,
    r2c_pencils,
    c2r_points,
    dft3d_c2c_direct,
    c2c,
    max_threads,
)
from .slab_layout import (  # noqa: F401
    slab_index,
    natural_to_slab,
    slab_to_natural,
    simulate_paper_steps_2_to_4,
    pencil_cz,
    pencil_index,
    natural_to_pencil,
    pencil_to_natural,
    simulate_pencil_transposes,
)
