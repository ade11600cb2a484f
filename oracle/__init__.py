"""CPU oracle for the mphv hot path -- TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package. It shares no code with
``paper_2305_01487_b200`` (the CUDA path) and neither imports the other.
"""
from .binding import (  # noqa: F401
    Grid, Box, build, lib, sweep_pencil, sweep_x, sweep_v, step, moments, total, num_threads, set_num_threads,
    boris_map, backsub_foot, sweep_pencil_faces, sweep_v_backsub, step_backsub,
    maxwellian, exchange_maxwellian, match_moments,
    BC_PERIODIC, BC_OUTFLOW, BC_WALL, OK, ERR_ARG, ERR_RANGE,
)
from . import fields  # noqa: F401,E402  (FDTD Maxwell update and the coupled step)
