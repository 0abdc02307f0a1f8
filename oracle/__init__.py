"""CPU oracle for libaffinescan — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` /
``--impl reference`` legs of ``bench.py`` may import this package.  It shares no
code with ``paper_2606_00601_b200`` (the CUDA path) and never imports it.
"""
from .oracle import (  # noqa: F401
    affine_scan,
    blelloch_scan,
    build,
    compose,
    fold_pairs,
    selective_scan_bwd,
    selective_scan_fwd,
    selective_scan_fwd_ext,
)
