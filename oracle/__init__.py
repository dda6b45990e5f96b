"""CPU oracle for the hybrid-FFT demagnetization field (arXiv 1910.07054).

TEST INFRASTRUCTURE ONLY.  Nothing under ``paper_1910_07054_b200/`` imports this
package; only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs do.  See ``oracle/oracle.py``.
"""
from .oracle import (  # noqa: F401
    build,
    newell_f,
    newell_g,
    tensor_point,
    nxx_fp64,
    tensor_row,
    tensor_spectrum,
    direct_field,
    direct_cells,
    hybrid_field,
    hybrid_layers,
    threads,
)
