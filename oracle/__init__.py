"""CPU oracle for the stroke-expansion hot path (TEST INFRASTRUCTURE, see stroke_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It never imports paper_2405_00127_b200's CUDA binding, and that package never imports this.
"""
from .binding import build as _build_stroke, expand, lib, piece_expand, OracleResult  # noqa: F401
from .binning import bin_lines, build as _build_bin  # noqa: F401


def build(force=False):
    """Compile every C source of the oracle (stroke_oracle.c, bin_oracle.c)."""
    _build_bin(force)
    return _build_stroke(force)
