"""Multi-GPU plan of the pointwise path: every grid point is independent, so the only
multi-rank logic is a partition of the points.  Elements (512 GLL points at
order 7) are dealt to ranks in contiguous ranges, as the paper's MPI
decomposition over elements does; the mechanism tables are replicated on
every rank; there is no data-path collective.  ``torch.distributed`` is used by callers only
for the timing barrier and the max-over-ranks reduction of the measured time.
"""
from __future__ import annotations

from .workloads import POINTS_PER_ELEMENT


def element_range(n_elements: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [first, last) element range of ``rank``: sizes differ by at most one element."""
    if not (0 <= rank < world) or n_elements < 0:
        raise ValueError("bad rank/world/n_elements")
    base, extra = divmod(n_elements, world)
    first = rank * base + min(rank, extra)
    return first, first + base + (1 if rank < extra else 0)


def point_range(n_elements: int, rank: int, world: int) -> tuple[int, int]:
    """[first, last) point range of ``rank`` (strong scaling: one field split over the ranks)."""
    a, b = element_range(n_elements, rank, world)
    return a * POINTS_PER_ELEMENT, b * POINTS_PER_ELEMENT


def weak_range(points_per_rank: int, rank: int, world: int) -> tuple[int, int, int]:
    """(offset, n, total) of ``rank`` under weak scaling: each rank owns ``points_per_rank``
    points of a field of ``world * points_per_rank`` points."""
    if not (0 <= rank < world):
        raise ValueError("bad rank/world")
    return rank * points_per_rank, points_per_rank, world * points_per_rank
