"""z-slab bookkeeping of an ahs_group: which planes a slab owns, who its neighbours are, and
which plane of which slab feeds which ghost plane after every step.

The rules themselves live in ONE place, csrc/ahs_api.cu (`slab_layout`, which `ahs_group_create` wires into the step kernel's peer
stores); `layout` below reads them through the C ABI (`ahs_slab_layout`, no GPU needed) and only wraps them in records: slab r of P
owns the global planes [r N/P, (r+1) N/P) at its local planes 1 .. N/P; local plane 0 is the ghost below (the top own plane of slab
r-1, periodically), local plane N/P + 1 the ghost above (the bottom own plane of slab r+1).  `binding.Group.layout` returns these
records; a driver that spreads the slabs over several processes (one rank per GPU) uses `owner` and `exchange_plan` to know which
transfers are local copies and which cross ranks (tests/test_slabs_host.py runs that plan over gloo, world_size 2, on CPU).
"""
from __future__ import annotations

from dataclasses import dataclass

# the five arrays whose boundary planes cross a slab face every step (new phi, theta of Eqs. 6-7), and the one extra array the
# Gauss residual of the slab above needs (eps_2 of the top plane); indices into the 10-field order of include/ahs.h
FACE_FIELDS = (0, 1, 4, 5, 6)
GAUSS_FIELD = 9


@dataclass(frozen=True)
class Slab:
    rank: int          # slab index r
    nslabs: int        # P
    N: int
    z_offset: int      # first own global plane
    nz: int            # own planes
    lo: int            # slab below (periodic)
    hi: int            # slab above (periodic)
    nz_alloc: int      # planes allocated per array: own planes at local 1 .. nz between the two ghost planes

    def local_plane(self, z_global: int) -> int:
        """Local index of an own global plane."""
        z = (z_global - self.z_offset) % self.N
        if not 0 <= z < self.nz:
            raise ValueError("plane %d is not owned by slab %d" % (z_global, self.rank))
        return z + 1

    def ghost_planes(self) -> dict:
        """{local ghost plane: global plane it mirrors}"""
        return {0: (self.z_offset - 1) % self.N, self.nz + 1: (self.z_offset + self.nz) % self.N}


def layout(N: int, nslabs: int) -> list:
    from . import binding
    try:
        return [Slab(r, nslabs, N, *binding.slab_layout(N, nslabs, r)) for r in range(max(nslabs, 1))]
    except binding.AhsError as e:
        raise ValueError(str(e))


def exchange_plan(N: int, nslabs: int) -> list:
    """The face transfers of one step, in a fixed order: (src slab, src local plane, dst slab, dst local plane, field indices).
    The bottom own plane of slab r goes to the ghost above of slab r-1, the top own plane to the ghost below of slab r+1 (with
    eps_2 for the Gauss residual)."""
    plan = []
    for s in layout(N, nslabs):
        plan.append((s.rank, 1, s.lo, s.nz + 1, FACE_FIELDS))
        plan.append((s.rank, s.nz, s.hi, 0, FACE_FIELDS + (GAUSS_FIELD,)))
    return plan


def owner(slab_rank: int, nslabs: int, world: int) -> int:
    """Process that drives slab `slab_rank` when P slabs are spread over `world` processes in contiguous blocks."""
    if nslabs % world != 0:
        raise ValueError("the number of slabs must be a multiple of the number of processes")
    return slab_rank // (nslabs // world)
