"""Host logic of the domain decomposition (tmw_options.domains_z / domains_t of include/tmw.h).

The lattice L^3 x T is cut into Pz x Pt sub-lattices L x L x (L/Pz) x (T/Pt), t first, then z (the paper ran on 4-36 GPUs:
PAPER.md:52, the "Nodes" columns of Table 2 :71-76; "the network has much stronger impact on the performance", :315).
This module restates, on the host, the index maps the CUDA kernels of csrc/ use, so that they can be checked without a
GPU and so that bench.py can report the bytes a cut moves:

  * domain (iz, it) has index iz + Pz * it and owns the global sites with z in [iz*Lz, (iz+1)*Lz), t in [it*Tl, (it+1)*Tl);
  * a hop in direction z or t that leaves a domain arrives through a ghost buffer: "lo" (the backward hop of the sites at
    local coordinate 0, sent by the neighbour BEHIND from its last slice) or "hi" (the forward hop of the sites at the last
    local coordinate, sent by the neighbour AHEAD from its first slice);
  * face index f = xh + Lh*(y + L*t_local) for a z cut and xh + Lh*(y + L*z_local) for a t cut, xh = x // 2; it is the same
    number for the output site and for the site whose spinor it receives;
  * the antiperiodic sign multiplies a ghost term only on the physical time boundary: the lo ghost of the domains with
    it = 0 and the hi ghost of those with it = Pt - 1 (reading C6), never on an internal cut;
  * with several ranks the domains are dealt in contiguous blocks, so that z-neighbours share a rank first.

Only arithmetic on indices; nothing here touches a spinor or a link.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

Z, T_DIR = 0, 1       # the two directions that may be cut
LO, HI = 0, 1         # ghost sides
HALF_SPINOR_REALS = 12


@dataclass(frozen=True)
class Partition:
    L: int
    T: int
    pz: int = 1
    pt: int = 1

    def __post_init__(self):
        if self.pz < 1 or self.pt < 1 or self.L % (2 * self.pz) or self.T % (2 * self.pt):
            raise ValueError("domains_z / domains_t must divide L / T into even local extents")

    # ---- shapes ----
    @property
    def ndom(self) -> int:
        return self.pz * self.pt

    @property
    def Lz(self) -> int:
        return self.L // self.pz

    @property
    def Tl(self) -> int:
        return self.T // self.pt

    @property
    def local_volume(self) -> int:
        return self.L * self.L * self.Lz * self.Tl

    def cut(self, direction: int) -> bool:
        return (self.pz if direction == Z else self.pt) > 1

    def nface(self, direction: int) -> int:
        """face sites of ONE parity on a cut of this direction"""
        return (self.L // 2) * self.L * (self.Tl if direction == Z else self.Lz)

    def face_bytes(self, direction: int, real_bytes: int = 4) -> int:
        """bytes one domain sends through ONE side of a cut per stencil application and column: 12 reals per face site"""
        return HALF_SPINOR_REALS * real_bytes * self.nface(direction)

    def exchange_bytes(self, real_bytes: int = 4) -> int:
        """bytes all domains together move per stencil application and column (2 sides per cut direction)"""
        return sum(2 * self.face_bytes(d, real_bytes) * self.ndom for d in (Z, T_DIR) if self.cut(d))

    # ---- domains ----
    def index(self, iz: int, it: int) -> int:
        return iz + self.pz * it

    def coords(self, d: int) -> tuple[int, int]:
        return d % self.pz, d // self.pz

    def origin(self, d: int) -> tuple[int, int]:
        iz, it = self.coords(d)
        return iz * self.Lz, it * self.Tl

    def domain_of(self, z: int, t: int) -> int:
        return self.index(z // self.Lz, t // self.Tl)

    def behind(self, d: int, direction: int) -> int:
        iz, it = self.coords(d)
        return self.index((iz - 1) % self.pz, it) if direction == Z else self.index(iz, (it - 1) % self.pt)

    def ahead(self, d: int, direction: int) -> int:
        iz, it = self.coords(d)
        return self.index((iz + 1) % self.pz, it) if direction == Z else self.index(iz, (it + 1) % self.pt)

    def ghost_sign(self, d: int, direction: int, side: int) -> int:
        if direction != T_DIR:
            return 1
        _, it = self.coords(d)
        return -1 if (side == LO and it == 0) or (side == HI and it == self.pt - 1) else 1

    # ---- faces ----
    def face_sites(self, d: int, direction: int, side: int, parity: int) -> np.ndarray:
        """GLOBAL coordinates (x, y, z, t), shape (nface, 4), of the sites of `parity` on the slice of domain d at local
        coordinate 0 (side = LO) or the last one (side = HI) in `direction`, ordered by face index."""
        L, Lh = self.L, self.L // 2
        oz, ot = self.origin(d)
        n_other = self.Tl if direction == Z else self.Lz
        f = np.arange(Lh * L * n_other)
        xh, y, o = f % Lh, (f // Lh) % L, f // (Lh * L)
        if direction == Z:
            z = np.full_like(f, oz + (self.Lz - 1 if side == HI else 0))
            t = ot + o
        else:
            z = oz + o
            t = np.full_like(f, ot + (self.Tl - 1 if side == HI else 0))
        x = 2 * xh + ((y + z + t + parity) & 1)
        return np.stack([x, y, z, t], axis=1)

    def messages(self) -> list[tuple[int, int, int, int]]:
        """(source domain, destination domain, direction, ghost side filled at the destination) of one stencil application:
        a domain's first slice goes to the hi ghost of the neighbour behind, its last slice to the lo ghost of the one ahead"""
        out = []
        for d in range(self.ndom):
            for direction in (Z, T_DIR):
                if self.cut(direction):
                    out.append((d, self.behind(d, direction), direction, HI))
                    out.append((d, self.ahead(d, direction), direction, LO))
        return out


def domains_for_rank(rank: int, world: int, ndom: int) -> list[int]:
    """Domains held by `rank`: contiguous blocks (ndom must be a multiple of world), so that the z-neighbours of a time
    slab share a rank before t-neighbours do."""
    if world < 1 or not 0 <= rank < world or ndom % world:
        raise ValueError(f"cannot deal {ndom} domains to rank {rank} of {world}")
    per = ndom // world
    return list(range(rank * per, (rank + 1) * per))


def rank_of_domain(d: int, world: int, ndom: int) -> int:
    if ndom % world or not 0 <= d < ndom:
        raise ValueError("bad domain / world")
    return d // (ndom // world)
