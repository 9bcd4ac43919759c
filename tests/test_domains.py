"""Host-side checks of the domain-decomposition index maps (paper_2201_09004_b200/domains.py = the maps the CUDA kernels of
SURVEY §8(f4) use): no GPU. Plus the world_size-2 gloo test of the rank <-> domain map."""
import itertools
import os
import socket

import numpy as np
import pytest

from paper_2201_09004_b200 import domains as D

GRIDS = [(8, 8, 1, 2), (8, 8, 2, 1), (8, 16, 2, 2), (4, 8, 2, 4), (8, 8, 4, 1), (4, 4, 2, 2)]


@pytest.mark.parametrize("L,T,pz,pt", GRIDS)
def test_domains_tile_the_lattice(L, T, pz, pt):
    p = D.Partition(L, T, pz, pt)
    owner = np.full((T, L), -1)
    for d in range(p.ndom):
        oz, ot = p.origin(d)
        assert oz % 2 == 0 and ot % 2 == 0  # even origins: local parity = global parity
        assert np.all(owner[ot:ot + p.Tl, oz:oz + p.Lz] == -1)
        owner[ot:ot + p.Tl, oz:oz + p.Lz] = d
        assert p.index(*p.coords(d)) == d
    assert np.all(owner >= 0)
    for z, t in itertools.product(range(L), range(T)):
        assert p.domain_of(z, t) == owner[t, z]
    assert p.ndom * p.local_volume == L ** 3 * T


@pytest.mark.parametrize("L,T,pz,pt", GRIDS)
def test_every_cut_hop_arrives_exactly_once_with_the_right_sign(L, T, pz, pt):
    """For every output site and every hop in +-z, +-t: either the neighbour is in the same domain (no ghost), or exactly
    one message delivers it: the sender's face site with the SAME face index is the neighbour site, and the sign on the
    ghost term is -1 exactly when the hop wraps around the global time extent."""
    p = D.Partition(L, T, pz, pt)
    ext = {D.Z: L, D.T_DIR: T}
    axis = {D.Z: 2, D.T_DIR: 3}
    msgs = p.messages()
    assert len(msgs) == len(set(msgs)) == sum(2 * p.ndom for d in (D.Z, D.T_DIR) if p.cut(d))
    delivered = {(dst, direction, side): src for src, dst, direction, side in msgs}
    for par in (0, 1):
        for d in range(p.ndom):
            for direction in (D.Z, D.T_DIR):
                for side in (D.LO, D.HI):
                    out = p.face_sites(d, direction, side, par)          # output sites on this slice, parity par
                    assert len(out) == p.nface(direction) and np.all(out.sum(axis=1) % 2 == par)
                    step = -1 if side == D.LO else +1
                    nb = out.copy()
                    nb[:, axis[direction]] = (nb[:, axis[direction]] + step) % ext[direction]
                    wraps = (out[:, axis[direction]] + step < 0) | (out[:, axis[direction]] + step >= ext[direction])
                    nb_dom = np.array([p.domain_of(z, t) for z, t in nb[:, 2:4]])
                    if not p.cut(direction):
                        assert np.all(nb_dom == d)   # periodic inside the domain, no ghost
                        assert (d, direction, side) not in delivered
                        continue
                    src = delivered[(d, direction, side)]
                    assert np.all(nb_dom == src)
                    # the sender packs its LAST slice for our lo ghost, its FIRST slice for our hi ghost, input parity 1 - par
                    sent = p.face_sites(src, direction, D.HI if side == D.LO else D.LO, 1 - par)
                    assert np.array_equal(sent, nb)  # same face index on both sides
                    sign = p.ghost_sign(d, direction, side)
                    if direction == D.T_DIR:
                        assert np.all(wraps == (sign == -1))
                    else:
                        assert sign == 1
    # sites that are on no cut slice have all their z, t neighbours inside their own domain
    if p.Lz > 2 and p.Tl > 2:
        z, t = p.origin(p.ndom - 1)
        assert p.domain_of(z + 1 + 1, t + 1 + 1) == p.domain_of(z + 1, t + 1) == p.ndom - 1


def test_face_bytes_and_errors():
    p = D.Partition(48, 144, 1, 2)
    assert p.nface(D.T_DIR) == 24 * 48 * 48 and p.face_bytes(D.T_DIR, 4) == 12 * 4 * 24 * 48 * 48
    assert p.exchange_bytes(4) == 2 * 2 * p.face_bytes(D.T_DIR, 4)
    assert not p.cut(D.Z) and p.cut(D.T_DIR)
    for bad in ((8, 8, 3, 1), (8, 8, 1, 3), (8, 8, 8, 1), (8, 8, 0, 1)):
        with pytest.raises(ValueError):
            D.Partition(*bad)
    assert D.domains_for_rank(1, 2, 4) == [2, 3] and D.rank_of_domain(3, 2, 4) == 1
    with pytest.raises(ValueError):
        D.domains_for_rank(0, 3, 4)


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        p = D.Partition(8, 16, 2, 2)
        mine = D.domains_for_rank(rank, world, p.ndom)
        # what this rank sends to / expects from other ranks in one stencil application
        sends = sorted((s, d, direction, side) for s, d, direction, side in p.messages()
                       if s in mine and D.rank_of_domain(d, world, p.ndom) != rank)
        recvs = sorted((s, d, direction, side) for s, d, direction, side in p.messages()
                       if d in mine and D.rank_of_domain(s, world, p.ndom) != rank)
        gathered = [None] * world
        dist.all_gather_object(gathered, dict(rank=rank, mine=mine, sends=sends, recvs=recvs))
        q.put(gathered)
    finally:
        dist.destroy_process_group()


def test_rank_domain_map_two_ranks_gloo():
    """2 ranks x 2 domains each on a 2 x 2 grid: the domains partition over the ranks, every off-rank send of one rank is an
    expected receive of the other, and only the t cut crosses ranks (the z-neighbours of a time slab share a rank)."""
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    views = [q.get(timeout=120) for _ in procs]
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    g = sorted(views[0], key=lambda v: v["rank"])
    assert sorted(views[1], key=lambda v: v["rank"]) == g  # both ranks saw the same picture
    assert g[0]["mine"] == [0, 1] and g[1]["mine"] == [2, 3]
    assert g[0]["sends"] == g[1]["recvs"] and g[1]["sends"] == g[0]["recvs"]
    assert len(g[0]["sends"]) == 4 and all(direction == D.T_DIR for _, _, direction, _ in g[0]["sends"])
