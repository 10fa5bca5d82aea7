"""Host logic of the block decomposition over GPUs (paper_2006_15698_b200/decomposed.py) on the
CPU: who owns what, who neighbours whom, message order, and the face exchange itself over torch.distributed with the
gloo backend and world_size 2 and 4 (the kernels that produce and consume the faces are tested on the GPU in
tests/test_gpu_halo.py, several ranks' contexts in one process)."""
import socket

import pytest

from paper_2006_15698_b200.decomposed import HALO, PERIODIC, WALL, FARFIELD, Decomposition, choose_variant

torch = pytest.importorskip("torch")


def test_blocks_tile_the_mesh_and_neighbours_are_mutual():
    for n, procs, bc in [((7, 6, 5), (2, 2, 2), (0,) * 6), ((9, 4, 4), (3, 1, 2), (1, 2, 0, 0, 1, 1)), ((5, 5, 5), (1, 1, 1), (0,) * 6)]:
        d = Decomposition(n, procs, bc)
        owned = set()
        for r in range(d.size):
            (x0, x1), (y0, y1), (z0, z1) = d.local_box(r)
            cells = {(x, y, z) for x in range(x0, x1) for y in range(y0, y1) for z in range(z0, z1)}
            assert not (cells & owned)
            owned |= cells
            assert d.rank_of(d.coords(r)) == r
            for f in range(6):
                nb = d.neighbour(r, f)
                if nb is None:
                    assert bc[f] != PERIODIC and d.local_bc(r)[f] == bc[f]
                else:
                    assert d.neighbour(nb, f ^ 1) == r                 # mutual, across the opposite face
                    a = f // 2                                         # and the shared face has the same transverse size
                    assert [d.local_n(r)[t] for t in range(3) if t != a] == [d.local_n(nb)[t] for t in range(3) if t != a]
                    assert d.local_bc(r)[f] == (PERIODIC if nb == r else HALO)
        assert len(owned) == n[0] * n[1] * n[2]


def test_receives_are_posted_in_the_order_the_peer_sends():
    for procs in [(2, 1, 1), (2, 2, 1), (3, 2, 2), (1, 1, 2)]:
        d = Decomposition((6, 6, 6), procs)
        for a in range(d.size):
            for b in range(d.size):
                if a == b:
                    continue
                sent = [f for f, nb in d.sends(a) if nb == b]            # faces of a, in posting order
                got = [f for f, nb in d.recvs(b) if nb == a]             # faces of b, in posting order
                assert got == [f ^ 1 for f in sent]
    # two ranks along a periodic axis: each is the other's neighbour on BOTH faces
    d = Decomposition((4, 4, 4), (2, 1, 1))
    assert d.sends(0) == [(0, 1), (1, 1)] and d.recvs(0) == [(1, 1), (0, 1)]
    assert d.local_bc(0) == (HALO, HALO, PERIODIC, PERIODIC, PERIODIC, PERIODIC)
    d = Decomposition((4, 4, 4), (2, 1, 1), (WALL, FARFIELD, 0, 0, 0, 0))
    assert d.local_bc(0) == (WALL, HALO, 0, 0, 0, 0) and d.local_bc(1) == (HALO, FARFIELD, 0, 0, 0, 0)
    with pytest.raises(ValueError):
        Decomposition((4, 4, 4), (5, 1, 1))
    with pytest.raises(ValueError):
        Decomposition((4, 4, 4), (2, 1, 1), (WALL, 0, 0, 0, 0, 0))


def test_one_column_shape_for_all_ranks():
    d = Decomposition((64, 64, 64), (2, 2, 2))                                # blocks of 32: 2x3 pads 33/32 = 3 %: accepted
    assert choose_variant(d, 4, [(2, 3), (3, 2), (2, 2), (1, 1)]) == 0
    d = Decomposition((32, 32, 32), (2, 2, 2))                                # blocks of 16: 2x3 and 3x2 pad 18/16 = 12.5 %
    assert choose_variant(d, 4, [(2, 3), (3, 2), (2, 2), (1, 1)]) == 2
    d = Decomposition((9, 9, 9), (2, 1, 1))                                   # blocks of 5 and 4 elements along x
    assert choose_variant(d, 1, [(4, 4), (1, 1)]) == 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, procs, out):
    import torch.distributed as dist
    from paper_2006_15698_b200.decomposed import Decomposition, exchange_torch_distributed
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    d = Decomposition((6, 5, 4), procs)
    # stand-ins for the face buffers: every export is tagged with (rank, face); sizes differ per face like the real ones
    size = lambda f: 10 + 3 * (f // 2)
    sends = [(f, nb, torch.full((size(f),), 100.0 * rank + f, dtype=torch.float64)) for f, nb in d.sends(rank)]
    recvs = [(f, nb, torch.zeros(size(f), dtype=torch.float64)) for f, nb in d.recvs(rank)]
    for _ in range(3):                                                       # several rounds, like several stages
        exchange_torch_distributed(dist)(rank, sends, recvs)
    ok = all(bool((buf == 100.0 * nb + (f ^ 1)).all()) for f, nb, buf in recvs)
    lam = torch.tensor([1.0 + rank], dtype=torch.float64)
    dist.all_reduce(lam, op=dist.ReduceOp.MAX)
    out[rank] = (ok, len(recvs), float(lam.item()))
    dist.destroy_process_group()


@pytest.mark.parametrize("procs", [(2, 1, 1), (1, 1, 2), (2, 2, 1)])
def test_face_exchange_over_gloo(procs):
    import torch.multiprocessing as mp
    world = procs[0] * procs[1] * procs[2]
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), procs, out), nprocs=world, join=True)
        res = dict(out)
    assert len(res) == world
    for rank in range(world):
        ok, nrecv, lam = res[rank]
        assert ok and nrecv == 2 * sum(1 for p in procs if p > 1) and lam == float(world)
