"""The N > 1 plumbing of the t-decomposition (paper_1212_0785_b200/slabs.py) on CPU with
world_size 2 and 3 over gloo: slab partition, neighbour messages, halos, reductions in fixed rank order.  No GPU
and no kernels: a slab here is a plain tensor [t_count + 2][sites per timeslice][reals], faces are its rows."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_partition_covers_the_lattice_with_even_slabs():
    from paper_1212_0785_b200.slabs import partition
    for Lt, n in ((16, 2), (16, 4), (96, 8), (10, 3), (8, 4), (64, 1), (12, 5)):
        p = partition(Lt, n)
        assert len(p) == n and p[0][0] == 0 and sum(c for _, c in p) == Lt
        assert all(c % 2 == 0 and c >= 2 for _, c in p)
        assert all(p[i + 1][0] == p[i][0] + p[i][1] for i in range(n - 1))
        assert max(c for _, c in p) - min(c for _, c in p) <= 2
    for Lt, n in ((16, 9), (15, 2), (8, 0)):
        with pytest.raises(ValueError):
            partition(Lt, n)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1212_0785_b200.slabs import SlabComm, partition
    Lt, Vs, k = 12, 10, 3
    g = torch.arange(Lt * Vs * k, dtype=torch.float64).reshape(Lt, Vs, k) * 0.5 + 1.0  # the "global field"
    tb, tc = partition(Lt, world)[rank]
    slab = torch.full((tc + 2, Vs, k), -1.0, dtype=torch.float64)
    slab[1: tc + 1] = g[tb: tb + tc]
    comm = SlabComm(rank, world, dist)
    lo, up = comm.exchange(slab[1].clone(), slab[tc].clone())  # first interior row down, last interior row up
    slab[0], slab[tc + 1] = lo, up
    ok_halo = bool(torch.equal(slab[0], g[(tb - 1) % Lt]) and torch.equal(slab[tc + 1], g[(tb + tc) % Lt]))
    # reductions: rank-ordered sum and per-timeslice concatenation
    local = slab[1: tc + 1].sum(dim=(1, 2))
    total = comm.combine(local.sum().reshape(1))
    per_t = comm.gather_concat(local)
    torch.save({"ok_halo": ok_halo, "total": total, "per_t": per_t, "want_per_t": g.sum(dim=(1, 2)),
                "lower": comm.lower, "upper": comm.upper}, f"{out}.{rank}")
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_halo_exchange_and_rank_ordered_reductions_over_gloo(tmp_path, world):
    out = str(tmp_path / "s")
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    res = [torch.load(f"{out}.{r}") for r in range(world)]
    for r, x in enumerate(res):
        assert x["ok_halo"], r
        assert x["lower"] == (r - 1) % world and x["upper"] == (r + 1) % world
        assert torch.equal(x["per_t"], x["want_per_t"])  # global timeslice order
        assert torch.equal(x["total"], res[0]["total"])  # the same bits on every rank
    assert abs(res[0]["total"].item() - res[0]["want_per_t"].sum().item()) < 1e-9


def test_single_slab_wraps_onto_itself():
    from paper_1212_0785_b200.slabs import SlabComm
    comm = SlabComm(0, 1)
    a, b = torch.tensor([1.0, 2.0]), torch.tensor([3.0, 4.0])
    lo, up = comm.exchange(a, b)  # what I send up comes back from below
    assert torch.equal(lo, b) and torch.equal(up, a)
    assert torch.equal(comm.combine(a), a) and torch.equal(comm.gather_concat(b), b)
