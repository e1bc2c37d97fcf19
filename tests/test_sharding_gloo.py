"""N > 1 path on CPU: world size 2 over gloo (DESIGN.md sec. 7 "Multi-GPU").

The path shards with NO data-path collective: every rank evaluates a contiguous row slab of the
grid (or a slice of the models of a batch) with the whole lens list.  What has to be right on the
host side is the slab arithmetic (lens_inputs.row_slab / model_slab) and the layout in which slabs
are put together; a gather exists only to assemble one contiguous map.  Here each rank evaluates
its slab with the CPU oracle (the CUDA path needs a GPU) and rank 0 checks that the gathered map is
bit-identical to the one-process map."""
import os
import socket

import numpy as np
import pytest

import lens_inputs as li

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import oracle

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # ---- one map, row slabs
        c = li.config(2, scale=32)  # 64 x 64, 500 mixed lenses
        g = li.Grid(x0=c.grid.x0 + 0.1, y0=c.grid.y0 + 0.3, dx=c.grid.dx * 1.1, nx=c.grid.nx, ny=c.grid.ny)  # not dyadic
        j0, nrows = li.row_slab(g, rank, world)
        # a slab is (grid, j0, nrows): the oracle evaluates rows [j0, j0 + nrows) of the FULL grid definition
        mine = oracle.grid(c.lenses, g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "kappa", "mu"), rows=(j0, j0 + nrows))
        mine = {n: v[j0:j0 + nrows] for n, v in mine.items()}
        rows = [li.row_slab(g, r, world)[1] for r in range(world)]
        ok = True
        for name in ("ax", "kappa", "mu"):
            parts = [torch.empty((rows[r], g.nx), dtype=torch.float64) for r in range(world)]
            dist.all_gather(parts, torch.from_numpy(np.ascontiguousarray(mine[name])))
            if rank == 0:
                full = oracle.grid(c.lenses, g.x0, g.y0, g.dx, g.nx, g.ny, planes=(name,))[name]
                ok = ok and np.array_equal(torch.cat(parts).numpy(), full, equal_nan=True)
        # ---- a batch, model slices
        b = li.config(4, scale=64)  # 64 models x 300 lenses on 16 x 16
        m0, m1 = li.model_slab(b.nmodel, rank, world)
        loc = np.stack([oracle.grid(b.lenses[m * b.nlens:(m + 1) * b.nlens], b.grid.x0, b.grid.y0, b.grid.dx, b.grid.nx,
                                    b.grid.ny, planes=("ay",))["ay"] for m in range(m0, m1)])
        parts = [torch.empty((li.model_slab(b.nmodel, r, world)[1] - li.model_slab(b.nmodel, r, world)[0], b.grid.ny,
                              b.grid.nx), dtype=torch.float64) for r in range(world)]
        dist.all_gather(parts, torch.from_numpy(loc))
        if rank == 0:
            m = b.nmodel - 1
            ref = oracle.grid(b.lenses[m * b.nlens:], b.grid.x0, b.grid.y0, b.grid.dx, b.grid.nx, b.grid.ny,
                              planes=("ay",))["ay"]
            ok = ok and np.array_equal(torch.cat(parts)[m].numpy(), ref)
        # ---- the bench's timing reduction: MAX over ranks
        t = torch.tensor([10.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ok = ok and float(t.item()) == 10.0 + world - 1
        if rank == 0:
            q.put(bool(ok))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_world_size_2_row_slabs_and_model_slices_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    mp.spawn(_worker, args=(world, port, q), nprocs=world, join=True)
    assert q.get() is True


@pytest.mark.parametrize("ny,world", [(64, 2), (7, 3), (2, 4), (1, 1), (4096, 8)])
def test_row_slabs_tile_the_grid(ny, world):
    g = li.Grid(x0=-3.0, y0=1.5, dx=0.25, nx=5, ny=ny)
    nxt = 0
    for r in range(world):
        j0, nrows = li.row_slab(g, r, world)
        assert j0 == nxt and 0 <= nrows <= -(-ny // world)
        nxt += nrows
    assert nxt == ny
    with pytest.raises(ValueError):
        li.row_slab(g, world, world)


def test_model_slices_tile_the_batch():
    for n, w in [(64, 2), (64, 8), (5, 3), (1, 4)]:
        ends = [li.model_slab(n, r, w) for r in range(w)]
        assert ends[0][0] == 0 and ends[-1][1] == n
        assert all(ends[i][1] == ends[i + 1][0] for i in range(w - 1))
