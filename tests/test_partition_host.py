"""CPU tests of the NEXT-2 host logic (paper_2409_10383_b200/partition.py): the z-slab partition map, the neighbour
table, and the 8-double all-reduce of the constraint norms on a world_size-2 gloo group, checked against the oracle's
mesh-wide norms (PAPER.md:285-309 is the scaling section; the exchange itself is PAPER.md:65, 75-76)."""
import os
import socket
from dataclasses import replace

import numpy as np
import pytest

from paper_2409_10383_b200 import inputs as I
from paper_2409_10383_b200 import partition as PT


def test_slab_partition_is_a_balanced_cover():
    for nbz in range(1, 20):
        for R in range(1, nbz + 1):
            parts = PT.slab_partition(nbz, R)
            assert len(parts) == R and parts[0][0] == 0
            assert all(parts[r][0] + parts[r][1] == parts[r + 1][0] for r in range(R - 1))
            assert parts[-1][0] + parts[-1][1] == nbz
            sizes = [t for _, t in parts]
            assert min(sizes) >= 1 and max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        PT.slab_partition(3, 4)


def test_slab_neighbours_and_params():
    assert PT.slab_neighbours(0, 1, 0) == (None, None)
    assert PT.slab_neighbours(0, 2, 0) == (1, 1) and PT.slab_neighbours(1, 2, 0) == (0, 0)
    assert PT.slab_neighbours(0, 4, 0) == (3, 1) and PT.slab_neighbours(3, 4, 0) == (2, 0)
    assert PT.slab_neighbours(0, 4, 1) == (None, 1) and PT.slab_neighbours(3, 4, 1) == (2, None)
    p = I.params_noise(8, (2, 3, 5), dx=0.1)
    u = np.arange(I.NF * 40 * 24 * 16, dtype=np.float64).reshape(I.NF, 40, 24, 16)
    got = []
    for r in range(3):
        ps = PT.slab_params(p, r, 3)
        bz0, nbz = PT.slab_partition(5, 3)[r]
        assert ps.nb == (2, 3, nbz) and abs(ps.xmin[2] - (p.xmin[2] + bz0 * 8 * 0.1)) < 1e-15
        got.append(PT.slab_interior(u, p, r, 3))
        assert got[-1].shape == (I.NF, nbz * 8, 24, 16)
    assert np.array_equal(np.concatenate(got, axis=1), u)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _norm_worker(rank, world, port, tmp):
    import torch
    import torch.distributed as dist
    from oracle import oracle as O
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = replace(I.params_noise(8, (1, 1, 4), dx=0.05), bc=0)
    u = O.enforce(p, I.smooth_random_data(p, 5, 0.05))[0]
    want, pc = O.constraints(p, u, percell=True)                   # oracle on the whole mesh (every rank computes it)
    bz0, nbz = PT.slab_partition(4, world)[rank]
    sl = slice(bz0 * 8, (bz0 + nbz) * 8)
    # this rank's raw share, from the oracle's per-cell values (the GPU's z4c_constraints_raw has this shape)
    H, M2 = pc[0][sl], (pc[1][sl] ** 2 + pc[2][sl] ** 2 + pc[3][sl] ** 2)
    raw = np.array([np.sum(H * H), np.abs(H).max(), 0.0, 0.0, np.sum(u[I.THETA][sl] ** 2), np.abs(u[I.THETA][sl]).max(),
                    0.0, 0.0])
    sums, maxs = torch.from_numpy(raw[0::2].copy()), torch.from_numpy(raw[1::2].copy())
    dist.all_reduce(sums, op=dist.ReduceOp.SUM)
    dist.all_reduce(maxs, op=dist.ReduceOp.MAX)
    red = np.empty(8)
    red[0::2], red[1::2] = sums.numpy(), maxs.numpy()
    got = PT.combine_raw_norms(red, p.ncells)
    ok = (abs(got[0] - want[0]) <= 1e-13 * want[0] and got[1] == want[1] and
          abs(got[4] - want[4]) <= 1e-13 * want[4] and got[5] == want[5])
    with open(os.path.join(tmp, f"ok{rank}"), "w") as f:
        f.write("1" if ok else f"0 {got} {want}")
    dist.destroy_process_group()


def test_constraint_norms_allreduce_world2_gloo(tmp_path, oracle):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_norm_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    for r in range(2):
        assert open(tmp_path / f"ok{r}").read() == "1"
