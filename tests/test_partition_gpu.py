"""GPU tests of NEXT-2 (one mesh over several packs; ghost exchange at every stage, PAPER.md:65,
75-76): the partitioned data path -- ghost images written into the z-neighbour's pack by the stage kernels -- must
reproduce the unpartitioned pack BIT FOR BIT, because every cell runs the same arithmetic on the same neighbour values.
Run on one GPU: all slabs in one process on one stream (SlabSet), and two processes on the same device that open each
other's buffers through CUDA IPC (DistributedSlab on the gloo backend). The 1 -> 8 GPU curve itself needs a node."""
import os
import socket
from dataclasses import replace

import numpy as np
import pytest

from paper_2409_10383_b200 import inputs as I
from tests.parity import padded_reference

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Z():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2409_10383_b200 import build, z4c
    build.build()
    return z4c


CASES = {
    # params, number of slabs
    "periodic_2": (lambda: I.params_noise(16, (2, 1, 4), dx=0.05), 2),
    "periodic_3_uneven": (lambda: I.params_noise(8, (1, 2, 5), dx=0.05), 3),
    "outflow_4": (lambda: replace(I.params_noise(10, (2, 2, 4), dx=0.05), bc=1, shift_eta=1.0), 4),
    "o6_periodic_2": (lambda: replace(I.params_noise(16, (1, 1, 2), dx=0.05), ng=4), 2),
}


@pytest.mark.parametrize("mode", [2, 1])
@pytest.mark.parametrize("name", list(CASES))
def test_slabs_reproduce_the_single_pack_bitwise(Z, oracle, name, mode):
    from paper_2409_10383_b200 import partition as PT
    mk, R = CASES[name]
    p = mk()
    u = I.smooth_random_data(p, 21, 0.1)
    one = Z.Z4c(p)
    one.set_fused(mode)
    one.set_initial_data(u)
    many = PT.SlabSet(p, R)
    many.set_fused(mode)
    many.set_initial_data(u)
    many.sync()
    # ghosts after set-up: every slab's padded state equals the global padding rule (O2) cut at the slab
    ref0 = padded_reference(one.get_interior(), p)
    nbxy = p.nb[0] * p.nb[1]
    for r, s in enumerate(many.slabs):
        bz0, nbz = many.parts[r]
        assert np.array_equal(s.state.cpu().numpy(), ref0[:, bz0 * nbxy:(bz0 + nbz) * nbxy])
    one.step(5)
    many.step(5)
    one.sync()
    many.sync()
    got, want = many.get_interior(), one.get_interior()
    assert np.array_equal(got, want)
    assert np.abs(want - I.minkowski(p)).max() > 1e-3                  # the data really evolved
    ref5 = padded_reference(want, p)
    for r, s in enumerate(many.slabs):                                  # ghosts too, after the last stage
        bz0, nbz = many.parts[r]
        assert np.array_equal(s.state.cpu().numpy(), ref5[:, bz0 * nbxy:(bz0 + nbz) * nbxy])
        assert abs(s.time() - one.time()) < 1e-15
    c1, cm = one.constraints(), many.constraints()
    assert np.all(np.abs(cm - c1) <= 1e-12 * np.abs(c1)) and np.array_equal(cm[1::2], c1[1::2])
    with pytest.raises(Z.Z4cError):
        many.slabs[0].step(1)                                           # a slab does not step on its own
    one.close()
    many.close()


def test_config3_in_four_slabs_at_full_size_bitwise(Z):
    """BASELINE configs[3] (two punctures, 512 blocks of 32^3, outflow) as `bench.py --gpus 4` would cut it -- four
    z-slabs of 2 block layers, mode 2, one stage kernel per slab and stage writing ghost images into the neighbouring
    slabs' buffers -- against the single pack after 2 steps: padded states (interior and every ghost) bit for bit,
    compared on the device."""
    import torch
    import bench
    from paper_2409_10383_b200 import partition as PT
    p, u, _ = bench.workload("bbh_256")
    one = Z.Z4c(p)
    one.set_initial_data(u)
    many = PT.SlabSet(p, 4)
    many.set_initial_data(u)
    del u
    assert one.effective_mode()[1] == 2 and all(s.effective_mode()[1] == 2 for s in many.slabs)
    nbxy = p.nb[0] * p.nb[1]
    for nsteps in (0, 2):
        one.step(nsteps)
        many.step(nsteps)
        one.sync()
        many.sync()
        for r, s in enumerate(many.slabs):
            bz0, nbz = many.parts[r]
            assert torch.equal(s.state, one.state[:, bz0 * nbxy:(bz0 + nbz) * nbxy]), (nsteps, r)
    assert float((one.state[I.CHI] - 1.0).abs().max()) > 0.5           # punctures: chi -> 0 near them
    c1, cm = one.constraints(), many.constraints()
    assert np.array_equal(cm[1::2], c1[1::2]) and np.all(np.abs(cm - c1) <= 1e-12 * np.abs(c1))
    one.close()
    many.close()


def test_enable_peer_on_the_own_device_and_on_a_missing_one(Z):
    import torch
    p = I.params_noise(16, (1, 1, 1), dx=0.05)
    sim = Z.Z4c(p)
    sim.set_initial_data(I.noise_data(p, 3))
    sim.enable_peer(torch.cuda.current_device())        # the own device needs nothing
    sim.enable_peer(torch.cuda.current_device())        # twice is not an error either
    with pytest.raises(Z.Z4cError):
        sim.enable_peer(torch.cuda.device_count() + 7)
    for other in range(torch.cuda.device_count()):      # on a multi-GPU node: every reachable peer, twice
        if other != torch.cuda.current_device() and torch.cuda.can_device_access_peer(torch.cuda.current_device(), other):
            sim.enable_peer(other)
            sim.enable_peer(other)
    sim.step(1)                                          # the context still works (no sticky error left behind)
    sim.sync()
    sim.close()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _ipc_worker(rank, world, port, tmp):
    import torch
    import torch.distributed as dist
    from paper_2409_10383_b200 import partition as PT
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = I.params_noise(16, (1, 2, 4), dx=0.05)
    u = I.smooth_random_data(p, 33, 0.1)
    slab = PT.DistributedSlab(p, "cuda:0")                              # both ranks on the one GPU of this box
    slab.set_initial_data(PT.slab_interior(u, p, rank, world))
    slab.step(3)
    slab.sim.sync()
    np.save(os.path.join(tmp, f"u{rank}.npy"), slab.sim.get_interior())
    np.save(os.path.join(tmp, f"c{rank}.npy"), slab.constraints())
    slab.close()
    dist.destroy_process_group()


def test_two_processes_exchange_ghosts_through_cuda_ipc(Z, tmp_path):
    """The multi-process plumbing on one device: IPC handles exchanged with all_gather_object, the neighbour's two
    state buffers opened in this process, ghost images stored into them by the stage kernel, a barrier per stage."""
    import torch.multiprocessing as mp
    p = I.params_noise(16, (1, 2, 4), dx=0.05)
    u = I.smooth_random_data(p, 33, 0.1)
    one = Z.Z4c(p)
    one.set_initial_data(u)
    one.step(3)
    one.sync()
    want, cwant = one.get_interior(), one.constraints()
    one.close()
    mp.spawn(_ipc_worker, args=(2, _free_port(), str(tmp_path)), nprocs=2, join=True)
    got = np.concatenate([np.load(tmp_path / f"u{r}.npy") for r in range(2)], axis=1)
    assert np.array_equal(got, want)
    for r in range(2):
        c = np.load(tmp_path / f"c{r}.npy")
        assert np.all(np.abs(c - cwant) <= 1e-12 * np.abs(cwant))
