"""Host-side logic of bench.py without a GPU: the multi-rank aggregation (MAX time, SUM units) on a 2-rank gloo
group, the workload table, the CPU reference arm."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sys.path.insert(0, ROOT)
    import bench
    ms, units = bench.aggregate(10.0 + 5.0 * rank, 1000.0 * (rank + 1), dist)
    q.put((rank, ms, units))
    dist.destroy_process_group()


def test_aggregate_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29731, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(2)]
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for _, ms, units in res:
        assert ms == 15.0 and units == 3000.0        # max over ranks, sum over ranks (replicas, weak scaling)


def test_aggregate_single_rank():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(3.0, 7.0, None) == (3.0, 7.0)


def test_workload_table_matches_baseline_configs():
    sys.path.insert(0, ROOT)
    import bench
    p, u, label = bench.workload("linear_wave_64")
    assert p.N == (64, 64, 64) and p.n == 16 and p.nblocks == 64 and "configs[1]" in label
    p, u, _ = bench.workload("noise_16_2x2x2")
    assert p.nblocks == 8 and u.shape == (22, 32, 32, 32)
    ps, us, what = bench.oracle_sample("linear_wave_64")
    assert ps.N == (64, 16, 16)


def test_default_workload_is_the_largest_fixed_config():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.DEFAULT_WORKLOAD == "bbh_256" and "configs[3]" in bench.WORKLOAD_LABELS["bbh_256"]
    ps, us, what = bench.oracle_sample("bbh_256")
    assert ps.N == (32, 32, 32) and abs(ps.dx - 48.0 / 256) < 1e-15 and ps.bc == 1 and ps.shift_eta == 1.0
    assert us[0].min() < 0.05                      # the sample really contains the puncture (chi -> 0)
    ps1, _, _ = bench.oracle_sample("bbh_256", small=True)
    assert ps1.N == (16, 16, 16)
    assert (64, (8, 8, 8)) in bench.SWEEP_POINT and len(bench.SWEEP_FULL) >= 12


def test_gpus_flag_spawns_the_ranks_itself():
    """`python bench.py --gpus 2` must be a complete command (it re-launches itself under torch.distributed.run,
    127.0.0.1 rendezvous). Checked on the CPU-only reference arm: rank 0 prints the one line, rank 1 exits 0 silently."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "1", "--workload", "linear_wave_64"],
                         capture_output=True, text=True, timeout=900, cwd=ROOT, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2


def test_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "zone-cycles/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


def test_workload_params_and_slab_data_agree_with_the_configs():
    """bench.py's per-slab generators (NEXT-2 weak scaling) give the same cells as the whole-mesh generators."""
    from dataclasses import replace
    import numpy as np
    import bench
    from paper_2409_10383_b200 import inputs as I
    from paper_2409_10383_b200 import partition as PT
    for idx, name in ((2, "puncture_128"), (3, "bbh_256")):
        p_cfg = I.config(idx)[0] if idx == 2 else None
        p, _, _ = bench.workload(name, params_only=True)
        if p_cfg is not None:
            assert p == p_cfg
    # a shrunk two-puncture mesh: whole-mesh data cut into z-slabs == data generated slab by slab
    p = replace(bench.workload("bbh_256", params_only=True)[0], n=8, nb=(2, 2, 4), dx=0.75, xmin=(-6.0, -6.0, -12.0))
    whole = bench.workload_data("bbh_256", p)
    for r in range(3):
        ps = PT.slab_params(p, r, 3)
        assert np.array_equal(bench.workload_data("bbh_256", ps), PT.slab_interior(whole, p, r, 3))


def test_two_level_workload_geometry():
    """bench.py --workload two_level_wave_256: the fine pack is the 2:1 refinement of a box of whole coarse blocks
    inside the coarse mesh, both levels share one dt, and the small (oracle-sized) variant has the same shape."""
    sys.path.insert(0, ROOT)
    import bench
    for small in (False, True):
        pc, pf, origin = bench.two_level_workload(small=small)
        assert abs(2.0 * pf.dx - pc.dx) < 1e-15 and abs(pc.dt - pf.dt) < 1e-18
        assert pc.bc == 0 and pf.bc == 1 and pc.ng == pf.ng
        for d in range(3):
            Mc = pf.N[d] // 2
            assert pf.N[d] % 2 == 0
            if not small:                                   # the timed mesh refines whole coarse blocks
                assert origin[d] % pc.n == 0 and Mc % pc.n == 0
            assert 0 <= origin[d] and origin[d] + Mc <= pc.N[d]
            assert abs(pf.xmin[d] - (pc.xmin[d] + origin[d] * pc.dx)) < 1e-14                # same physical corner
    pc, pf, origin = bench.two_level_workload()
    assert pc.nblocks == 512 and pf.nblocks == 512 and pc.n == 32 and pf.n == 32
