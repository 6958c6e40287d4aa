"""Host-side logic of bench.py: byte accounting, and the N>1 aggregation (max time over ranks,
sum of units) under a 2-rank gloo group on CPU.  The path itself does not shard ("replicas only")."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench
import synth


def test_compulsory_bytes_match_survey_table():
    # C2 169,728 / C3 1,189,888 / C4 152,612 / C5 1,343,488 bytes per site
    assert bench.compulsory_bytes_per_site(48, "c64", 1) == 169_728
    assert bench.compulsory_bytes_per_site(128, "c64", 1) == 1_189_888
    assert bench.compulsory_bytes_per_site(64, "i16", 1) == 152_612
    assert bench.compulsory_bytes_per_site(128, "c64", 16) == 1_343_488


def test_oracle_sample_is_bounded():
    for name in synth.CONFIGS:
        cfg = synth.config(name)
        d = bench.oracle_sample_dims(cfg)
        assert all(a <= b for a, b in zip(d, cfg["dims"]))
        assert synth.lattice_volume(d) * 9 * cfg["Nc"] ** 2 * cfg["nrhs"] <= 1.6e8


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, units = bench.reduce_max_sum(10.0 + 5.0 * rank, 100.0 * (rank + 1))
    bench.barrier()
    q.put((rank, ms, units))
    dist.destroy_process_group()


def test_two_rank_aggregation_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29611 + os.getpid() % 200
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for _, ms, units in res:
        assert ms == 15.0 and units == 300.0


def test_single_process_aggregation_is_identity():
    assert bench.reduce_max_sum(3.0, 7.0) == (3.0, 7.0)


def test_paper_per_gpu_volume_configs_follow_from_table_1():
    """synth.CONFIGS P2 / P3 are the paper's own per-GPU coarse volumes: derived here from the numbers the
    paper prints (tests/golden/per_gpu_coarse_volumes.txt), not typed in twice."""
    g = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "per_gpu_coarse_volumes.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split("=")
            g[k.strip()] = [int(x) for x in v.split()]
    local = [a // b for a, b in zip(g["global_lattice"], g["gpu_grid"])]
    assert local == g["local_volume"]
    lvl2 = [a // b for a, b in zip(local, g["aggregate_level2"])]
    lvl3 = [a // b for a, b in zip(lvl2, g["aggregate_level3"])]
    assert tuple(lvl2) == synth.config("P2")["dims"] and synth.config("P2")["Nc"] == g["Nc_level2"][0]
    assert tuple(lvl3) == synth.config("P3")["dims"] and synth.config("P3")["Nc"] == g["Nc_level3"][0]
    assert synth.lattice_volume(lvl2) == 1152 and synth.lattice_volume(lvl3) == 32
