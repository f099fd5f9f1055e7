"""Host logic of bench.py on CPU: the roofline numerator and the N > 1 aggregation (max over ranks through
torch.distributed; gloo here, nccl on the GPU box)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_alg_flops_formula():
    st = {"alg_sum_n2": 1000, "alg_sum_n": 100, "alg_incidence": 10}
    # unique orbital pairs n(n+1) + V dV scaling n + 120 per (point, atom)
    assert bench.alg_flops(st) == 1000 + 100 + 100 + 120 * 10


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t = bench.max_over_ranks([0.1 * (rank + 1), 1.0 - 0.25 * rank], torch.device("cpu"), world)
    out[rank] = t
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29613, out), nprocs=world, join=True)
        for r in range(world):
            assert np.allclose(out[r], [0.2, 1.0])
    # whole-job value for replicas: N * points / slowest rank
    assert bench.job_value(1000, 0.2, world) == 2 * 1000 / 0.2


def test_force_alg_flops_formula():
    st = {"alg_sum_n2": 1000, "alg_sum_n": 100, "alg_incidence": 10}
    # Psi over every ordered orbital pair 2 n^2, three gradient components times Psi 6 n, values + gradients 360 per (point, atom)
    assert bench.force_alg_flops(st) == 2 * 1000 + 6 * 100 + 360 * 10


def test_traffic_lookup_is_keyed_by_batch_shape_and_source_digest(tmp_path, monkeypatch):
    """roofline.traffic comes from the committed ncu capture only when BOTH the grid-batch shape of the run and the digest of the
    kernel sources match the capture; otherwise it is None with a reason (never a figure that describes another launch)."""
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    os.makedirs(tmp_path / "profiles")
    monkeypatch.setattr(bench, "csrc_digest", lambda: "abc123")
    (tmp_path / "profiles" / "r3_traffic.csv").write_text(
        "# comment\ncfg,batch,call,dram_bytes_read,dram_bytes_write,csrc_digest\n4,8x8x16,rho_main,100,50,abc123\n4,4x8x16,rho_main,70,30,zzz\n")
    assert bench.ncu_traffic(4, (8, 8, 16), "rho_main")[0] == 150
    v, why = bench.ncu_traffic(4, (8, 8, 8), "rho_main")
    assert v is None and "no capture" in why
    v, why = bench.ncu_traffic(4, (4, 8, 16), "rho_main")
    assert v is None and "stale" in why
    assert bench.ncu_traffic(3, (8, 8, 16), "rho_main")[0] is None


def test_committed_traffic_capture_is_reported_only_for_matching_sources():
    """The committed capture of the headline config: reported when it was taken on the sources in the tree (csrc/ without the force
    kernels), withheld as stale otherwise."""
    rows = [ln.split(",") for ln in open(os.path.join(ROOT, "profiles", "r3_traffic.csv")) if ln[0] not in "#c"]
    assert rows and {r[2].strip() for r in rows} == {"vlocal_main", "rho_main"}
    v, why = bench.ncu_traffic(4, (8, 8, 16), "rho_main")
    if all(r[5].strip() == bench.csrc_digest() for r in rows):
        assert v > 1e11
    else:
        assert v is None and "stale" in why
