"""Host logic of bench.py (-m "not gpu"): whole-job accounting over ranks (world_size 2, gloo, CPU), and the
bounded reference arm's JSON contract."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r: time 10 + 5r ms, its own frame of 100 (+r) input px and 70 (+2r) output px
    out = bench.reduce_over_ranks(10.0 + 5.0 * rank, 100 + rank, 70 + 2 * rank, dist, None)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, out))


def test_reduce_over_ranks_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(2):  # MAX of the times, SUM of the pixels, identical on every rank
        assert res[r] == (15.0, 201.0, 142.0)


def test_reduce_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(3.5, 10, 7) == (3.5, 10.0, 7.0)


def test_reference_arm_nonzero_rank_is_silent():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_reference_arm_json_contract(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setattr(bench, "SAMPLE_SIDE", {"bilinear": 256, "lanczos3": 128})
    import io
    from contextlib import redirect_stdout
    buf = io.StringIO()
    ns = type("A", (), dict(gpus=1, steps=1, warmup=0, impl="reference", workload="config1"))()
    monkeypatch.setenv("RANK", "0")
    with redirect_stdout(buf):
        assert bench.run_reference(ns) == 0
    line = json.loads(buf.getvalue())
    assert line["impl"] == "reference" and line["unit"] == "Mpix/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": "Mpix/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    # both arms print the same `config` for a workload (the driver compares them)
    import synth
    assert line["config"] == bench.public_config("config1", synth.config0(), 1)
    assert line["config"]["workload"] == bench.WORKLOADS["config1"][0] and line["config"]["W"] == 9576


def test_rooflines_pick_the_binding_resource():
    sys.path.insert(0, ROOT)
    import bench
    px_in, n1, n4 = 9576 * 6388, 44887802, 179550640
    # bilinear configs[1]: HBM binds (1215.5 MB per frame)
    r = bench.rooflines("bilinear", px_in, n1, False, 0.29, 1965.0, 6450.9, "test")
    assert r["bound"] == "hbm" and abs(r["algorithmic_bytes"] - 1215503248) < 1 and 0.6 < r["frac"] < 0.7
    # fused coadd: 14 B per input px + 16 B per output px = 1574.6 MB
    assert abs(bench.algorithmic_work("bilinear", px_in, n1, True)[0] - 1574605664) < 1
    # Lanczos-3 at nside 2^18: the shared-memory gather (36 taps per output) has the longest time at peak
    r4 = bench.rooflines("lanczos3", px_in, n4, False, 2.5, 1965.0, 6450.9, "test")
    assert r4["bound"].startswith("smem") and r4["fractions"]["smem"] > r4["fractions"]["fp32"] > r4["fractions"]["hbm"]
    assert abs(r4["frac"] - r4["time_at_peak_ms"]["smem"] / 2.5) < 1e-12
