"""The N > 1 host logic of bench.py on CPU: two gloo ranks shard the workload by seed (independent
catalogues, no data-path collective), the step time is the max over ranks and the job total the sum.
The per-rank "device time" here is faked (there is no GPU in this test); what is checked is the
sharding rule and the reductions bench.py applies to the numbers it prints."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    import catalogues as cat
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cats = bench.workload("cfg1", seed_shift=bench.rank_seed_shift(rank))
    pts = cats[0]["points"]
    fake_ms = 10.0 + 5.0 * rank                   # rank 1 is the slow one
    fake_units = float(pts.shape[0] + rank)
    t = bench.max_over_ranks(fake_ms)
    u = bench.sum_over_ranks(fake_units)
    # strong-scaling mode: partial histograms of the hub shards are summed with one all-reduce
    part = np.arange(12, dtype=np.int64) * (rank + 1)
    full = bench.allreduce_hist(part)
    assert np.array_equal(full, np.arange(12, dtype=np.int64) * 3), full
    wfull = bench.allreduce_hist(np.full(5, 0.25 * (rank + 1)))
    assert np.allclose(wfull, 0.75)
    # per-rank enumeration times of a strong-scaling step and their imbalance (max / mean - 1)
    times = bench.gather_over_ranks(fake_ms)
    assert times == [10.0, 15.0] and abs(bench.imbalance(times) - 0.2) < 1e-12
    dist.barrier()
    np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([t, u, pts[0, 0], float(len(cats))]))
    dist.destroy_process_group()


def test_two_rank_sharding_and_reductions(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    r0 = np.load(tmp_path / "r0.npy")
    r1 = np.load(tmp_path / "r1.npy")
    assert r0[0] == r1[0] == 15.0                 # max over ranks, identical on every rank
    assert r0[1] == r1[1] == 2000 + 2001          # whole-job units = sum over ranks
    assert r0[2] != r1[2]                         # different seeds -> different catalogues per rank
    assert r0[3] == r1[3] == 1.0


def test_single_process_reductions_are_identity():
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.sum_over_ranks(7.0) == 7.0
    assert bench.rank_seed_shift(0) == 0 and bench.rank_seed_shift(3) != bench.rank_seed_shift(2)
    assert bench.gather_over_ranks(2.0) == [2.0] and bench.imbalance([2.0]) == 0.0


def test_roofline_arithmetic_reproduces_by_hand():
    """S:8(d): frac = max(5 E / BW_HBM, (4 sum len N+(j) + hits) / BW_L2) / t -- the figure of the bench line must follow
    from the units it prints."""
    import bench
    w = dict(name="x", weighted=False, edges=1.0e8, spoke=1.0e10, tail=8.0e9, hits=6.0e9)
    peaks = dict(l2_read_gbs=12000.0, smem_atom_gops=800.0, red_f64_gops=180.0, red_u64_gops=185.0)
    r = bench.roofline_3pcf("cfg2", w, 20.0, 6500.0, "test", peaks)
    t_l2 = (4 * 1.0e10 + 6.0e9) / 12000e9
    assert r["bound"] == "l2" and abs(r["frac"] - t_l2 * 1e3 / 20.0) < 1e-12
    assert abs(r["achieved"] / r["peak"] - r["frac"]) < 1e-12
    r4 = bench.roofline_4pcf("x", dict(name="y", hits=1.5e9), 10.0, 1, peaks)
    assert r4["bound"] == "l2-atomics" and abs(r4["frac"] - (1.5e9 / 10e-3 / 1e9) / 185.0) < 1e-12


def test_traffic_comes_from_the_committed_capture():
    """roofline.traffic = DRAM bytes of the launch from profiles/dram_traffic.json, whose sources are committed csv files."""
    import json
    import bench
    table = json.load(open(os.path.join(ROOT, "profiles", "dram_traffic.json")))
    for key in ("cfg5:cfg5", "cfg2:cfg2D", "cfg2:cfg2R", "cfg3:cfg3"):
        b, src = bench.dram_traffic(key)
        assert b == table[key]["bytes"] > 0 and src.startswith("profiles/dram_traffic.json")
        assert os.path.exists(os.path.join(ROOT, "profiles", table[key]["source"].split(" ")[0]))
    assert bench.dram_traffic("nothing:here") == (None, None)
    w = dict(name="cfg5", weighted=False, edges=8.4e9, spoke=1.8e13, tail=1.4e13, hits=7.1e12)
    peaks = dict(l2_read_gbs=13500.0, smem_atom_gops=2000.0, red_f64_gops=190.0, red_u64_gops=185.0)
    assert bench.roofline_3pcf("cfg5", w, 9560.0, 6465.0, "test", peaks)["traffic"] == table["cfg5:cfg5"]["bytes"]


def test_reference_arm_line_schema():
    """bench.py --impl reference (the oracle on the host cores) prints one JSON line with the contract's keys."""
    import json
    import subprocess
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, check=True, cwd=ROOT)
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in line, key
    assert line["impl"] == "reference" and line["value"] > 0 and line["vs_baseline"] is None
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["config"]["workload"] == "cfg1"
