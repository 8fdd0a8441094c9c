"""N > 1 is "replicas only": no data-path collective exists.  What N > 1 adds is host
logic in bench.py -- MAX over ranks of the device times, SUM of the counters, whole-job value, rank-0-only
output of the reference arm -- covered here with world_size 2 over gloo on CPU.  The one exchange that does exist
is opt-in (the two-GPU Phi / Psi split of PAPER.md:167): exchange_halves of the binding, run
here by two gloo processes on CPU tensors."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% os.environ["PORT"],
                        rank=int(os.environ["RANK"]), world_size=2)
rank = dist.get_rank()
mx, sm = bench.reduce_over_ranks([100.0 + 50.0 * rank, 7.0 - rank], [1000 + rank], dist, "cpu")
print(json.dumps({"rank": rank, "max": mx, "sum": sm, "value": bench.job_value(2, 8, mx[0])}))
dist.destroy_process_group()
""" % ROOT


def test_reduce_over_ranks_world2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = str(29500 + os.getpid() % 2000)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), PORT=port)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs)
    for out in outs:
        d = json.loads(out.strip().splitlines()[-1])
        assert d["max"] == [150.0, 7.0]          # slowest replica, per quantity
        assert d["sum"] == [2001.0]
        assert abs(d["value"] - 2 * 8 / 0.150) < 1e-9


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks([3.0, 4.0], [5], None, "cpu") == ([3.0, 4.0], [5])
    assert bench.job_value(1, 8, 1000.0) == 8.0


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_timed_steps_stay_inside_the_schedule():
    """bench.py times steps of the config's own 40-step schedule only (BASELINE.json c3: 'steps 9...40'): the
    driver's K = 20, W = 5 is one segment, steps 14..33; a K that does not fit is split into segments that each
    start from a fresh init + ramp-up + warm-up."""
    sys.path.insert(0, ROOT)
    import bench
    assert bench.timed_segments(8, 5, 20) == [list(range(13, 33))]
    segs = bench.timed_segments(8, 5, 40)
    assert [len(s) for s in segs] == [27, 13] and all(s[0] == 13 and s[-1] < 40 for s in segs)
    assert bench.timed_segments(4, 1, 3, sched=8) == [[5, 6, 7]]
    import pytest
    with pytest.raises(ValueError):
        bench.timed_segments(8, 32, 1)


SPLIT_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import paper_2412_14104_b200 as t
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% os.environ["PORT"],
                        rank=int(os.environ["RANK"]), world_size=2)
rank = dist.get_rank()
ok = True
for group in (None, dist.new_group([0, 1])):
    n = 100003
    full_phi = torch.arange(n, dtype=torch.float64) * 0.5 + 1.0      # what rank 0 contracted
    full_psi = -torch.arange(n, dtype=torch.float64) / 3.0 - 2.0     # what rank 1 contracted
    phi = full_phi.clone() if rank == 0 else torch.full((n,), float("nan"), dtype=torch.float64)
    psi = full_psi.clone() if rank == 1 else torch.full((n,), float("nan"), dtype=torch.float64)
    t.exchange_halves(phi, psi, rank, group)
    ok = ok and torch.equal(phi, full_phi) and torch.equal(psi, full_psi)
print(json.dumps({"rank": rank, "ok": bool(ok)}))
dist.destroy_process_group()
""" % ROOT


def test_phi_psi_exchange_world2_gloo(tmp_path):
    """After exchange_halves both processes hold both halves, bit for bit: rank 0's Phi, rank 1's Psi."""
    script = tmp_path / "split_worker.py"
    script.write_text(SPLIT_WORKER)
    port = str(31500 + os.getpid() % 2000)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), PORT=port)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs)
    for out in outs:
        assert json.loads(out.strip().splitlines()[-1])["ok"] is True
