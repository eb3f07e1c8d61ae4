"""Host-side multi-process logic (CPU, gloo, world_size 2): the replicas helper that bench.py uses to line up
N independent replicas and to combine their timings (max over ranks of the time, sum of the units), and the
alg_slots / alg_bytes accounting of bench.py."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
from paper_1510_06340_b200.replicas import Replicas
rep = Replicas(backend="gloo")
rank = rep.rank
rep.barrier()
units, secs = 1000.0 * (rank + 1), 0.5 * (rank + 1)          # rank 1 is slower and did more
out = dict(rank=rank, world=rep.world, mx=rep.max(secs), sm=rep.sum(units), thr=rep.throughput(units, secs))
rep.barrier()
rep.close()
print(json.dumps(out))
"""


def test_two_replicas_over_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29533")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        so, se = p.communicate(timeout=120)
        assert p.returncode == 0, se
        outs.append(json.loads(so.strip().splitlines()[-1]))
    for o in outs:
        assert o["world"] == 2
        assert o["mx"] == 1.0                      # max over ranks
        assert o["sm"] == 3000.0                   # sum over ranks
        assert o["thr"] == 3000.0                  # whole-job units / slowest rank's time


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    from paper_1510_06340_b200.replicas import Replicas
    env = {k: os.environ.pop(k, None) for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE")}
    try:
        rep = Replicas()
        assert rep.world == 1 and rep.max(2.5) == 2.5 and rep.sum(7) == 7.0
        assert rep.throughput(10.0, 2.0) == 5.0
    finally:
        for k, v in env.items():
            if v is not None:
                os.environ[k] = v


def test_reference_arm_under_two_ranks_prints_once(tmp_path):
    """bench.py --impl reference under torchrun-style env: rank 0 prints the line, rank 1 exits 0 silently."""
    outs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29534")
        p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                            "--warmup", "1", "--ref-crop", "16"], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=300)
        assert p.returncode == 0, p.stderr
        outs.append(p.stdout.strip())
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0
    assert outs[1] == ""


def test_algorithmic_work_matches_survey_table():
    """~3.7 k slots (RK2, k=2), ~7.2 k slots (RK3, k=3) per cell-update; 200 / 320 B (+32 B CFL)."""
    sys.path.insert(0, ROOT)
    import bench
    s22, L22, m22 = bench.alg_slots("minmod", 2, 2, 3)
    s33, L33, m33 = bench.alg_slots("superbee", 3, 3, 3)
    assert m22 == 3 * 478 and m33 == 3 * 644
    assert 3500 <= s22 <= 3800 and 7000 <= s33 <= 7400
    assert bench.alg_bytes(2) == 232 and bench.alg_bytes(3) == 352
    # the second convention (the sequences the product code issues: reciprocal 3, root 6, flux 24) is below the survey's and counts the same
    # pieces: per MUSTA interface (k+1)(3*24 + 50) + 20k
    n33, _, mm33 = bench.alg_slots("superbee", 3, 3, 3, minimal=True)
    assert mm33 == 3 * (4 * (3 * 24 + 50) + 60) and n33 < s33 and 6000 <= n33 <= 6500
    # single-precision state: the state's bytes halve, the slots do not change
    assert bench.alg_bytes(3, state_bytes=4) == 176
    # tabulated EOS: 201 slots per flux evaluation in both conventions (they differ only in the root and divide of the CFL pass)
    t33 = bench.alg_slots("superbee", 3, 3, 3, table=True)[0]
    assert abs(t33 - bench.alg_slots("superbee", 3, 3, 3, table=True, minimal=True)[0]) < 20 and t33 > 3 * s33
    w = bench.class_work("staged", "superbee", 3, 3, True, True, state_bytes=4)
    assert w["cell_stage"][1] == 20 + 160 and w["combine"][1] == 160 + 60
