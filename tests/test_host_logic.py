"""Host-side logic that needs no GPU: batch sharding, the multi-rank path under gloo (world_size 2),
the parity rule itself, and bench.py's reference arm."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_range_partitions_exactly():
    from paper_2501_00675_b200.sharding import shard_range
    for batch in (0, 1, 7, 512, 16384, 16385):
        for world in (1, 2, 3, 8):
            spans = [shard_range(batch, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == batch
            for (a0, a1), (b0, b1) in zip(spans, spans[1:]):
                assert a1 == b0
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


_WORKER = r'''
import os, sys
sys.path.insert(0, os.environ["COS_ROOT"])
import numpy as np, torch, torch.distributed as dist
from paper_2501_00675_b200 import sharding
from harness import workloads as wl
import oracle
dist.init_process_group("gloo")
rank, _, world = sharding.env_rank_world()
w = wl.baseline_config(2, batch=101)
lo, hi = sharding.shard_range(w.batch, rank, world)
G, _ = oracle.build_G(w.xy[lo:hi], w.tau[lo:hi], w.table, None, w.beta, 0.0)
_, c = oracle.eval_all_connected(G, None, U=w.U, threads=1)
# the job's only collectives: MAX of the time, SUM of the unit count (sharding.py)
t = sharding.max_over_ranks(1.0 + rank, dist)
units = sharding.sum_over_ranks(float(hi - lo), dist)
parts = [None] * world
dist.all_gather_object(parts, (lo, hi, c))
if rank == 0:
    full = np.concatenate([p[2] for p in sorted(parts)])
    Gf, _ = oracle.build_G(w.xy, w.tau, w.table, None, w.beta, 0.0)
    _, ref = oracle.eval_all_connected(Gf, None, U=w.U, threads=1)
    assert np.array_equal(full, ref), "sharded evaluation differs from the unsharded one"
    assert t == float(world) and units == float(w.batch)
    print("GLOO_OK")
dist.destroy_process_group()
'''


def test_two_rank_gloo_sharding(tmp_path, oracle_mod):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    env = dict(os.environ, COS_ROOT=ROOT, OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", "29533", str(script)]
    res = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    assert "GLOO_OK" in res.stdout


def test_parity_rule_accepts_fp64_reorderings_and_rejects_errors(oracle_mod):
    """A second FP64 evaluation of the same exact sums (vertices relabelled) must pass the rule, and
    a result that is wrong in the 8th digit must fail it."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity_util import CLUSTERED_EXCEPTION_FRACTION, check_parity
    from harness import workloads as wl
    w = wl.baseline_config(4, batch=512)                       # clustered times: the hardest config
    G, _ = oracle_mod.build_G(w.xy, w.tau, w.table, None, w.beta, 0.0)
    p = np.random.default_rng(0).permutation(w.n)
    Gp = np.ascontiguousarray(G[:, p][:, :, p])
    for which, pick in (("all", 0), ("connected", 1)):
        other = oracle_mod.eval_all_connected(Gp, None, U=w.U)[pick]
        st = check_parity(oracle_mod, other, G, None, w.U, None, which, max_fraction=CLUSTERED_EXCEPTION_FRACTION,
                          label="oracle vs relabelled oracle, cfg4")
        assert st["exceptions"] <= 5
        wrong = other * (1.0 + 3e-8)
        with pytest.raises(AssertionError):
            check_parity(oracle_mod, wrong, G, None, w.U, None, which, max_fraction=CLUSTERED_EXCEPTION_FRACTION,
                         label="(wrong in the 8th digit)")


def test_bench_reference_arm_prints_contract_line(oracle_mod):
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                          "--warmup", "1", "--workload", "cfg2"], capture_output=True, text=True, timeout=600)
    assert res.returncode == 0, res.stderr[-2000:]
    line = json.loads(res.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "configurations/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["higher_is_better"] is True
