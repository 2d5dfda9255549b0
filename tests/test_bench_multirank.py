"""-m "not gpu": host logic of bench.py's N>1 path (replicas, no data-path collective) under gloo, world_size 2.

Covers: per-rank input selection (rank r takes member r of the perturbed-charge batch on the same operator),
the whole-job aggregation (sum of units over ranks / max of time over ranks), and the reference arm's
"rank 0 alone runs" rule."""
import os
import subprocess
import sys
import textwrap

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import numpy as np
    import torch.distributed as dist
    import bench
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    inp, rhs, bc = bench.build_inputs(2, rank, world, "cpu")
    units, ms = bench.aggregate(100 + rank, 10.0 * (rank + 1), world, None)
    args = bench.parse_args(["--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0", "--gpus", "2"])
    line = bench.run_reference(args, rank, world)
    print(json.dumps({"rank": rank, "units": units, "ms": ms, "rhs_sum": float(rhs.sum()), "bc0": float(bc[0]),
                      "eps_sum": float(inp.eps_x.sum()), "ref_line": line is not None}), flush=True)
    dist.destroy_process_group()
""") % ROOT


def test_two_rank_replicas_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29631", WORLD_SIZE="2", OMP_NUM_THREADS="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e[-2000:]
        outs.append(__import__("json").loads(o.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    # whole-job aggregate: units summed, time = max over ranks, identical on both ranks
    for d in outs:
        assert d["units"] == 201.0 and d["ms"] == 20.0
    # same operator on every rank, a different right-hand side per rank (batch members 0 and 1)
    assert outs[0]["eps_sum"] == outs[1]["eps_sum"]
    assert outs[0]["rhs_sum"] != outs[1]["rhs_sum"] or outs[0]["bc0"] != outs[1]["bc0"]
    # the reference arm prints on rank 0 only
    assert outs[0]["ref_line"] is True and outs[1]["ref_line"] is False


def test_single_rank_aggregate_is_identity():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.aggregate(7, 3.5, 1) == (7.0, 3.5)
    assert bench.workload_name(5, "f32", 1e-5) == "config5_385^3_f32_tol1e-05"


def test_gpus_flag_launches_its_own_ranks():
    """`python bench.py --gpus 2` started WITHOUT a launcher must start two local ranks itself (torch.distributed.run on
    127.0.0.1) and report n_gpus 2; on the reference arm rank 0 alone works and prints, rank 1 exits 0."""
    import json
    import subprocess

    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    env["OMP_NUM_THREADS"] = "2"
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "1",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [json.loads(l) for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # one JSON line, from rank 0
    assert lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2 and lines[0]["value"] > 0
