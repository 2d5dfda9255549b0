"""NEXT row f4 -- one solve over several GPUs by z-slabs (the paper's node had two GPUs).

-m "not gpu": the partition arithmetic, the slicing of the inputs (every unknown and every face owned exactly as the
library expects) and the ranks' exchange protocol (SlabComm) under gloo with world_size 2 on CPU tensors.
-m gpu: all slabs in one process on one GPU (the library kernels + the same exchange code with device copies) against
the oracle's solve of the undivided problem."""
import json
import os
import subprocess
import sys
import textwrap

import numpy as np
import pytest

from workloads import make_config, random_operator

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_and_input_slices():
    from paper_1704_02745_b200.slab import partition, slab_inputs

    assert partition(10, 3) == [(0, 4), (4, 3), (7, 3)]
    assert partition(5, 5) == [(z, 1) for z in range(5)]
    assert partition(385, 8)[0] == (0, 49) and sum(n for _, n in partition(385, 8)) == 385
    with pytest.raises(ValueError):
        partition(3, 4)
    inp = random_operator(7, 5, 9, seed=3)
    parts = partition(inp.nz, 3)
    rebuilt = np.empty_like(inp.rhs)
    for s, (z0, nzl) in enumerate(parts):
        ex, ey, ez, kb, rh, bc = slab_inputs(inp.nx, inp.ny, inp.nz, inp.eps_x, inp.eps_y, inp.eps_z, inp.kbar2,
                                             inp.rhs, inp.bc, z0, nzl)
        assert ex.shape == (nzl, inp.ny, inp.nx + 1) and ey.shape == (nzl, inp.ny + 1, inp.nx)
        assert ez.shape == (nzl + 1, inp.ny, inp.nx) and kb.shape == rh.shape == (nzl, inp.ny, inp.nx)
        assert bc.size == 2 * (nzl * inp.ny + nzl * inp.nx + inp.ny * inp.nx)
        # interface faces are shared: the top face plane of slab s is the bottom face plane of slab s + 1
        assert np.array_equal(ez[0], inp.eps_z[z0]) and np.array_equal(ez[-1], inp.eps_z[z0 + nzl])
        zm, zp = bc[-2 * inp.ny * inp.nx:-inp.ny * inp.nx], bc[-inp.ny * inp.nx:]
        gzm, gzp = inp.bc[-2 * inp.ny * inp.nx:-inp.ny * inp.nx], inp.bc[-inp.ny * inp.nx:]
        assert np.array_equal(zm, gzm if s == 0 else np.zeros_like(zm))
        assert np.array_equal(zp, gzp if s == len(parts) - 1 else np.zeros_like(zp))
        assert np.array_equal(bc[:nzl * inp.ny].reshape(nzl, inp.ny), inp.bc[:inp.nz * inp.ny].reshape(inp.nz, inp.ny)[z0:z0 + nzl])
        rebuilt[z0:z0 + nzl] = rh
    assert np.array_equal(rebuilt, inp.rhs)


WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import torch, torch.distributed as dist
    from paper_1704_02745_b200.slab import SlabComm
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    owner = [0, 0, 1]                       # three slabs: two on process 0 (local copies), one on process 1 (gloo)
    comm = SlabComm(owner, rank, dist)
    ids = comm.local()
    half = 4
    send = {s: torch.arange(2 * half, dtype=torch.float64) + 100.0 * s for s in ids}
    recv = {s: torch.full((2 * half,), -1.0, dtype=torch.float64) for s in ids}
    comm.exchange(send, recv, half)
    scal = {s: torch.tensor([1.0 + s, 10.0 * (s + 1)], dtype=torch.float64) for s in ids}
    comm.all_reduce(scal)
    print(json.dumps({"rank": rank, "recv": {str(s): recv[s].tolist() for s in ids},
                      "scal": {str(s): scal[s].tolist() for s in ids}}), flush=True)
    dist.destroy_process_group()
""") % ROOT


def test_exchange_protocol_two_processes_gloo(tmp_path):
    """Slab s's lower half must land in the upper half of slab s-1's receive buffer and its upper half in the lower
    half of slab s+1's, across the process boundary (gloo) exactly as inside a process (copies); outer halves stay
    untouched; the all-reduce leaves the sum over ALL slabs in every slab's scalars."""
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29641", WORLD_SIZE="2", OMP_NUM_THREADS="1")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    recv, scal = {}, {}
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e[-2000:]
        d = json.loads(o.strip().splitlines()[-1])
        recv.update({int(k): v for k, v in d["recv"].items()})
        scal.update({int(k): v for k, v in d["scal"].items()})
    lo = lambda s: [100.0 * s + i for i in range(4)]           # what slab s sends down
    hi = lambda s: [100.0 * s + 4 + i for i in range(4)]       # what slab s sends up
    assert recv[0] == [-1.0] * 4 + lo(1)                        # nothing below slab 0; slab 1's lower half above it
    assert recv[1] == hi(0) + lo(2)
    assert recv[2] == hi(1) + [-1.0] * 4
    for s in range(3):
        assert scal[s] == [1.0 + 2.0 + 3.0, 10.0 + 20.0 + 30.0]


@pytest.mark.gpu
@pytest.mark.parametrize("nslabs", [2, 3])
@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_slab_solve_matches_oracle(cuda_device, nslabs, prec, tol):
    """All slabs in one process on one GPU: library kernels per slab (ghost planes, interface faces not folded into b,
    local sums) + SlabComm with device copies, against the oracle's solve of the UNDIVIDED problem -- north-star bars,
    iteration count within 5 % (the dot products are summed slab by slab, so the last bits of alpha / beta differ)."""
    import torch

    from oracle import pbref
    from paper_1704_02745_b200 import build as pb_build
    from paper_1704_02745_b200.slab import SlabComm, SlabRank, partition, slab_inputs, solve_slabs

    pb_build.build()
    inp = make_config(2) if nslabs == 2 else random_operator(45, 23, 31, seed=8)
    ref = pbref.from_inputs(inp)
    o = ref.solve(tol, 5000)
    o7 = ref.solve(tol, 7)
    ref.close()
    stream = torch.cuda.Stream()
    parts = partition(inp.nz, nslabs)
    with torch.cuda.stream(stream):
        ranks = {}
        for s, (z0, nzl) in enumerate(parts):
            ranks[s] = SlabRank(s, nslabs, inp.nx, inp.ny, nzl, inp.h,
                                *slab_inputs(inp.nx, inp.ny, inp.nz, inp.eps_x, inp.eps_y, inp.eps_z, inp.kbar2,
                                             inp.rhs, inp.bc, z0, nzl), stream=stream.cuda_stream)
        comm = SlabComm([0] * nslabs, 0, None)
        res = solve_slabs(ranks, comm, tol, 5000, prec, check_every=8)
        res2 = solve_slabs(ranks, comm, tol, 5000, prec, check_every=32)
        short = solve_slabs(ranks, comm, tol, 7, prec, check_every=3)
        for r in ranks.values():
            r.close()
    phi = np.concatenate([res[s]["phi"] for s in range(nslabs)], axis=0)
    scale = np.max(np.abs(o["phi"]))
    assert all(res[s]["status"] == 0 for s in range(nslabs))
    assert len({res[s]["iters"] for s in range(nslabs)}) == 1                  # every rank took the same decision
    assert abs(res[0]["iters"] - o["iters"]) <= max(1, round(0.05 * o["iters"])), (res[0]["iters"], o["iters"])
    assert res[0]["relres"] < tol
    assert np.max(np.abs(phi - o["phi"])) <= (1e-8 if prec == "f64" else 1e-4) * scale
    assert np.array_equal(phi, np.concatenate([res2[s]["phi"] for s in range(nslabs)], axis=0))   # repeatable
    assert all(short[s]["status"] == 6 and short[s]["iters"] == 7 for s in range(nslabs))
    phi7 = np.concatenate([short[s]["phi"] for s in range(nslabs)], axis=0)
    assert np.max(np.abs(phi7 - o7["phi"])) <= (1e-8 if prec == "f64" else 1e-4) * scale
