"""world_size-2 `gloo` tests (CPU) of the N>1 paths of bench.py.

Default ("replicas only"): with --gpus N every rank runs an independent
replica, and the only cross-rank steps are the barrier around the timed region and the max over
ranks of the device time.  These tests run exactly that logic (bench.Ranks) with the gloo backend,
and the rank discipline of `--impl reference` (rank 0 alone runs and prints; the others exit 0
without work).  The opt-in aux-sharded mode (`--shard-aux`, paper_2505_03755_b200/sharded.py) adds
one sum all-reduce of the partial J, K: its host logic and the collective run here with a local
path written in numpy (the handles themselves are covered on the GPU by tests/test_gpu_sharded.py).
"""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, time
sys.path.insert(0, sys.argv[1])
import bench
r = bench.Ranks("gloo", None)
assert r.world == 2 and r.dist is not None
r.barrier()
# every rank contributes its own "device time"; all must see the slowest one
mine = 10.0 + 5.0 * r.rank
got = r.max_over_ranks(mine)
assert got == 15.0, got
# a rank that arrives late at the barrier holds the others
t0 = time.perf_counter()
if r.rank == 1:
    time.sleep(0.5)
r.barrier()
waited = time.perf_counter() - t0
assert waited >= 0.45, waited
r.close()
print("rank %d ok" % r.rank)
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(argv, world=2, extra_env=None):
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
        env.update(extra_env or {})
        procs.append(subprocess.Popen(argv, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True,
                                      cwd=ROOT))
    outs = [p.communicate(timeout=300) for p in procs]
    return [(p.returncode, o, e) for p, (o, e) in zip(procs, outs)]


def test_barrier_and_max_over_ranks_gloo_world2():
    res = _spawn([sys.executable, "-c", WORKER, ROOT])
    for rank, (rc, out, err) in enumerate(res):
        assert rc == 0, (rank, err[-2000:])
        assert f"rank {rank} ok" in out


def test_reference_arm_runs_on_rank0_only():
    res = _spawn([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "tiny",
                  "--gpus", "2", "--steps", "1", "--warmup", "1"])
    (rc0, out0, err0), (rc1, out1, err1) = res
    assert rc0 == 0 and rc1 == 0, (err0[-2000:], err1[-2000:])
    assert out1.strip() == ""                     # the other ranks exit 0 without work
    lines = [ln for ln in out0.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "ms" and d["higher_is_better"] is False
    assert d["cpu_baseline"]["kind"].startswith("oracle") and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


SHARD_WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
import dfjk_inputs, oracle
from paper_2505_03755_b200.sharded import AuxShardedJK, aux_range
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
inp = dfjk_inputs.make_random(23, 17, [6, 3], 77, L=5.0)          # 17 aux rows over 2 ranks: 9 + 8
lo, hi = aux_range(inp.naux, rank, world)
assert (lo, hi) == ((0, 9) if rank == 0 else (9, 17))
def unpack(Bp, nao):
    sq = np.zeros((Bp.shape[0], nao, nao))
    mu, nu = np.tril_indices(nao)
    sq[:, mu, nu] = Bp
    sq[:, nu, mu] = Bp
    return sq
def local(Cs, occs):                         # stands in for DFJK.get_jk on B[lo:hi]: numpy on this rank's rows only
    sq = unpack(inp.B_packed[lo:hi], inp.nao)
    J, K = [], []
    for C, occ in zip(Cs, occs):
        D = (C * occ) @ C.T
        J.append(np.einsum("p,pmn->mn", np.einsum("pmn,mn->p", sq, D), sq))
        K.append(np.einsum("pml,ls,pns->mn", sq, D, sq))
    return torch.from_numpy(np.stack(J)), torch.from_numpy(np.stack(K))
J, K = AuxShardedJK(local).get_jk(inp.C, inp.occ)
Jo, Ko = oracle.get_jk_inputs(inp)
assert np.abs(J.numpy() - Jo).max() <= 1e-13 * np.abs(Jo).max()
assert np.abs(K.numpy() - Ko).max() <= 1e-13 * np.abs(Ko).max()
Jn, Kn = AuxShardedJK(lambda: (None, local(inp.C, inp.occ)[1])).get_jk()
assert Jn is None and np.abs(Kn.numpy() - Ko).max() <= 1e-13 * np.abs(Ko).max()
dist.destroy_process_group()
print("rank %d ok" % rank)
"""


def test_aux_range_partitions_the_rows():
    from paper_2505_03755_b200.sharded import aux_range
    for naux, world in [(4000, 8), (17, 2), (5, 8), (0, 3), (4001, 4)]:
        r = [aux_range(naux, k, world) for k in range(world)]
        assert r[0][0] == 0 and r[-1][1] == naux
        assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
        sizes = [b - a for a, b in r]
        assert max(sizes) - min(sizes) <= 1


def test_aux_sharded_partials_sum_to_the_full_result_gloo_world2():
    """each rank's partial J, K over its aux slice, one sum all-reduce (gloo here, NCCL on GPUs)"""
    res = _spawn([sys.executable, "-c", SHARD_WORKER, ROOT])
    for rank, (rc, out, err) in enumerate(res):
        assert rc == 0, (rank, err[-3000:])
        assert f"rank {rank} ok" in out
