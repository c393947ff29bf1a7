"""Aux-sharded mode on real handles, on ONE GPU.

J and K are sums over the aux index P, so handles bound to disjoint contiguous ranges of aux rows
(`sharded.aux_range`, the paper's block-to-GPU "hashing") return partial J, K whose sum in rank
order is the full result.  Here the "ranks" are handles on row-slice VIEWS of one resident tensor
and the all-reduce is a device-side sum in rank order; the collective itself is covered by the
world_size-2 gloo tests (tests/test_multirank_cpu.py).  No N > 1 hardware run exists for this
build (unmeasured).
"""
import numpy as np
import pytest

import dfjk_inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10


def rel(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


@pytest.mark.parametrize("nao,naux,nocc,seed,world", [
    (67, 45, [23, 7], 201, 2),          # npair even: every slice 16-byte aligned
    (67, 45, [23, 7], 201, 3),
    (5, 7, [2], 202, 2),                # npair = 15 odd, lo = 4 even
    (6, 9, [3, 2], 203, 3),             # npair = 21 odd, lo = 3 odd: the slice is only 8-byte aligned
    (150, 61, [37, 10], 204, 4),        # 16 + 15 + 15 + 15 rows
    (40, 3, [9], 205, 4),               # more ranks than some can fill: one rank holds no rows
])
def test_partials_of_row_slices_sum_to_the_full_result(nao, naux, nocc, seed, world):
    import oracle
    import torch
    import paper_2505_03755_b200 as dfjk
    from paper_2505_03755_b200.sharded import aux_range, make_sharded
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(3.0, nao / 6))
    inp.occ[0][0] = -0.7                                   # a signed occupation rides along
    Jo, Ko = oracle.get_jk_inputs(inp)
    B = torch.from_numpy(inp.B_packed).cuda()
    Cs = [torch.from_numpy(c).cuda() for c in inp.C]
    occs = [torch.from_numpy(o).cuda() for o in inp.occ]
    with dfjk.DFJK(B, nao) as h:
        J1, K1 = h.get_jk(Cs, occs)
        torch.cuda.synchronize()
    Jsum, Ksum = torch.zeros_like(J1), torch.zeros_like(K1)
    misaligned = 0
    for rank in range(world):                              # rank order: the order an all-reduce ring would not
        lo, hi = aux_range(naux, rank, world)              # guarantee, hence the 1e-13 against one handle
        rows = B[lo:hi]                                    # a view, not a copy
        misaligned += int(rows.data_ptr() % 16 != 0)
        sh, hr = make_sharded(rows, nao, naux, rank=rank, world=world)
        Jr, Kr = sh.get_jk(Cs, occs)                       # no process group: the local partial
        torch.cuda.synchronize()
        Jsum += Jr
        Ksum += Kr
        hr.close()
    if (nao * (nao + 1) // 2) % 2 == 1 and world == 3 and nao == 6:
        assert misaligned > 0                              # the case the 16-byte check used to reject
    J, K = Jsum.cpu().numpy(), Ksum.cpu().numpy()
    for s in range(inp.nset):
        assert rel(J[s], Jo[s]) <= TOL and rel(K[s], Ko[s]) <= TOL
        assert rel(J[s], J1[s].cpu().numpy()) <= 1e-13 and rel(K[s], K1[s].cpu().numpy()) <= 1e-13


def test_sharded_large_slices_take_the_fast_paths():
    """4 ranks x 250 aux rows of a nao=300 tensor (npair even): bulk-copy J passes, the re-tiled copy
    and several SYRK splits per slice; partials against the oracle on every element"""
    import oracle
    import torch
    import paper_2505_03755_b200 as dfjk
    from paper_2505_03755_b200.sharded import aux_range
    inp = dfjk_inputs.make_config("small")
    Jo, Ko = oracle.get_jk_inputs(inp)
    B = torch.from_numpy(inp.B_packed).cuda()
    Cs = [torch.from_numpy(c).cuda() for c in inp.C]
    occs = [torch.from_numpy(o).cuda() for o in inp.occ]
    Jsum = torch.zeros((1, inp.nao, inp.nao), dtype=torch.float64, device="cuda")
    Ksum = torch.zeros_like(Jsum)
    for rank in range(4):
        lo, hi = aux_range(inp.naux, rank, 4)
        with dfjk.DFJK(B[lo:hi], inp.nao) as h:
            Jr, Kr = h.get_jk(Cs, occs)
            torch.cuda.synchronize()
            assert h.plan()["retiled"] == 1
        Jsum += Jr
        Ksum += Kr
    assert rel(Jsum[0].cpu().numpy(), Jo[0]) <= TOL and rel(Ksum[0].cpu().numpy(), Ko[0]) <= TOL


def test_handles_on_two_devices_in_one_process():
    """the >48 KB shared-memory opt-in is per device: a second handle on another GPU of the same
    process must work (skipped on a one-GPU box), and a call with the wrong current device is refused"""
    import torch
    import paper_2505_03755_b200 as dfjk
    inp = dfjk_inputs.make_random(70, 40, [15, 6], 206, L=10.0)
    outs = []
    ndev = torch.cuda.device_count()
    for d in range(min(ndev, 2)):
        dev = torch.device("cuda", d)
        B = torch.from_numpy(inp.B_packed).to(dev)
        Cs = [torch.from_numpy(c).to(dev) for c in inp.C]
        occs = [torch.from_numpy(o).to(dev) for o in inp.occ]
        with dfjk.DFJK(B, inp.nao) as h:
            J, K = h.get_jk(Cs, occs)
            torch.cuda.synchronize(dev)
            outs.append((J.cpu(), K.cpu()))
    if ndev < 2:
        pytest.skip("one GPU: the second-device leg needs two")
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
