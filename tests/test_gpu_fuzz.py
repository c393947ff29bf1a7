"""Seeded random shapes and options through dfjk_get_jk / dfjk_get_jk_dm / dfjk_ao2mo against the oracle.

Every case draws a basis size, an aux count, a set structure (empty sets, thin sets, signed occupations)
and a combination of the scheduling options that must not change the result (N_blk, split-K, two-pass J,
gather vs re-tiled half-transform, single-launch path, one-pass thin half-transform).  Bar: 1e-10.
"""
import numpy as np
import pytest

import dfjk_inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10


def rel(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def draw_case(seed):
    rs = np.random.default_rng(seed)
    nao = int(rs.choice([rs.integers(1, 20), rs.integers(20, 100), rs.integers(100, 280)]))
    naux = int(rs.integers(1, 70))
    nset = int(rs.integers(1, 7))
    nocc = [int(min(nao, rs.choice([0, rs.integers(1, 9), rs.integers(1, max(2, nao // 2))]))) for _ in range(nset)]
    while sum(nocc) > nao:
        nocc[int(np.argmax(nocc))] //= 2
    if sum(nocc) == 0:
        nocc[0] = 1
    opts = {}
    if rs.random() < 0.3:
        opts["two_pass_j"] = True
    if rs.random() < 0.3:
        opts["no_retile"] = True
    if rs.random() < 0.4:
        opts["nblk"] = int(rs.integers(1, naux + 1))
    if rs.random() < 0.3:
        opts["ksplit"] = int(rs.integers(1, 6))
    if rs.random() < 0.5:
        opts["no_small_path"] = True
    if rs.random() < 0.3:
        opts["no_symm_thin"] = True
    return nao, naux, nocc, opts


@pytest.mark.parametrize("seed", range(5000, 5040))
def test_random_get_jk(seed):
    import oracle
    import torch
    import paper_2505_03755_b200 as dfjk
    nao, naux, nocc, opts = draw_case(seed)
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(3.0, nao / 6))
    rs = np.random.default_rng(seed + 1)
    for o in inp.occ:
        o *= rs.choice([-1.0, 1.0, 1.0], size=o.shape)
    Jo, Ko = oracle.get_jk_inputs(inp)
    B = torch.from_numpy(inp.B_packed).cuda()
    Cs = [torch.from_numpy(c).cuda() for c in inp.C]
    occs = [torch.from_numpy(o).cuda() for o in inp.occ]
    with dfjk.DFJK(B, nao, **opts) as h:
        J, K = h.get_jk(Cs, occs)
        Jonly, _ = h.get_jk(Cs, occs, with_k=False)
        _, Konly = h.get_jk(Cs, occs, with_j=False)
        torch.cuda.synchronize()
    assert torch.equal(K, Konly), (nao, naux, nocc, opts)
    for s in range(len(nocc)):
        if nocc[s] == 0:
            assert not J[s].any() and not K[s].any() and not Jonly[s].any()
            continue
        ej, ek, ej1 = rel(J[s].cpu().numpy(), Jo[s]), rel(K[s].cpu().numpy(), Ko[s]), rel(Jonly[s].cpu().numpy(), Jo[s])
        assert ej <= TOL and ek <= TOL and ej1 <= TOL, (nao, naux, nocc, opts, s, ej, ek, ej1)
        assert torch.equal(J[s], J[s].T) and torch.equal(K[s], K[s].T)


@pytest.mark.parametrize("seed", range(5100, 5116))
def test_random_ao2mo_and_dm_form(seed):
    import oracle
    import torch
    import paper_2505_03755_b200 as dfjk
    rs = np.random.default_rng(seed)
    nao = int(rs.integers(2, 160))
    naux = int(rs.integers(1, 40))
    nmo = int(rs.integers(1, nao + 1))
    nact = int(rs.integers(1, min(nmo, 10) + 1))
    a0 = int(rs.integers(0, nmo - nact + 1))
    opts = {}
    if rs.random() < 0.5:
        opts["ao2mo_route"] = int(rs.integers(1, 3))
    if rs.random() < 0.3:
        opts["no_symm_thin"] = True
    if rs.random() < 0.3:
        opts["nblk"] = int(rs.integers(1, naux + 1))
    inp = dfjk_inputs.make_random(nao, naux, [1], seed, L=max(3.0, nao / 6))
    M = rs.standard_normal((nao, nmo))
    o_bpa, o_ppaa, o_papa = oracle.ao2mo(inp.B_packed, nao, M, a0, nact)
    D = rs.standard_normal((1, nao, nao))
    D = D + D.transpose(0, 2, 1)
    Jo = oracle.get_jk(inp.B_packed, nao, [np.eye(nao)], [np.ones(nao)])[0] * 0.0    # shape only
    Kd_o = oracle.get_k_dform(inp.B_packed, nao, D[0])
    B = torch.from_numpy(inp.B_packed).cuda()
    with dfjk.DFJK(B, nao, **opts) as h:
        bpa, ppaa, papa = h.ao2mo(torch.from_numpy(M).cuda(), a0, nact)
        Jd, Kd = h.get_jk_dm(torch.from_numpy(D).cuda())
        torch.cuda.synchronize()
    assert rel(bpa.cpu().numpy(), o_bpa) <= TOL, (nao, naux, nmo, a0, nact, opts)
    assert rel(ppaa.cpu().numpy(), o_ppaa) <= TOL and rel(papa.cpu().numpy(), o_papa) <= TOL, (nao, naux, nmo, a0, nact, opts)
    assert rel(Kd[0].cpu().numpy(), Kd_o) <= TOL, (nao, naux, opts)
    assert Jo.shape == tuple(Jd.shape)
