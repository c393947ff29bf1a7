"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default options).

All five configs are compared with the full oracle on EVERY element (R7: per set,
max|dJ|/max|J| and max|dK|/max|K| over all nao^2 entries <= 1e-10); tiny and small live in
test_gpu_parity.py, medium / large / lasscf here.  The oracle needs about two minutes of the GPU
box's 16 host cores for each of the two nao=1200 configs (plus a minute to draw the 23 GB tensor).
AO2MO (Eq. 18-21) at the bench's size is compared on sampled elements that the oracle computes one
by one from the definitions (oracle.ao2mo_sample) and on whole aux rows of bpa.
"""
import numpy as np
import pytest

import dfjk_inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _gpu_jk(inp, B, **opts):
    import torch
    import paper_2505_03755_b200 as dfjk
    Cs = [torch.from_numpy(c).cuda() for c in inp.C]
    occs = [torch.from_numpy(o).cuda() for o in inp.occ]
    with dfjk.DFJK(B, inp.nao, **opts) as h:
        J, K = h.get_jk(Cs, occs)
        torch.cuda.synchronize()
        plan = h.plan()
    out = J.cpu().numpy(), K.cpu().numpy(), plan
    del J, K
    torch.cuda.empty_cache()
    return out


def _assert_every_element(inp, J, K, Jo, Ko, plan):
    for s in range(inp.nset):
        ej = np.abs(J[s] - Jo[s]).max() / np.abs(Jo[s]).max()
        ek = np.abs(K[s] - Ko[s]).max() / np.abs(Ko[s]).max()
        print(f"{inp.name} set {s}: max|dJ|/max|J| = {ej:.2e}, max|dK|/max|K| = {ek:.2e} over all "
              f"{inp.nao}^2 entries, plan {plan}")
        assert ej <= TOL and ek <= TOL, (inp.name, s, ej, ek, plan)
        assert np.isfinite(J[s]).all() and np.isfinite(K[s]).all()
        assert np.array_equal(J[s], J[s].T) and np.array_equal(K[s], K[s].T)    # bitwise symmetric


@pytest.mark.parametrize("name", ["medium", "large", "lasscf"])
def test_config_every_element(name):
    """native fp64 path at the default options, then the opt-in FP64-emulated K path (int8 tensor
    cores) on the same resident tensor against the same oracle result"""
    import oracle
    import torch
    inp = dfjk_inputs.make_config(name)
    B = torch.from_numpy(inp.B_packed).cuda()
    J, K, plan = _gpu_jk(inp, B)
    Jo, Ko = oracle.get_jk_inputs(inp)
    _assert_every_element(inp, J, K, Jo, Ko, plan)
    if name != "medium":
        # the launch configuration the bench times: several aux blocks, split-K, the re-tiled copy
        assert plan["nblk"] < inp.naux and plan["ksplit"] > 1 and plan["retiled"] == 1, plan
    for S in (6, 5):
        Je, Ke, plan_e = _gpu_jk(inp, B, ht_emulation_slices=S, k_emulation_slices=S)
        errs = [np.abs(Ke[s] - Ko[s]).max() / np.abs(Ko[s]).max() for s in range(inp.nset)]
        ej = max(np.abs(Je[s] - Jo[s]).max() / np.abs(Jo[s]).max() for s in range(inp.nset))
        print(f"{inp.name} emulated K (half-transform and SYRK on the int8 tensor cores, {S} slices): "
              f"max|dK|/max|K| = {max(errs):.2e} over all entries of all sets, J {ej:.2e}, plan {plan_e}")
        assert ej <= TOL                                         # J is never emulated
        assert all(np.array_equal(Ke[s], Ke[s].T) for s in range(inp.nset))
        if S == 6:
            assert max(errs) <= TOL, (name, errs)                # the stated slice count for 1e-10
        else:
            assert max(errs) <= 1e-8, (name, errs)
    del B
    torch.cuda.empty_cache()


def test_ao2mo_at_bench_size_sampled():
    """nao = 1200, nmo = 340, nact = 8 (the bench's AO2MO call, active-first route) on the first 400
    aux rows of the `large` tensor: ppaa / papa at sampled (p1, p2, a1, a2) against the oracle's
    element sampler, bpa of two whole aux rows against the full oracle (Eq. 18-19)."""
    import oracle
    import torch
    import paper_2505_03755_b200 as dfjk
    naux = 400
    inp = dfjk_inputs.make_config("large", aux_rows=naux)
    nao, nmo, nact = inp.nao, 340, 8
    a0 = nmo - nact
    M = np.ascontiguousarray(dfjk_inputs.make_orbitals("large", all_columns=True)[:, :nmo])
    B = torch.from_numpy(inp.B_packed).cuda()
    with dfjk.DFJK(B, nao) as h:
        bpa, ppaa, papa = h.ao2mo(torch.from_numpy(M).cuda(), a0, nact)
        torch.cuda.synchronize()
        assert h.last_ao2mo_route == 2
    bpa, ppaa, papa = bpa.cpu().numpy(), ppaa.cpu().numpy(), papa.cpu().numpy()
    rs = np.random.default_rng(17)
    samples = [(int(rs.integers(nmo)), int(rs.integers(nmo)), int(rs.integers(nact)), int(rs.integers(nact)))
               for _ in range(8)]
    samples += [(0, 0, 0, 0), (nmo - 1, nmo - 1, nact - 1, nact - 1), (nmo - 1, 0, 0, nact - 1), (a0 + 3, a0 + 5, 5, 3),
                (63, 64, 1, 2), (128, 127, 7, 0)]
    v20, v21 = oracle.ao2mo_sample(inp.B_packed, nao, M, a0, nact, samples)
    s20, s21 = np.abs(ppaa).max(), np.abs(papa).max()
    for t, (p1, p2, a1, a2) in enumerate(samples):
        assert abs(ppaa[p1, p2, a1, a2] - v20[t]) <= TOL * s20, (samples[t], ppaa[p1, p2, a1, a2], v20[t])
        assert abs(papa[p1, a1, p2, a2] - v21[t]) <= TOL * s21, (samples[t], papa[p1, a1, p2, a2], v21[t])
    rows = [0, naux - 1]
    o_bpa, _, _ = oracle.ao2mo(inp.B_packed[rows], nao, M, a0, nact)
    assert np.abs(bpa[rows] - o_bpa).max() <= TOL * np.abs(o_bpa).max()
    # properties that hold at any size: (p1 p2|a1 a2) is symmetric in p1 <-> p2 and in a1 <-> a2,
    # (p1 a1|p2 a2) under the pair exchange (p1 a1) <-> (p2 a2)
    assert np.abs(ppaa - ppaa.transpose(1, 0, 2, 3)).max() <= 1e-12 * s20
    assert np.abs(ppaa - ppaa.transpose(0, 1, 3, 2)).max() <= 1e-12 * s20
    assert np.abs(papa - papa.transpose(2, 3, 0, 1)).max() <= 1e-12 * s21


def test_basis_beyond_the_bench_sizes_every_element():
    """nao = 2000 (system C of the paper has 1378 AOs): 32 row blocks, 508 padded columns in two N
    tiles of the half-transform, 25 x 25 SYRK tiles, a thin second set; AO2MO's active-first route with the tiled
    half-transform (the one-pass kernel stops at nao = 1280).  Every element against the oracle."""
    import oracle
    import torch
    import paper_2505_03755_b200 as dfjk
    nao, naux = 2000, 40
    inp = dfjk_inputs.make_random(nao, naux, [500, 8], 601, L=120.0)
    inp.occ[1][::2] *= -1.0
    B = torch.from_numpy(inp.B_packed).cuda()
    J, K, plan = _gpu_jk(inp, B)
    Jo, Ko = oracle.get_jk_inputs(inp)
    _assert_every_element(inp, J, K, Jo, Ko, plan)
    M = np.ascontiguousarray(np.linalg.qr(np.random.default_rng(602).standard_normal((nao, 64)))[0])
    with dfjk.DFJK(B, nao, ao2mo_route=2) as h:
        bpa, ppaa, papa = h.ao2mo(torch.from_numpy(M).cuda(), 50, 6)
        torch.cuda.synchronize()
    o_bpa, o_ppaa, o_papa = oracle.ao2mo(inp.B_packed, nao, M, 50, 6)
    for a, b in ((bpa, o_bpa), (ppaa, o_ppaa), (papa, o_papa)):
        assert np.abs(a.cpu().numpy() - b).max() <= TOL * np.abs(b).max()
