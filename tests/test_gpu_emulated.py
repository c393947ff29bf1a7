"""Opt-in FP64-emulated K path on the int8 tensor cores against
the same oracle: the achieved error is printed and asserted against the stated bound
   |dK[mu][nu]| <= (S + 2) 2^(-7S) sum_pg n_pg 2^(e(pg,mu) + e(pg,nu))
(include/dfjk.h, csrc/emu.cu), which the test evaluates with numpy from an independent half-transform,
and against north_star's 1e-10 at 6 slices.  J does not take part in the emulation.
"""
import numpy as np
import pytest

import dfjk_inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10


def rel(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def unpack_np(Bp, nao):
    sq = np.zeros((Bp.shape[0], nao, nao))
    mu, nu = np.tril_indices(nao)
    sq[:, mu, nu] = Bp
    sq[:, nu, mu] = Bp
    return sq


def stated_bound(inp, s, S, pgroup, nblk):
    """(S+2) 2^(-7S) sum over scale groups of (terms) 2^(e_mu + e_nu), e = exponent of the group's row
    maximum of |X| + 1, X = B_P C sqrt|occ| (numpy, independent of both the oracle and the CUDA path)"""
    sq = unpack_np(inp.B_packed, inp.nao)
    X = np.einsum("pml,li->pmi", sq, inp.C[s] * np.sqrt(np.abs(inp.occ[s])))
    bound = np.zeros((inp.nao, inp.nao))
    for b0 in range(0, inp.naux, nblk):
        for p0 in range(b0, min(inp.naux, b0 + nblk), pgroup):
            p1 = min(inp.naux, b0 + nblk, p0 + pgroup)
            vmax = np.abs(X[p0:p1]).max(axis=(0, 2))
            e2 = np.where(vmax > 0, 2.0 ** (np.floor(np.log2(np.maximum(vmax, 1e-300))) + 1), 0.0)
            bound += (p1 - p0) * X.shape[2] * np.outer(e2, e2)
    return (S + 2) * 2.0 ** (-7 * S) * bound


@pytest.mark.parametrize("nao,naux,nocc,seed,opts", [
    (48, 160, [12], 401, {}),                                        # one tile
    (67, 45, [23, 7], 402, {}),                                      # two sets sharing a 32-column chunk
    (150, 61, [37, 10], 403, dict(nblk=20, k_emulation_group=8)),    # several aux blocks, ragged last scale group
    (200, 40, [9, 8, 8, 1, 40, 3], 404, {}),                         # six sets, three row tiles
    (330, 35, [40, 9], 405, dict(ksplit=3)),                         # 3 x 5 tiles, forced split cap
    (257, 33, [64], 406, dict(k_emulation_group=1)),                 # one scale per aux row
])
def test_emulated_k_against_the_oracle_and_the_stated_bound(nao, naux, nocc, seed, opts):
    import oracle
    import torch
    import paper_2505_03755_b200 as dfjk
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(4.0, nao / 6))
    Jo, Ko = oracle.get_jk_inputs(inp)
    B = torch.from_numpy(inp.B_packed).cuda()
    Cs = [torch.from_numpy(c).cuda() for c in inp.C]
    occs = [torch.from_numpy(o).cuda() for o in inp.occ]
    with dfjk.DFJK(B, nao, no_small_path=True) as h:               # the same J kernels as the emulated handles
        Jn, Kn = h.get_jk(Cs, occs)
        torch.cuda.synchronize()
    errs = {}
    for S in (3, 4, 5, 6):
        with dfjk.DFJK(B, nao, k_emulation_slices=S, **opts) as h:
            J, K = h.get_jk(Cs, occs)
            torch.cuda.synchronize()
            plan = h.plan()
        assert torch.equal(J, Jn)                                    # J is not emulated
        K = K.cpu().numpy()
        pgroup = opts.get("k_emulation_group", 16)
        for s in range(inp.nset):
            if nocc[s] == 0:
                continue
            assert np.array_equal(K[s], K[s].T)
            d = np.abs(K[s] - Ko[s])
            bound = stated_bound(inp, s, S, pgroup, plan["nblk"])
            assert (d <= bound + 1e-13 * np.abs(Ko[s]).max()).all(), (S, s, d.max(), bound.max())
            errs[(S, s)] = d.max() / np.abs(Ko[s]).max()
    print(f"emulated K nao={nao} naux={naux} nocc={nocc}: " +
          ", ".join(f"S={S} set {s}: {e:.1e}" for (S, s), e in sorted(errs.items())))
    assert all(e <= TOL for (S, s), e in errs.items() if S == 6)
    assert all(errs[(3, s)] > errs[(6, s)] for s in range(inp.nset) if (3, s) in errs)   # more slices, smaller error


def test_emulated_k_with_signed_occupations():
    import oracle
    import torch
    import paper_2505_03755_b200 as dfjk
    inp = dfjk_inputs.make_random(150, 40, [37, 10, 5], 407, L=20.0)
    rs = np.random.default_rng(408)
    for o in inp.occ[:2]:
        o *= rs.choice([-1.0, 1.0], size=o.shape)                    # the third set stays non-negative
    Jo, Ko = oracle.get_jk_inputs(inp)
    B = torch.from_numpy(inp.B_packed).cuda()
    Cs = [torch.from_numpy(c).cuda() for c in inp.C]
    occs = [torch.from_numpy(o).cuda() for o in inp.occ]
    with dfjk.DFJK(B, inp.nao, k_emulation_slices=6) as h:
        J, K = h.get_jk(Cs, occs)
        _, Konly = h.get_jk(Cs, occs, with_j=False)
        torch.cuda.synchronize()
        assert torch.equal(K, Konly)
    for s in range(3):
        assert rel(J[s].cpu().numpy(), Jo[s]) <= TOL and rel(K[s].cpu().numpy(), Ko[s]) <= TOL


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_emulated_configs_every_element(name):
    """BASELINE.json's two small configs (medium / large / lasscf: test_gpu_full_size.py): SYRK alone and
    half-transform + SYRK on the int8 tensor cores against the oracle, every element"""
    import oracle
    import torch
    import paper_2505_03755_b200 as dfjk
    inp = dfjk_inputs.make_config(name)
    Jo, Ko = oracle.get_jk_inputs(inp)
    B = torch.from_numpy(inp.B_packed).cuda()
    Cs = [torch.from_numpy(c).cuda() for c in inp.C]
    occs = [torch.from_numpy(o).cuda() for o in inp.occ]
    for ht, S in ((0, 5), (0, 6), (5, 5), (6, 6)):
        with dfjk.DFJK(B, inp.nao, k_emulation_slices=S, ht_emulation_slices=ht) as h:
            J, K = h.get_jk(Cs, occs)
            torch.cuda.synchronize()
        e = rel(K[0].cpu().numpy(), Ko[0])
        print(f"emulated K, {name} config, half-transform slices {ht}, SYRK slices {S}: max|dK|/max|K| = {e:.2e}")
        assert rel(J[0].cpu().numpy(), Jo[0]) <= TOL
        if S == 6:
            assert e <= TOL


def test_emulation_option_range():
    import torch
    import paper_2505_03755_b200 as dfjk
    B = torch.zeros((2, 10), dtype=torch.float64, device="cuda")
    for bad in (1, 2, 7):
        with pytest.raises(dfjk.DFJKError):
            dfjk.DFJK(B, 4, k_emulation_slices=bad)


@pytest.mark.parametrize("nao,naux,nocc,seed,opts", [
    (48, 160, [12], 411, {}),
    (67, 45, [23, 7], 412, {}),                                      # ragged: 3 k-blocks of lam, the last with 3 columns
    (150, 61, [37, 10], 413, dict(nblk=20)),
    (330, 35, [40, 9, 60], 414, {}),                                 # 128 padded columns: two 80-column tiles
    (260, 12, [130, 129], 415, {}),                                  # 264 padded columns: four N tiles
])
def test_emulated_half_transform(nao, naux, nocc, seed, opts):
    """Eq. 16 on the int8 tensor cores (ht_emulation_slices), alone and together with the emulated
    SYRK; J (two-pass in this mode) is untouched by the emulation."""
    import oracle
    import torch
    import paper_2505_03755_b200 as dfjk
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(4.0, nao / 6))
    inp.occ[0][0] = -0.3                                             # a signed occupation rides along
    Jo, Ko = oracle.get_jk_inputs(inp)
    B = torch.from_numpy(inp.B_packed).cuda()
    Cs = [torch.from_numpy(c).cuda() for c in inp.C]
    occs = [torch.from_numpy(o).cuda() for o in inp.occ]
    out = []
    for ht, ks in ((6, 0), (6, 6), (5, 5), (4, 0)):
        with dfjk.DFJK(B, nao, ht_emulation_slices=ht, k_emulation_slices=ks, **opts) as h:
            J, K = h.get_jk(Cs, occs)
            _, Konly = h.get_jk(Cs, occs, with_j=False)
            torch.cuda.synchronize()
            assert h.plan()["retiled"] == 0 and torch.equal(K, Konly)
        J, K = J.cpu().numpy(), K.cpu().numpy()
        ej = max(rel(J[s], Jo[s]) for s in range(inp.nset))
        ek = max(rel(K[s], Ko[s]) for s in range(inp.nset))
        out.append(f"ht={ht} syrk={ks}: {ek:.1e}")
        assert ej <= TOL
        assert all(np.array_equal(K[s], K[s].T) for s in range(inp.nset))
        if ht == 6:
            assert ek <= TOL, (ht, ks, ek)
        if ht == 4:
            assert ek <= 1e-5
    print(f"emulated half-transform nao={nao} naux={naux} nocc={nocc}: " + ", ".join(out))
