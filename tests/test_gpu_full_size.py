"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default options).

medium: every element against the full oracle.  large / lasscf: the oracle would need ~2 minutes of
16 host cores each, so sampled outputs are computed one by one from the definitions
(oracle.sample) plus properties that hold at any size (bitwise symmetry, Tr(D J) = sum rho^2 >= 0 is
implied by the sampled J; linearity across the lasscf sets is covered at small size).
"""
import numpy as np
import pytest

import dfjk_inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _gpu_jk(inp):
    import torch
    import paper_2505_03755_b200 as dfjk
    B = torch.from_numpy(inp.B_packed).cuda()
    Cs = [torch.from_numpy(c).cuda() for c in inp.C]
    occs = [torch.from_numpy(o).cuda() for o in inp.occ]
    with dfjk.DFJK(B, inp.nao) as h:
        J, K = h.get_jk(Cs, occs)
        torch.cuda.synchronize()
        plan = h.plan()
    out = J.cpu().numpy(), K.cpu().numpy(), plan
    del B, J, K
    torch.cuda.empty_cache()
    return out


def test_medium_config_every_element():
    import oracle
    inp = dfjk_inputs.make_config("medium")
    J, K, plan = _gpu_jk(inp)
    Jo, Ko = oracle.get_jk_inputs(inp)
    for s in range(inp.nset):
        ej = np.abs(J[s] - Jo[s]).max() / np.abs(Jo[s]).max()
        ek = np.abs(K[s] - Ko[s]).max() / np.abs(Ko[s]).max()
        assert ej <= TOL and ek <= TOL, (s, ej, ek, plan)
        assert np.array_equal(J[s], J[s].T) and np.array_equal(K[s], K[s].T)


@pytest.mark.parametrize("name", ["large", "lasscf"])
def test_full_size_sampled(name):
    import oracle
    inp = dfjk_inputs.make_config(name)
    J, K, plan = _gpu_jk(inp)
    nao, nset = inp.nao, inp.nset
    rs = np.random.default_rng(11)
    samples = [(int(rs.integers(nset)), int(rs.integers(nao)), int(rs.integers(nao))) for _ in range(6)]
    samples += [(0, 0, 0), (nset - 1, nao - 1, nao - 1), (0, nao - 1, 0), (nset - 1, 63, 64), (0, 80, 79),
                (nset - 1, 1199, 1120)]
    Jv, Kv = oracle.sample(inp.B_packed, nao, inp.C, inp.occ, samples)
    for t, (s, mu, nu) in enumerate(samples):
        assert abs(J[s, mu, nu] - Jv[t]) <= TOL * np.abs(J[s]).max(), (name, samples[t], plan)
        assert abs(K[s, mu, nu] - Kv[t]) <= TOL * np.abs(K[s]).max(), (name, samples[t], plan)
    for s in range(nset):
        assert np.isfinite(J[s]).all() and np.isfinite(K[s]).all()
        assert np.array_equal(J[s], J[s].T) and np.array_equal(K[s], K[s].T)
        # K is positive semidefinite for occ >= 0: its diagonal is non-negative
        assert (np.diagonal(K[s]) >= 0).all()
