"""GPU parity of dfjk_get_jk_dm (Eq. 14-17 as printed, general symmetric density matrices) against the
oracle's D-form evaluation (oracle.get_k_dform: Eq. 16 then Eq. 17, literally) and, for J, the
brute-force-pinned C-form oracle on the eigen-decomposition of D.  Bar 1e-10."""
import numpy as np
import pytest

import dfjk_inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10


def rel(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def sym_indefinite(nao, seed):
    """a symmetric matrix with eigenvalues of both signs (no C sqrt(occ) form exists)"""
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((nao, nao))
    return 0.5 * (A + A.T)


def oracle_j_of_dm(Bp, nao, D):
    import oracle
    w, U = np.linalg.eigh(D)                      # J is linear in D: J[D] = J[D+] - J[D-]
    pos, neg = w > 0, w < 0
    J = np.zeros((nao, nao))
    if pos.any():
        J += oracle.get_jk(Bp, nao, [np.ascontiguousarray(U[:, pos])], [w[pos]], with_k=False)[0][0]
    if neg.any():
        J -= oracle.get_jk(Bp, nao, [np.ascontiguousarray(U[:, neg])], [-w[neg]], with_k=False)[0][0]
    return J


@pytest.mark.parametrize("nao,naux,nset,seed,opts", [
    (12, 5, 1, 301, {}),
    (67, 45, 2, 302, {}),
    (130, 40, 1, 303, {}),                        # one row past a 128 boundary, several N passes impossible here
    (150, 33, 3, 304, dict(nblk=7)),              # several aux blocks, three sets
    (200, 21, 1, 305, dict(ksplit=3)),
    (400, 8, 1, 306, {}),                         # 400 columns: two N passes of the half-transform
])
def test_density_matrix_form(nao, naux, nset, seed, opts):
    import torch
    import oracle
    import paper_2505_03755_b200 as dfjk
    inp = dfjk_inputs.make_random(nao, naux, [1], seed, L=max(4.0, nao / 6))
    Ds = np.stack([sym_indefinite(nao, seed + 10 * s) for s in range(nset)])
    B = torch.from_numpy(inp.B_packed).cuda()
    with dfjk.DFJK(B, nao, **opts) as h:
        J, K = h.get_jk_dm(torch.from_numpy(Ds).cuda())
        torch.cuda.synchronize()
        assert h.last_launch_count > 0
        Jonly, _ = h.get_jk_dm(torch.from_numpy(Ds).cuda(), with_k=False)
        _, Konly = h.get_jk_dm(torch.from_numpy(Ds).cuda(), with_j=False)
        torch.cuda.synchronize()
        assert torch.equal(J, Jonly) and torch.equal(K, Konly)
    J, K = J.cpu().numpy(), K.cpu().numpy()
    for s in range(nset):
        Ko = oracle.get_k_dform(inp.B_packed, nao, Ds[s])
        Jo = oracle_j_of_dm(inp.B_packed, nao, Ds[s])
        assert rel(K[s], Ko) <= TOL, (s, rel(K[s], Ko))
        assert rel(J[s], Jo) <= TOL, (s, rel(J[s], Jo))
        assert np.array_equal(J[s], J[s].T) and np.array_equal(K[s], K[s].T)


def test_dm_form_agrees_with_c_form_on_a_psd_density():
    import torch
    import paper_2505_03755_b200 as dfjk
    inp = dfjk_inputs.make_random(96, 50, [20], 311, L=12.0)
    D = (inp.C[0] * inp.occ[0]) @ inp.C[0].T
    B = torch.from_numpy(inp.B_packed).cuda()
    with dfjk.DFJK(B, 96) as h:
        J1, K1 = h.get_jk([torch.from_numpy(inp.C[0]).cuda()], [torch.from_numpy(inp.occ[0]).cuda()])
        J2, K2 = h.get_jk_dm(torch.from_numpy(D[None]).cuda())
        torch.cuda.synchronize()
    assert rel(J2.cpu().numpy(), J1.cpu().numpy()) < 1e-12 and rel(K2.cpu().numpy(), K1.cpu().numpy()) < 1e-12
