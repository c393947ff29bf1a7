"""Pins for the AO2MO oracle (oracle/ao2mo_oracle.c, Eq. 18-21).

The paper prints no value for this kernel either, so the pins are definitional: the direct 4-index
transformation of the Eq. 12 tensor (brute force, itself checked against numpy.einsum), M = I
(the outputs are slices of the AO tensor), permutational symmetries, the overlap of the two outputs
on all-active indices, an independent BLAS-backed einsum evaluation of Eq. 18-21, and the
contraction with an active-space density against the (independently pinned) JK oracle.  A wrong
index pattern in Eq. 20 vs Eq. 21, a transposed M, or a wrong active offset fails at least one.
"""
import numpy as np
import pytest

import dfjk_inputs
import oracle


def unpack_np(Bp, nao):
    naux = Bp.shape[0]
    sq = np.zeros((naux, nao, nao))
    mu, nu = np.tril_indices(nao)
    sq[:, mu, nu] = Bp
    sq[:, nu, mu] = Bp
    return sq


def relerr(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


def make(nao, naux, nmo, seed, L=0.0):
    rng = np.random.default_rng(seed)
    inp = dfjk_inputs.make_random(nao, naux, [1], seed, L=L)
    M = rng.standard_normal((nao, nmo))
    return inp.B_packed, M


def test_bruteforce_matches_numpy_four_index_transform():
    nao, naux, nmo, a0, nact = 5, 4, 4, 1, 2
    Bp, M = make(nao, naux, nmo, 21)
    sq = unpack_np(Bp, nao)
    g = np.einsum("pab,pcd->abcd", sq, sq)                                  # Eq. 12
    Ma = M[:, a0:a0 + nact]
    ppaa = np.einsum("ai,bj,ck,dl,abcd->ijkl", M, M, Ma, Ma, g, optimize=True)
    papa = np.einsum("ai,bk,cj,dl,abcd->ikjl", M, Ma, M, Ma, g, optimize=True)
    bf_ppaa, bf_papa = oracle.ao2mo_bruteforce(Bp, nao, M, a0, nact)
    assert relerr(bf_ppaa, ppaa) < 1e-13 and relerr(bf_papa, papa) < 1e-13


@pytest.mark.parametrize("nao,naux,nmo,a0,nact,seed", [(6, 5, 5, 2, 2, 31), (7, 3, 7, 0, 3, 32), (8, 9, 4, 1, 3, 33)])
def test_oracle_matches_bruteforce(nao, naux, nmo, a0, nact, seed):
    Bp, M = make(nao, naux, nmo, seed)
    bpa, ppaa, papa = oracle.ao2mo(Bp, nao, M, a0, nact)
    bf_ppaa, bf_papa = oracle.ao2mo_bruteforce(Bp, nao, M, a0, nact)
    assert relerr(ppaa, bf_ppaa) < 1e-13
    assert relerr(papa, bf_papa) < 1e-13
    # the two index patterns differ: Eq. 20 is not Eq. 21 with axes swapped
    assert relerr(ppaa.transpose(0, 2, 1, 3), papa) > 1e-3


def test_identity_coefficients_give_slices_of_the_ao_tensor():
    nao, naux, a0, nact = 9, 6, 3, 4
    Bp, _ = make(nao, naux, nao, 41)
    sq = unpack_np(Bp, nao)
    g = np.einsum("pab,pcd->abcd", sq, sq)
    bpa, ppaa, papa, bmo = oracle.ao2mo(Bp, nao, np.eye(nao), a0, nact, with_bmo=True)
    assert np.array_equal(bmo, sq)                                          # M = I: nothing changes
    assert relerr(ppaa, g[:, :, a0:a0 + nact, a0:a0 + nact]) < 1e-14
    assert relerr(papa, g[:, a0:a0 + nact, :, a0:a0 + nact]) < 1e-14
    assert np.array_equal(bpa, sq[:, :, a0:a0 + nact])


def test_symmetries_overlap_and_bpa():
    nao, naux, nmo, a0, nact = 14, 11, 10, 4, 3
    Bp, M = make(nao, naux, nmo, 51, L=5.0)
    bpa, ppaa, papa, bmo = oracle.ao2mo(Bp, nao, M, a0, nact, with_bmo=True)
    assert relerr(bmo, bmo.transpose(0, 2, 1)) < 1e-14                      # b^P_{p1 p2} symmetric
    assert np.array_equal(bpa, bmo[:, :, a0:a0 + nact])
    assert relerr(ppaa, ppaa.transpose(1, 0, 2, 3)) < 1e-14                 # (p1 p2|a1 a2) = (p2 p1|a1 a2)
    assert relerr(ppaa, ppaa.transpose(0, 1, 3, 2)) < 1e-14                 #              = (p1 p2|a2 a1)
    assert relerr(papa, papa.transpose(2, 3, 0, 1)) < 1e-14                 # (p1 a1|p2 a2) = (p2 a2|p1 a1)
    act = slice(a0, a0 + nact)
    assert relerr(ppaa[act, act], papa[act, :, act, :].transpose(0, 1, 2, 3)) < 1e-14   # (a b|c d) both ways
    # positivity: (p a|p a) = sum_P bpa^2 >= 0
    d = np.einsum("papa->pa", papa)
    assert (d >= 0).all() and relerr(d, (bpa ** 2).sum(0)) < 1e-14


def test_independent_einsum_evaluation():
    nao, naux, nmo, a0, nact = 20, 17, 13, 5, 4
    Bp, M = make(nao, naux, nmo, 61, L=6.0)
    sq = unpack_np(Bp, nao)
    bh = np.einsum("Pef,ep->Pfp", sq, M)                                    # Eq. 18
    bmo = np.einsum("Pfp,fq->Ppq", bh, M)                                   # Eq. 19
    act = slice(a0, a0 + nact)
    ppaa = np.einsum("Ppq,Pab->pqab", bmo, bmo[:, act, act])                # Eq. 20
    papa = np.einsum("Ppa,Pqb->paqb", bmo[:, :, act], bmo[:, :, act])       # Eq. 21
    o_bpa, o_ppaa, o_papa, o_bmo = oracle.ao2mo(Bp, nao, M, a0, nact, with_bmo=True)
    assert relerr(o_bmo, bmo) < 1e-13 and relerr(o_bpa, bmo[:, :, act]) < 1e-13
    assert relerr(o_ppaa, ppaa) < 1e-13 and relerr(o_papa, papa) < 1e-13


def test_contraction_with_active_density_reproduces_the_jk_oracle():
    """sum_{a1 a2} (p1 p2|a1 a2) D[a1][a2] = (M^T J[D_ao] M)[p1][p2] and
    sum_{a1 a2} (p1 a1|p2 a2) D[a1][a2] = (M^T K[D_ao] M)[p1][p2], D_ao = M_act D M_act^T:
    ties Eq. 20-21 to Eq. 14-17, whose oracle is pinned by its own brute force."""
    nao, naux, nmo, a0, nact = 16, 12, 11, 3, 5
    Bp, M = make(nao, naux, nmo, 71, L=4.0)
    rng = np.random.default_rng(72)
    occ = rng.uniform(0, 2, nact)
    U = np.linalg.qr(rng.standard_normal((nact, nact)))[0]
    D = (U * occ) @ U.T                                                     # a non-diagonal active 1-RDM
    Cact = M[:, a0:a0 + nact] @ U                                           # natural orbitals in the AO basis
    J, K = oracle.get_jk(Bp, nao, [Cact], [occ])
    _, ppaa, papa = oracle.ao2mo(Bp, nao, M, a0, nact)
    assert relerr(np.einsum("pqab,ab->pq", ppaa, D), M.T @ J[0] @ M) < 1e-12
    assert relerr(np.einsum("paqb,ab->pq", papa, D), M.T @ K[0] @ M) < 1e-12


def test_edge_shapes():
    Bp, M = make(6, 4, 5, 81)
    bpa, ppaa, papa = oracle.ao2mo(Bp, 6, M, 2, 0)                          # no active orbitals
    assert bpa.shape == (4, 5, 0) and ppaa.size == 0 and papa.size == 0
    bpa, ppaa, papa = oracle.ao2mo(Bp[:0], 6, M, 1, 2)                      # no aux rows
    assert not ppaa.any() and not papa.any()
    with pytest.raises(RuntimeError):
        oracle.ao2mo(Bp, 6, M, 4, 2)                                        # active range past nmo


def test_element_sampler_against_the_full_oracle_and_the_brute_force():
    """dfjk_oracle_ao2mo_sample (single elements of Eq. 20-21 from the definitions, used for parity at
    bench size) against the full oracle at a ragged small size (every element of both outputs), and
    against the direct 4-index transformation of the Eq. 12 tensor at a tiny size.  A wrong index
    order between ppaa[p1][p2][a1][a2] and papa[p1][a1][p2][a2] fails: the case is non-symmetric
    in all four indices (non-orthonormal M, a0 > 0, nact < nmo)."""
    nao, naux, nmo, a0, nact = 19, 11, 9, 2, 3
    Bp, M = make(nao, naux, nmo, 91, L=5.0)
    _, ppaa, papa = oracle.ao2mo(Bp, nao, M, a0, nact)
    samples = [(p1, p2, a1, a2) for p1 in range(nmo) for p2 in range(nmo) for a1 in range(nact) for a2 in range(nact)]
    v20, v21 = oracle.ao2mo_sample(Bp, nao, M, a0, nact, samples)
    assert relerr(v20.reshape(nmo, nmo, nact, nact), ppaa) < 1e-13
    assert relerr(v21.reshape(nmo, nmo, nact, nact).transpose(0, 2, 1, 3), papa) < 1e-13
    assert relerr(ppaa, papa.transpose(0, 2, 1, 3)) > 1e-2          # the two outputs really differ
    nao, naux, nmo, a0, nact = 7, 5, 6, 1, 4
    Bp, M = make(nao, naux, nmo, 92)
    b20, b21 = oracle.ao2mo_bruteforce(Bp, nao, M, a0, nact)
    samples = [(5, 0, 3, 1), (0, 5, 1, 3), (2, 2, 0, 0), (4, 1, 2, 3)]
    v20, v21 = oracle.ao2mo_sample(Bp, nao, M, a0, nact, samples)
    for t, (p1, p2, a1, a2) in enumerate(samples):
        assert abs(v20[t] - b20[p1, p2, a1, a2]) < 1e-12 * np.abs(b20).max()
        assert abs(v21[t] - b21[p1, a1, p2, a2]) < 1e-12 * np.abs(b21).max()
    with pytest.raises(RuntimeError):
        oracle.ao2mo_sample(Bp, nao, M, a0, nact, [(0, 0, nact, 0)])        # active index out of range
