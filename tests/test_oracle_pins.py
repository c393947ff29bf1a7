"""Pins for the CPU oracle (oracle/dfjk_oracle.c) against what the paper and the mathematics fix.

The paper prints no worked example, matrix element or energy for the JK call, so the
pins are definitional: the brute-force 4-index contraction (Eq. 12 + Eq. 5), closed
forms, invariants, an independent BLAS-backed numpy.einsum evaluation, and the values SURVEY.md
8(c) recorded from a throw-away numpy evaluation of the definitions (tests/golden/tiny_survey.txt).
A dropped term, wrong sign/index or transposed operand in the oracle fails at least one of them.
"""
import os

import numpy as np
import pytest

import dfjk_inputs
import oracle

HERE = os.path.dirname(os.path.abspath(__file__))


def unpack_np(Bp, nao):
    """independent unpack via numpy.tril_indices (the packing convention of DESIGN.md R1)"""
    naux = Bp.shape[0]
    sq = np.zeros((naux, nao, nao))
    mu, nu = np.tril_indices(nao)
    sq[:, mu, nu] = Bp
    sq[:, nu, mu] = Bp
    return sq


def einsum_jk(Bp, nao, C, occ):
    """third opinion: Eq. 14-17 through numpy.einsum / BLAS"""
    sq = unpack_np(Bp, nao)
    D = (C * occ) @ C.T
    rho = np.einsum("pmn,mn->p", sq, D)
    J = np.einsum("p,pmn->mn", rho, sq)
    V = np.einsum("pml,ls->pms", sq, D, optimize=True)       # Eq. 16
    K = np.einsum("pms,pns->mn", V, sq, optimize=True)       # Eq. 17
    return D, rho, J, K


def relerr(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


# ---------------------------------------------------------------- packing convention
def test_unpack_roundtrip_and_convention():
    nao = 7
    Bp = np.arange(nao * (nao + 1) // 2, dtype=np.float64) + 1.0
    sq = oracle.unpack_slice(Bp, nao)
    assert np.array_equal(sq, sq.T)
    mu, nu = np.tril_indices(nao)
    assert np.array_equal(sq[mu, nu], Bp)                    # pack(unpack(x)) == x
    # idx(mu,nu) = mu(mu+1)/2 + nu: element (3,1) is packed entry 7, (6,6) the last one
    assert sq[3, 1] == Bp[3 * 4 // 2 + 1] == 8.0
    assert sq[1, 3] == 8.0 and sq[6, 6] == Bp[-1]


def test_density_definition():
    rng = np.random.default_rng(5)
    C, occ = rng.standard_normal((9, 4)), rng.uniform(0, 2, 4)
    assert np.allclose(oracle.density(C, occ), (C * occ) @ C.T, rtol=0, atol=1e-14)


# ---------------------------------------------------------------- brute force (Eq. 12 + Eq. 5)
@pytest.mark.parametrize("nao,naux,nocc,seed", [(5, 3, 2, 11), (12, 7, 5, 12), (9, 1, 9, 13)])
def test_jk_vs_bruteforce_4index(nao, naux, nocc, seed):
    inp = dfjk_inputs.make_random(nao, naux, [nocc], seed)    # non-orthonormal C, occ in [0,2]
    J, K = oracle.get_jk_inputs(inp)
    D = oracle.density(inp.C[0], inp.occ[0])
    Jb, Kb = oracle.bruteforce(inp.B_packed, nao, D)
    assert relerr(J[0], Jb) < 1e-13
    assert relerr(K[0], Kb) < 1e-13
    # and the brute force itself against a numpy 4-index tensor built independently
    sq = unpack_np(inp.B_packed, nao)
    g = np.einsum("pab,pcd->abcd", sq, sq)                    # g^{a c}_{b d} = b_ab b_cd
    assert relerr(Jb, np.einsum("abcd,cd->ab", g, D)) < 1e-13
    assert relerr(Kb, np.einsum("adcb,cd->ab", g, D)) < 1e-13


def test_bruteforce_distinguishes_j_from_k():
    inp = dfjk_inputs.make_random(8, 5, [3], 21)
    D = oracle.density(inp.C[0], inp.occ[0])
    Jb, Kb = oracle.bruteforce(inp.B_packed, 8, D)
    assert relerr(Jb, Kb) > 1e-2                               # a swapped index pattern would be seen


# ---------------------------------------------------------------- closed forms
def packed_from_square(sq):
    nao = sq.shape[-1]
    mu, nu = np.tril_indices(nao)
    return np.ascontiguousarray(sq[..., mu, nu])


def test_closed_form_identity_slice():
    """naux=1, B_0 = I: rho = Tr D, J = Tr(D) I, K = D exactly."""
    nao = 11
    inp = dfjk_inputs.make_random(nao, 1, [4], 31)
    Bp = packed_from_square(np.eye(nao)[None])
    assert np.array_equal(np.nonzero(Bp[0])[0], np.array([m * (m + 3) // 2 for m in range(nao)]))
    J, K, rho = oracle.get_jk(Bp, nao, inp.C, inp.occ, with_rho=True)
    D = (inp.C[0] * inp.occ[0]) @ inp.C[0].T
    assert abs(rho[0, 0] - np.trace(D)) < 1e-13
    assert np.allclose(J[0], np.trace(D) * np.eye(nao), rtol=0, atol=1e-13)
    assert np.allclose(K[0], D, rtol=0, atol=1e-13)


def test_closed_form_rank_one_slices_j_equals_k():
    """B_P = u_P u_P^T makes (mu nu|lam sig) fully symmetric, so J = K."""
    nao, naux = 10, 6
    rng = np.random.default_rng(32)
    u = rng.standard_normal((naux, nao))
    Bp = packed_from_square(np.einsum("pm,pn->pmn", u, u))
    inp = dfjk_inputs.make_random(nao, naux, [4], 33)
    J, K = oracle.get_jk(Bp, nao, inp.C, inp.occ)
    assert relerr(J[0], K[0]) < 1e-13
    D = (inp.C[0] * inp.occ[0]) @ inp.C[0].T
    w = np.einsum("pm,mn,pn->p", u, D, u)                      # u_P^T D u_P
    assert relerr(J[0], np.einsum("p,pm,pn->mn", w, u, u)) < 1e-13


def test_closed_form_diagonal_slices():
    """B_P = diag(d_P): J = diag(sum_P (d_P . diag D) d_P), K[m][n] = D[m][n] sum_P d_P[m] d_P[n]."""
    nao, naux = 9, 5
    rng = np.random.default_rng(34)
    d = rng.standard_normal((naux, nao))
    sq = np.zeros((naux, nao, nao))
    sq[:, np.arange(nao), np.arange(nao)] = d
    inp = dfjk_inputs.make_random(nao, naux, [3], 35)
    J, K = oracle.get_jk(packed_from_square(sq), nao, inp.C, inp.occ)
    D = (inp.C[0] * inp.occ[0]) @ inp.C[0].T
    assert np.allclose(J[0], np.diag((d @ np.diag(D)) @ d), rtol=0, atol=1e-13)
    assert np.allclose(K[0], D * (d.T @ d), rtol=0, atol=1e-13)


def test_closed_form_identity_orbitals():
    """C = I (nocc = nao), n = 1: D = I, rho_P = Tr B_P, K = sum_P B_P^2."""
    nao, naux = 8, 4
    inp = dfjk_inputs.make_random(nao, naux, [nao], 36)
    J, K, rho = oracle.get_jk(inp.B_packed, nao, [np.eye(nao)], [np.ones(nao)], with_rho=True)
    sq = unpack_np(inp.B_packed, nao)
    assert np.allclose(rho[0], np.trace(sq, axis1=1, axis2=2), rtol=0, atol=1e-13)
    assert relerr(K[0], np.einsum("pml,pln->mn", sq, sq)) < 1e-13
    assert relerr(J[0], np.einsum("p,pmn->mn", rho[0], sq)) < 1e-13


# ---------------------------------------------------------------- invariants
def test_invariants_symmetry_traces_and_forms():
    nao, naux = 20, 13
    inp = dfjk_inputs.make_random(nao, naux, [6, 3], 41)
    J, K, rho = oracle.get_jk_inputs(inp, with_rho=True)
    sq = unpack_np(inp.B_packed, nao)
    for s in range(2):
        C, occ = inp.C[s], inp.occ[s]
        D = (C * occ) @ C.T
        assert np.abs(J[s] - J[s].T).max() <= 1e-14 * np.abs(J[s]).max()
        assert np.abs(K[s] - K[s].T).max() <= 1e-14 * np.abs(K[s]).max()
        # Tr(D J) = sum_P rho_P^2 >= 0
        assert np.isclose(np.sum(D * J[s]), np.sum(rho[s] ** 2), rtol=1e-13)
        # Tr(D K) = sum_P || C'^T B_P C' ||_F^2 with C' = C sqrt(occ)  (R8)
        Cp = C * np.sqrt(occ)
        M = np.einsum("mi,pmn,nj->pij", Cp, sq, Cp)
        assert np.isclose(np.sum(D * K[s]), np.sum(M ** 2), rtol=1e-13)
        assert np.sum(D * K[s]) >= 0
        # K from C (Eq. 16-17 with gamma = C occ C^T) == K from D (Eq. 16-17 as printed)
        assert relerr(K[s], oracle.get_k_dform(inp.B_packed, nao, D)) < 1e-13


def test_north_star_trace_identity_needs_unit_occupations():
    """north_star's Tr(DK) = sum_P ||C^T B_P C||_F^2 holds as written only for n_i = 1 (R8)."""
    nao, naux, nocc = 14, 6, 5
    inp = dfjk_inputs.make_random(nao, naux, [nocc], 42, orthonormal=True)
    C = inp.C[0]
    sq = unpack_np(inp.B_packed, nao)
    M = np.einsum("mi,pmn,nj->pij", C, sq, C)
    _, K1 = oracle.get_jk(inp.B_packed, nao, [C], [np.ones(nocc)], with_j=False)
    assert np.isclose(np.sum((C @ C.T) * K1[0]), np.sum(M ** 2), rtol=1e-13)
    _, K2 = oracle.get_jk(inp.B_packed, nao, [C], [np.full(nocc, 2.0)], with_j=False)
    assert np.isclose(np.sum((2 * C @ C.T) * K2[0]), 4 * np.sum(M ** 2), rtol=1e-13)


def test_linearity_in_density():
    """JK[a D1 + b D2] = a JK[D1] + b JK[D2]: stack the two orbital sets into one set."""
    nao, naux = 16, 9
    inp = dfjk_inputs.make_random(nao, naux, [4, 5], 43)
    a, b = 0.7, 1.9
    J, K = oracle.get_jk_inputs(inp)
    Cst = np.concatenate(inp.C, axis=1)
    ost = np.concatenate([a * inp.occ[0], b * inp.occ[1]])
    Js, Ks = oracle.get_jk(inp.B_packed, nao, [Cst], [ost])
    assert relerr(Js[0], a * J[0] + b * J[1]) < 1e-13
    assert relerr(Ks[0], a * K[0] + b * K[1]) < 1e-13


def test_batched_sets_equal_one_at_a_time_and_empty_set():
    nao, naux = 15, 8
    inp = dfjk_inputs.make_random(nao, naux, [5, 0, 2], 44)
    J, K = oracle.get_jk_inputs(inp)
    assert not J[1].any() and not K[1].any()                  # nocc = 0: zero density (R12)
    for s in (0, 2):
        J1, K1 = oracle.get_jk(inp.B_packed, nao, [inp.C[s]], [inp.occ[s]])
        assert np.array_equal(J1[0], J[s]) and np.array_equal(K1[0], K[s])
    Jo, _ = oracle.get_jk_inputs(inp, with_k=False)
    _, Ko = oracle.get_jk_inputs(inp, with_j=False)
    assert np.array_equal(Jo, J) and np.array_equal(Ko, K)


def test_thread_count_does_not_change_bits():
    """OpenMP splits output rows only, so every output element is summed in the same order whatever
    the thread count: the oracle run with 1 thread and with 4 threads (separate processes, the
    runtime reads OMP_NUM_THREADS at start-up) gives bit-identical J, K and rho."""
    import hashlib
    import subprocess
    import sys
    code = ("import sys, hashlib; sys.path.insert(0, %r); import dfjk_inputs, oracle; "
            "inp = dfjk_inputs.make_random(67, 45, [23, 7], 45, L=9.0); "
            "J, K, rho = oracle.get_jk_inputs(inp, with_rho=True); "
            "print(oracle.num_threads(), hashlib.sha256(J.tobytes() + K.tobytes() + rho.tobytes()).hexdigest())"
            % os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    got = {}
    for nt in (1, 4):
        env = dict(os.environ, OMP_NUM_THREADS=str(nt), OMP_DYNAMIC="false")
        out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=300)
        assert out.returncode == 0, out.stderr[-2000:]
        threads, digest = out.stdout.split()
        assert int(threads) == nt                              # the runs really differ in thread count
        got[nt] = digest
    assert got[1] == got[4]


# ---------------------------------------------------------------- library third opinion
@pytest.mark.parametrize("name", ["tiny"])
def test_config_vs_einsum(name):
    inp = dfjk_inputs.make_config(name)
    J, K, rho = oracle.get_jk_inputs(inp, with_rho=True)
    for s in range(inp.nset):
        D, rho_e, Je, Ke = einsum_jk(inp.B_packed, inp.nao, inp.C[s], inp.occ[s])
        assert relerr(rho[s], rho_e) < 1e-13
        assert relerr(J[s], Je) < 1e-13
        assert relerr(K[s], Ke) < 1e-13


def test_midsize_multi_set_vs_einsum():
    """ragged sizes (nao, nocc, naux multiples of nothing), two sets, fractional occupations"""
    inp = dfjk_inputs.make_random(67, 45, [23, 7], 45, L=9.0)
    J, K = oracle.get_jk_inputs(inp)
    for s in range(2):
        _, _, Je, Ke = einsum_jk(inp.B_packed, inp.nao, inp.C[s], inp.occ[s])
        assert relerr(J[s], Je) < 1e-13 and relerr(K[s], Ke) < 1e-13


def test_fp32_cannot_meet_the_bar(tiny_inputs):
    """precision floor: an fp32 evaluation of K misses 1e-10 by orders of magnitude (R-prec)"""
    inp = tiny_inputs
    _, K = oracle.get_jk_inputs(inp, with_j=False)
    sq = unpack_np(inp.B_packed, inp.nao).astype(np.float32)
    Cp = (inp.C[0] * np.sqrt(inp.occ[0])).astype(np.float32)
    X = np.einsum("pml,li->pmi", sq, Cp)
    K32 = np.einsum("pmi,pni->mn", X, X)
    assert relerr(K32.astype(np.float64), K[0]) > 1e-8


# ---------------------------------------------------------------- recorded values
def read_golden(path):
    out = {}
    with open(path) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                out[k.strip()] = [float(t) for t in v.split(",")]
    return out


def test_tiny_config_matches_survey_recorded_values(tiny_inputs):
    g = read_golden(os.path.join(HERE, "golden", "tiny_survey.txt"))
    inp = tiny_inputs
    B = inp.B_packed
    assert np.isclose(B.sum(), g["sum_B"][0], rtol=1e-12)
    assert np.isclose((B ** 2).sum(), g["sum_B2"][0], rtol=1e-12)
    assert np.allclose(B[0, :3], g["B0_first3"], rtol=1e-12)
    J, K, rho = oracle.get_jk_inputs(inp, with_rho=True)
    D = (inp.C[0] * inp.occ[0]) @ inp.C[0].T
    J, K = J[0], K[0]
    assert np.allclose(rho[0, :3], g["rho_first3"], rtol=1e-11)
    got = dict(J_0_0=J[0, 0], J_5_3=J[5, 3], J_47_0=J[47, 0], K_0_0=K[0, 0], K_5_3=K[5, 3],
               K_47_0=K[47, 0], trJ=np.trace(J), trK=np.trace(K), trDJ=np.sum(D * J),
               trDK=np.sum(D * K), maxabsJ=np.abs(J).max(), maxabsK=np.abs(K).max())
    for k, v in got.items():
        assert np.isclose(v, g[k][0], rtol=1e-11, atol=1e-14), (k, v, g[k][0])


# ---------------------------------------------------------------- element sampler
def test_sampler_matches_full_oracle():
    inp = dfjk_inputs.make_random(33, 21, [9, 4], 46, L=6.0)
    J, K = oracle.get_jk_inputs(inp)
    samples = [(0, 0, 0), (0, 32, 0), (0, 5, 17), (1, 17, 5), (1, 32, 32), (0, 12, 12)]
    Jv, Kv = oracle.sample(inp.B_packed, inp.nao, inp.C, inp.occ, samples)
    for t, (s, mu, nu) in enumerate(samples):
        assert abs(Jv[t] - J[s, mu, nu]) <= 1e-13 * np.abs(J[s]).max()
        assert abs(Kv[t] - K[s, mu, nu]) <= 1e-13 * np.abs(K[s]).max()
    # and against einsum directly (the sampler is pinned on its own, not only via get_jk)
    _, _, Je, Ke = einsum_jk(inp.B_packed, inp.nao, inp.C[1], inp.occ[1])
    assert abs(Jv[3] - Je[17, 5]) <= 1e-13 * np.abs(Je).max()
    assert abs(Kv[3] - Ke[17, 5]) <= 1e-13 * np.abs(Ke).max()
