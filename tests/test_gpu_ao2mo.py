"""GPU parity of dfjk_ao2mo (Eq. 18-21) against oracle/ao2mo_oracle.c, element by element.

Bar: max|d|/max|.| <= 1e-10 for bpa, ppaa and papa (fp64 sums in a different order; observed ~1e-15).
"""
import numpy as np
import pytest

import dfjk_inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10


def rel(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def run_case(nao, naux, nmo, a0, nact, seed, L=0.0, orth=False, **opts):
    import torch
    import oracle
    import paper_2505_03755_b200 as dfjk
    inp = dfjk_inputs.make_random(nao, naux, [1], seed, L=L)
    rng = np.random.default_rng(seed + 7)
    M = rng.standard_normal((nao, nmo))
    if orth:
        M = np.linalg.qr(rng.standard_normal((nao, nao)))[0][:, :nmo].copy()
    o_bpa, o_ppaa, o_papa = oracle.ao2mo(inp.B_packed, nao, M, a0, nact)
    B = torch.from_numpy(inp.B_packed).cuda()
    with dfjk.DFJK(B, nao, **opts) as h:
        bpa, ppaa, papa = h.ao2mo(torch.from_numpy(M).cuda(), a0, nact)
        torch.cuda.synchronize()
        assert h.last_launch_count > 0 or naux == 0 or nmo == 0
        bpa2, ppaa2, papa2 = h.ao2mo(torch.from_numpy(M).cuda(), a0, nact)     # deterministic
        torch.cuda.synchronize()
        assert torch.equal(bpa, bpa2) and torch.equal(ppaa, ppaa2) and torch.equal(papa, papa2)
    bpa, ppaa, papa = bpa.cpu().numpy(), ppaa.cpu().numpy(), papa.cpu().numpy()
    if o_bpa.size:
        assert rel(bpa, o_bpa) <= TOL, rel(bpa, o_bpa)
        assert rel(ppaa, o_ppaa) <= TOL, rel(ppaa, o_ppaa)
        assert rel(papa, o_papa) <= TOL, rel(papa, o_papa)
    return bpa, ppaa, papa


@pytest.mark.parametrize("nao,naux,nmo,a0,nact,seed", [
    (16, 9, 12, 3, 4, 201),         # everything smaller than one tile
    (67, 45, 50, 11, 5, 202),       # ragged, nmo*nact odd
    (130, 70, 130, 60, 8, 203),     # nmo = nao, one row past a 128 tile
    (150, 33, 97, 0, 3, 204),       # active block at the start, odd nmo
    (96, 20, 40, 34, 6, 205),       # active block at the end (a0 + nact = nmo)
    (48, 1, 48, 20, 2, 206),        # single aux row
])
def test_ragged_shapes(nao, naux, nmo, a0, nact, seed):
    run_case(nao, naux, nmo, a0, nact, seed, L=max(4.0, nao / 6))


@pytest.mark.parametrize("opts", [dict(nblk=1), dict(nblk=7), dict(workspace_cap_bytes=1 << 21),
                                  dict(ao2mo_route=1), dict(ao2mo_route=2), dict(ao2mo_route=1, nblk=5),
                                  dict(ao2mo_route=2, nblk=5)])
def test_blocking_and_route_do_not_change_the_result(opts):
    """route 1 = Eq. 18-21 in the printed order, route 2 = active first (never forms bmo)"""
    run_case(120, 61, 90, 30, 6, 210, L=15.0, **opts)


@pytest.mark.parametrize("route", [1, 2])
@pytest.mark.parametrize("nao,naux,nmo,a0,nact,seed", [(67, 45, 50, 11, 5, 241), (130, 70, 130, 60, 8, 242),
                                                       (150, 33, 97, 0, 3, 243), (48, 1, 48, 20, 2, 244)])
def test_both_routes_on_ragged_shapes(route, nao, naux, nmo, a0, nact, seed):
    run_case(nao, naux, nmo, a0, nact, seed, L=max(4.0, nao / 6), ao2mo_route=route)


def test_small_config_shape_with_orthonormal_orbitals():
    """nao=300, naux=1000 (BASELINE.json's `small` B), all 300 MOs, (8 active) -- several tiles and aux blocks"""
    bpa, ppaa, papa = run_case(300, 1000, 300, 80, 8, 220, L=20.0, orth=True)
    # permutational symmetry of the CUDA result itself
    assert rel(ppaa, ppaa.transpose(1, 0, 2, 3)) < 1e-12 and rel(papa, papa.transpose(2, 3, 0, 1)) < 1e-12


def test_edges_and_errors():
    import torch
    import paper_2505_03755_b200 as dfjk
    inp = dfjk_inputs.make_random(20, 6, [1], 230)
    B = torch.from_numpy(inp.B_packed).cuda()
    M = torch.from_numpy(np.random.default_rng(1).standard_normal((20, 10))).cuda()
    with dfjk.DFJK(B, 20) as h:
        bpa, ppaa, papa = h.ao2mo(M, 4, 0)                      # no active orbitals
        assert bpa.shape == (6, 10, 0) and ppaa.numel() == 0
        with pytest.raises(dfjk.DFJKError):
            h.ao2mo(M, 8, 4)                                    # active range past nmo
        J, K = h.get_jk([M[:, :3].contiguous()], [torch.ones(3, dtype=torch.float64, device="cuda")])
        torch.cuda.synchronize()                                # the handle still serves get_jk
        assert torch.isfinite(J).all() and torch.isfinite(K).all()


def test_route_follows_the_flop_model():
    """few active orbitals: active first (route 2); an active space as large as the MO space: the
    printed order (route 1); both against the oracle"""
    import torch
    import oracle
    import paper_2505_03755_b200 as dfjk
    inp = dfjk_inputs.make_random(64, 30, [1], 251, L=10.0)
    M = np.random.default_rng(252).standard_normal((64, 40))
    B = torch.from_numpy(inp.B_packed).cuda()
    with dfjk.DFJK(B, 64) as h:
        assert h.last_ao2mo_route == 0
        for a0, nact, want in ((10, 3, 2), (0, 40, 1)):
            bpa, ppaa, papa = h.ao2mo(torch.from_numpy(M).cuda(), a0, nact)
            torch.cuda.synchronize()
            assert h.last_ao2mo_route == want
            o_bpa, o_ppaa, o_papa = oracle.ao2mo(inp.B_packed, 64, M, a0, nact)
            assert rel(bpa.cpu().numpy(), o_bpa) <= TOL
            assert rel(ppaa.cpu().numpy(), o_ppaa) <= TOL and rel(papa.cpu().numpy(), o_papa) <= TOL


@pytest.mark.parametrize("route", [1, 2])
def test_more_mo_columns_than_one_n_tile(route):
    """nmo = 380 > 352: Eq. 18 (route 1) needs two N tiles of the half-transform; k_gemm_tn two N tiles"""
    run_case(400, 9, 380, 100, 4, 261, L=40.0, ao2mo_route=route)


# ---- the one-pass symmetric thin half-transform (symm.cu) behind the active-first route, nact <= 8
@pytest.mark.parametrize("nao,naux,nmo,a0,nact,seed", [
    (5, 3, 5, 1, 2, 301),           # smaller than one row group; naux * npair odd (plain-load tail of the last row)
    (33, 7, 20, 4, 8, 302),         # one row past a super-group of 32 rows; npair odd: odd aux rows start 8-byte aligned
    (129, 5, 60, 10, 7, 303),       # one column past a 128-column chunk, nao % 4 == 1
    (130, 4, 64, 0, 1, 304),        # nao % 4 == 2, a single active column
    (263, 6, 100, 50, 8, 305),      # three chunks, ragged last row group, nao % 4 == 3
    (520, 3, 48, 40, 8, 306),       # five chunks: every warp owns several column blocks
])
def test_symm_thin_shapes(nao, naux, nmo, a0, nact, seed):
    """route 2 with at most 8 active columns streams the packed triangle once (k_symm_thin); every shape
    is also run with the tiled half-transform (no_symm_thin) and both must match the oracle"""
    a = run_case(nao, naux, nmo, a0, nact, seed, L=max(4.0, nao / 6), ao2mo_route=2)
    b = run_case(nao, naux, nmo, a0, nact, seed, L=max(4.0, nao / 6), ao2mo_route=2, no_symm_thin=True)
    for x, y in zip(a, b):
        assert rel(x, y) <= 1e-12


def test_symm_thin_large_basis_every_block():
    """nao = 1203 (ragged, 10 chunks, all 20 register-resident column blocks per warp), white-noise B so
    that a wrong block anywhere shows; more aux rows than SMs so the persistent loop wraps"""
    run_case(1203, 150, 24, 8, 8, 307, L=0.0, ao2mo_route=2)


@pytest.mark.parametrize("nao,naux,nmo,a0,nact,seed", [
    (1300, 3, 16, 4, 4, 308),       # two column panels of 1280: 20 columns in the second
    (1400, 4, 12, 2, 8, 311),       # the second panel holds 15 column blocks, ragged last row group (1400 = 175 x 8)
    (2570, 2, 10, 1, 3, 312),       # three panels: the first two add direct sums for the rows of the third
])
def test_symm_thin_column_panels(nao, naux, nmo, a0, nact, seed):
    """a basis beyond 1280 (system C of the paper: 1378 AOs) takes one launch per panel of 1280 columns; the first
    panel stores every row of Z, later panels add; against the oracle and against the tiled half-transform"""
    a = run_case(nao, naux, nmo, a0, nact, seed, L=100.0, ao2mo_route=2)
    b = run_case(nao, naux, nmo, a0, nact, seed, L=100.0, ao2mo_route=2, no_symm_thin=True)
    for x, y in zip(a, b):
        assert rel(x, y) <= 1e-12


def test_symm_thin_unaligned_tensor_falls_back():
    """a row slice of an odd-npair tensor is only 8-byte aligned: the tiled path must be taken"""
    import torch
    import oracle
    import paper_2505_03755_b200 as dfjk
    nao, naux = 33, 9                                           # npair = 561, odd
    inp = dfjk_inputs.make_random(nao, naux, [1], 309, L=8.0)
    M = np.random.default_rng(310).standard_normal((nao, 12))
    Bfull = torch.from_numpy(inp.B_packed).cuda()
    Bs = Bfull[1:]                                              # data_ptr = base + 561 * 8
    assert Bs.data_ptr() % 16 == 8
    with dfjk.DFJK(Bs, nao, ao2mo_route=2) as h:
        bpa, ppaa, papa = h.ao2mo(torch.from_numpy(M).cuda(), 2, 6)
        torch.cuda.synchronize()
    o_bpa, o_ppaa, o_papa = oracle.ao2mo(inp.B_packed[1:], nao, M, 2, 6)
    assert rel(bpa.cpu().numpy(), o_bpa) <= TOL and rel(ppaa.cpu().numpy(), o_ppaa) <= TOL
    assert rel(papa.cpu().numpy(), o_papa) <= TOL


@pytest.mark.parametrize("nao,naux,nmo,a0,nact,seed", [
    (200, 40, 60, 5, 9, 321),       # 45 active pairs (padded to 46): 48-row tiles of the transposed W product
    (203, 64, 70, 20, 10, 322),     # 55 pairs: 56-row tiles
    (120, 72, 50, 3, 11, 323),      # 66 pairs: beyond 64, the W product runs in the other orientation
    (200, 41, 60, 5, 8, 324),       # naux % 4 != 0: no bulk copies, the gather producer
])
def test_active_first_route_with_more_active_orbitals(nao, naux, nmo, a0, nact, seed):
    """the W contraction over the packed active pairs a1 >= a2 in both orientations, the packed index transformations
    and the lower-tile Eq. 21, for 8 to 11 active orbitals"""
    bpa, ppaa, papa = run_case(nao, naux, nmo, a0, nact, seed, L=max(4.0, nao / 6), ao2mo_route=2)
    assert np.array_equal(papa, papa.transpose(2, 3, 0, 1))                  # mirrored: bitwise symmetric
    assert np.array_equal(ppaa, ppaa.transpose(0, 1, 3, 2))                  # one packed pair serves (a1, a2) and (a2, a1)
