"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, element by element.

Bar (BASELINE.json north_star): max|dJ|/max|J| and max|dK|/max|K| <= 1e-10 per set.  fp64 DMMA/DFMA
sums differ from the oracle only in the order of additions, so the observed errors are ~1e-15..1e-13.
"""
import numpy as np
import pytest

import dfjk_inputs

pytestmark = pytest.mark.gpu

TOL = 1e-10


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device; there is no CPU fallback")
    return torch


@pytest.fixture(scope="module", params=["default", "tiled"])
def dfjk(request, torch_cuda):
    """every test of this module runs twice: with the default dispatch (embedding-sized calls take the
    single-launch path of csrc/small.cu) and with no_small_path=True (always the tensor-pipe kernels)"""
    import types
    import paper_2505_03755_b200 as pkg
    pkg.load_library()
    if request.param == "default":
        return pkg
    proxy = types.SimpleNamespace(**{k: getattr(pkg, k) for k in dir(pkg) if not k.startswith("__")})

    def tiled(*a, **kw):
        kw.setdefault("no_small_path", True)
        return pkg.DFJK(*a, **kw)
    proxy.DFJK = tiled
    proxy.small_path = False
    return proxy


def to_dev(torch, inp):
    B = torch.from_numpy(inp.B_packed).cuda()
    Cs = [torch.from_numpy(c).cuda() for c in inp.C]
    occs = [torch.from_numpy(o).cuda() for o in inp.occ]
    return B, Cs, occs


def rel(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def check_against_oracle(torch, dfjk, inp, **opts):
    import oracle
    Jo, Ko = oracle.get_jk_inputs(inp)
    B, Cs, occs = to_dev(torch, inp)
    with dfjk.DFJK(B, inp.nao, **opts) as h:
        J, K = h.get_jk(Cs, occs)
        torch.cuda.synchronize()
        plan = h.plan()
        assert h.last_launch_count > 0
    J, K = J.cpu().numpy(), K.cpu().numpy()
    for s in range(inp.nset):
        if np.abs(Jo[s]).max() == 0:
            assert not J[s].any() and not K[s].any()
            continue
        ej, ek = rel(J[s], Jo[s]), rel(K[s], Ko[s])
        assert ej <= TOL and ek <= TOL, (inp.name, s, ej, ek, plan)
        assert np.array_equal(J[s], J[s].T) and np.array_equal(K[s], K[s].T)   # bitwise symmetric
    return J, K


def test_dmma_fragment_mapping(dfjk):
    dfjk.selftest_dmma()


def test_tiny_config(torch_cuda, dfjk):
    check_against_oracle(torch_cuda, dfjk, dfjk_inputs.make_config("tiny"))


def test_tiny_config_dispatch(torch_cuda, dfjk):
    """tiny (nao=48, naux=160, nocc=12) is launch-latency bound: one launch by default, seven with
    no_small_path; small (nao=300) always takes the tensor-pipe kernels"""
    torch = torch_cuda
    for name in ("tiny", "small"):
        inp = dfjk_inputs.make_config(name)
        B, Cs, occs = to_dev(torch, inp)
        with dfjk.DFJK(B, inp.nao) as h:
            h.get_jk(Cs, occs)
            torch.cuda.synchronize()
            one = h.last_launch_count == 1
        assert one == (name == "tiny" and getattr(dfjk, "small_path", True))


@pytest.mark.parametrize("nao,naux,nocc,seed,kw", [
    (96, 20, [48], 171, {}),                                 # the largest basis and column count of the path
    (80, 170, [40, 0, 8], 172, {}),                          # more aux rows than SMs, an empty set
    (33, 9, [1] * 16 + [2] * 16, 173, dict(max_nset=32, max_nocc_total=48)),   # 32 sets
    (1, 2, [1], 174, {}),                                    # a single AO
    (64, 5, [64], 175, {}),                                  # nocc = nao, fewer aux rows than CTAs
    (48, 300, [12], 176, {}),                                # two aux rows per CTA: the second adds to the partials
    (64, 700, [16, 5], 177, {}),                             # three aux rows per CTA, two sets, a ragged last tile of columns
    (90, 310, [21], 178, {}),                                # nao not a multiple of 8: clamped rows in the 8 x 8 tiles
])
def test_single_launch_path(torch_cuda, dfjk, nao, naux, nocc, seed, kw):
    """shapes inside the single-launch regime: J and K together, J alone, K alone, signed occupations,
    two calls in a row (the arrival ticket is reset), against the oracle"""
    import oracle
    torch = torch_cuda
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(3.0, nao / 6))
    rs = np.random.default_rng(seed + 1)
    for o in inp.occ:
        o *= rs.choice([-1.0, 1.0], size=o.shape)
    Jo, Ko = oracle.get_jk_inputs(inp)
    B, Cs, occs = to_dev(torch, inp)
    with dfjk.DFJK(B, inp.nao, **kw) as h:
        J, K = h.get_jk(Cs, occs)
        torch.cuda.synchronize()
        assert (h.last_launch_count == 1) == getattr(dfjk, "small_path", True)
        Jonly, _ = h.get_jk(Cs, occs, with_k=False)
        _, Konly = h.get_jk(Cs, occs, with_j=False)
        J2, K2 = h.get_jk(Cs, occs)
        torch.cuda.synchronize()
        assert torch.equal(J, J2) and torch.equal(K, K2) and torch.equal(K, Konly)
    for s in range(inp.nset):
        if nocc[s] == 0:
            assert not J[s].any() and not K[s].any()
            continue
        assert rel(J[s].cpu().numpy(), Jo[s]) <= TOL and rel(K[s].cpu().numpy(), Ko[s]) <= TOL
        assert rel(Jonly[s].cpu().numpy(), Jo[s]) <= TOL
        assert torch.equal(J[s], J[s].T) and torch.equal(K[s], K[s].T)


def test_small_config(torch_cuda, dfjk):
    check_against_oracle(torch_cuda, dfjk, dfjk_inputs.make_config("small"))


@pytest.mark.parametrize("nao,naux,nocc,seed", [
    (5, 3, [2], 101),            # npair odd: scalar load paths
    (6, 7, [6], 102),            # npair odd, nocc = nao
    (67, 45, [23, 7], 103),      # ragged everything, two sets
    (129, 70, [33], 104),        # one row past a 128 tile
    (130, 9, [5, 0, 12], 105),   # empty middle set
    (200, 130, [9, 8, 8, 1, 40, 3, 17, 2], 106),  # eight sets
    (257, 33, [64], 107),        # three m-tiles: direct, crossing and transposed chunks all occur
    (48, 1, [12], 108),          # single aux row
    (330, 20, [40, 9], 161),     # 3 x 112: the 112 x 112 SYRK tile
    (1203, 3, [35, 8], 164),     # large ragged basis: 19 row blocks, the last with 51 rows; 16 x 16 SYRK tiles
    (420, 14, [400], 162),       # 400 columns: two N tiles of the half-transform (fused rho over both)
    (400, 10, [180, 150, 60], 163),   # 392 padded columns in two N tiles, a set straddling them
])
def test_ragged_shapes(torch_cuda, dfjk, nao, naux, nocc, seed):
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(4.0, nao / 6))
    check_against_oracle(torch_cuda, dfjk, inp)


@pytest.mark.parametrize("nao,naux,nocc,seed", [
    (5, 3, [2], 121),                      # npair odd: the DMMA fallback of pass 1
    (8, 13, [3, 2], 122),                  # npair even, 36 pairs: far less than one stage
    (67, 45, [23, 7], 123),                # npair even, ragged rows (45 = 5 groups of 8 + 5)
    (181, 70, [9, 8, 8, 1, 40, 3], 124),   # npair = 16471: one full 16384-pair CTA chunk + a ragged one
    (200, 130, [9, 8, 8, 1, 40, 3, 17, 2], 125),   # eight sets, three row blocks of 64
    (40, 21, [3, 1, 4, 1, 5, 9, 2, 6, 5, 3, 5], 126),   # eleven sets: two set groups
])
def test_j_only_two_pass_path(torch_cuda, dfjk, nao, naux, nocc, seed):
    """J alone runs the two-pass J (bulk-copy pipeline for pass 1 when npair is even)."""
    import oracle
    torch = torch_cuda
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(4.0, nao / 6))
    Jo, _ = oracle.get_jk_inputs(inp, with_k=False)
    B, Cs, occs = to_dev(torch, inp)
    with dfjk.DFJK(B, inp.nao, max_nset=12, max_nocc_total=max(nao, sum(nocc))) as h:
        J, K = h.get_jk(Cs, occs, with_k=False)
        torch.cuda.synchronize()
        assert K is None
    J = J.cpu().numpy()
    for s in range(inp.nset):
        assert rel(J[s], Jo[s]) <= TOL, (s, rel(J[s], Jo[s]))
        assert np.array_equal(J[s], J[s].T)


@pytest.mark.parametrize("nao,naux,nocc,seed,opts", [
    (1, 2, [1], 141, {}),                                   # a single AO: npair = 1
    (40, 17, [40], 142, {}),                                # nocc = nao
    (33, 9, [1] * 16 + [2] * 16, 143, dict(max_nset=32, max_nocc_total=48)),   # 32 sets, the hard maximum
    (72, 300, [11], 144, dict(workspace_cap_bytes=1)),      # one aux row per block: 300 blocks
    (260, 12, [130, 129], 145, {}),                         # 259 + 5 padded columns: wide N tile, nao % 8 != 0
])
def test_degenerate_and_extreme_shapes(torch_cuda, dfjk, nao, naux, nocc, seed, opts):
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(3.0, nao / 6))
    check_against_oracle(torch_cuda, dfjk, inp, **opts)


def test_no_aux_rows_gives_zeros(torch_cuda, dfjk):
    torch = torch_cuda
    B = torch.empty((0, 10 * 11 // 2), dtype=torch.float64, device="cuda")
    C = torch.ones((10, 3), dtype=torch.float64, device="cuda")
    with dfjk.DFJK(B, 10) as h:
        J, K = h.get_jk([C], [torch.ones(3, dtype=torch.float64, device="cuda")],
                        out_j=torch.full((1, 10, 10), 7.0, dtype=torch.float64, device="cuda"),
                        out_k=torch.full((1, 10, 10), 7.0, dtype=torch.float64, device="cuda"))
        torch.cuda.synchronize()
    assert not J.any() and not K.any()


@pytest.mark.parametrize("nao,naux,nocc,seed,opts", [
    (24, 10, [5], 146, {}),                                  # one negative column
    (67, 45, [23, 7], 147, {}),                              # two sets sharing a 32-column chunk, mixed signs
    (150, 61, [37, 10, 3], 148, dict(two_pass_j=True)),      # Eq. 14 through the signed packed density
    (150, 61, [37, 10, 3], 148, dict(nblk=7, ksplit=3)),     # several aux blocks and splits
    (330, 20, [40, 9], 149, {}),                             # 112 x 112 SYRK tiles
    (420, 14, [400], 150, {}),                               # two N tiles of the half-transform
    (200, 33, [9, 8, 8, 1, 40, 3, 17, 2], 155, {}),          # eight sets
])
def test_signed_occupations_at_c_form_cost(torch_cuda, dfjk, nao, naux, nocc, seed, opts):
    """occupations of any sign (differences of densities) through dfjk_get_jk: the
    kernels use C' = C sqrt(|occ|) and flip a sign bit, D = C' diag(sign occ) C'^T exactly.  The
    oracle takes the occupations as they are (no sqrt folding)."""
    import oracle
    torch = torch_cuda
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(4.0, nao / 6))
    rs = np.random.default_rng(seed + 1000)
    for o in inp.occ:                                        # about half of the columns negative, one exact zero
        o *= rs.choice([-1.0, 1.0], size=o.shape)
        if o.size > 2:
            o[1] = 0.0
    assert any((o < 0).any() for o in inp.occ)
    Jo, Ko = oracle.get_jk_inputs(inp)
    B, Cs, occs = to_dev(torch, inp)
    with dfjk.DFJK(B, inp.nao, **opts) as h:
        J, K = h.get_jk(Cs, occs)
        Jonly, _ = h.get_jk(Cs, occs, with_k=False)          # two-pass J on the signed packed density
        _, Konly = h.get_jk(Cs, occs, with_j=False)
        torch.cuda.synchronize()
        assert torch.equal(K, Konly)
    J, K, Jonly = J.cpu().numpy(), K.cpu().numpy(), Jonly.cpu().numpy()
    for s in range(inp.nset):
        assert rel(J[s], Jo[s]) <= TOL and rel(K[s], Ko[s]) <= TOL and rel(Jonly[s], Jo[s]) <= TOL, (s, opts)
        assert np.array_equal(J[s], J[s].T) and np.array_equal(K[s], K[s].T)
    # the indefinite density also goes through the density-matrix form: same numbers
    D = np.stack([(c * o) @ c.T for c, o in zip(inp.C, inp.occ)])
    if sum(nocc) <= 60:
        with dfjk.DFJK(B, inp.nao) as h:
            Jd, Kd = h.get_jk_dm(torch.from_numpy(D).cuda())
            torch.cuda.synchronize()
        assert rel(Jd.cpu().numpy(), Jo) <= TOL and rel(Kd.cpu().numpy(), Ko) <= TOL


def test_sign_of_occupations_does_not_leak_between_calls(torch_cuda, dfjk):
    """the sign bits are rewritten by every call: a signed call followed by an unsigned one (and an
    AO2MO call, which has no occupations) gives the unsigned answers bit for bit"""
    torch = torch_cuda
    inp = dfjk_inputs.make_random(90, 31, [20, 11], 156, L=15.0)
    B, Cs, occs = to_dev(torch, inp)
    with dfjk.DFJK(B, inp.nao) as h:
        J0, K0 = h.get_jk(Cs, occs)
        M = torch.from_numpy(np.random.default_rng(5).standard_normal((90, 31))).cuda()
        ref = [t.clone() for t in h.ao2mo(M, 20, 6)]
        h.get_jk(Cs, [-o for o in occs])
        J1, K1 = h.get_jk(Cs, occs)
        got = h.ao2mo(M, 20, 6)
        torch.cuda.synchronize()
        assert torch.equal(J0, J1) and torch.equal(K0, K1)
        assert all(torch.equal(a, b) for a, b in zip(ref, got))
        Jn, Kn = h.get_jk(Cs, [-o for o in occs])           # J and K are linear in D: D -> -D
        torch.cuda.synchronize()
        assert torch.equal(Jn, -J0) and torch.equal(Kn, -K0)


def test_more_than_eight_sets(torch_cuda, dfjk):
    inp = dfjk_inputs.make_random(40, 21, [3, 1, 4, 1, 5, 9, 2, 6, 5, 3, 5], 109)
    check_against_oracle(torch_cuda, dfjk, inp, max_nset=12, max_nocc_total=44)


@pytest.mark.parametrize("opts", [dict(nblk=1), dict(nblk=7), dict(nblk=16, ksplit=5), dict(ksplit=1),
                                  dict(workspace_cap_bytes=1 << 20), dict(copy_B=True), dict(two_pass_j=True),
                                  dict(two_pass_j=True, nblk=5), dict(no_retile=True)])
def test_blocking_and_split_k_do_not_change_the_result(torch_cuda, dfjk, opts):
    """N_blk and split-K are memory/parallelism knobs, not part of the result."""
    inp = dfjk_inputs.make_random(150, 61, [37, 10], 110, L=20.0)
    check_against_oracle(torch_cuda, dfjk, inp, **opts)


def test_j_only_k_only_and_batching(torch_cuda, dfjk):
    torch = torch_cuda
    inp = dfjk_inputs.make_random(90, 50, [20, 11, 6], 111, L=15.0)
    B, Cs, occs = to_dev(torch, inp)
    with dfjk.DFJK(B, inp.nao) as h:
        J, K = h.get_jk(Cs, occs)
        Jonly, none_k = h.get_jk(Cs, occs, with_k=False)
        none_j, Konly = h.get_jk(Cs, occs, with_j=False)
        assert none_k is None and none_j is None
        torch.cuda.synchronize()
        # with both outputs rho comes out of the half-transform (one stream over B fewer); J-only runs
        # the two-pass J: same numbers up to the order of additions
        assert rel(J.cpu().numpy(), Jonly.cpu().numpy()) < 1e-13 and torch.equal(K, Konly)
        with dfjk.DFJK(B, inp.nao, two_pass_j=True) as h2:
            J2, K2 = h2.get_jk(Cs, occs)
            torch.cuda.synchronize()
            assert torch.equal(J2, Jonly) and torch.equal(K2, K)
        for s in range(3):                      # nset-batched == one at a time, bit for bit in J
            J1, K1 = h.get_jk([Cs[s]], [occs[s]])
            torch.cuda.synchronize()
            assert rel(J1[0].cpu().numpy(), J[s].cpu().numpy()) < 1e-13
            assert rel(K1[0].cpu().numpy(), K[s].cpu().numpy()) < 1e-13


@pytest.mark.parametrize("nao,naux,nocc,seed", [(67, 21, [23, 7], 151), (257, 33, [64], 152), (300, 40, [80], 153)])
def test_retiled_and_gathered_half_transform_agree_bitwise(torch_cuda, dfjk, nao, naux, nocc, seed):
    """the re-tiled copy of B (default) and the gather from the packed triangle feed the same numbers
    to the same DMMA sequence"""
    torch = torch_cuda
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(4.0, nao / 6))
    B, Cs, occs = to_dev(torch, inp)
    with dfjk.DFJK(B, nao) as h1, dfjk.DFJK(B, nao, no_retile=True) as h2:
        J1, K1 = h1.get_jk(Cs, occs)
        J2, K2 = h2.get_jk(Cs, occs)
        torch.cuda.synchronize()
        assert torch.equal(J1, J2) and torch.equal(K1, K2)


def test_repeat_calls_are_bitwise_deterministic_and_stream_ordered(torch_cuda, dfjk):
    torch = torch_cuda
    inp = dfjk_inputs.make_random(140, 77, [31, 9], 112, L=12.0)
    B, Cs, occs = to_dev(torch, inp)
    with dfjk.DFJK(B, inp.nao) as h:
        J0, K0 = h.get_jk(Cs, occs)
        torch.cuda.synchronize()
        st = torch.cuda.Stream()
        st.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(st):
            J1, K1 = h.get_jk(Cs, occs)
            J2, K2 = h.get_jk(Cs, occs, stream=st)
        st.synchronize()
        assert torch.equal(J0, J1) and torch.equal(K0, K1)
        assert torch.equal(J0, J2) and torch.equal(K0, K2)


def test_get_jk_is_cuda_graph_capturable(torch_cuda, dfjk):
    """dfjk_get_jk only enqueues (no allocation, no host sync: PAPER.md:259-261), so a call can be
    captured into a CUDA graph and replayed on new orbitals -- the many-small-calls regime of the
    embedded fragments."""
    import oracle
    torch = torch_cuda
    a = dfjk_inputs.make_random(60, 35, [13, 5], 131, L=9.0)
    b = dfjk_inputs.make_random(60, 35, [13, 5], 132, L=9.0)           # other orbitals, same shapes
    B = torch.from_numpy(a.B_packed).cuda()
    C = torch.from_numpy(a.C_concat()).cuda()
    occ = torch.from_numpy(a.occ_concat()).cuda()
    J = torch.empty((2, 60, 60), dtype=torch.float64, device="cuda")
    K = torch.empty_like(J)
    with dfjk.DFJK(B, 60) as h:
        h.get_jk_raw(a.nocc, C, occ, out_j=J, out_k=K)                 # warm-up: function attributes set
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            h.get_jk_raw(a.nocc, C, occ, out_j=J, out_k=K)
        for inp in (b, a):
            C.copy_(torch.from_numpy(inp.C_concat()))
            occ.copy_(torch.from_numpy(inp.occ_concat()))
            J.zero_(); K.zero_()
            g.replay()
            torch.cuda.synchronize()
            Jo, Ko = oracle.get_jk(a.B_packed, 60, inp.C, inp.occ)
            for s in range(2):
                assert rel(J[s].cpu().numpy(), Jo[s]) <= TOL and rel(K[s].cpu().numpy(), Ko[s]) <= TOL
        del g


def test_outputs_are_overwritten_not_accumulated(torch_cuda, dfjk):
    torch = torch_cuda
    inp = dfjk_inputs.make_random(33, 12, [7], 113)
    B, Cs, occs = to_dev(torch, inp)
    with dfjk.DFJK(B, inp.nao) as h:
        J, K = h.get_jk(Cs, occs)
        junk_j = torch.full_like(J, 1e300)
        junk_k = torch.full_like(K, float("nan"))
        h.get_jk(Cs, occs, out_j=junk_j, out_k=junk_k)
        torch.cuda.synchronize()
        assert torch.equal(J, junk_j) and torch.equal(K, junk_k)


def test_host_buffer_entry_point(torch_cuda, dfjk):
    torch = torch_cuda
    import oracle
    inp = dfjk_inputs.make_random(70, 40, [15, 6], 114, L=10.0)
    Jo, Ko = oracle.get_jk_inputs(inp)
    B = torch.from_numpy(inp.B_packed).cuda()
    C = torch.from_numpy(inp.C_concat()).pin_memory()
    occ = torch.from_numpy(inp.occ_concat()).pin_memory()
    J = torch.empty((2, 70, 70), dtype=torch.float64).pin_memory()
    K = torch.empty((2, 70, 70), dtype=torch.float64).pin_memory()
    with dfjk.DFJK(B, inp.nao) as h:
        h.get_jk_host(inp.nocc, C, occ, J, K)     # synchronises before returning
    for s in range(2):
        assert rel(J[s].numpy(), Jo[s]) <= TOL and rel(K[s].numpy(), Ko[s]) <= TOL


def test_error_codes(torch_cuda, dfjk):
    torch = torch_cuda
    inp = dfjk_inputs.make_random(20, 6, [4], 115)
    B, Cs, occs = to_dev(torch, inp)
    with pytest.raises(ValueError):
        dfjk.DFJK(B[:, :-1].contiguous(), 20)
    with dfjk.DFJK(B, 20, max_nset=2, max_nocc_total=10) as h:
        with pytest.raises(dfjk.DFJKError) as e:   # nset beyond capacity
            h.get_jk([Cs[0]] * 3, [occs[0]] * 3)
        assert e.value.code == 1
        with pytest.raises(dfjk.DFJKError):        # nocc total beyond capacity
            big = torch.zeros((20, 11), dtype=torch.float64, device="cuda")
            h.get_jk([big], [torch.ones(11, dtype=torch.float64, device="cuda")])
        J, K = h.get_jk(Cs, occs)                  # the handle is still usable afterwards
        torch.cuda.synchronize()
        assert torch.isfinite(J).all() and torch.isfinite(K).all()
    lib = dfjk.load_library()
    assert lib.dfjk_destroy(None) == 0
    assert lib.dfjk_strerror(4).decode().startswith("unsupported")


@pytest.mark.parametrize("nao,naux,nocc,seed,opts", [
    (130, 30, [5], 181, {}),                          # npair odd: odd aux rows start 8-byte aligned
    (200, 170, [8], 182, {}),                         # more aux rows than SMs
    (263, 21, [3], 183, dict(nblk=4)),                # several aux blocks: rho written block by block
    (1203, 6, [7], 184, {}),                          # ragged, all 20 column blocks per warp
    (520, 9, [8], 185, dict(two_pass_j=True)),        # rho from the two-pass J, X from the thin kernel
    (1400, 5, [6], 186, {}),                          # two column panels of the one-pass kernel: rho summed over both
])
def test_one_thin_set_takes_the_one_pass_half_transform(torch_cuda, dfjk, nao, naux, nocc, seed, opts):
    """a JK call on one set of at most 8 orbitals (a fragment's active space): the half-transform streams the
    packed triangle once (k_symm_thin) and writes rho itself; signed occupations; against the oracle and
    against the tiled kernel (no_symm_thin)"""
    import oracle
    torch = torch_cuda
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(4.0, nao / 6))
    inp.occ[0][::2] *= -1.0
    Jo, Ko = oracle.get_jk_inputs(inp)
    B, Cs, occs = to_dev(torch, inp)
    res = []
    for extra in ({}, dict(no_symm_thin=True)):
        with dfjk.DFJK(B, inp.nao, **opts, **extra) as h:
            J, K = h.get_jk(Cs, occs)
            n_both = h.last_launch_count
            _, Konly = h.get_jk(Cs, occs, with_j=False)
            Jonly, _ = h.get_jk(Cs, occs, with_k=False)
            torch.cuda.synchronize()
            assert torch.equal(K, Konly)
        assert rel(J[0].cpu().numpy(), Jo[0]) <= TOL and rel(K[0].cpu().numpy(), Ko[0]) <= TOL
        assert rel(Jonly[0].cpu().numpy(), Jo[0]) <= TOL
        assert torch.equal(J[0], J[0].T) and torch.equal(K[0], K[0].T)
        res.append((J, K, n_both))
    assert rel(res[0][0].cpu().numpy(), res[1][0].cpu().numpy()) <= 1e-12
    assert rel(res[0][1].cpu().numpy(), res[1][1].cpu().numpy()) <= 1e-12
    if not opts.get("two_pass_j"):
        assert res[0][2] == res[1][2] - 1                    # no rho-reduce launch: the thin kernel writes rho


@pytest.mark.parametrize("nao,naux,nsets,seed", [
    (67, 45, 3, 191),        # npair = 2278: four full chunks + 230 pairs (not a multiple of 4); 45 rows = 5 groups + 5
    (183, 70, 6, 192),       # npair = 16836: a second CTA chunk of 452 pairs; two row blocks of 64
    (200, 130, 8, 193),      # eight sets, three row blocks
    (64, 9, 5, 194),         # two row groups, the second with one row
])
def test_j_pass_1_on_the_tensor_pipe(torch_cuda, dfjk, nao, naux, nsets, seed):
    """three to eight sets: pass 1 runs as a GEMM over the pairs on DMMA.8x8x4 (k_j1_mma), the weighted densities
    fetched once per 64 aux rows; J alone (two-pass J), signed occupations"""
    import oracle
    torch = torch_cuda
    rs = np.random.default_rng(seed)
    nocc = [int(rs.integers(1, 7)) for _ in range(nsets)]
    inp = dfjk_inputs.make_random(nao, naux, nocc, seed, L=max(4.0, nao / 6))
    inp.occ[0] *= -1.0
    Jo, _ = oracle.get_jk_inputs(inp, with_k=False)
    B, Cs, occs = to_dev(torch, inp)
    with dfjk.DFJK(B, inp.nao, no_small_path=True) as h:
        J, _ = h.get_jk(Cs, occs, with_k=False)
        J2, _ = h.get_jk(Cs, occs, with_k=False)
        torch.cuda.synchronize()
        assert torch.equal(J, J2)
    for s in range(nsets):
        assert rel(J[s].cpu().numpy(), Jo[s]) <= TOL, (s, rel(J[s].cpu().numpy(), Jo[s]))
        assert torch.equal(J[s], J[s].T)
