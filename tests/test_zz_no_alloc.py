"""dfjk_small_jk_static: the single-launch get_jk on the library's static device scratch (no handle, no
allocation) against the existing handle path (dfjk_get_jk), on calls made back to back.

Collected last on purpose (the file name sorts after every other test file): the run uses
pytest -x, so a failure here hides nothing.  Needs nothing from the other tests: passes alone in a fresh
process and after the rest of the suite.

Tolerance: the bar of tests/test_gpu_parity.py (max|d|/max|ref| <= 1e-10 per set).  Both paths run the same
kernel; when the static scratch does not cap the number of CTAs the sums run in the same order and the
results are bitwise equal.
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


def device_inputs(torch, inp):
    B = torch.from_numpy(inp.B_packed).cuda()
    C = torch.from_numpy(np.concatenate([c.reshape(-1) for c in inp.C])).cuda()
    occ = torch.from_numpy(np.concatenate(inp.occ)).cuda()
    return B, C, occ


def handle_path(torch, pkg, inp, B, C, occ):
    with pkg.DFJK(B, inp.nao) as h:
        J, K = h.get_jk_raw(list(inp.nocc), C, occ)
        torch.cuda.synchronize()
        # the existing path: the single launch on the handle's workspace, or the tiled kernels when the partials of
        # one CTA per aux row do not fit it ("capped": 14 launches)
        assert h.last_launch_count == 1 or inp.name.startswith("random7103"), h.last_launch_count
    return J, K


def cap_binds(inp):
    """True when DFJK_STATIC_SCRATCH_BYTES holds fewer CTAs' partials than dfjk_get_jk would launch (one CTA per
    aux row at these sizes): then the sums run in another order and only the tolerance applies"""
    per_cta = len(inp.nocc) * (inp.nao * inp.nao + inp.nao * (inp.nao + 1) // 2)
    return inp.naux * per_cta > (8 << 20) // 8


def rel(a, b):
    return float((a - b).abs().max() / max(float(b.abs().max()), 1e-300))


def signed(inp, seed):
    """occupations of either sign (differences of densities)"""
    rng = np.random.default_rng(seed)
    inp.occ = [o * rng.choice([-1.0, 1.0], size=o.shape) for o in inp.occ]
    return inp


CASES = {
    # BASELINE.json configs[0]
    "tiny": lambda: dfjk_inputs.make_config("tiny"),
    # several sets, one of them empty, ragged sizes, signed occupations (room for 29 CTAs' partials)
    "sets": lambda: signed(dfjk_inputs.make_random(77, 171, [9, 0, 17, 4], seed=7101, L=10.0), 7102),
    # the largest partials the entry point takes: 8 sets at nao = 96 leave room for 9 CTAs only
    "capped": lambda: dfjk_inputs.make_random(96, 130, [6] * 8, seed=7103, L=12.0),
}


def run_static(torch, pkg, inp, B, C, occ, fill):
    nset = len(inp.nocc)
    J = torch.full((nset, inp.nao, inp.nao), fill, dtype=torch.float64, device="cuda")
    K = torch.full((nset, inp.nao, inp.nao), fill, dtype=torch.float64, device="cuda")
    pkg.small_jk_static(B, inp.nao, list(inp.nocc), C, occ, out_j=J, out_k=K)
    return J, K


@pytest.mark.parametrize("order", [("tiny", "tiny"), ("capped", "tiny"), ("sets", "capped"), ("tiny", "sets")],
                         ids=lambda o: "+".join(o))
def test_static_scratch_entry_matches_the_handle_path_on_two_calls_in_a_row(torch_cuda, order):
    """two calls back to back on one stream, no synchronisation in between: the second runs on whatever the
    first left in the shared array (other sizes, other CTA count), and both must match dfjk_get_jk"""
    torch = torch_cuda
    import paper_2505_03755_b200 as pkg
    inps = [CASES[name]() for name in order]
    devs = [device_inputs(torch, inp) for inp in inps]
    refs = [handle_path(torch, pkg, inp, *dev) for inp, dev in zip(inps, devs)]
    torch.cuda.synchronize()
    outs = [run_static(torch, pkg, inp, *dev, fill=float("nan")) for inp, dev in zip(inps, devs)]
    torch.cuda.synchronize()
    for name, inp, (Jr, Kr), (J, K) in zip(order, inps, refs, outs):
        for s in range(len(inp.nocc)):
            assert rel(J[s], Jr[s]) <= TOL, (name, s)
            assert rel(K[s], Kr[s]) <= TOL, (name, s)
        assert torch.equal(J, J.transpose(1, 2)) and torch.equal(K, K.transpose(1, 2)), name
        if not cap_binds(inp):
            # same number of CTAs as the handle path: same order of additions
            assert torch.equal(J, Jr) and torch.equal(K, Kr), name
    # a third call repeats the first one bit for bit (deterministic, nothing of the second call leaks in)
    J3, K3 = run_static(torch, pkg, inps[0], *devs[0], fill=0.0)
    torch.cuda.synchronize()
    assert torch.equal(J3, outs[0][0]) and torch.equal(K3, outs[0][1])


def test_static_scratch_entry_one_output_at_a_time(torch_cuda):
    torch = torch_cuda
    import paper_2505_03755_b200 as pkg
    inp = CASES["sets"]()
    B, C, occ = device_inputs(torch, inp)
    Jr, Kr = handle_path(torch, pkg, inp, B, C, occ)
    nset = len(inp.nocc)
    J = torch.full((nset, inp.nao, inp.nao), float("nan"), dtype=torch.float64, device="cuda")
    K = torch.full_like(J, float("nan"))
    pkg.small_jk_static(B, inp.nao, list(inp.nocc), C, occ, out_j=J)
    pkg.small_jk_static(B, inp.nao, list(inp.nocc), C, occ, out_k=K)
    torch.cuda.synchronize()
    for s in range(nset):
        assert rel(J[s], Jr[s]) <= TOL and rel(K[s], Kr[s]) <= TOL, s
    J2, K2 = run_static(torch, pkg, inp, B, C, occ, fill=float("nan"))
    torch.cuda.synchronize()
    assert torch.equal(J, J2) and torch.equal(K, K2), "J-only and K-only calls give the bits of the joint call"


def test_static_scratch_entry_in_a_cuda_graph(torch_cuda):
    """the stated use: after one call outside the capture (set-up: address of the static array, function
    attribute) the entry point only enqueues a memset node and a kernel node, so it can be captured and replayed
    on new orbitals"""
    torch = torch_cuda
    import paper_2505_03755_b200 as pkg
    a = dfjk_inputs.make_random(60, 35, [13, 5], seed=7201, L=9.0)
    b = dfjk_inputs.make_random(60, 35, [13, 5], seed=7202, L=9.0)           # other orbitals, same shapes
    B, C, occ = device_inputs(torch, a)
    refs = []
    for inp in (a, b):
        _, Ci, oi = device_inputs(torch, inp)
        refs.append(handle_path(torch, pkg, inp, B, Ci, oi))
    J = torch.empty((2, 60, 60), dtype=torch.float64, device="cuda")
    K = torch.empty_like(J)
    pkg.small_jk_static(B, 60, a.nocc, C, occ, out_j=J, out_k=K)             # set-up happens here
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        pkg.small_jk_static(B, 60, a.nocc, C, occ, out_j=J, out_k=K, stream=torch.cuda.current_stream())
    for inp, (Jr, Kr) in ((b, refs[1]), (a, refs[0]), (b, refs[1])):
        _, Ci, oi = device_inputs(torch, inp)
        C.copy_(Ci)
        occ.copy_(oi)
        J.fill_(float("nan"))
        K.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(J, Jr) and torch.equal(K, Kr)
    del g


def test_static_scratch_entry_allocates_no_device_memory(torch_cuda):
    """free device memory as the driver reports it does not shrink over a call (after one warm-up call, which
    loads the kernel and looks up the address of the static array)"""
    torch = torch_cuda
    import paper_2505_03755_b200 as pkg
    inp = CASES["capped"]()
    B, C, occ = device_inputs(torch, inp)
    J, K = run_static(torch, pkg, inp, B, C, occ, fill=0.0)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        pkg.small_jk_static(B, inp.nao, list(inp.nocc), C, occ, out_j=J, out_k=K)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0


@pytest.mark.parametrize("nao,naux,nocc,word", [
    (97, 10, [4], "nao = 97"),                 # nao beyond 96
    (48, 10, [2] * 9, "nset = 9"),             # more than DFJK_STATIC_MAX_NSET sets
    (96, 10, [49], "nao * sum(nocc)"),         # 96 * 49 > 4608
    (96, 400, [24], "2^26"),                   # 400 * 96^2 * 25 > 2^26
    (48, 10, [0], "at least one occupied"),    # nothing to do is the caller's mistake here
    (48, 10, [49], "nocc[0]"),                 # more columns than rows
])
def test_static_scratch_entry_rejects_sizes_beyond_its_maximum(torch_cuda, nao, naux, nocc, word):
    torch = torch_cuda
    import paper_2505_03755_b200 as pkg
    B = torch.zeros((naux, nao * (nao + 1) // 2), dtype=torch.float64, device="cuda")
    C = torch.zeros(max(nao * sum(nocc), 1), dtype=torch.float64, device="cuda")
    occ = torch.ones(max(sum(nocc), 1), dtype=torch.float64, device="cuda")
    J = torch.full((len(nocc), nao, nao), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(pkg.DFJKError) as ei:
        pkg.small_jk_static(B, nao, nocc, C, occ, out_j=J)
    assert ei.value.code == 1 and word in str(ei.value), str(ei.value)
    torch.cuda.synchronize()
    assert bool((J == 7.0).all()), "a rejected call must not touch the outputs"
