#!/usr/bin/env python
"""bench.py -- DF get_jk milliseconds at nao=1200 / naux=4000 on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config large] [--impl reference]

A step is one pass of the whole hot path: one dfjk_get_jk producing J
and K of the `large` config (nao=1200, naux=4000, nocc=300, ~23 GB packed B resident in HBM).
`value` is the device-timed milliseconds per step with inputs resident; `e2e` is the same call
through dfjk_get_jk_host with pinned HOST buffers for C, occ, J, K (copies inside the timed
region; B stays resident as the paper prescribes).  `roofline` describes the
dominant kernel (the DMMA half-transform), `cpu_baseline` the oracle on the host cores on a
bounded sample of aux rows.  north_star names no sharding ("replicas only"): with
--gpus N every rank runs an independent replica and the max over ranks is reported; --shard-aux is the
opt-in, unmeasured aux-sharded mode (one all-reduce of the partial J, K).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import dfjk_inputs  # noqa: E402

METRIC = "DF get_jk ms at nao=1200/naux=4000; K FP64 TFLOP/s & J HBM GB/s vs peak"
# measured on this pool (profiles/r01_calib.md): DMMA.8x8x4 issue-rate peak, burst == sustained
FP64_DMMA_PEAK_TFLOPS = 37.1
FP64_CUBLAS_TFLOPS = 35.47
HBM_READ_STREAM_GBS = 7430.0
# ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum of k_half_transform<19,1> at `large`:
# 9.41 + 3.26 GB per 1122-aux-row launch (profiles/r02_ncu_large.md; the re-tiled Bt is 1.35x the packed bytes)
HT_DRAM_BYTES_PER_AUX_ROW_LARGE = 12.66e9 / 1122


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16=float(d["bf16_tflops"]),
                    bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), source="measured")
    return dict(hbm_gbs=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")


def flops_bytes(cfg):
    nao, naux = cfg["nao"], cfg["naux"]
    nocc_tot, nset = sum(cfg["nocc"]), len(cfg["nocc"])
    npair = nao * (nao + 1) // 2
    ht = 2.0 * naux * nao * nao * nocc_tot
    syrk = 1.0 * naux * nao * (nao + 1) * nocc_tot
    jbytes = 2.0 * naux * npair * 8 + nset * (2 * npair + 2 * naux) * 8.0
    return dict(ht=ht, syrk=syrk, k=ht + syrk, j_bytes=jbytes, j_flops=4.0 * naux * npair * nset,
                b_bytes=naux * npair * 8.0)


class ClockSampler:
    """nvidia-smi clock / throttle-reason sampler running during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0, power_w_max=None)
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            t = [x.strip() for x in line.split(",")]
            if len(t) < 7:
                continue
            try:
                sm.append(float(t[0])); smax.append(float(t[1])); pw.append(float(t[2]))
            except ValueError:
                continue
            for n, v in zip(names, t[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(smax)), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=float(max(pw)))
        return out


class Ranks:
    """One process per GPU, replicas only: the only cross-rank traffic is the
    barrier around the timed region and the max over ranks of the device time.  backend "nccl" on
    the GPU box; "gloo" with device=None runs the same logic on CPU (tests/test_multirank_cpu.py)."""

    def __init__(self, backend: str = "nccl", device=None):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.device = device
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            kw = {"device_id": device} if device is not None else {}
            dist.init_process_group(backend, **kw)
            self.dist = dist

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()
        if self.device is not None:
            import torch
            torch.cuda.synchronize()

    def max_over_ranks(self, x: float) -> float:
        if self.dist is None:
            return x
        import torch
        t = torch.tensor([x], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()
            self.dist = None


def upload_B(torch, cfg, keep_host: bool):
    """Generate packed B on the host in row chunks (the canonical recipe) and upload it."""
    nao, naux, L, k = cfg["nao"], cfg["naux"], cfg["L"], cfg["k"]
    npair = dfjk_inputs.npair_of(nao)
    Bd = torch.empty((naux, npair), dtype=torch.float64, device="cuda")
    env = dfjk_inputs.gen.decay_envelope(nao, naux, L)
    rng = np.random.default_rng(1000 + k)
    Bh = np.empty((naux, npair)) if keep_host else None
    rows = max(1, min(naux, (1 << 28) // npair))          # ~2 GiB chunks
    stage = torch.empty((rows, npair), dtype=torch.float64).pin_memory()
    sv = stage.numpy()
    for r0 in range(0, naux, rows):
        r1 = min(naux, r0 + rows)
        torch.cuda.synchronize()                           # the previous async copy has left `stage`
        rng.standard_normal(out=sv[: r1 - r0])
        sv[: r1 - r0] *= env
        if keep_host:
            Bh[r0:r1] = sv[: r1 - r0]
        Bd[r0:r1].copy_(stage[: r1 - r0], non_blocking=True)
    torch.cuda.synchronize()
    return Bd, Bh


def oracle_sample_time(cfg, C, occ, Bh_rows, target_s: float):
    """Time the oracle (as it stands) on a bounded sample: the first R aux rows of the workload.
    Returns (seconds, R).  R is calibrated from a 2-row probe to land near target_s."""
    import oracle
    nao = cfg["nao"]
    t0 = time.perf_counter()
    oracle.get_jk(Bh_rows[:2], nao, C, occ)
    per_row = (time.perf_counter() - t0) / 2
    R = int(max(2, min(Bh_rows.shape[0], target_s / max(per_row, 1e-9))))
    t0 = time.perf_counter()
    oracle.get_jk(Bh_rows[:R], nao, C, occ)
    return time.perf_counter() - t0, R


def run_reference(args, cfg, name):
    """--impl reference: the CPU oracle on the host cores, bounded sample per step (rank 0 only)."""
    import oracle
    if int(os.environ.get("RANK", "0")) != 0:
        return
    C, occ = dfjk_inputs.make_orbitals(name)
    nao, naux = cfg["nao"], cfg["naux"]
    probe_rows = min(naux, 64)
    Bh = dfjk_inputs.make_B_packed(nao, naux, cfg["L"], 1000 + cfg["k"], rows=probe_rows)
    t0 = time.perf_counter()
    oracle.get_jk(Bh[:2], nao, C, occ)
    per_row = (time.perf_counter() - t0) / 2
    R = int(max(2, min(probe_rows, 4.0 / max(per_row, 1e-9))))      # ~4 s of CPU work per step
    for _ in range(args.warmup):
        oracle.get_jk(Bh[:2], nao, C, occ)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.get_jk(Bh[:R], nao, C, occ)
    dt = (time.perf_counter() - t0) / args.steps
    ms_full = dt * 1e3 * naux / R
    sample = f"first {R} of {naux} aux rows per step, time scaled by {naux}/{R} (cost is linear in aux rows)"
    line = {
        "impl": "reference", "metric": METRIC, "value": ms_full, "unit": "ms", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_full, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "nao": nao, "naux": naux, "nocc": cfg["nocc"], "sample": sample},
        "cpu_baseline": {"value": ms_full, "unit": "ms", "cores": oracle.num_threads(),
                         "kind": f"oracle, extrapolated from {R} of {naux} aux rows", "sample": sample},
        "e2e": {"value": ms_full, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="large", choices=list(dfjk_inputs.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-parity", action="store_true", help="skip the sampled parity check")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=20.0)
    ap.add_argument("--shard-aux", action="store_true",
                    help="with --gpus N > 1: shard the aux rows over the ranks and sum-all-reduce J, K (strong scaling) "
                         "instead of N independent replicas")
    ap.add_argument("--no-small-calls", action="store_true", help="skip the small-call (CUDA graph) section")
    ap.add_argument("--no-emulated", action="store_true", help="skip the opt-in FP64-emulated K path (int8 tensor cores) section")
    ap.add_argument("--no-dm-form", action="store_true", help="skip the density-matrix-form (Eq. 16-17 as printed) section")
    ap.add_argument("--no-ao2mo", action="store_true", help="skip the AO2MO (Eq. 18-21) section")
    ap.add_argument("--workspace-gib", type=float, default=0.0, help="dfjk_options.workspace_cap_bytes (0 = default)")
    args = ap.parse_args()
    name = args.config
    cfg = dfjk_inputs.CONFIGS[name]
    if args.impl == "reference":
        run_reference(args, cfg, name)
        return

    import torch
    import paper_2505_03755_b200 as dfjk          # raises if libdfjk.so is missing: no CPU fallback
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (B200); there is no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    ranks = Ranks("nccl", torch.device("cuda", local))
    barrier, max_over_ranks = ranks.barrier, ranks.max_over_ranks

    nao, naux, nocc = cfg["nao"], cfg["naux"], cfg["nocc"]
    nset = len(nocc)
    fb = flops_bytes(cfg)
    lead = rank == 0
    want_host_B = lead and world == 1 and not (args.no_parity and args.no_cpu_baseline)
    t_gen = time.perf_counter()
    Bd, Bh = upload_B(torch, cfg, keep_host=want_host_B)
    shard = args.shard_aux and world > 1
    if shard:
        from paper_2505_03755_b200.sharded import AuxShardedJK, aux_range
        lo, hi = aux_range(naux, rank, world)
        Bd = Bd[lo:hi].clone()                     # this rank's contiguous aux rows
        torch.cuda.empty_cache()
        fb = flops_bytes(dict(cfg, naux=hi - lo))  # per-kernel rooflines are per rank
        args.no_ao2mo = True
    t_gen = time.perf_counter() - t_gen
    C_list, occ_list = dfjk_inputs.make_orbitals(name)
    C_host = torch.from_numpy(np.concatenate([c.ravel() for c in C_list])).pin_memory()
    occ_host = torch.from_numpy(np.concatenate(occ_list)).pin_memory()
    C_dev, occ_dev = C_host.cuda(), occ_host.cuda()
    J = torch.empty((nset, nao, nao), dtype=torch.float64, device="cuda")
    K = torch.empty_like(J)
    J_host = torch.empty((nset, nao, nao), dtype=torch.float64).pin_memory()
    K_host = torch.empty_like(J_host).pin_memory()

    h = dfjk.DFJK(Bd, nao, workspace_cap_bytes=int(args.workspace_gib * (1 << 30)))
    stream = torch.cuda.current_stream()

    def timed(fn, steps):
        """device milliseconds per step over exactly `steps` calls, events on the launching stream"""
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        for _ in range(steps):
            fn()
        e1.record(stream)
        barrier()
        return e0.elapsed_time(e1) / steps

    full = lambda: h.get_jk_raw(nocc, C_dev, occ_dev, out_j=J, out_k=K, stream=stream)
    if shard:
        local_full = full
        full = lambda: AuxShardedJK(local_full, None).get_jk()   # partial J, K + one NCCL sum all-reduce each
    j_only = lambda: h.get_jk_raw(nocc, C_dev, occ_dev, with_k=False, out_j=J, stream=stream)
    k_only = lambda: h.get_jk_raw(nocc, C_dev, occ_dev, with_j=False, out_k=K, stream=stream)
    host = lambda: h.get_jk_host(nocc, C_host, occ_host, J_host, K_host, stream=stream)

    for _ in range(args.warmup):
        full()
    barrier()

    # ---- the timed region: exactly K steps of the whole path, clocks sampled meanwhile
    h.set_profiling(True)
    phases = {p: [0.0, 0] for p in dfjk.api.PHASES}
    launches = 0
    clocks = ClockSampler(local)
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    marks[0].record(stream)
    for i in range(args.steps):
        full()
        marks[i + 1].record(stream)
        launches += h.last_launch_count
        for p, (ms, n) in h.profile().items():     # waits for this step's last event only
            phases[p][0] += ms
            phases[p][1] += n
    barrier()
    ms_step = max_over_ranks(marks[0].elapsed_time(marks[-1]) / args.steps)     # mean over exactly K steps
    per_step = [marks[i].elapsed_time(marks[i + 1]) for i in range(args.steps)]
    ms_median = max_over_ranks(float(np.median(per_step)))
    ms_best = max_over_ranks(float(min(per_step)))
    clk = clocks.stop()
    h.set_profiling(False)
    plan = h.plan()

    # ---- the same call through the host-buffer entry point (H2D of C/occ, D2H of J/K inside)
    for _ in range(2):
        host()
    t0 = time.perf_counter()
    ms_e2e_dev = timed(host, args.steps)
    ms_e2e_wall = (time.perf_counter() - t0) * 1e3 / args.steps
    ms_e2e = max_over_ranks(max(ms_e2e_dev, ms_e2e_wall))
    h2d = int(C_host.numel() * 8 + occ_host.numel() * 8)
    d2h = int(2 * J_host.numel() * 8)

    # ---- J pass and K path alone (K_out = NULL / J_out = NULL), for the two rooflines
    nrep = max(3, min(args.steps, 5))
    j_only(); k_only()
    ms_j = max_over_ranks(timed(j_only, nrep))
    ms_k = max_over_ranks(timed(k_only, nrep))
    h.set_profiling(True)                       # phases of the two-pass J (the fused call has no pass 1)
    j_only()
    jprof = h.profile()
    h.set_profiling(False)
    j1_only_ms, j2_only_ms = jprof["j1"][0], jprof["j2"][0]
    # ---- signed occupations (differences of densities): the same call with every
    # third occupation negated must cost what the unsigned call costs
    occ_signed = occ_dev.clone()
    occ_signed[::3] *= -1.0
    signed = lambda: h.get_jk_raw(nocc, C_dev, occ_signed, out_j=J, out_k=K, stream=stream)
    signed()
    ms_signed = max_over_ranks(timed(signed, nrep))
    ms_unsigned = max_over_ranks(timed(full, nrep)) if not shard else ms_step

    # ---- AO2MO (Eq. 18-21) on the same resident B: an embedding-sized MO set
    ao = None
    if not args.no_ao2mo:
        nmo = min(nao, sum(nocc) + (40 if name in ("large", "medium", "small") else 0))
        nact = min(8, nmo)
        a0 = nmo - nact if name != "lasscf" else nocc[0]
        Q = dfjk_inputs.make_orbitals(name, all_columns=True)
        M_host = np.ascontiguousarray(Q[:, :nmo])
        M_dev = torch.from_numpy(M_host).cuda()
        ao_fn = lambda: h.ao2mo(M_dev, a0, nact, stream=stream)
        outs = ao_fn()
        torch.cuda.synchronize()
        ao_launches = h.last_launch_count
        ao_route = h.last_ao2mo_route
        del outs
        ms_ao = max_over_ranks(timed(lambda: ao_fn() and None, max(2, min(args.steps, 3))))
        h.set_profiling(True)                       # Eq. 18 (the thin half-transform of the active-first route) alone
        ao_fn()
        aprof = h.profile()
        h.set_profiling(False)
        ht_ao_ms = aprof["half_transform"][0]
        ht_ao_bytes = naux * (nao * (nao + 1) // 2 * 8.0 + nao * 8 * 8.0)
        ao_flops = (2.0 * naux * nao * nao * nmo + 2.0 * naux * nao * nmo * nmo
                    + 2.0 * naux * nmo * nmo * nact * nact + 2.0 * naux * (nmo * nact) ** 2)
        ntri = nact * (nact + 1) // 2
        ao_exec = (2.0 * naux * nao * nao * nact + 2.0 * naux * nao * nmo * nact + 2.0 * naux * (nao * (nao + 1) // 2) * ntri
                   + 2.0 * nao * nmo * ntri * (nao + nmo) + 1.0 * naux * (nmo * nact) ** 2) if ao_route == 2 else ao_flops
        ao = {"ms": ms_ao, "nmo": nmo, "a0": a0, "nact": nact, "launches_per_call": ao_launches,
              "route": {1: "Eq. 18-21 in the printed order", 2: "active first (bmo never formed)"}.get(ao_route, "?"),
              "eq18_ms": ht_ao_ms, "contractions_ms": aprof["syrk"][0],
              "eq18_gbs": (ht_ao_bytes / (ht_ao_ms * 1e-3) * 1e-9) if (ao_route == 2 and nact <= 8 and ht_ao_ms > 0) else None,
              "eq18_note": "active-first route with <= 8 active columns: one pass over the packed triangle (k_symm_thin), "
                           "algorithmic bytes = packed B once + Z; HBM-bound",
              "executed_flops": ao_exec, "executed_tflops": ao_exec / (ms_ao * 1e-3) * 1e-12,
              "frac_of_fp64_peak": ao_exec / (ms_ao * 1e-3) * 1e-12 / FP64_DMMA_PEAK_TFLOPS,
              "algorithmic_flops_as_printed": ao_flops,
              "flops_note": "executed_* (and the fraction) count what the chosen route really computes; "
                            "algorithmic_flops_as_printed counts Eq. 18 + Eq. 19 (full square) + Eq. 20 + Eq. 21 in the "
                            "printed order, which the active-first route avoids"}
    # ---- the density-matrix form (Eq. 14-17 exactly as printed) on the first set's
    # density D = C n C^T, checked against the C-form result of the same density
    dmf = None
    if not args.no_dm_form and not shard:
        n0 = nocc[0]
        C0 = C_dev[: nao * n0].view(nao, n0)
        D_dev = ((C0 * occ_dev[:n0]) @ C0.T).contiguous()[None]      # input construction only
        Jd = torch.empty((1, nao, nao), dtype=torch.float64, device="cuda")
        Kd = torch.empty_like(Jd)
        dm_fn = lambda: h.get_jk_dm(D_dev, out_j=Jd, out_k=Kd, stream=stream)
        dm_fn()
        torch.cuda.synchronize()
        dm_launches = h.last_launch_count
        ms_dm = max_over_ranks(timed(dm_fn, 2))
        full()
        torch.cuda.synchronize()
        dm_flops = 2.0 * naux * nao * nao * nao + 1.0 * naux * nao * (nao + 1) * nao
        dmf = {"ms": ms_dm, "launches_per_call": dm_launches, "algorithmic_flops": dm_flops,
               "tflops": dm_flops / (ms_dm * 1e-3) * 1e-12,
               "frac_of_fp64_peak": dm_flops / (ms_dm * 1e-3) * 1e-12 / FP64_DMMA_PEAK_TFLOPS,
               "max_rel_diff_vs_c_form_J": float((Jd[0] - J[0]).abs().max() / J[0].abs().max()),
               "max_rel_diff_vs_c_form_K": float((Kd[0] - K[0]).abs().max() / K[0].abs().max()),
               "flops_note": "Eq. 16 (2 naux nao^3) + Eq. 17 on the lower triangle (naux nao^2 (nao+1))"}
        del D_dev, Jd, Kd
    # ---- the many-small-calls regime of the embedded fragments:
    # the `small` config called directly and as a replayed CUDA graph (dfjk_get_jk only enqueues)
    # ---- opt-in FP64 emulation of the K path on the int8 tensor cores:
    # the same call on a second handle, error of K against the native fp64 result over every element
    emulated = None
    if not args.no_emulated and not shard:
        full()
        torch.cuda.synchronize()
        K_native = K.clone()
        emulated = []
        for ht_s, k_s in ((6, 6), (5, 5)):
            he = dfjk.DFJK(Bd, nao, ht_emulation_slices=ht_s, k_emulation_slices=k_s,
                           workspace_cap_bytes=int(args.workspace_gib * (1 << 30)))
            Je, Ke = torch.empty_like(J), torch.empty_like(K)
            e_full = lambda: he.get_jk_raw(nocc, C_dev, occ_dev, out_j=Je, out_k=Ke, stream=stream)
            e_konly = lambda: he.get_jk_raw(nocc, C_dev, occ_dev, with_j=False, out_k=Ke, stream=stream)
            for _ in range(2):
                e_full()
            ms_e = max_over_ranks(timed(e_full, nrep))
            ms_ek = max_over_ranks(timed(e_konly, nrep))
            he.set_profiling(True)
            e_full()
            ep = he.profile()
            he.set_profiling(False)
            errs = [float((Ke[s_] - K_native[s_]).abs().max() / K_native[s_].abs().max()) for s_ in range(nset)]
            emulated.append({"ht_slices": ht_s, "syrk_slices": k_s, "ms": ms_e, "k_path_ms": ms_ek,
                             "half_transform_ms": ep["half_transform"][0], "syrk_ms": ep["syrk"][0],
                             "launches_per_call": he.last_launch_count, "plan": he.plan(),
                             "equivalent_fp64_tflops": fb["k"] / (ms_ek * 1e-3) * 1e-12,
                             "max_rel_err_K_vs_native_every_element": max(errs),
                             "kernels": "tcgen05.mma kind::i8 (UTCIMMA), TMEM int32 accumulators, bulk-copied core-matrix images"})
            he.close()
            del Je, Ke
        del K_native
        torch.cuda.empty_cache()
    small = None
    if not args.no_small_calls:
        small = {}
        # the two small configs of BASELINE.json and one fragment-sized call with two sets (nao 80, naux 300: the
        # embedding-sized regime of PAPER.md:84-86 between them)
        frag = dict(nao=80, naux=300, nocc=[10, 8])
        for sname in ("tiny", "fragment", "small"):
            sinp = (dfjk_inputs.make_random(frag["nao"], frag["naux"], frag["nocc"], seed=8080, L=12.0)
                    if sname == "fragment" else dfjk_inputs.make_config(sname))
            sB = torch.from_numpy(sinp.B_packed).cuda()
            sC = torch.from_numpy(sinp.C_concat()).cuda()
            socc = torch.from_numpy(sinp.occ_concat()).cuda()
            sJ = torch.empty((sinp.nset, sinp.nao, sinp.nao), dtype=torch.float64, device="cuda")
            sK = torch.empty_like(sJ)
            hs = dfjk.DFJK(sB, sinp.nao)
            s_fn = lambda: hs.get_jk_raw(sinp.nocc, sC, socc, out_j=sJ, out_k=sK, stream=stream)
            for _ in range(3):
                s_fn()
            torch.cuda.synchronize()
            s_launches = hs.last_launch_count
            ms_direct = max_over_ranks(timed(s_fn, 100))
            cap = torch.cuda.Stream()
            cap.wait_stream(stream)
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.stream(cap):
                with torch.cuda.graph(graph, stream=cap):
                    hs.get_jk_raw(sinp.nocc, sC, socc, out_j=sJ, out_k=sK, stream=cap)
            stream.wait_stream(cap)
            graph.replay()
            torch.cuda.synchronize()
            ms_graph = max_over_ranks(timed(graph.replay, 100))
            sfb = flops_bytes(frag if sname == "fragment" else dfjk_inputs.CONFIGS[sname])
            small[sname] = {"nao": sinp.nao, "naux": sinp.naux, "nocc": sinp.nocc, "l2": "L2-warm",
                            "launches_per_call": s_launches, "ms_direct": ms_direct, "ms_cuda_graph": ms_graph,
                            "k_tflops_graph": sfb["k"] / (ms_graph * 1e-3) * 1e-12}
            del graph
            hs.close()
            if s_launches == 1:
                # the single-launch path (csrc/small.cu) served this call: the tiled kernels for comparison
                ht_ = dfjk.DFJK(sB, sinp.nao, no_small_path=True)
                t_fn = lambda: ht_.get_jk_raw(sinp.nocc, sC, socc, out_j=sJ, out_k=sK, stream=stream)
                for _ in range(3):
                    t_fn()
                torch.cuda.synchronize()
                small[sname]["path"] = "single launch (small.cu)"
                small[sname]["tiled_kernels_launches_per_call"] = ht_.last_launch_count
                small[sname]["tiled_kernels_ms_direct"] = max_over_ranks(timed(t_fn, 100))
                ht_.close()
                # the allocation-free entry point (same kernel on the library's static scratch; one 8-byte memset more)
                n_fn = lambda: dfjk.small_jk_static(sB, sinp.nao, sinp.nocc, sC, socc, out_j=sJ, out_k=sK, stream=stream)
                for _ in range(3):
                    n_fn()
                torch.cuda.synchronize()
                small[sname]["static_scratch_ms_direct"] = max_over_ranks(timed(n_fn, 100))
    if not lead:
        h.close()
        ranks.close()
        return
    pk = measured_peaks()
    npair_bytes = nao * (nao + 1) // 2 * 8.0
    ht_ms, ht_n = phases["half_transform"]
    sy_ms, sy_n = phases["syrk"]
    ht_tflops = fb["ht"] * args.steps / (ht_ms * 1e-3) * 1e-12 if ht_ms > 0 else 0.0
    sy_tflops = fb["syrk"] * args.steps / (sy_ms * 1e-3) * 1e-12 if sy_ms > 0 else 0.0
    line = {
        "metric": METRIC, "value": ms_step, "unit": "ms", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "ms_per_step_median": ms_median, "ms_per_step_best": ms_best,
        "higher_is_better": False,
        "scaling": "strong" if shard else "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "nao": nao, "naux": naux, "nset": nset, "nocc": nocc,
                   "B_packed_GB": fb["b_bytes"] * 1e-9, "parallelism": ("aux-sharded + all-reduce" if shard else "replicas only") if world > 1 else "1 gpu",
                   "l2": "inputs (packed B) far larger than the 126 MB L2, no flush needed" if fb["b_bytes"] > 1e9
                         else "L2-warm (inputs fit the L2)",
                   "plan": plan, "input_gen_s": round(t_gen, 1)},
        "clocks": {"sm_mhz": clk["sm_mhz"], "sm_max_mhz": clk["sm_max_mhz"], "reasons": clk["reasons"],
                   "samples": clk["samples"], "power_w_max": clk["power_w_max"]},
        "e2e": {"value": ms_e2e, "unit": "ms", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "api": "dfjk_get_jk_host (pinned C, occ, J, K; B resident)"},
        "gpu_launches": launches,
        "roofline": {"kernel": "k_half_transform", "bound": "tensor", "achieved": ht_tflops,
                     "peak": FP64_DMMA_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": ht_tflops / FP64_DMMA_PEAK_TFLOPS,
                     "traffic": (HT_DRAM_BYTES_PER_AUX_ROW_LARGE * naux * args.steps / max(ht_n, 1)
                                 if (nao, sum(nocc)) == (1200, 300) else None),
                     "traffic_unit": "bytes per launch (constant from one ncu --set full capture: dram read + write, profiles/r02_ncu_large.md)",
                     "algorithmic_bytes_per_launch": (npair_bytes + nao * sum(nocc) * 8.0) * naux * args.steps / max(ht_n, 1),
                     "launches": ht_n, "avg_launch_ms": ht_ms / max(ht_n, 1),
                     "algorithmic_flops_per_step": fb["ht"],
                     "peak_source": "measured DMMA.8x8x4 issue-rate peak on this pool (profiles/r01_calib.md); "
                                    "cuBLAS fp64 8192^3 reaches %.2f; MEASURED_PEAKS bf16 %.1f x nominal 45/2250 = %.1f"
                                    % (FP64_CUBLAS_TFLOPS, pk["bf16"], pk["bf16"] * 45.0 / 2250.0)},
        "k_path": {"ms": ms_k, "tflops": fb["k"] / (ms_k * 1e-3) * 1e-12,
                   "frac_of_fp64_peak": fb["k"] / (ms_k * 1e-3) * 1e-12 / FP64_DMMA_PEAK_TFLOPS,
                   "half_transform_tflops": ht_tflops, "syrk_tflops": sy_tflops,
                   "algorithmic_flops": fb["k"]},
        "j_pass": {"ms": ms_j, "gbs": fb["j_bytes"] / (ms_j * 1e-3) * 1e-9,
                   "frac_of_measured_hbm": fb["j_bytes"] / (ms_j * 1e-3) * 1e-9 / pk["hbm_gbs"],
                   "frac_of_8TBs": fb["j_bytes"] / (ms_j * 1e-3) * 1e-9 / 8000.0,
                   "pass1_gbs": fb["b_bytes"] / (j1_only_ms * 1e-3) * 1e-9 if j1_only_ms > 0 else None,
                   "pass2_gbs": fb["b_bytes"] / (j2_only_ms * 1e-3) * 1e-9 if j2_only_ms > 0 else None,
                   "pass_note": "per-pass GB/s from the event profile of one J-only (two-pass) call",
                   "algorithmic_bytes": fb["j_bytes"], "hbm_peak_source": pk["source"]},
        "signed_occ": {"ms": ms_signed, "ms_unsigned": ms_unsigned, "ratio": ms_signed / ms_unsigned,
                       "note": "same call with every third occupation negated (C' = C sqrt|occ|, sign-bit flip in the SYRK)"},
        "phases_ms_per_step": {p: v[0] / args.steps for p, v in phases.items()},
    }

    if emulated is not None:
        line["k_emulated"] = emulated
    if small is not None:
        line["small_calls"] = small
    if dmf is not None:
        line["dm_form"] = dmf
    if ao is not None:
        line["ao2mo"] = ao
        if Bh is not None and not args.no_parity:
            import oracle
            bpa, ppaa, papa = h.ao2mo(M_dev, ao["a0"], ao["nact"], stream=stream)
            torch.cuda.synchronize()
            rows = [0, naux - 1]
            o_bpa, _, _ = oracle.ao2mo(Bh[rows], nao, M_host, ao["a0"], ao["nact"])
            g_bpa = bpa[rows].cpu().numpy()
            nm, na = ao["nmo"], ao["nact"]
            smp = [(0, 0, 0, 0), (nm - 1, nm // 2, na - 1, 0), (nm // 3, nm - 1, na // 2, na - 1), (ao["a0"], 1, 1, 1)]
            v20, v21 = oracle.ao2mo_sample(Bh, nao, M_host, ao["a0"], na, smp)
            s20, s21 = float(ppaa.abs().max()), float(papa.abs().max())
            e20 = max(abs(float(ppaa[p1, p2, a1, a2]) - v20[t]) / s20 for t, (p1, p2, a1, a2) in enumerate(smp))
            e21 = max(abs(float(papa[p1, a1, p2, a2]) - v21[t]) / s21 for t, (p1, p2, a1, a2) in enumerate(smp))
            ao["parity"] = {"kind": "oracle.ao2mo bpa of aux rows 0 and naux-1 (Eq. 18-19), every element; "
                                    "oracle.ao2mo_sample on %d elements of ppaa and papa (Eq. 20-21)" % len(smp),
                            "max_rel_err": float(np.abs(g_bpa - o_bpa).max() / np.abs(o_bpa).max()),
                            "max_rel_err_ppaa": float(e20), "max_rel_err_papa": float(e21), "tolerance": 1e-10}
            del bpa, ppaa, papa
    if Bh is not None and not args.no_parity:
        import oracle
        torch.cuda.synchronize()
        rs = np.random.default_rng(7)
        samples = [(int(rs.integers(nset)), int(rs.integers(nao)), int(rs.integers(nao))) for _ in range(4)]
        samples += [(0, 0, 0), (nset - 1, nao - 1, nao - 1), (0, nao - 1, 0), (0, min(127, nao - 1), min(128, nao - 1))]
        t0 = time.perf_counter()
        Jv, Kv = oracle.sample(Bh, nao, C_list, occ_list, samples)
        Jg, Kg = J.cpu().numpy(), K.cpu().numpy()
        ej = max(abs(Jg[s, m, n] - Jv[t]) / np.abs(Jg[s]).max() for t, (s, m, n) in enumerate(samples))
        ek = max(abs(Kg[s, m, n] - Kv[t]) / np.abs(Kg[s]).max() for t, (s, m, n) in enumerate(samples))
        line["parity"] = {"kind": "oracle.sample on %d elements" % len(samples), "max_rel_err_J": float(ej),
                          "max_rel_err_K": float(ek), "tolerance": 1e-10, "ok": bool(ej <= 1e-10 and ek <= 1e-10),
                          "seconds": round(time.perf_counter() - t0, 1)}
    if Bh is not None and not args.no_cpu_baseline:
        import oracle
        secs, R = oracle_sample_time(cfg, C_list, occ_list, Bh, args.cpu_seconds)
        line["cpu_baseline"] = {"value": secs * 1e3 * naux / R, "unit": "ms", "cores": oracle.num_threads(),
                                "kind": f"oracle, extrapolated from {R} of {naux} aux rows",
                                "sample": f"first {R} of {naux} aux rows in {secs:.1f} s, scaled by {naux}/{R} "
                                          "(the oracle's cost is linear in aux rows)"}
    print(json.dumps(line), flush=True)
    h.close()
    ranks.close()


if __name__ == "__main__":
    main()
