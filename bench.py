#!/usr/bin/env python
"""bench.py -- H|psi> applies/s (complex128) and achieved HBM GB/s vs the measured B200 peak.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]
                    [--per-config q12,q24,...|none] [--sharded]

Headline workload (config.workload): BASELINE.json configs[2], the 28-qubit Fermi-Hubbard chain
(sector dim 11,778,624; 188.5 MB per vector, larger than the 126 MB L2, so no L2 flush is needed).
A "step" is one pass of the hot path over one state vector: one order-12 shifted Taylor step of
exp(-i H dt) (a7: 12 fused apply+axpby launches of the a4 kernel, terms accumulated in pairs) followed by one fused energy
(a5: bs_expect) = 13 H applications.  a1-a3 (grouping, sector tables) are built once per operator and
reported as setup_ms; a6 (rotations) is timed in the q24 entry of `per_config`.
value = H applications per second over all ranks (each rank propagates its own state: weak scaling,
no data-path collective).  See DESIGN.md "Measurement" for the byte counts behind `roofline`.
With --workload q12 | q24 | q32 | q56 (molecular configs) a step is one bs_apply + one bs_expect = 2 H applications
 and `roofline` is reported against the FP64 pipe, which is what binds them.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import synth_inputs as si  # noqa: E402

SMEM_PEAK_TBS = 128 * 148 * 1.965e9 / 1e12        # shared-memory / L1 data path: 128 B/clk/SM
DFMA_PEAK = 64 * 148 * 1.965e9                     # FP64 pipe: 64 DFMA/clk/SM, measured (profiles/r02_fp64_peak.md)
METRIC = "H|psi> applies/s (fp64 complex)"
UNIT = "applies/s"
TAYLOR_ORDER = 12
DT = 0.05


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc = index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])), mx.append(float(f[1])), pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def build_operator(name: str, bs):
    """a1 + a2 on the device, fed by the device-side JW construction (bs_jw_*): returns (op, raw term count)."""
    cfg = si.CONFIGS[name]
    if cfg.kind == "hubbard":
        L = cfg.n_orb
        return bs.bs_jw_hubbard(L, cfg.hubbard_t, cfg.hubbard_u), (L - 1) * 16 + L * 16
    h, g = si.integrals(cfg.n_orb, cfg.seed_ints)
    n = cfg.n_orb
    return bs.bs_jw_molecular(h, g), 8 * n * n + 64 * n ** 4


def nnz_per_row(cfg) -> int:
    """Non-zeros per row of a molecular H in the sector for generic integrals (closed form)."""
    from math import comb
    oa, va, ob, vb = cfg.n_alpha, cfg.n_orb - cfg.n_alpha, cfg.n_beta, cfg.n_orb - cfg.n_beta
    return 1 + oa * va + ob * vb + comb(oa, 2) * comb(va, 2) + comb(ob, 2) * comb(vb, 2) + oa * va * ob * vb


def table_bytes(op) -> int:
    """Group-table bytes of the a2 layout: xg u64[G] + offs i64[G+1] + z u64[M] + w c128[M]."""
    return 8 * op.n_groups + 8 * (op.n_groups + 1) + 24 * op.n_terms


def _median(v):
    return float(np.median(np.asarray(v, dtype=np.float64)))


def per_config_entry(name: str, bs, torch, peak_gbs: float, flush_buf, with_cpu: bool = False):
    """Plain bs_apply / bs_expect timings of one BASELINE.json config (CUDA events, median)."""
    cfg = si.CONFIGS[name]
    t0 = time.perf_counter()
    op, m_raw = build_operator(name, bs)
    sec = bs.bs_sector_build(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t0
    psi = torch.from_numpy(si.random_state(cfg.dim, cfg.seed_psi)).cuda()
    out = torch.empty_like(psi)
    flush = 16 * cfg.dim * 2 < 126e6                      # both vectors would sit in the 126 MB L2
    ev = lambda: torch.cuda.Event(enable_timing=True)     # noqa: E731
    a, b = ev(), ev()
    a.record()
    bs.bs_apply(op, sec, psi, out)                         # first call also builds the cached plan
    b.record()
    torch.cuda.synchronize()
    first_ms = a.elapsed_time(b)
    reps = 0 if first_ms > 30000 else (2 if first_ms > 2000 else (3 if first_ms > 500 else 10))
    times = []
    for _ in range(reps):
        if flush:
            flush_buf.zero_()
        a, b = ev(), ev()
        a.record()
        bs.bs_apply(op, sec, psi, out)
        b.record()
        torch.cuda.synchronize()
        times.append(a.elapsed_time(b))
    apply_ms = _median(times) if times else first_ms
    ent = {"n_qubits": cfg.n_qubits, "dim": cfg.dim, "groups": op.n_groups, "strings": op.n_terms,
           "plan": bs.bs_plan_describe(op, sec), "plan_info": bs.bs_plan_info(op, sec),
           "raw_terms": m_raw, "setup_s": round(t_setup, 3),
           "plan_build_ms": max(0.0, first_ms - apply_ms) if times else None,    # first call builds the cached plan
           "apply_ms": apply_ms, "applies_per_s": 1e3 / apply_ms, "reps": max(reps, 1),
           "l2_flush_between_reps": bool(flush)}
    if cfg.kind == "molecular":       # non-zeros per row of H in the sector for generic integrals
        ent["nonzeros_per_s"] = nnz_per_row(cfg) * cfg.dim / (apply_ms * 1e-3)
        ent["gather_gbs"] = 16 * ent["nonzeros_per_s"] / 1e9      # 16-byte amplitude gathers through L2 / shared memory
        # Resources that bind these configs: one 16-byte amplitude per non-zero through the
        # shared-memory / L1 path (128 B/clk/SM) and 2 DFMA per non-zero (real weight x complex amplitude) on the FP64
        # pipe (64 DFMA/clk/SM measured, profiles/r02_fp64_peak.md); SM clock from MEASURED_PEAKS (1965 MHz).
        ent["binding"] = {
            "smem_gather": {"achieved_tbs": ent["gather_gbs"] / 1e3, "peak_tbs": SMEM_PEAK_TBS,
                            "frac": ent["gather_gbs"] / 1e3 / SMEM_PEAK_TBS,
                            "note": "16 B x non-zeros/s against 128 B/clk/SM x 148 SMs x 1.965 GHz; the K-resolved kernel "
                                    "gathers once per n - N_beta + 1 non-zeros, so this is an equivalent rate"},
            "fp64": {"useful_dfma_per_s": 2 * ent["nonzeros_per_s"], "peak_dfma_per_s": DFMA_PEAK,
                     "frac": 2 * ent["nonzeros_per_s"] / DFMA_PEAK}}
    bytes_alg = 32 * cfg.dim + table_bytes(op)
    ent["hbm_gbs_algorithmic"] = bytes_alg / apply_ms / 1e6
    ent["hbm_frac_of_measured_peak"] = ent["hbm_gbs_algorithmic"] / peak_gbs
    ent["traffic_ncu"] = TRAFFIC_NCU.get(name)
    if reps:
        bs.bs_expect(op, sec, psi)                         # first call may allocate library scratch
        t0 = time.perf_counter()
        e = bs.bs_expect(op, sec, psi)
        ent["expect_ms"] = (time.perf_counter() - t0) * 1e3
        ent["energy"] = e.real
    if name in ("q24", "q32"):
        # a6: first-order Trotterised UCCSD state preparation (Eq. 39), generator order of reading U10.
        # A run = consecutive generators with one alpha mask (or all with x_b = 0): ONE launch; the floor of a run is one
        # read + write of the state vector.  q24: cells in shared memory; q32: cells in place (L2), see DESIGN.md 5.2.
        from paper_2606_28952_b200 import jw_terms as jw
        ex = si.uccsd_excitations(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
        th = si.thetas(len(ex), cfg.seed_theta or 3004)
        X, Z, Cc, offs = jw.excitation_generator_terms(ex)
        gens = bs.bs_group_xmask(X, Z, Cc, cfg.n_qubits, 0.0, bs.BS_MODE_SEQUENCE, offs)
        rt, launches = [], 0
        for i in range(3):
            psi.zero_()
            psi[0] = 1.0
            a, b = ev(), ev()
            n0 = bs.bs_launch_count()
            a.record()
            bs.bs_apply_pauli_rotations(gens, sec, th, psi)
            b.record()
            torch.cuda.synchronize()
            launches = bs.bs_launch_count() - n0
            if i:
                rt.append(a.elapsed_time(b))
        ent["uccsd_generators"] = len(ex)
        ent["uccsd_pauli_strings"] = int(len(X))
        ent["uccsd_prep_ms"] = _median(rt)
        ent["rotations_per_s"] = len(ex) / (_median(rt) * 1e-3)
        ent["uccsd_launches"] = int(launches)
        ent["uccsd_hbm_floor_ms"] = launches * 32 * cfg.dim / peak_gbs / 1e6   # one read + write of psi per launch (run)
        del gens
    del psi, out, op, sec
    torch.cuda.empty_cache()
    if with_cpu and cfg.dim > 1000:
        ent["cpu_baseline"] = cpu_baseline(name, max_seconds=12.0)
    return ent


def tfim_entry(bs, torch, peak_gbs: float, flush_buf, n_qubits: int = 20):
    """NEXT-2: the paper's dynamics model in the FULL 2^N space (Eq. 40),
    a number-non-conserving operator: plain bs_apply / bs_expect through the full-space kernel (k_apply_full)."""
    x, z, c = si.tfim_terms(n_qubits)
    op = bs.bs_group_xmask(x, z, c, n_qubits, 0.0)
    sec = bs.bs_sector_build(n_qubits)
    D = 1 << n_qubits
    psi = torch.from_numpy(si.random_state(D, 40 + n_qubits)).cuda()
    out = torch.empty_like(psi)
    bs.bs_apply(op, sec, psi, out)
    times = []
    for _ in range(10):
        flush_buf.zero_()                                  # 2 x 16 MB would sit in the 126 MB L2
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        bs.bs_apply(op, sec, psi, out)
        b.record()
        torch.cuda.synchronize()
        times.append(a.elapsed_time(b))
    ms = _median(times)
    e = bs.bs_expect(op, sec, psi)
    bytes_alg = 32 * D + table_bytes(op)
    return {"n_qubits": n_qubits, "dim": D, "groups": op.n_groups, "strings": op.n_terms, "space": "full 2^N",
            "plan": bs.bs_plan_describe(op, sec), "apply_ms": ms, "applies_per_s": 1e3 / ms,
            "l2_flush_between_reps": True, "hbm_gbs_algorithmic": bytes_alg / ms / 1e6,
            "hbm_frac_of_measured_peak": bytes_alg / ms / 1e6 / peak_gbs, "energy": e.real,
            "gathers_per_target": op.n_groups}


def cpu_baseline(name: str, max_seconds: float = 30.0):
    """The oracle's Eq. 27 gather (OpenMP over target rows, as it stands) on this host's cores, on a bounded sample.
    Small sectors: orc_apply_grouped on an alpha-row slab, scaled linearly in rows.  configs 4-5: the per-row beta
    search makes that function take minutes per row, so the slab function with the search hoisted
    (orc_apply_grouped_slab, the writer of the full-size goldens) is timed on two slabs; its per-call setup is
    separated from the per-row cost by the difference and counted once."""
    from oracle import oracle as orc
    cfg = si.CONFIGS[name]
    if cfg.kind == "hubbard":
        ref = orc.hubbard_h(cfg.n_orb, cfg.hubbard_t, cfg.hubbard_u)
    else:
        ref = orc.molecular_h(*si.integrals(cfg.n_orb, cfg.seed_ints))
    osec = orc.Sector(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    psi = si.random_state(cfg.dim, cfg.seed_psi)
    rows = osec.dim_alpha
    cores = orc.num_threads()
    if cfg.dim > 5e7:
        r1, r2 = min(rows, cores), min(rows, 3 * cores)
        t0 = time.perf_counter()
        osec.apply_grouped_slab(ref, psi, 0, r1)
        t1 = time.perf_counter() - t0
        t0 = time.perf_counter()
        osec.apply_grouped_slab(ref, psi, 0, r2)
        t2 = time.perf_counter() - t0
        per_row = max(1e-9, (t2 - t1) / max(1, r2 - r1))
        fixed = max(0.0, t1 - r1 * per_row)
        t_full = fixed + rows * per_row
        sample = (f"oracle orc_apply_grouped_slab on alpha rows [0,{r1}) and [0,{r2}) of {rows}: {t1:.1f} s and {t2:.1f} s "
                  f"-> {per_row:.3f} s per row + {fixed:.1f} s setup, extrapolated linearly in rows")
        return {"value": 1.0 / t_full, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    out = np.zeros_like(psi)
    probe = max(1, rows // 64)
    t0 = time.perf_counter()
    osec.apply_grouped(ref, psi, 0, probe, out)
    t_probe = time.perf_counter() - t0
    n_rows = int(min(rows, max(probe, (max_seconds * 0.6) / (t_probe / probe))))
    t0 = time.perf_counter()
    osec.apply_grouped(ref, psi, 0, n_rows, out)
    t = time.perf_counter() - t0
    applies_per_s = (n_rows / rows) / t
    sample = (f"oracle orc_apply_grouped on alpha rows [0,{n_rows}) of {rows} ({n_rows * osec.dim_beta} of "
              f"{cfg.dim} targets) in {t:.2f} s, scaled linearly in rows")
    return {"value": applies_per_s, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_28952_b200 import bs          # raises if libbs.so is missing: no CPU fallback

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (libbs has no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peak_gbs, peak_src = _peaks()
    name = args.workload
    cfg = si.CONFIGS[name]
    D = cfg.dim

    # ---- setup (a1-a3), outside the timed region ------------------------------------------------
    t0 = time.perf_counter()
    op, _ = build_operator(name, bs)
    sec = bs.bs_sector_build(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    torch.cuda.synchronize()
    setup_ms = (time.perf_counter() - t0) * 1e3
    psi_h = torch.from_numpy(si.random_state(D, cfg.seed_psi + rank)).pin_memory()   # one state per rank
    out_h = torch.empty_like(psi_h).pin_memory()
    psi = psi_h.cuda()
    work = torch.empty(2 * D, dtype=torch.complex128, device="cuda")
    e_shift = bs.bs_expect(op, sec, psi).real            # also builds the cached plan
    tb = table_bytes(op)
    ev = lambda: torch.cuda.Event(enable_timing=True)    # noqa: E731

    # What a step is ("Work timed"): the lattice model is propagated (configs[2]: Taylor-12
    # steps); the molecular configs time one H application + one expectation (their order-12 series at dt = 0.05 does
    # not converge: the spectrum of the synthetic molecular H is two orders of magnitude wider than the chain's).
    taylor = cfg.kind == "hubbard"
    outs_dev = [work[:D], work[D:]]      # molecular steps: H psi lands here (bs_apply uses no work space)

    def main_op(vec, k=0):
        if taylor:
            bs.bs_taylor_step(op, sec, vec, work, DT, TAYLOR_ORDER, e_shift)
        else:
            bs.bs_apply(op, sec, vec, outs_dev[k])

    def step():
        main_op(psi)
        return bs.bs_expect(op, sec, psi)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing ------------------------------------------------------------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()            # nvidia-smi needs ~0.5 s to deliver its first sample: start before warm-up
    for _ in range(args.warmup):
        step()
    t_w = time.perf_counter()
    while time.perf_counter() - t_w < 0.6:      # keep the GPU under load until the sampler is live
        step()
    barrier()
    n0 = bs.bs_launch_count()
    marks = [ev() for _ in range(2 * args.steps + 1)]
    marks[0].record()
    energy = None
    for i in range(args.steps):
        main_op(psi)
        marks[2 * i + 1].record()
        energy = bs.bs_expect(op, sec, psi)
        marks[2 * i + 2].record()
    barrier()
    launches = bs.bs_launch_count() - n0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = marks[0].elapsed_time(marks[-1])
    taylor_ms = sum(marks[2 * i].elapsed_time(marks[2 * i + 1]) for i in range(args.steps))
    expect_ms = sum(marks[2 * i + 1].elapsed_time(marks[2 * i + 2]) for i in range(args.steps))
    norm_drift = abs(bs.bs_vdot(sec, psi, psi).real - 1.0)

    # ---- end to end: host buffers, H2D + D2H inside the timed region ---------------------------------
    # Every step copies its input state from pinned host memory and its propagated state (+ energy) back.
    # Steps are independent (same host input), so the copies are pipelined against compute: two device
    # buffers, H2D of step i+1 and D2H of step i-1 run on their own streams while step i computes.
    e2e_steps = max(2, min(args.steps, 20))
    s_main = torch.cuda.current_stream()
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    bufs = [psi, torch.empty_like(psi)]
    outs_h = [out_h, torch.empty_like(psi_h).pin_memory()]
    ev_in = [torch.cuda.Event() for _ in range(e2e_steps + 1)]
    ev_c = [torch.cuda.Event() for _ in range(e2e_steps)]
    ev_out = [torch.cuda.Event() for _ in range(e2e_steps)]

    def h2d(i):
        with torch.cuda.stream(s_in):
            if i >= 2:
                s_in.wait_event(ev_out[i - 2])          # buffer i % 2 was last read by the D2H of step i-2
            bufs[i % 2].copy_(psi_h, non_blocking=True)
            ev_in[i].record(s_in)

    barrier()
    a, b = ev(), ev()
    a.record()
    s_in.wait_event(a)
    h2d(0)
    for i in range(e2e_steps):
        if i + 1 < e2e_steps:
            h2d(i + 1)
        s_main.wait_event(ev_in[i])
        main_op(bufs[i % 2], i % 2)
        bs.bs_expect(op, sec, bufs[i % 2])                 # 16-byte result, synchronises the compute stream
        ev_c[i].record(s_main)
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_c[i])
            # the step's result: the propagated state, or H psi.  Output half i % 2 is next written by step i + 2,
            # which waits for ev_out[i] through its input buffer (h2d), so this copy may overlap step i + 1
            outs_h[i % 2].copy_(bufs[i % 2] if taylor else outs_dev[i % 2], non_blocking=True)
            ev_out[i].record(s_out)
    s_main.wait_event(ev_out[e2e_steps - 1])
    if e2e_steps > 1:
        s_main.wait_event(ev_out[e2e_steps - 2])
    b.record()
    barrier()
    e2e_ms = a.elapsed_time(b)
    psi = bufs[0]

    t = torch.tensor([total_ms, e2e_ms, taylor_ms, expect_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms, e2e_ms, taylor_ms, expect_ms = t.tolist()
    applies_per_step = TAYLOR_ORDER + 1 if taylor else 2
    if rank == 0:
        value = world * applies_per_step * args.steps / (total_ms * 1e-3)
        # dominant kernel: the apply kernel of the Taylor launches. Algorithmic bytes per Taylor step (bs_taylor_step
        # accumulates terms in pairs): odd k: 32 D (in, out); even k: 64 D (in, out, acc r+w); the last launch writes no
        # out (48 D even, 48 D odd: in + acc r+w); + tables each launch.  Order 12: (6*32 + 5*64 + 48) D = 560 D.
        per_launch = [(32 if k % 2 else 64) for k in range(1, TAYLOR_ORDER + 1)]
        per_launch[-1] = 48
        bytes_taylor = sum(per_launch) * D + TAYLOR_ORDER * tb
        launch_ms = taylor_ms / (args.steps * TAYLOR_ORDER)
        achieved = bytes_taylor / TAYLOR_ORDER / launch_ms / 1e6
        plan = bs.bs_plan_describe(op, sec)
        if taylor:
            step_txt = (f"1 Taylor-{TAYLOR_ORDER} step (dt={DT}, shifted) + 1 bs_expect = {applies_per_step} H applies")
            roofline = {"bound": "hbm", "kernel": ("k_light<0>" if "+light" in plan else "k_rows<MODE_FINAL>")
                        + " (the 12 apply+axpby launches of bs_taylor_step)",
                        "achieved": achieved, "peak": peak_gbs, "unit": "GB/s", "frac": achieved / peak_gbs,
                        "peak_source": peak_src, "bytes_per_launch": bytes_taylor / TAYLOR_ORDER,
                        "launch_ms": launch_ms, "traffic": (TRAFFIC_NCU.get(name) or {}).get("bytes_per_launch"),
                        "traffic_source": (TRAFFIC_NCU.get(name) or {}).get("profile")}
        else:
            # Molecular configs: thousands of non-zeros per target, the compulsory-bytes roofline is out of reach of any
            # exact method; what binds is the FP64 pipe (k_ab / k_aa on the FP64 tensor
            # instruction).  2 FMA = 4 flops per non-zero (real weight x complex amplitude) over the plain bs_apply;
            # peak = 64 FMA/clk/SM measured (profiles/r02_fp64_peak.md) x 148 SMs x 1.965 GHz x 2 flops.
            step_txt = "1 bs_apply + 1 bs_expect = 2 H applies"
            apply_ms = taylor_ms / args.steps
            flops = 4.0 * nnz_per_row(cfg) * D
            roofline = {"bound": "alu", "kernel": "k_ab + k_aa_mma (FP64 tensor instruction) of one bs_apply",
                        "achieved": flops / (apply_ms * 1e-3) / 1e12, "peak": 2 * DFMA_PEAK / 1e12, "unit": "TFLOP/s",
                        "frac": flops / (apply_ms * 1e-3) / (2 * DFMA_PEAK),
                        "peak_source": "derived: measured 64 FP64 FMA/clk/SM (profiles/r02_fp64_peak.md) x 148 SMs x 1.965 GHz",
                        "flops_per_launch": flops, "launch_ms": apply_ms, "useful_flops_only": True,
                        "traffic": (TRAFFIC_NCU.get(name) or {}).get("bytes_per_launch"),
                        "traffic_source": (TRAFFIC_NCU.get(name) or {}).get("profile")}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
            "config": {"workload": f"{name}: BASELINE.json configs[{si.CONFIG_ORDER.index(name)}]",
                       "n_qubits": cfg.n_qubits, "sector": [cfg.n_orb, cfg.n_alpha, cfg.n_beta], "dim": D,
                       "groups": op.n_groups, "strings": op.n_terms,
                       "step": step_txt,
                       "l2": (f"vectors of {16 * D / 1e6:.1f} MB each exceed the 126 MB L2, no flush needed" if 16 * D > 126e6
                              else f"vectors of {16 * D / 1e6:.1f} MB fit the 126 MB L2 and are NOT flushed between steps "
                                   "(the per_config sweep flushes)"),
                       "parallelism": f"{world} independent state vector(s), one per GPU",
                       "plan": plan},
            "setup_ms": setup_ms, ("taylor_ms_per_step" if taylor else "apply_ms_per_step"): taylor_ms / args.steps,
            "expect_ms_per_call": expect_ms / args.steps, "energy": energy.real, "norm_drift": norm_drift,
            "gpu_launches": int(launches), "clocks": clocks,
            "e2e": {"value": world * applies_per_step * e2e_steps / (e2e_ms * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": 16 * D, "d2h_bytes_per_step": 16 * D + 16, "steps": e2e_steps,
                    "pipeline": "H2D of step i+1 and D2H of step i-1 overlap step i (2 device buffers, 3 streams)"},
            "roofline": roofline,
        }
        want = [] if args.per_config == "none" else args.per_config.split(",")
        if want and world == 1:
            del psi, work
            torch.cuda.empty_cache()
            flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
            line["per_config"] = {n: per_config_entry(n, bs, torch, peak_gbs, flush_buf, not args.no_cpu_baseline)
                                  for n in want}
            line["per_config"]["tfim20_full_space"] = tfim_entry(bs, torch, peak_gbs, flush_buf)
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(name)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
# `ncu --set full` capture (profiles/); None until a capture exists for that workload.
# Each entry names the committed capture it was read from (profiles/); refreshed whenever the kernel changes.
TRAFFIC_NCU = {
    "q28_hubbard": {"bytes_per_launch": 6.74e8, "kernel": "k_light<0>", "profile": "profiles/r02_q28_k_light_full.md",
                    "note": "Taylor-12 launch mix: 6 odd launches at 487 MB, 5 even at 894 MB, the last (48 D) taken as their mean"},
    "q24": {"bytes_per_launch": None, "kernel": "k_ab<12>", "profile": None},
    "q32": {"bytes_per_launch": 2.96e10, "kernel": "k_ab<16> (one slab of 1,456 rows; 9 slabs per apply)",
            "profile": "profiles/r02b_q32_k_ab_k_aa_full.md",
            "note": "dram__bytes_read + dram__bytes_write of two launches: 28.66e9 and 30.58e9"},
    "q56": {"bytes_per_launch": 9.74e10, "kernel": "k_ab<28> (one slab of 2,880 rows; 8 slabs per apply)",
            "profile": "profiles/r02c_q56_k_ab_full.md"},
}


def run_sharded(args):
    """--sharded: ONE state vector, alpha-row slabs over the ranks (bs_apply_rows), NCCL all-gather of the slabs
    (paper_2606_28952_b200/dist.py).  Strong scaling: value = applies/s of the one vector; per-phase device times
    (max over ranks) are reported so that the parts that do not shrink with N are visible."""
    import torch
    import torch.distributed as dist
    from paper_2606_28952_b200 import bs
    from paper_2606_28952_b200.dist import row_slabs, sharded_apply, sharded_expect

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (libbs has no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:  # one rank: the same code path through a single-process group
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29577")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", local))
    name = args.workload
    cfg = si.CONFIGS[name]
    op, _ = build_operator(name, bs)
    sec = bs.bs_sector_build(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    psi = torch.from_numpy(si.random_state(cfg.dim, cfg.seed_psi)).cuda()      # identical on every rank
    out = torch.empty_like(psi)
    Da, Db = cfg.dim_alpha, cfg.dim_beta

    def apply_rows(pin, pout, lo, hi):
        bs.bs_apply_rows(op, sec, pin, pout, lo, hi)

    evs = []

    def marks(what):
        e = torch.cuda.Event(enable_timing=True)
        e.record()
        evs.append(e)

    for _ in range(max(args.warmup, 3)):
        sharded_apply(apply_rows, psi, out, Da, Db)
    dist.barrier()
    torch.cuda.synchronize()
    n0 = bs.bs_launch_count()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(args.steps):
        sharded_apply(apply_rows, psi, out, Da, Db, marks=marks)
    b.record()
    dist.barrier()
    torch.cuda.synchronize()
    launches = bs.bs_launch_count() - n0
    total_ms = a.elapsed_time(b)
    comp_ms = sum(evs[3 * i].elapsed_time(evs[3 * i + 1]) for i in range(args.steps)) / args.steps
    gath_ms = sum(evs[3 * i + 1].elapsed_time(evs[3 * i + 2]) for i in range(args.steps)) / args.steps
    e = sharded_expect(apply_rows, psi, out, Da, Db)
    t = torch.tensor([total_ms, comp_ms, gath_ms], dtype=torch.float64, device="cuda")
    tmin = t.clone()
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(tmin, op=dist.ReduceOp.MIN)
    if rank == 0:
        total_ms, comp_ms, gath_ms = t.tolist()
        line = {"metric": METRIC, "value": args.steps / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
                "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64 (complex128)",
                "data": "synthetic", "mode": "sharded",
                "config": {"workload": f"{name}: BASELINE.json configs[{si.CONFIG_ORDER.index(name)}]",
                           "dim": cfg.dim, "step": "1 H application of ONE state vector",
                           "parallelism": f"alpha-row slabs over {world} rank(s) (bs_apply_rows) + all-gather of the slabs",
                           "slabs": row_slabs(Da, world), "plan": bs.bs_plan_describe(op, sec)},
                "compute_ms_max": comp_ms, "compute_ms_min": tmin[1].item(), "allgather_ms_max": gath_ms,
                "allgather_bytes": 16 * cfg.dim, "energy": e.real, "gpu_launches": int(launches)}
        print(json.dumps(line), flush=True)
    dist.barrier()
    dist.destroy_process_group()


def run_reference(args):
    """--impl reference: the oracle as it stands (OpenMP grouped apply) on this host's cores.
    Each step is one H application on a bounded sample (an alpha-row slab) of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as orc
    name = args.workload
    cfg = si.CONFIGS[name]
    if cfg.kind == "hubbard":
        ref = orc.hubbard_h(cfg.n_orb, cfg.hubbard_t, cfg.hubbard_u)
    else:
        ref = orc.molecular_h(*si.integrals(cfg.n_orb, cfg.seed_ints))
    osec = orc.Sector(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    psi = si.random_state(cfg.dim, cfg.seed_psi)
    out = np.zeros_like(psi)
    rows = osec.dim_alpha
    probe = max(1, rows // 64)
    t0 = time.perf_counter()
    osec.apply_grouped(ref, psi, 0, probe, out)
    per_row = (time.perf_counter() - t0) / probe
    budget = 150.0 / max(1, args.steps + args.warmup)      # whole run within a few minutes
    n_rows = int(min(rows, max(1, budget / per_row)))
    for _ in range(args.warmup):
        osec.apply_grouped(ref, psi, 0, n_rows, out)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        osec.apply_grouped(ref, psi, 0, n_rows, out)
    t = time.perf_counter() - t0
    value = args.steps * (n_rows / rows) / t
    sample = f"alpha rows [0,{n_rows}) of {rows} per step, scaled linearly in rows"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
            "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 (complex128)", "data": "synthetic",
            "config": {"workload": f"{name}: BASELINE.json configs[{si.CONFIG_ORDER.index(name)}]",
                       "n_qubits": cfg.n_qubits, "sector": [cfg.n_orb, cfg.n_alpha, cfg.n_beta], "dim": cfg.dim,
                       "step": "1 H application by the CPU oracle (orc_apply_grouped) on a row slab"},
            "cpu_baseline": {"value": value, "unit": UNIT, "kind": "oracle", "cores": orc.num_threads(),
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="q28_hubbard", choices=si.CONFIG_ORDER)
    ap.add_argument("--per-config", default="q12,q24,q28_hubbard,q32,q56",
                    help="comma list of configs to time with plain bs_apply (N=1 only), or 'none'")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sharded", action="store_true",
                    help="one state vector sharded by alpha-row slabs over the ranks + NCCL all-gather (dist.py)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    elif args.sharded:
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
