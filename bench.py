#!/usr/bin/env python
"""bench.py -- one JSON line for the EmuGEMM hot path on N B200s (contract: see DESIGN.md "Measurement").

A step = one pass of the whole hot path (pre-pass + fused tensor-core GEMM + reconstruction) =
one C-ABI call on one batch of synthetic input of the paper's distribution (Eq. 19).
Default workload: BASELINE.json configs[1] point m=n=k=8192, phi=0.5, seed 1, p=8 (Scheme I DGEMM).
`value` = emulated FP64 TFLOP/s = 2mnk/t with inputs resident in HBM; `e2e` = the same metric through
the C-ABI call with HOST (pinned) buffers, H2D/D2H copies inside the timed region.
N > 1: independent problems per rank (weak scaling), no data-path collective.
--impl reference times the CPU oracle (deliberately slow) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

NOMINAL_INT8_TOPS = 4500.0  # PAPER.md:276, the denominator of the 75 % target
METRIC = "emulated FP64 TFLOP/s (2mnk/t) & INT8 Top/s as % of B200 dense INT8 peak"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)  # median of >= 30 runs
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scheme", default="oz1", choices=["oz1", "oz1s", "oz2", "oz2z"])
    ap.add_argument("--size", type=int, default=8192, help="m = n = k")
    ap.add_argument("--m", type=int, default=0)
    ap.add_argument("--n", type=int, default=0)
    ap.add_argument("--k", type=int, default=0)
    ap.add_argument("--p", type=int, default=0, help="slices (oz1) or moduli (oz2); default 8 / 16")
    ap.add_argument("--phi", type=float, default=-1.0)
    ap.add_argument("--slice-bits", type=int, default=7, choices=[7, 8], help="Scheme I digit width (8: balanced base 256, DESIGN.md R23)")
    ap.add_argument("--slice-form", type=int, default=0, choices=[0, 1],
                    help="7-bit Scheme I digits: 0 = two's-complement fields (R24, PAPER.md:345; default), 1 = sign-magnitude (R1, round 1's default)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-probe", action="store_true")
    ap.add_argument("--cpu-sample", type=int, default=0, help="rows = cols of the oracle sample")
    ap.add_argument("--probe-flags", type=lambda x: int(x, 0), default=0,
                    help="A/B experiments only (results may be WRONG): run the PROBES build of the library with these "
                         "emugemm_dbg_set_flags bits (include/emugemm.h), e.g. 0x10000 = no wave barrier")
    ap.add_argument("--oracle-table", action="store_true",
                    help="with --impl reference: time the oracle IN FULL on 1024^3 instances of every config family (BASELINE.md 3)")
    ap.add_argument("--inputs", default="eq19", choices=["eq19", "nonneg", "a_nonneg", "ones"],
                    help="eq19 (default): the paper's signed distribution; nonneg: |A|, |B| of the same draw; a_nonneg: |A|, B; ones: all ones -- "
                         "power experiments only (operand sign bits cost clock under the power cap, profiles/r2_operand_sign_power.md)")
    ap.add_argument("--fusion", action="store_true", help="Scheme II: fused reconstruction inside the GEMM kernel (default: separate CRT kernel)")
    return ap.parse_args()


def workload(a):
    m = a.m or a.size
    n = a.n or a.size
    k = a.k or a.size
    if a.scheme in ("oz1", "oz1s"):
        p = a.p or (8 if a.scheme == "oz1" else 4)
        seed, phi = (1, 0.5) if a.scheme == "oz1" else (4, 1.0)
        ops = p * (p + 1) * m * n * k  # INT8 ops (p(p+1)/2 products of 2mnk)
        flops = 2.0 * m * n * k
        alg = p * (m + n) * k + (8 if a.scheme == "oz1" else 4) * m * n  # Eq. 10: fused GEMM bytes
        name = f"{'OZ1 DGEMM' if a.scheme == 'oz1' else 'OZ1 SGEMM'} m={m} n={n} k={k} p={p}"
    else:
        p = a.p or (16 if a.scheme == "oz2" else 14)
        seed, phi = (2, 1.0) if a.scheme == "oz2" else (3, 1.0)
        ops = (1 if a.scheme == "oz2" else 3) * p * 2 * m * n * k
        flops = (2.0 if a.scheme == "oz2" else 8.0) * m * n * k
        # Eq. 15 / 18: per modulus (m+n)k + mn, 3M 3(m+n)k + 2mn
        alg = p * ((m + n) * k + m * n) if a.scheme == "oz2" else p * (3 * (m + n) * k + 2 * m * n)
        name = f"{'OZ2 DGEMM' if a.scheme == 'oz2' else 'OZ2 ZGEMM-3M'} m={m} n={n} k={k} N={p}"
    if a.phi >= 0:
        phi = a.phi
    return dict(m=m, n=n, k=k, p=p, seed=seed, phi=phi, ops=float(ops), flops=float(flops), name=name, alg_bytes=float(alg))


def make_inputs(a, w, seed_offset=0):
    import numpy as np
    import emugemm_inputs as G
    if a.scheme == "oz2z":
        A, B = G.complex_pair(w["m"], w["n"], w["k"], w["phi"], w["seed"] + seed_offset)
    else:
        A, B = G.real_pair(w["m"], w["n"], w["k"], w["phi"], w["seed"] + seed_offset,
                           dtype=np.float32 if a.scheme == "oz1s" else np.float64)
    if a.inputs == "nonneg":   # same magnitudes, no sign bits (complex: both parts)
        A, B = (np.abs(A.real) + 1j * np.abs(A.imag), np.abs(B.real) + 1j * np.abs(B.imag)) if a.scheme == "oz2z" else (np.abs(A), np.abs(B))
    elif a.inputs == "a_nonneg" and a.scheme != "oz2z":
        A = np.abs(A)
    elif a.inputs == "ones":
        A, B = np.ones_like(A), np.ones_like(B)
    return A, B


class ClockSampler:
    """nvidia-smi clocks line of B200_PROFILING.md, sampled every 50 ms; only samples whose timestamp falls inside
    the timed window [t0, t1] (host clock, taken right after / before a device synchronize) are used."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        self.idx = gpu_index

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={self.idx}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self, t0, t1):
        import datetime
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, pw, reasons, n_all = [], [], [], set(), 0
        for r in rows:
            if len(r) < 9:
                continue
            try:
                ts = datetime.datetime.strptime(r[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                c, m, w = float(r[1]), float(r[2]), float(r[3])
            except ValueError:
                continue
            n_all += 1
            if not (t0 <= ts <= t1):
                continue
            sm.append(c); mx.append(m); pw.append(w)
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if v.strip().lower() == "active":
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples in the timed window"], "samples_total": n_all}
        return {"sm_mhz": statistics.median(sm), "sm_min_mhz": min(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_oracle_leg(a, w, sample):
    """The oracle as it stands, on this box's host cores, on a bounded sample of the same workload:
    `sample` rows x `sample` columns of the output, full k (every sampled element costs O(k p^2))."""
    import numpy as np
    import emugemm_inputs as G
    from oracle import oracle as O
    A, B = make_inputs(a, w)
    rows = G.sample_indices(w["m"], sample, 1)[:sample]
    cols = G.sample_indices(w["n"], sample, 2)[:sample]
    t0 = time.perf_counter()
    if a.scheme == "oz1":
        O.oz1_sampled(A, B, w["p"], rows, cols)
    elif a.scheme == "oz1s":
        O.oz1_sampled(A.astype(np.float64), B.astype(np.float64), w["p"], rows, cols, is_f32=True)
    elif a.scheme == "oz2":
        O.oz2_sampled(A, B, w["p"], rows, cols)
    else:
        O.oz2_sampled(A, B, w["p"], rows, cols, is3m=True)
    dt = time.perf_counter() - t0
    per_out = w["flops"] / (w["m"] * w["n"])
    val = per_out * len(rows) * len(cols) / dt / 1e12
    return {"value": val, "unit": "TFLOP/s", "cores": O.threads(), "kind": "oracle", "seconds": dt,
            "sample": f"{len(rows)} rows x {len(cols)} cols of the {w['name']} output, full k"}


def calibrated_oracle_leg(a, w, target_s=15.0):
    """cpu_oracle_leg on a sample sized for ~target_s seconds of CPU work: calibrate on 96 x 96 sampled outputs (fixed
    per-call slicing cost included, so small samples are pessimistic), then run the sized sample.  The SAME routine
    serves `cpu_baseline` of the main arm and every step of `--impl reference`, so the two figures agree."""
    cal = cpu_oracle_leg(a, w, 96)
    per_elem = cal["seconds"] / (96 * 96)
    side = int(min(w["m"], w["n"], max(96, (2.7 * target_s / max(per_elem, 1e-9)) ** 0.5)))
    return cpu_oracle_leg(a, w, side), side


def oracle_context(a, w):
    """SURVEY 8(d) / BASELINE.md 3: the oracle single-threaded on a small sample of this workload, and BASELINE config 1
    (Scheme I DGEMM 256^3, p = 6) IN FULL with one thread and with all threads.  Context beside `cpu_baseline`."""
    import emugemm_inputs as G
    from oracle import oracle as O
    out = {}
    nthreads = O.threads()
    try:
        O.set_threads(1)
        st = cpu_oracle_leg(a, w, 48)
        out["single_thread"] = {"value": st["value"], "unit": "TFLOP/s", "cores": 1, "seconds": st["seconds"], "sample": st["sample"]}
        A, B = G.real_pair(256, 256, 256, 0.5, 0)
        t0 = time.perf_counter(); O.dgemm_oz1(A, B, 6); t1 = time.perf_counter() - t0
        O.set_threads(nthreads)
        t0 = time.perf_counter(); O.dgemm_oz1(A, B, 6); tn = time.perf_counter() - t0
        fl = 2.0 * 256 ** 3
        out["config1_full_256_p6"] = {"seconds_1_thread": t1, "gflops_1_thread": fl / t1 / 1e9, "seconds_all": tn,
                                      "gflops_all": fl / tn / 1e9, "cores": nthreads,
                                      "int_mac_per_s_all": 21.0 * 256 ** 3 / tn}
    finally:
        O.set_threads(nthreads)
    return out


def oracle_table():
    """BASELINE.md 3 / SURVEY 8(d): the oracle in full on config 1 and on 1024^3 instances of configs 2-5 (p / N unchanged),
    all host threads, plus one thread on 512^3; seconds, emulated GFLOP/s, integer MAC/s.  One JSON line."""
    import numpy as np
    import emugemm_inputs as G
    from oracle import oracle as O
    nthreads = O.threads()
    rows = []

    def timed(name, fn, flops, macs):
        t0 = time.perf_counter(); fn(); dt = time.perf_counter() - t0
        rows.append({"case": name, "threads": O.threads(), "seconds": round(dt, 3), "emulated_gflops": round(flops / dt / 1e9, 3),
                     "int_gmac_per_s": round(macs / dt / 1e9, 2)})

    A0, B0 = G.real_pair(256, 256, 256, 0.5, 0)
    timed("config 1: OZ1 DGEMM 256^3 p=6 (full)", lambda: O.dgemm_oz1(A0, B0, 6), 2.0 * 256 ** 3, 21.0 * 256 ** 3)
    for s_ in (1024, 512):
        O.set_threads(nthreads if s_ == 1024 else 1)
        A, B = G.real_pair(s_, s_, s_, 0.5, 1)
        for p_ in ((3, 6, 8) if s_ == 1024 else (8,)):
            timed(f"config 2: OZ1 DGEMM {s_}^3 p={p_}", lambda: O.dgemm_oz1(A, B, p_), 2.0 * s_ ** 3, p_ * (p_ + 1) / 2.0 * s_ ** 3)
        A, B = G.real_pair(s_, s_, s_, 1.0, 2)
        for N_ in ((12, 16, 20) if s_ == 1024 else (16,)):
            timed(f"config 3: OZ2 DGEMM {s_}^3 N={N_}", lambda: O.dgemm_oz2(A, B, N_), 2.0 * s_ ** 3, float(N_) * s_ ** 3)
        Az, Bz = G.complex_pair(s_, s_, s_, 1.0, 3)
        for N_ in ((14, 18) if s_ == 1024 else (14,)):
            timed(f"config 4: OZ2 ZGEMM-3M {s_}^3 N={N_}", lambda: O.zgemm_oz2_3m(Az, Bz, N_), 8.0 * s_ ** 3, 3.0 * N_ * s_ ** 3)
        Af, Bf = G.real_pair(s_, s_, s_, 1.0, 4, dtype=np.float32)
        timed(f"config 5: OZ1 SGEMM {s_}^3 p=4", lambda: O.sgemm_oz1(Af, Bf, 4), 2.0 * s_ ** 3, 10.0 * s_ ** 3)
    O.set_threads(nthreads)
    print(json.dumps({"impl": "reference", "oracle_table": rows, "cores": nthreads}))


def reference_leg(a, w):
    """--impl reference: the oracle on host cores; each step = the same bounded sample of the workload that the main
    arm's `cpu_baseline` uses (calibrated to ~15 s), repeated for `steps` steps or until ~150 s are spent."""
    vals, cb = [], None
    cpu_oracle_leg(a, w, 32)  # warm-up (library load, page-in)
    first, side = calibrated_oracle_leg(a, w)
    vals.append(first["value"]); cb = first
    t_all = time.perf_counter()
    for _ in range(max(0, a.steps - 1)):
        if time.perf_counter() - t_all + first["seconds"] > 150:
            break
        cb = cpu_oracle_leg(a, w, side)
        vals.append(cb["value"])
    v = statistics.median(vals)
    cb["value"] = v
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": "TFLOP/s", "n_gpus": a.gpus, "steps": len(vals),
            "warmup": a.warmup, "ms_per_step": 1e3 * cb["seconds"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int8", "data": "synthetic",
            "config": {"workload": w["name"], "phi": w["phi"], "seed": w["seed"], "note": "CPU oracle, sampled outputs"},
            "cpu_baseline": cb, "e2e": {"value": v, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    a = parse()
    w = workload(a)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    if a.impl == "reference":
        if rank == 0:
            if a.oracle_table:
                oracle_table()
            else:
                reference_leg(a, w)
        return

    import numpy as np
    import torch
    import paper_2606_25453_b200 as E
    from paper_2606_25453_b200 import shard

    assert torch.cuda.is_available(), "bench.py needs a GPU: the product path has no CPU fallback"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # independent problem per rank (weak scaling): same recipe, seed offset by rank
    A, B = make_inputs(a, w, seed_offset=shard.rank_seed(0, rank))
    cdtype = {"oz1": torch.float64, "oz1s": torch.float32, "oz2": torch.float64, "oz2z": torch.complex128}[a.scheme]
    hA, hB = torch.from_numpy(A).pin_memory(), torch.from_numpy(B).pin_memory()
    hC = torch.empty((w["m"], w["n"]), dtype=cdtype).pin_memory()
    dA, dB = hA.cuda(), hB.cuda()
    dC = torch.empty((w["m"], w["n"]), dtype=cdtype, device="cuda")
    h = E.EmuGemm(probes=bool(a.probe_flags))
    stream = torch.cuda.current_stream()
    h.set_stream(stream)
    h.set_slice_bits(a.slice_bits)
    if a.slice_form:
        h.set_slice_form(a.slice_form)
    if a.probe_flags:
        h.dbg_set_flags(a.probe_flags)
    if a.fusion:
        h.set_oz2_fusion(True)
    call = {"oz1": h.dgemm_oz1, "oz1s": h.sgemm_oz1, "oz2": h.dgemm_oz2, "oz2z": h.zgemm_oz2_3m}[a.scheme]

    def step():
        call(dA, dB, dC, w["p"])

    def step_e2e():
        dA.copy_(hA, non_blocking=True)
        dB.copy_(hB, non_blocking=True)
        call(dA, dB, dC, w["p"])
        hC.copy_(dC, non_blocking=True)

    step()  # sizes the workspace outside every timed region
    torch.cuda.synchronize()

    # ---- device-resident timing: W warm-ups, then exactly K steps between barriers ----
    sampler = ClockSampler(local)
    sampler.start()
    for _ in range(max(a.warmup, 3)):
        step()
    h.enable_stage_timing(True)
    barrier()
    t_win0 = time.time()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage = [[], [], []]
    cycles = []
    launches = 0
    e0.record(stream)
    for _ in range(a.steps):
        step()
        # stage events sit on the same stream; reading them synchronises after the step, before the next launch
        ms, nl = h.stage_ms()
        for i in range(3):
            stage[i].append(ms[i])
        launches += nl
        cycles.append(h.last_gemm_cycles())
    e1.record(stream)
    barrier()
    total_ms = e0.elapsed_time(e1)
    h.enable_stage_timing(False)

    # a second pass without the per-step synchronisation gives the back-to-back step time
    barrier()
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(a.steps + 1)]
    marks[0].record(stream)
    for i in range(a.steps):
        step()
        marks[i + 1].record(stream)   # an event record does not synchronise: the steps still run back to back
    barrier()
    clocks = sampler.stop(t_win0, time.time())
    per_step = [marks[i].elapsed_time(marks[i + 1]) for i in range(a.steps)]
    ms_step = shard.max_over_ranks(marks[0].elapsed_time(marks[-1]) / a.steps, dist, "cuda")
    ms_median = statistics.median(per_step)
    ms_q = statistics.quantiles(per_step, n=4) if len(per_step) >= 4 else [ms_median] * 3
    value = shard.aggregate_throughput(w["flops"], world, ms_step) / 1e12

    # ---- end to end: host (pinned) buffers, H2D + call + D2H inside the timed region ----
    # Every step copies its own inputs host -> device and its result device -> host.  Serial leg: all on one stream.
    # Pipelined leg (the reported e2e): double-buffered device operands, the copies of step i+1 / i-1 run on two
    # copy streams while the C-ABI call of step i runs on the compute stream (PCIe is full duplex), ordered by events.
    e2e = None
    if not a.no_e2e:
        for _ in range(2):
            step_e2e()
        barrier()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_e2e = max(3, min(a.steps, 10))
        g0.record(stream)
        for _ in range(n_e2e):
            step_e2e()
        g1.record(stream)
        barrier()
        ms_serial = shard.max_over_ranks(g0.elapsed_time(g1) / n_e2e, dist, "cuda")

        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
        bufA, bufB, bufC = [dA, torch.empty_like(dA)], [dB, torch.empty_like(dB)], [dC, torch.empty_like(dC)]
        hC2 = [hC, torch.empty_like(hC).pin_memory()]

        def pipelined(n_steps):
            h2d, comp, d2h = [], [], []
            for i in range(n_steps):
                b = i & 1
                ev_in = torch.cuda.Event()
                with torch.cuda.stream(s_in):
                    if i >= 2:
                        s_in.wait_event(comp[i - 2])   # operands of step i-2 consumed: buffer b is free
                    bufA[b].copy_(hA, non_blocking=True)
                    bufB[b].copy_(hB, non_blocking=True)
                    ev_in.record(s_in)
                h2d.append(ev_in)
                stream.wait_event(ev_in)
                if i >= 2:
                    stream.wait_event(d2h[i - 2])       # result of step i-2 copied out: C buffer b is free
                call(bufA[b], bufB[b], bufC[b], w["p"])
                ev_c = torch.cuda.Event()
                ev_c.record(stream)
                comp.append(ev_c)
                ev_o = torch.cuda.Event()
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_c)
                    hC2[b].copy_(bufC[b], non_blocking=True)
                    ev_o.record(s_out)
                d2h.append(ev_o)
            return d2h[-1]

        pipelined(2)
        barrier()
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_pipe = max(4, min(a.steps, 10))
        p0.record(stream)
        s_in.wait_event(p0)
        last = pipelined(n_pipe)
        stream.wait_event(last)
        p1.record(stream)
        barrier()
        ms_e2e = shard.max_over_ranks(p0.elapsed_time(p1) / n_pipe, dist, "cuda")
        e2e = {"value": shard.aggregate_throughput(w["flops"], world, ms_e2e) / 1e12, "unit": "TFLOP/s",
               "ms_per_step": ms_e2e, "mode": "double-buffered: H2D / call / D2H of consecutive steps overlap on 3 streams",
               "serial_ms_per_step": ms_serial,
               "serial_value": shard.aggregate_throughput(w["flops"], world, ms_serial) / 1e12,
               "h2d_bytes_per_step": int(hA.numel() * hA.element_size() + hB.numel() * hB.element_size()),
               "d2h_bytes_per_step": int(hC.numel() * hC.element_size())}
        del bufA, bufB, bufC, hC2

    # every collective is done: all ranks leave the process group together (rank 0 goes on alone with the probe leg and the
    # CPU oracle, which take tens of seconds; the other ranks must not sit in a half-torn-down group meanwhile)
    if dist is not None:
        barrier()
        dist.destroy_process_group()
        dist = None
    if rank != 0:
        return

    # ---- roofline of the dominant kernel (the fused tensor-core GEMM), measured live ----
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        pass
    bf16_burst = peaks.get("bf16_tflops", 1590.0)
    peak_src = "measured bf16 burst x2 (guide's nominal int8:bf16 ratio 4.5:2.25)" if peaks else \
        "fallback 1.59 PF bf16 x2 (guide's nominal int8:bf16 ratio)"
    gemm_ms = statistics.median(stage[1])
    gemm_q = statistics.quantiles(stage[1], n=4) if len(stage[1]) >= 4 else [gemm_ms] * 3
    achieved = w["ops"] / (gemm_ms * 1e-3) / 1e12
    peak = 2.0 * bf16_burst
    # dram__bytes_read.sum + dram__bytes_write.sum of the GEMM kernel, per launch, from the committed ncu capture of this
    # command at this commit (profiles/traffic.csv: workload, kernel, bytes, capture file); ncu cannot run inside a timed run
    traffic, traffic_src = None, None
    try:
        for row in open(os.path.join(ROOT, "profiles", "traffic.csv")):
            f = [x.strip() for x in row.split(",")]
            if len(f) >= 3 and f[0] == w["name"]:
                traffic = float(f[2])
                traffic_src = f[3] if len(f) > 3 else "profiles/traffic.csv"
    except (OSError, ValueError):
        pass
    roof = {"bound": "tensor", "kernel": "oz1_gemm_kernel" if a.scheme.startswith("oz1") else "oz2_gemm_kernel",
            "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic,
            "traffic_source": traffic_src, "algorithmic_bytes": w["alg_bytes"],
            "peak_source": peak_src, "kernel_ms": gemm_ms, "kernel_ms_iqr": gemm_q[2] - gemm_q[0], "int8_ops_per_launch": w["ops"],
            "frac_of_nominal_4500": achieved / NOMINAL_INT8_TOPS}
    if peaks.get("bf16_tflops_sustained"):
        roof["frac_of_sustained"] = achieved / (2.0 * peaks["bf16_tflops_sustained"])
    if clocks.get("sm_mhz"):
        roof["frac_of_clock_scaled"] = achieved / (148 * 16384 * clocks["sm_mhz"] * 1e6 / 1e12)
    if cycles and min(cycles) > 0:
        # SM cycle counter of the GEMM kernel (CTA 0): INT8 ops per clock per SM against 16384, clock-independent
        cyc = statistics.median(cycles)
        roof["per_clock_efficiency"] = w["ops"] / (cyc * 148) / 16384.0
        roof["sm_ghz_during_kernel"] = cyc / (gemm_ms * 1e-3) / 1e9

    detail = {"stage_ms_median": {"prepass": statistics.median(stage[0]), "gemm": gemm_ms, "recon": statistics.median(stage[2])},
              "synced_ms_per_step": total_ms / a.steps,
              "int8_tops_end_to_end": world * w["ops"] / (ms_step * 1e-3) / 1e12}
    elem = {"oz1": 8, "oz1s": 4, "oz2": 8, "oz2z": 16}[a.scheme]
    planes = w["p"] * (3 if a.scheme == "oz2z" else 1)
    kpad = (w["k"] + 127) // 128 * 128
    pre_bytes = elem * (w["m"] * w["k"] + w["k"] * w["n"]) + planes * kpad * (w["m"] + w["n"])
    detail["prepass_algorithmic_GBps"] = pre_bytes / (detail["stage_ms_median"]["prepass"] * 1e-3) / 1e9
    detail["prepass_frac_of_hbm"] = detail["prepass_algorithmic_GBps"] / peaks.get("hbm_gbs", 6650.0)
    if not a.no_probe:
        try:
            # the kernel's own MMA issue schedule on operands resident in shared memory (no TMA, no epilogue):
            # what the tensor pipe sustains for this p; Scheme II uses the plain N = 256 schedule (p = 1)
            pp = w["p"] if a.scheme in ("oz1", "oz1s") else 1
            hp = E.EmuGemm(probes=True)   # the PROBES build of the same sources (probe kernels are not in the product)
            hp.set_stream(stream)
            _, tops, eff = hp.dbg_oz1_issue_probe(pp, True, 4000)
            hp.close()
            detail["issue_probe_per_clock_efficiency"] = eff
            detail["issue_probe_tops"] = tops
            roof["frac_of_probe"] = achieved / tops
        except Exception as ex:  # the probe is context, never the product
            detail["i8_issue_probe_error"] = str(ex)
    if a.scheme == "oz1" and w["p"] == 8 and a.slice_bits == 7 and not a.no_probe:
        # NEXT item f1 (R23): the same problem with 7 balanced 8-bit slices (28 instead of 36 products),
        # which reaches the accuracy of 8 slices of 7 bits; context only, the headline stays BASELINE's p = 8
        h.set_slice_bits(8)
        for _ in range(3):
            call(dA, dB, dC, 7)
        q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        q0.record(stream)
        for _ in range(5):
            call(dA, dB, dC, 7)
        q1.record(stream)
        torch.cuda.synchronize()
        h.set_slice_bits(7)
        ms8 = q0.elapsed_time(q1) / 5
        detail["f1_8bit_slices_p7"] = {"ms_per_step": ms8, "emulated_tflops": w["flops"] / (ms8 * 1e-3) / 1e12,
                                       "int8_tops": 56.0 * w["m"] * w["n"] * w["k"] / (ms8 * 1e-3) / 1e12}
        # NEXT item f2: 64 products of 512^3 through ONE strided batched call; context only
        try:
            gb = torch.Generator(device="cuda")
            gb.manual_seed(w["seed"] + 7)
            Ab = torch.rand((64, 512, 512), device="cuda", dtype=torch.float64, generator=gb) - 0.5
            Bb = torch.rand((64, 512, 512), device="cuda", dtype=torch.float64, generator=gb) - 0.5
            Cb = torch.empty((64, 512, 512), device="cuda", dtype=torch.float64)
            for _ in range(3):
                h.dgemm_oz1_strided_batched(Ab, Bb, Cb, 8)
            q0.record(stream)
            for _ in range(10):
                h.dgemm_oz1_strided_batched(Ab, Bb, Cb, 8)
            q1.record(stream)
            torch.cuda.synchronize()
            msb = q0.elapsed_time(q1) / 10
            detail["f2_strided_batched_64x512_p8"] = {"ms_per_call": msb,
                                                      "emulated_tflops": 2.0 * 64 * 512 ** 3 / (msb * 1e-3) / 1e12}
            del Ab, Bb, Cb
        except Exception as ex:  # context, never the product
            detail["f2_strided_batched_error"] = str(ex)
    detail["paper_context"] = "paper: 3654 Top/s (81% of 4500) EmuGEMM-I end-to-end on B200, other machine (PAPER.md:293)"

    line = {"metric": METRIC, "value": value, "unit": "TFLOP/s", "n_gpus": world, "steps": a.steps, "warmup": max(a.warmup, 3),
            "ms_per_step": ms_step, "ms_per_step_median": ms_median, "ms_per_step_iqr": ms_q[2] - ms_q[0],
            "value_at_median": w["flops"] / (ms_median * 1e-3) / 1e12,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int8", "data": "synthetic",
            "config": {"workload": w["name"] + ("" if a.inputs == "eq19" else f" [inputs: {a.inputs}]"), "phi": w["phi"], "seed": w["seed"], "alpha": 1, "beta": 0, "slice_bits": a.slice_bits, "slice_form": a.slice_form, "probe_flags": hex(a.probe_flags), "oz2_fusion": bool(a.fusion), "inputs": a.inputs,
                       "l2": "inputs (A, B, slices > 1 GB) exceed the 126 MB L2, no flush needed",
                       "parallelism": f"{world} independent problems" if world > 1 else "1 GPU"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roof, "detail": detail}
    if not a.no_cpu:
        if a.cpu_sample:
            line["cpu_baseline"] = cpu_oracle_leg(a, w, a.cpu_sample)
        else:  # the same calibrated sample `--impl reference` times
            line["cpu_baseline"], _ = calibrated_oracle_leg(a, w)
        try:
            line["cpu_baseline"]["context"] = oracle_context(a, w)
        except Exception as ex:  # context, never the product
            line["cpu_baseline"]["context_error"] = str(ex)
    print(json.dumps(line))
    h.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
