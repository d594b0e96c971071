#!/usr/bin/env python
"""bench.py -- headline measurement of the Wilson-Dirac hot path (arXiv 2503.06721) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--prec f64] [--variant 0] [--impl ours|reference]

One "step" = one pass of the whole hot path over one set of synthetic fields:
    links_to_rep, Dphi_eo, Dphi_oe, Dphi, Dphi_hat, g5Dphi_sq            (8 stencil passes + 1 link build)
Default workload: BASELINE.json configs[1] -- SU(3) fundamental, 32^4, fp64 (the configuration the metric is quoted on).
`value` = algorithmic GFLOP (SURVEY.md 8(d) flop model) per step / device time per step, inputs resident in HBM.
`roofline` = the dominant kernel (the Dphi_eo stencil pass): compulsory bytes (2S+8K per output site) / its own
CUDA-event duration, against the measured copy bandwidth of MEASURED_PEAKS.json.
`e2e` = the same step through hirep_apply_host with pinned HOST buffers (H2D of links+spinors, D2H of results, timed).
`cpu_baseline` = the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
`per_config` = after the headline step, the same six operators on EVERY BASELINE configuration C2..C5 in fp64 and fp32 (C4 also
in link mode REBUILD), timed the way SURVEY.md 8(d) prescribes: >= 10 warm-ups, then n back-to-back launches (n = 100, fewer
for multi-millisecond kernels so that a repeat stays near 0.25 s; never < 10) over 4 rotating spinor buffer sets, median of 5
repeats -- next to the single-launch-inside-a-step number, so launch gaps are visible instead of folded into a fraction.
`--impl reference` times the oracle alone (this tier's reference arm).  N > 1: independent replicas.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Dphi_eo GFLOP/s & effective HBM GB/s (fraction of B200 peak), per N_g/rep"


# ------------------------------------------------------------------------------- cost model
def cost_model(cfg, prec, rebuild=False):
    d = cfg.d_R
    real = cfg.rep == 1
    w = 8 if prec == "f64" else 4
    S = 8 * d * w                                  # one spinor
    K = d * d * (1 if real else 2) * w             # one represented link
    KF = 2 * cfg.n_g ** 2 * w
    if rebuild:                                    # link mode REBUILD streams fundamental links
        K = KF
    F_hop = (64 if real else 128) * d * d + 56 * d
    V = cfg.volume
    ops = {
        # name: (flops, compulsory bytes as executed by this library's link layout, paper-ideal compulsory bytes)
        "Dphi_eo": (F_hop * V / 2, (2 * S + 8 * K) * V / 2, (2 * S + 8 * K) * V / 2),
        "Dphi_oe": (F_hop * V / 2, (2 * S + 8 * K) * V / 2, (2 * S + 8 * K) * V / 2),
        "Dphi": ((F_hop + 16 * d) * V, (2 * S + 8 * K) * V, (2 * S + 4 * K) * V),
        "Dphi_hat": ((2 * F_hop + 16 * d) * V / 2, (5 * S + 16 * K) * V / 2, (5 * S + 16 * K) * V / 2),
        "g5Dphi_sq": (2 * (F_hop + 16 * d) * V, 2 * (2 * S + 8 * K) * V, 2 * (2 * S + 4 * K) * V),
        "links_to_rep": (0.0, 8 * V * (KF + K), 4 * V * (KF + K)),
    }
    return dict(S=S, K=K, KF=KF, F_hop=F_hop, ops=ops)


OP_ORDER = ["links_to_rep", "Dphi_eo", "Dphi_oe", "Dphi", "Dphi_hat", "g5Dphi_sq"]


def ncu_traffic(config, prec, op):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `op`, from the committed ncu captures
    (profiles/r02_traffic.csv, else profiles/r01b_traffic.csv; the commands that made them are in the .md beside them)."""
    path = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    if not os.path.exists(path):
        path = os.path.join(ROOT, "profiles", "r01b_traffic.csv")
    if not os.path.exists(path):
        return None
    import csv
    for row in csv.DictReader(open(path)):
        if row["config"] == config and row["prec"] == prec and row["op"] == op:
            return int(row["dram_read_bytes"]) + int(row["dram_write_bytes"])
    return None


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def max_over_ranks(value, dist, device=None):
    """Timing rule of the bench contract: a multi-rank number is the MAX over ranks (all_reduce MAX; works for the
    nccl backend on a GPU and for gloo on CPU, where the world_size-2 test runs it)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(flops_per_replica_step, world, ms_step):
    """Whole-job GFLOP/s of `world` independent replicas (weak scaling): units of all ranks / max time."""
    return world * flops_per_replica_step / (ms_step * 1e-3) / 1e9


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region (B200_PROFILING.md 'clocks line') through NVML
    (nvidia_ml_py: a sample every few ms from a thread, no process start-up); falls back to one nvidia-smi query."""
    BAD = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40, "sw_power_cap": 0x4}

    def __init__(self, index):
        self.index, self.sm, self.mask, self.smax = index, [], 0, None
        self.stop_flag = threading.Event()
        self.thread = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            # NVML enumerates physical devices: honour CUDA_VISIBLE_DEVICES when it is a plain index list
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            phys = self.index
            if vis and all(v.strip().isdigit() for v in vis.split(",")):
                ids = [int(v) for v in vis.split(",")]
                phys = ids[self.index] if self.index < len(ids) else self.index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.thread = threading.Thread(target=self._loop, daemon=True)
            self.thread.start()
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        while not self.stop_flag.is_set():
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.mask |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            except Exception:
                pass
            time.sleep(0.003)

    def stop(self):
        if self.thread is not None:
            self.stop_flag.set()
            self.thread.join(timeout=2)
        if not self.sm:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=clocks.sm,clocks.max.sm",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=20).stdout
                f = [float(x) for x in out.strip().split(",")]
                return {"sm_mhz": f[0], "sm_max_mhz": f[1], "reasons": ["sampled after the timed region (NVML unavailable)"], "samples": 1}
            except Exception:
                return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml and nvidia-smi unavailable"], "samples": 0}
        sm = sorted(self.sm)
        reasons = sorted(k for k, bit in self.BAD.items() if self.mask & bit)
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": self.smax, "reasons": reasons, "samples": len(sm)}



# ------------------------------------------------------------------- all configurations (SURVEY.md 8(d) timing)
SWEEP = [("C2", "f64", False), ("C2", "f32", False), ("C3", "f64", False), ("C3", "f32", False), ("C4", "f64", False),
         ("C4", "f32", False), ("C4", "f64", True), ("C4", "f32", True), ("C5", "f64", False), ("C5", "f32", False),
         ("C5", "f64", True), ("C5", "f32", True)]
NSETS = 4          # rotating spinor buffer sets (C2 fp32 half spinors are 50 MB < L2: one set would be timed out of L2)


class Fields:
    """Device-resident native fields of one configuration: links (stored represented or fundamental for REBUILD) and NSETS
    independent input / output spinor sets."""

    def __init__(self, torch, hirep, synth, cfg, prec, rebuild, dev, variant=0, nsets=NSETS):
        cdt = torch.complex128 if prec == "f64" else torch.complex64
        links_c, (psi_c,) = synth.make_inputs_torch(cfg, dev, cdt, n_spinors=1)
        self.cfg, self.prec, self.rebuild = cfg, prec, rebuild
        self.geom = g = hirep.Geometry(cfg.T, cfg.L, cfg.n_g, cfg.rep, prec, device=dev)
        g.set_kernel_variant(variant)
        self.lf = g.links_import(links_c)
        self.links_c, self.psi_c = links_c, psi_c      # canonical tensors (the e2e leg copies them to the host); drop() frees them
        if rebuild:
            g.set_link_mode(hirep.LINKS_REBUILD)
            self.lr = self.lf
        else:
            self.lr = g.new_links_rep()
            g.links_to_rep(self.lf, out=self.lr)
        hb = g.sizes["spinor_half"]
        x0 = g.spinor_import(psi_c, hirep.FULL)
        self.x = [x0] + [x0.clone() for _ in range(nsets - 1)]
        self.y = [g.new_spinor(hirep.FULL) for _ in range(nsets)]
        self.hb = hb

    def drop_canonical(self):
        self.links_c = self.psi_c = None

    def op(self, name, k=0):
        """closure launching operator `name` on spinor set k"""
        g, m0, hb = self.geom, self.cfg.m0, self.hb
        x, y, lr, lf = self.x[k % len(self.x)], self.y[k % len(self.y)], self.lr, self.lf
        if name == "links_to_rep":
            return lambda: g.links_to_rep(lf, out=lr)
        if name == "Dphi_eo":
            return lambda: g.Dphi_eo(x[hb:], lr, out=y[:hb])
        if name == "Dphi_oe":
            return lambda: g.Dphi_oe(x[:hb], lr, out=y[hb:])
        if name == "Dphi":
            return lambda: g.Dphi(m0, x, lr, out=y)
        if name == "Dphi_hat":
            return lambda: g.Dphi_hat(m0, x[:hb], lr, out=y[:hb])
        if name == "g5Dphi_sq":
            return lambda: g.g5Dphi_sq(m0, x, lr, out=y)
        raise KeyError(name)


def op_row(cm, name, ms, peak):
    """Fractions are on SURVEY.md 8(d)'s COMPULSORY bytes (every datum crosses HBM once: Dphi (2S+4K)V, links_to_rep 4V(K_F+K)); the
    bytes the gather layout actually streams (every link stored twice) are reported beside them as `*_as_executed`."""
    fl, by_exec, by = cm["ops"][name]
    return {"ms": round(ms, 4), "gflops": round(fl / ms / 1e6, 1), "gbs": round(by / ms / 1e6, 1),
            "frac_hbm": round(by / ms / 1e6 / peak, 4), "frac_8TBs_nominal": round(by / ms / 1e6 / 8000.0, 4),
            "gbs_as_executed": round(by_exec / ms / 1e6, 1), "frac_as_executed": round(by_exec / ms / 1e6 / peak, 4)}


def time_back_to_back(torch, fields, name, target_s=0.25, repeats=5, warm=10, nmax=100, nmin=10):
    """warm-ups, then `repeats` x n back-to-back launches rotating over the spinor sets; median ms per launch."""
    fns = [fields.op(name, k) for k in range(NSETS)]
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for i in range(warm):
        fns[i % NSETS]()
    b.record()
    torch.cuda.synchronize()
    est = max(a.elapsed_time(b) / warm, 1e-3)
    n = int(max(nmin, min(nmax, target_s * 1e3 / est)))
    times = []
    for _ in range(repeats):
        a.record()
        for i in range(n):
            fns[i % NSETS]()
        b.record()
        torch.cuda.synchronize()
        times.append(a.elapsed_time(b) / n)
    times.sort()
    return times[len(times) // 2], n


def sweep_config(torch, hirep, synth, dev, name, prec, rebuild, peak, variant=0, fields=None):
    cfg = synth.CONFIGS[name]
    cm = cost_model(cfg, prec, rebuild)
    own = fields is None
    if own:
        fields = Fields(torch, hirep, synth, cfg, prec, rebuild, dev, variant)
        fields.drop_canonical()
        torch.cuda.empty_cache()
    ops = [k for k in OP_ORDER if not (rebuild and k == "links_to_rep")]
    # (i) single launches inside whole steps (what the headline's per_op reports): 3 steps, one event pair per launch
    in_step = {k: [] for k in ops}
    for it in range(2 + 3):
        for k in ops:
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fields.op(k, it)(); b.record()
            if it >= 2:
                in_step[k].append((a, b))
    torch.cuda.synchronize()
    out = {"d_R": cfg.d_R, "lattice": "%dx%d^3" % (cfg.T, cfg.L), "links": "rebuild" if rebuild else "stored", "ops": {}}
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    for k in ops:
        ms, n = time_back_to_back(torch, fields, k)
        row = op_row(cm, k, ms, peak)
        row["launches_per_repeat"] = n
        row["ms_in_step"] = round(sum(a.elapsed_time(b) for a, b in in_step[k]) / len(in_step[k]), 4)
        out["ops"][k] = row
    ck = sampler.stop()
    out["clocks"] = {"sm_mhz": ck.get("sm_mhz"), "reasons": ck.get("reasons")}   # sustained back-to-back load: the power cap shows here
    if own and not rebuild:   # the clover term per configuration (the headline configuration has the full block in next1_linalg_cg)
        try:
            out["clover"] = measure_clover(torch, hirep, fields.geom, cfg, prec, cm, cfg.m0, fields.x[0], fields.y[0], fields.lr, peak, light=True)
        except Exception as e:
            out["clover"] = {"error": "%s: %s" % (type(e).__name__, e)}
            torch.cuda.empty_cache()
    if own:
        del fields
        torch.cuda.empty_cache()
    return out

# -------------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    from harness import synth
    from paper_2503_06721_b200 import hirep

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    hirep.load()

    cfg = synth.CONFIGS[args.config]
    if args.custom:   # "N_g,rep,T,L": any other gauge group / representation / lattice (same recipe as C2: Haar links)
        n_g, rep, T, L = [int(v) for v in args.custom.split(",")]
        cfg = synth.Config("custom", T, L, n_g, rep, -0.2, "haar", 77, ("Dphi_eo", "Dphi_hat"))
    prec = args.prec
    rebuild = args.link_mode == "rebuild"
    cm = cost_model(cfg, prec, rebuild)
    ops_run = [k for k in OP_ORDER if not (rebuild and k == "links_to_rep")]
    F = Fields(torch, hirep, synth, cfg, prec, rebuild, dev, args.variant)
    geom, m0 = F.geom, cfg.m0
    ev = {k: [] for k in OP_ORDER}

    def step(it, record=False):
        for k in ops_run:
            fn = F.op(k, it)
            if record:
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); fn(); b.record()
                ev[k].append((a, b))
            else:
                fn()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for it in range(args.warmup):
        step(it)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = geom.launch_count()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0.record()
    for it in range(args.steps):
        step(it, record=True)
    t1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_total = t0.elapsed_time(t1)
    launches = geom.launch_count() - launches0
    ms_total = max_over_ranks(ms_total, dist, dev)
    ms_step = ms_total / args.steps

    flops_step = sum(cm["ops"][k][0] for k in ops_run)
    value = aggregate_value(flops_step, world, ms_step)
    peak, peak_src = peaks()
    per_op = {}
    for k in ops_run:
        ms = sum(a.elapsed_time(b) for a, b in ev[k]) / len(ev[k])
        per_op[k] = op_row(cm, k, ms, peak)
    eo = per_op["Dphi_eo"]
    traffic = ncu_traffic(args.config, prec, "Dphi_eo") if not rebuild else None
    roofline = {"bound": "hbm", "kernel": "hop stencil (Dphi_eo pass)", "achieved": eo["gbs"], "peak": peak,
                "unit": "GB/s", "frac": round(eo["gbs"] / peak, 4), "traffic": traffic, "peak_source": peak_src,
                "algorithmic_bytes": cm["ops"]["Dphi_eo"][1], "frac_of_8TBs_nominal": round(eo["gbs"] / 8000.0, 4),
                "timing": "one CUDA-event pair around the single launch inside each timed step (launch gap and pipeline fill included); "
                          "per_config has the back-to-back figure"}

    # ---- e2e: same step through hirep_apply_host with pinned host buffers
    e2e = None
    if not args.no_e2e and not rebuild:
        links_h = F.links_c.cpu().pin_memory()
        psi_h = F.psi_c.cpu().pin_memory()
        idx = torch.arange(cfg.volume)
        par = ((idx // cfg.L ** 3) + (idx // cfg.L ** 2) % cfg.L + (idx // cfg.L) % cfg.L + idx % cfg.L) % 2
        psi_e_h = psi_h[par == 0].contiguous().pin_memory()
        psi_o_h = psi_h[par == 1].contiguous().pin_memory()
        outs = {k: torch.empty_like(v).pin_memory() for k, v in (("f", psi_h), ("e", psi_e_h), ("o", psi_o_h))}
        H = hirep

        outs["e2"], outs["f2"] = torch.empty_like(outs["e"]).pin_memory(), torch.empty_like(outs["f"]).pin_memory()

        def host_step():
            # the five operators pipelined through hirep_apply_host_async (each result in its own pinned host buffer),
            # one hirep_sync at the end of the step: every input is copied host -> device and every result device -> host
            h = geom.handle
            H.hirep_apply_host_async(h, H.OP_DPHI_EO, m0, outs["e"].data_ptr(), psi_o_h.data_ptr(), links_h.data_ptr())
            H.hirep_apply_host_async(h, H.OP_DPHI_OE, m0, outs["o"].data_ptr(), psi_e_h.data_ptr(), None)
            H.hirep_apply_host_async(h, H.OP_DPHI, m0, outs["f"].data_ptr(), psi_h.data_ptr(), None)
            H.hirep_apply_host_async(h, H.OP_DPHI_HAT, m0, outs["e2"].data_ptr(), psi_e_h.data_ptr(), None)
            H.hirep_apply_host_async(h, H.OP_G5DPHI_SQ, m0, outs["f2"].data_ptr(), psi_h.data_ptr(), None)
            H.hirep_sync(h)

        nb = lambda t: t.numel() * t.element_size()
        h2d = nb(links_h) + 2 * nb(psi_h) + 2 * nb(psi_e_h) + nb(psi_o_h)
        d2h = 2 * nb(psi_h) + 2 * nb(psi_e_h) + nb(psi_o_h)
        ksteps = max(1, min(args.steps, 3))
        host_step()
        barrier()
        w0 = time.perf_counter()
        for _ in range(ksteps):
            host_step()
        torch.cuda.synchronize()
        w1 = time.perf_counter()
        ms_e2e = (w1 - w0) * 1e3 / ksteps
        ms_e2e = max_over_ranks(ms_e2e, dist, dev)
        e2e = {"value": round(aggregate_value(flops_step, world, ms_e2e), 2), "unit": "GFLOP/s", "ms_per_step": round(ms_e2e, 3),
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": ksteps,
               "api": "hirep_apply_host_async x5 + hirep_sync (pinned host canonical buffers; links copied once per step)"}
        del links_h, psi_h
    F.drop_canonical()
    torch.cuda.empty_cache()

    # ---- NEXT-1 row: linear algebra, reductions and CG on the same fields; outside the timed step
    extras = None
    if not args.no_extras and not rebuild:
        extras = measure_extras(torch, hirep, geom, cfg, prec, cm, m0, F.x[0], F.y[0], F.lr, peak)

    # ---- every BASELINE configuration x precision (+ C4 REBUILD), SURVEY 8(d) timing; rank 0 of a 1-GPU run only
    per_config, sweep_s = None, None
    if world == 1 and args.sweep != "none" and not args.custom:
        ts = time.perf_counter()
        per_config = {}
        wanted = SWEEP if args.sweep == "all" else [c for c in SWEEP if c[0] in args.sweep.split(",")]
        for name, pr, rb in wanted:
            key = "%s_%s%s" % (name, pr, "_rebuild" if rb else "")
            same = (name == args.config and pr == prec and rb == rebuild and not args.custom)
            if not same:
                need = sweep_bytes(synth.CONFIGS[name], pr, rb)
                if F is not None and torch.cuda.mem_get_info()[0] < need:
                    del geom
                    F = None            # the headline's fields make room for the big configurations
                    torch.cuda.empty_cache()
            try:
                per_config[key] = sweep_config(torch, hirep, synth, dev, name, pr, rb, peak, args.variant, F if same else None)
            except Exception as e:      # one configuration must not take the headline line down with it
                per_config[key] = {"error": "%s: %s" % (type(e).__name__, e)}
                torch.cuda.empty_cache()
        sweep_s = round(time.perf_counter() - ts, 1)

    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        cpu = cpu_baseline(args.config, prec)

    if rank == 0:
        roofline_c4 = None
        c4 = (per_config or {}).get("C4_f64", {}).get("ops", {}).get("Dphi_hat")
        if c4:
            roofline_c4 = {"bound": "hbm", "kernel": "C4 fp64 Dphi_hat (two hop stencil passes, d_R = 6)", "achieved": c4["gbs"], "peak": peak,
                           "unit": "GB/s", "frac": c4["frac_hbm"], "traffic": ncu_traffic("C4", "f64", "Dphi_hat"), "peak_source": peak_src,
                           "algorithmic_bytes": cost_model(synth.CONFIGS["C4"], "f64")["ops"]["Dphi_hat"][1],
                           "frac_of_8TBs_nominal": c4["frac_8TBs_nominal"],
                           "timing": "back-to-back launches, median of 5 repeats (sustained: the SM clock under the power cap is in per_config.C4_f64.clocks)",
                           "in_step": {"ms": c4["ms_in_step"], "frac": round(c4["frac_hbm"] * c4["ms"] / c4["ms_in_step"], 4)}}
        b2b = (per_config or {}).get("%s_%s%s" % (args.config, prec, "_rebuild" if rebuild else ""), {}).get("ops", {}).get("Dphi_eo")
        if b2b:
            roofline["back_to_back"] = {"ms": b2b["ms"], "achieved": b2b["gbs"], "frac": b2b["frac_hbm"]}
        out = {
            "metric": METRIC, "value": round(value, 1), "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": round(ms_step, 4), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": prec, "data": "synthetic",
            "config": {"workload": "%s: SU(%d) %s (d_R=%d) %dx%d^3 %s; step = links_to_rep + Dphi_eo + Dphi_oe + Dphi + Dphi_hat + g5Dphi_sq"
                                   % (cfg.name, cfg.n_g, synth.REP_NAMES[cfg.rep], cfg.d_R, cfg.T, cfg.L, prec),
                       "links": ("fundamental links, R rebuilt in registers (link mode REBUILD; no links_to_rep in the step)" if rebuild
                                 else "stored represented links (gather layout)"), "kernel_variant": args.variant,
                       "l2": "inputs larger than L2: each step streams %.2f GB of links and spinors (L2 = 126 MB) and rotates over %d spinor sets"
                             % (sum(cm["ops"][k][1] for k in ops_run) / 1e9, NSETS),
                       "parallelism": "replicas x%d (no sharding; DESIGN.md)" % world},
            "gpu_launches": launches,
            "per_op": per_op,
            "roofline": roofline,
            "roofline_C4_f64_Dphi_hat": roofline_c4,
            "e2e": e2e,
            "per_config": per_config,
            "per_config_seconds": sweep_s,
            "next1_linalg_cg": extras,
            "cpu_baseline": cpu,
            "clocks": clocks,
        }
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def sweep_bytes(cfg, prec, rebuild):
    """device memory one configuration of the sweep needs: links (fundamental + represented), canonical inputs while they
    are imported, 2 x NSETS full spinors, work space of the two-pass operators"""
    w = 8 if prec == "f64" else 4
    V, d, N = cfg.volume, cfg.d_R, cfg.n_g
    S = 8 * d * w
    K = d * d * (1 if cfg.rep == 1 else 2) * w
    KF = 2 * N * N * w
    return V * (8 * KF + (0 if rebuild else 8 * K) + 4 * KF + (2 * NSETS + 3) * S) + (2 << 30)


def measure_clover(torch, hirep, geom, cfg, prec, cm, m0, x_full, y_full, lr, peak, light=False):
    """NEXT-2: clover set-up kernels and operators on resident fields.  light: the per_config form (no CG, no exponential clover)."""
    V, S, d = cfg.volume, cm["S"], cfg.d_R
    iters = 20

    def timeit(fn, reps=20):
        fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    out = {}
    # NEXT-2, second part: clover term (Eq 47-49).  Algorithmic bytes per site: clover field 4 d^2 complex + spinor in/out.
    d = cfg.d_R
    cb = S * d                                          # clover bytes per site: 4 d^2 complex (S = 4 d complex)
    if torch.cuda.mem_get_info()[0] < 2 * cb * V + (4 << 30):
        out["clover"] = {"skipped": "clover field of %.1f GB does not fit beside the resident fields" % (cb * V / 1e9)}
    else:
        lbytes = geom.sizes["links_rep"] / V            # represented-link bytes per site
        cl = geom.clover_field(lr)
        ms = timeit(lambda: geom.clover_field(lr, out=cl), reps=3)
        out["clover_field"] = {"ms": round(ms, 3), "note": "once per gauge update; 72 d_R^3 complex MACs per site out of the gather-layout links"}
        ms = timeit(lambda: geom.Cphi(m0, 1.0, x_full, cl, out=y_full))
        by = (cb + 2 * S) * V
        out["Cphi"] = {"ms": round(ms, 4), "gbs": round(by / ms / 1e6, 1), "frac_hbm": round(by / ms / 1e6 / peak, 3)}
        # Site-diagonal matrices inside the stencil epilogues ("fused into the second pass") where the ring kernel carries
        # them (stored links, d_R <= 6: ring / pair kernels), else separate block-apply launches.  Fractions are on the compulsory bytes
        # of the fused form (every field once); the composed form moves 2S more per block application and is timed beside it.
        fused_diag = d <= 6

        def both_forms(fn, by, nl_fused, nl_composed):
            ms = timeit(fn, reps=10)
            r = {"ms": round(ms, 4), "gbs": round(by / ms / 1e6, 1), "frac_hbm": round(by / ms / 1e6 / peak, 3),
                 "launches": nl_fused if fused_diag else nl_composed, "fused_epilogue": bool(fused_diag)}
            if fused_diag:
                geom.set_tuning(hirep.TUNE_FUSE_DIAG, 0)
                r["ms_composed"] = round(timeit(fn, reps=10), 4)
                r["launches_composed"] = nl_composed
                geom.set_tuning(hirep.TUNE_FUSE_DIAG, 1)
            return r

        out["Dphi_clover"] = both_forms(lambda: geom.Dphi_clover(m0, 1.0, x_full, lr, cl, out=y_full), (cb + lbytes + 2 * S) * V, 1, 2)   # in is both neighbour data and self term: 2S
        # the Schur form Eq 43 with these blocks: block inverse (once per gauge update and mass), its application, D_hat
        hb = geom.sizes["spinor_half"]
        x_e, y_e = x_full[:hb], y_full[:hb]
        inv = geom.clover_inv_field(m0, 0.5, hirep.ODD, cl)
        ms = timeit(lambda: geom.clover_inv_field(m0, 0.5, hirep.ODD, cl, out=inv), reps=3)
        out["clover_inv_field"] = {"ms": round(ms, 3), "note": "in-place Gauss-Jordan of the 2 d_R x 2 d_R blocks of the odd sites"}
        ms = timeit(lambda: geom.Cphi_inv(hirep.ODD, x_e, inv, out=y_e))
        by = (2 * cb + 2 * S) * V / 2                    # full blocks: 8 d^2 complex per site, one parity
        out["Cphi_inv"] = {"ms": round(ms, 4), "gbs": round(by / ms / 1e6, 1), "frac_hbm": round(by / ms / 1e6 / peak, 3)}
        # two stencil passes (2S + 8K each) + the even input once more as the self term + inverse blocks (2 cb) + clover H, B (cb)
        by = cm["ops"]["Dphi_eo"][1] * 2 + S * V / 2 + 3 * cb * V / 2
        out["Dphi_clover_hat"] = both_forms(lambda: geom.Dphi_clover_hat(m0, 0.5, x_e, lr, cl, inv, out=y_e), by, 2, 4)
        try:    # even-odd preconditioned CG with the clover term: Q_hat^2 = 2 x (the launches above), then the CG's linear algebra
            if light:
                raise StopIteration
            geom.cg_g5Dphi_clover_hat_sq(m0, 0.5, x_e, lr, cl, inv, 1e-30, 2, out=y_e)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            _, it, res = geom.cg_g5Dphi_clover_hat_sq(m0, 0.5, x_e, lr, cl, inv, 1e-30, iters, out=y_e)
            torch.cuda.synchronize()
            ms_it = (time.perf_counter() - t0) * 1e3 / max(it, 1)
            # fused form: the CG's reductions ride in the epilogues of the second pass of each Q_hat (r read + write, x / p update, A p never stored)
            by_it = 2 * by + ((2 + 5 - 1) if fused_diag else (1 + 3 + 5)) * S * V / 2
            out["cg_g5Dphi_clover_hat_sq"] = {"iterations": it, "ms_per_iteration": round(ms_it, 4), "gbs": round(by_it / ms_it / 1e6, 1),
                                              "frac_hbm": round(by_it / ms_it / 1e6 / peak, 3), "launches_per_iteration": 7 if fused_diag else 13, "fused_reductions": bool(fused_diag),
                                              "relres_after": res}
        except StopIteration:
            pass
        except Exception as e:
            out["cg_g5Dphi_clover_hat_sq"] = {"error": str(e)}
        del inv
        # exponential clover (Eq 50): full 2 d_R x 2 d_R blocks on both parities (8 d^2 complex per site)
        if not light and d <= 10 and torch.cuda.mem_get_info()[0] > 6 * cb * V + (4 << 30):
            nb = hirep.hirep_clover_inv_bytes(geom.handle)
            E = geom.clover_exp_field(m0, 1.0, cl)
            ms = timeit(lambda: hirep.hirep_clover_exp_field(geom.handle, m0, 1.0, hirep.ODD, 0, E[nb:].data_ptr(), cl.data_ptr()), reps=3)
            out["clover_exp_field"] = {"ms": round(ms, 3), "note": "one parity; scaling and squaring, 18 block products per site and chirality"}
            Ei = geom.clover_exp_field(m0, 1.0, cl, inverse=True)
            out["Dphi_expclover"] = both_forms(lambda: geom.Dphi_blocks(x_full, lr, E, out=y_full), (2 * cb + lbytes + 2 * S) * V, 1, 2)
            by = cm["ops"]["Dphi_eo"][1] * 2 + S * V / 2 + 4 * cb * V / 2
            out["Dphi_expclover_hat"] = both_forms(lambda: geom.Dphi_blocks_hat(x_e, lr, E, Ei[nb:], out=y_e), by, 2, 4)
            del E, Ei
        del cl
    return out


def measure_extras(torch, hirep, geom, cfg, prec, cm, m0, x_full, y_full, lr, peak):
    """GB/s of the streaming kernels (full-lattice spinors) and ms per CG iteration of hirep_cg_g5Dphi_sq."""
    V, S, d = cfg.volume, cm["S"], cfg.d_R
    z_full = geom.new_spinor(hirep.FULL)
    z_full.copy_(x_full)

    def timeit(fn, reps=20):
        fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    out = {}
    ms = timeit(lambda: geom.lc(hirep.FULL, y_full, 0.5, x_full, -1.5, z_full))
    out["lc"] = {"ms": round(ms, 4), "gbs": round(3 * S * V / ms / 1e6, 1), "frac_hbm": round(3 * S * V / ms / 1e6 / peak, 3)}
    ms = timeit(lambda: geom.lc1(hirep.FULL, y_full, 0.5 + 0.25j, x_full))
    out["lc1"] = {"ms": round(ms, 4), "gbs": round(3 * S * V / ms / 1e6, 1), "frac_hbm": round(3 * S * V / ms / 1e6 / peak, 3)}
    ms = timeit(lambda: geom.sqnorm(hirep.FULL, x_full))
    out["sqnorm"] = {"ms": round(ms, 4), "gbs": round(S * V / ms / 1e6, 1), "frac_hbm": round(S * V / ms / 1e6 / peak, 3),
                     "note": "includes the result read-back and stream synchronisation"}
    ms = timeit(lambda: geom.prod(hirep.FULL, x_full, z_full))
    out["prod"] = {"ms": round(ms, 4), "gbs": round(2 * S * V / ms / 1e6, 1), "frac_hbm": round(2 * S * V / ms / 1e6 / peak, 3)}
    # CG: a fixed number of iterations on a well-conditioned mass so that every iteration does the same work
    iters = 20
    geom.cg_g5Dphi_sq(2.0, x_full, lr, 1e-30, 2, out=y_full)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    _, it, res = geom.cg_g5Dphi_sq(2.0, x_full, lr, 1e-30, iters, out=y_full)
    torch.cuda.synchronize()
    ms_it = (time.perf_counter() - t0) * 1e3 / max(it, 1)
    fl_it = cm["ops"]["g5Dphi_sq"][0]
    # compulsory bytes of one iteration: two full-lattice stencil passes (2S + 4K each; the fused form never stores A p: -S) plus the
    # linear algebra -- unfused: ||B p||^2 (1) + r update (3) + x, p update (5) spinor passes; fused into the stencil epilogues
    # (tile-pair kernel: complex links d_R <= 3, fp32 also d_R = 4, 6; real SU(2) adjoint in fp64): r read + write (2) + x, p update (5)
    fused = (d <= 3 and (prec == "f64" or cfg.rep != 1)) or (prec == "f32" and cfg.rep != 1 and d in (4, 6))
    by_it = cm["ops"]["g5Dphi_sq"][2] + ((2 + 5 - 1) if fused else (1 + 3 + 5)) * S * V
    out["cg_g5Dphi_sq"] = {"iterations": it, "ms_per_iteration": round(ms_it, 4), "gflops_operator": round(fl_it / ms_it / 1e6, 1),
                           "gbs": round(by_it / ms_it / 1e6, 1), "frac_hbm": round(by_it / ms_it / 1e6 / peak, 3),
                           "launches_per_iteration": 5 if fused else 7, "fused_reductions": fused, "relres_after": res}
    hb = geom.sizes["spinor_half"]
    x_e, y_e = x_full[:hb], y_full[:hb]
    geom.cg_g5Dphi_hat_sq(2.0, x_e, lr, 1e-30, 2, out=y_e)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    _, it, res = geom.cg_g5Dphi_hat_sq(2.0, x_e, lr, 1e-30, iters, out=y_e)
    torch.cuda.synchronize()
    ms_it = (time.perf_counter() - t0) * 1e3 / max(it, 1)
    fl_it = 2 * cm["ops"]["Dphi_hat"][0]
    # same accounting on the even sites; the ring / pair kernels (d_R <= 6, stored links) carry the reductions in the epilogue of the
    # second pass of each Q_hat: ||Q_hat p||^2 with the first, r -= alpha A p and ||r||^2 (A p never stored) with the second
    fused_eo = d <= 6
    by_it = 2 * cm["ops"]["Dphi_hat"][1] + ((2 + 5 - 1) if fused_eo else (1 + 3 + 5)) * S * V / 2
    out["cg_g5Dphi_hat_sq"] = {"iterations": it, "ms_per_iteration": round(ms_it, 4), "gflops_operator": round(fl_it / ms_it / 1e6, 1),
                               "gbs": round(by_it / ms_it / 1e6, 1), "frac_hbm": round(by_it / ms_it / 1e6 / peak, 3),
                               "launches_per_iteration": 7 if fused_eo else 9, "fused_reductions": fused_eo, "relres_after": res}
    ms = timeit(lambda: geom.Dphi_tm_hat(m0, 0.3, x_e, lr, out=y_e), reps=10)
    by = cm["ops"]["Dphi_hat"][1]                          # D_oo^-1 = (a - i mu gamma_5)/(a^2 + mu^2) rides in the epilogue of the D_oe pass
    out["Dphi_tm_hat"] = {"ms": round(ms, 4), "gbs": round(by / ms / 1e6, 1), "frac_hbm": round(by / ms / 1e6 / peak, 3),
                          "gflops": round(cm["ops"]["Dphi_hat"][0] / ms / 1e6, 1), "launches": 2}
    out.update(measure_clover(torch, hirep, geom, cfg, prec, cm, m0, x_full, y_full, lr, peak))
    # NEXT-4: fermion force of the hopping term (Eq 20-21): both fields and the forward links once, N^2-1 reals per link out
    try:
        na = cfg.n_g ** 2 - 1
        w = 8 if prec == "f64" else 4
        fbuf = geom.force_hopping(x_full, z_full, lr)
        ms = timeit(lambda: geom.force_hopping(x_full, z_full, lr, out=fbuf), reps=10)
        by = (2 * S + 4 * cm["K"] + 4 * na * w) * V
        out["force_hopping"] = {"ms": round(ms, 4), "gbs": round(by / ms / 1e6, 1), "frac_hbm": round(by / ms / 1e6 / peak, 3),
                                "note": "compulsory bytes (2S + 4K + 4(N^2-1)w) per site; d_R <= 4 (fp32: 6): one warp per tile walks the four mu, M in registers; fp64 d_R = 5, 6: two warps per tile; d_R >= 8: one warp per (tile, mu), vectors in shared memory"}
        del fbuf
    except Exception as e:
        out["force_hopping"] = {"error": str(e)}
    try:
        out["fma_peak_tflops"] = {"f64": round(hirep.hirep_fma_peak(hirep.F64), 2), "f32": round(hirep.hirep_fma_peak(hirep.F32), 2)}
    except Exception as e:   # measurement utility only
        out["fma_peak_tflops"] = {"error": str(e)}
    return out


# ------------------------------------------------------------------------------- oracle arm / cpu baseline
def prepare_sample(config, prec, T, L):
    from harness import synth
    cfg = synth.CONFIGS[config].resized(T, L)
    U, (psi,) = synth.make_inputs(cfg)
    U, psi = synth.round_to_precision(U, prec), synth.round_to_precision(psi, prec)
    return cfg, U, psi, synth.parity_sites(T, L, 0), synth.parity_sites(T, L, 1)


def oracle_step(prep):
    """One step (the same six ops) of the oracle, as it stands, on the prepared sample; returns seconds."""
    from oracle import oracle as orc
    cfg, U, psi, ev, od = prep
    T, L, d, m0 = cfg.T, cfg.L, cfg.d_R, cfg.m0
    t0 = time.perf_counter()
    R = orc.represent_field(cfg.n_g, cfg.rep, U)
    orc.Dphi_eo(T, L, d, R, psi[od]); orc.Dphi_oe(T, L, d, R, psi[ev]); orc.Dphi(T, L, d, m0, R, psi)
    orc.Dphi_hat(T, L, d, m0, R, psi[ev]); orc.g5Dphi_sq(T, L, d, m0, R, psi)
    return time.perf_counter() - t0


def sample_flops(prep):
    cm = cost_model(prep[0], "f64")
    return sum(cm["ops"][k][0] for k in OP_ORDER)


SAMPLE = {"C1": (4, 4), "C2": (16, 16), "C3": (16, 16), "C4": (8, 8), "C5": (4, 4)}   # small sub-lattice samples
SAMPLE_BIG = {"C1": (4, 4), "C2": (32, 32), "C3": (24, 24), "C4": (12, 12), "C5": (8, 4)}  # larger ones (C1, C2: the full lattice)


def pick_sample(config, prec, n_steps, budget_s):
    """The larger of the two sample lattices if n_steps oracle steps on it fit budget_s: one step of the small sample is
    timed and the big one extrapolated by volume (the oracle's cost is linear in the number of sites)."""
    small = prepare_sample(config, prec, *SAMPLE[config])
    t_small = oracle_step(small)
    Tb, Lb = SAMPLE_BIG[config]
    ratio = (Tb * Lb ** 3) / float(SAMPLE[config][0] * SAMPLE[config][1] ** 3)
    if ratio > 1 and t_small * ratio * n_steps * 1.3 <= budget_s:
        return prepare_sample(config, prec, Tb, Lb), (Tb, Lb)
    return small, SAMPLE[config]


def cpu_baseline(config, prec):
    """The oracle as it stands on the host cores: whole steps on a bounded sample, repeated for about 10-20 s."""
    from oracle import oracle as orc
    prep, (T, L) = pick_sample(config, prec, 3, 30.0)
    secs, n = 0.0, 0
    while n < 1 or (secs < 10.0 and n < 200):
        secs += oracle_step(prep)
        n += 1
    return {"value": round(n * sample_flops(prep) / secs / 1e9, 3), "unit": "GFLOP/s", "cores": orc.num_threads(), "kind": "oracle",
            "sample": "%d steps (same six ops) of %s on a %dx%d^3 lattice, %.1f s of oracle time" % (n, config, T, L, secs)}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as orc
    from harness import synth
    prep, (T, L) = pick_sample(args.config, args.prec, args.steps + min(args.warmup, 1), 150.0)
    for _ in range(min(args.warmup, 1)):
        oracle_step(prep)
    secs = [oracle_step(prep) for _ in range(args.steps)]
    ms_step = sum(secs) * 1e3 / len(secs)
    gf = sample_flops(prep) / (ms_step * 1e-3) / 1e9
    cores, cfg = orc.num_threads(), synth.CONFIGS[args.config]
    sample = "one step (same six ops) of %s on a %dx%d^3 lattice" % (args.config, T, L)
    out = {"impl": "reference", "metric": METRIC, "value": round(gf, 3), "unit": "GFLOP/s", "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(ms_step, 2), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": "%s: SU(%d) %s (d_R=%d) %dx%d^3 %s; step = links_to_rep + Dphi_eo + Dphi_oe + Dphi + Dphi_hat + g5Dphi_sq"
                                  % (cfg.name, cfg.n_g, synth.REP_NAMES[cfg.rep], cfg.d_R, cfg.T, cfg.L, args.prec),
                      "sample": sample},
           "gpu_launches": 0,
           "cpu_baseline": {"value": round(gf, 3), "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": round(gf, 3), "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C2", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--prec", default="f64", choices=["f64", "f32"])
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--custom", default="", help="N_g,rep,T,L instead of --config (rep: 0 FUND, 1 ADJ, 2 SYM, 3 2AS); per-op table only")
    ap.add_argument("--link-mode", default="stored", choices=["stored", "rebuild"])
    ap.add_argument("--sweep", default="all", help="per_config sweep after the headline: all | none | comma list of C2..C5")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the linear-algebra / CG measurements")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
