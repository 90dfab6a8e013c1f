#!/usr/bin/env python
"""bench.py -- throughput of the fused twisted-mass dslash hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--profile-brief]

One STEP = one pass of the whole hot path over the 32^3x64 lattice (BASELINE.json configs[2] and configs[3]):
  degenerate doublet (Haar links, 12-real, kappa=0.1632, mu=0.0015):   for fp64, fp32, half:  LHS of Eq. 2.2 (ASYM)
                                                                        and LHS of Eq. 2.3 (SYM)   [PAPER.md:60-62]
  non-degenerate doublet (exp(i 0.3 H) links, 12-real, mu=0.15, eps=0.19):  for fp32, half:  ASYM plain and ASYM dagger
i.e. 10 tm_mat_pc calls = 20 fused-kernel launches (kernel types A, B, A-xpay; plain and dagger; 1 and 2 flavors;
three precisions; 12-real link rebuild; half quantisation).  value = flops of a step / time, in GFLOPS, with the flop
counts of DESIGN.md section 7 (1320 per hop + local terms).  Inputs are seeded synthetic fields resident in HBM; the
gauge fields (201-805 MB each) and the sweep's working set are far larger than the 126 MB L2.

Multi-GPU: the path does not shard (BASELINE.json: one GPU, no halo exchange) -> replicas only; with --gpus N every
rank runs the same step on its own GPU, value = N x units / max-over-ranks time, scaling "weak".

--impl reference times the CPU oracle (oracle/, fp64, as it stands) on the host cores on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

DIMS = (32, 32, 32, 64)
KAPPA = 0.1632
DEG = dict(mu=0.0015, epsilon=0.0, twist_flavor=1)          # configs[2]
NDEG = dict(mu=0.15, epsilon=0.19, twist_flavor=0)          # configs[3]
SEED_DEG, SEED_NDEG = 3, 4
RECON = 12
PREC_NAME = {8: "fp64", 4: "fp32", 2: "half"}
KT_NAME = {0: "A", 1: "A-xpay", 2: "B", 3: "REC"}
ASYM, SYM = 0, 1

# Paper's Table 1 (GTX Titan, 12-real): context only, another machine.
PAPER_GFLOPS = {(1, 8): 190, (1, 4): 415, (1, 2): 759, (2, 8): 163, (2, 4): 516, (2, 2): 879}
PAPER_GFLOPS_8REAL = {(1, 8): 183, (1, 4): 487, (1, 2): 858, (2, 8): 115, (2, 4): 567, (2, 2): 624}


def flops_per_site(nf, kt):
    """hop 1320 / flavor; deg R 48, inverse scale +24, axpy +48; ndeg R 192, R^-1 240, axpy 96."""
    if nf == 1:
        return {0: 1392, 1: 1440, 2: 1416, 3: 1440}[kt]
    return {0: 2880, 1: 2976, 2: 2928, 3: 2976}[kt]


def bytes_per_site(nf, prec, recon, kt):
    """Algorithmic bytes per output site: every link once, input spinor once, output once, x once (+ half norms)."""
    x = 0 if kt == 0 else 1
    return 8 * recon * prec + nf * 24 * prec * (2 + x) + (4 * nf * (2 + x) if prec == 2 else 0)


def step_ops():
    """The composites of one step: (nf, prec, matpc type, dagger)."""
    ops = []
    for prec in (8, 4, 2):
        ops += [(1, prec, ASYM, 0), (1, prec, SYM, 0)]
    for prec in (4, 2):
        ops += [(2, prec, ASYM, 0), (2, prec, ASYM, 1)]
    return ops


def op_kernels(op):
    nf, prec, typ, dagger = op
    return [(nf, prec, 0, dagger), (nf, prec, 2 if typ == ASYM else 1, dagger)]


def op_flops(op, vh):
    return sum(flops_per_site(nf, kt) for nf, _, kt, _ in op_kernels(op)) * vh


def op_bytes(op, vh):
    return sum(bytes_per_site(nf, prec, RECON, kt) for nf, prec, kt, _ in op_kernels(op)) * vh


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons while the GPU is under load (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 <= t <= t1] or [r for _, r in self.rows[-3:]]
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            f = [c.strip() for c in r.split(",")]
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except Exception:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def reduce_over_ranks(ms_local, world):
    """Max over ranks of the device time (bench contract); gloo/nccl all_reduce, identity when world == 1."""
    if world == 1:
        return ms_local
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def ncu_traffic(name):
    """DRAM read+write bytes per launch of kernel `name` from the committed ncu --set full summary, or None."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None
    for line in open(path):
        f = [c.strip() for c in line.split(";")]
        if len(f) >= 2 and f[0] == name:
            try:
                return float(f[1])
            except ValueError:
                return None
    return None


class Workload:
    """Device-resident inputs of one step (seeded synthetic stand-ins for the paper's ensembles)."""

    def __init__(self, device, log, slab=None):
        import torch
        import paper_1311_4462_b200 as tm
        import synth_inputs as si
        self.tm, self.si, self.torch = tm, si, torch
        # --sharded: this rank's 32^3x64 slab of a 32^3 x (64 N) lattice (the same seeded fields on every slab: N copies stacked
        # along x4 are a valid gauge field), kernels with open time hops + face exchange (paper_1311_4462_b200/sharded.py)
        self.slab = slab
        self.lat = slab.lat if slab is not None else tm.Lattice(DIMS, device)
        self.vh = self.lat.Vh
        t = time.time()
        self.host_gauge = {1: si.gauge_field(DIMS, SEED_DEG, "haar"), 2: si.gauge_field(DIMS, SEED_NDEG, "near_identity")}
        self.host_in = {1: si.to_parity(si.spinor_field(DIMS, 1, SEED_DEG), DIMS, 0),
                        2: si.to_parity(si.spinor_field(DIMS, 2, SEED_NDEG), DIMS, 0)}
        log("host inputs generated in %.1f s" % (time.time() - t))
        self.params = {1: tm.params(KAPPA, **DEG), 2: tm.params(KAPPA, **NDEG)}
        self.gauge, self.fin, self.ftmp, self.fout = {}, {}, {}, {}
        for nf, prec, _, _ in step_ops():
            key = (nf, prec)
            if key in self.gauge:
                continue
            self.gauge[key] = self.lat.gauge(self.host_gauge[nf], prec, RECON)
            self.fin[key] = self.lat.field(prec, nf).upload_cb(0, self.host_in[nf])
            self.ftmp[key], self.fout[key] = self.lat.field(prec, nf), self.lat.field(prec, nf)
        self.lat.sync()

    def mat_pc(self, key, nf, typ, dagger):
        if self.slab is not None:
            self.slab.mat_pc(self.fout[key], self.fin[key], self.ftmp[key], self.gauge[key], self.params[nf], typ, dagger)
        else:
            self.tm.mat_pc(self.fout[key], self.fin[key], self.ftmp[key], self.gauge[key], self.params[nf], typ, dagger)

    def step(self):
        for nf, prec, typ, dagger in step_ops():
            self.mat_pc((nf, prec), nf, typ, dagger)

    def make_pinned(self):
        torch = self.torch
        self.pin_in, self.pin_out = {}, {}
        for nf in (1, 2):
            n = nf * self.vh * 24
            a = torch.empty(n, dtype=torch.float64, pin_memory=True)
            a.numpy()[:] = self.host_in[nf].view(np.float64).reshape(-1)
            self.pin_in[nf] = a
            self.pin_out[nf] = torch.empty(n, dtype=torch.float64, pin_memory=True)

    def step_e2e(self):
        """The same step through the C-ABI with HOST buffers: upload in_e, tm_mat_pc, download out_e, per composite.
        The asynchronous entry points overlap the H2D copy of the next input, the kernels and the D2H copy of the
        previous result; tm_sync at the end of the step: every result of the step is on the host when it returns."""
        tm = self.tm
        h2d = d2h = 0
        for nf, prec, typ, dagger in step_ops():
            key = (nf, prec)
            tm.tm_field_upload_cb_async(self.fin[key].h, 0, self.pin_in[nf].data_ptr())
            self.mat_pc(key, nf, typ, dagger)
            tm.tm_field_download_cb_async(self.fout[key].h, 0, self.pin_out[nf].data_ptr())
            h2d += self.pin_in[nf].numel() * 8
            d2h += self.pin_out[nf].numel() * 8
        self.lat.sync()
        return h2d, d2h


def oracle_step(ora, si, dims, gauge, inp, sample_desc):
    """One pass of the step's four distinct operators through the CPU oracle (fp64); returns (seconds, flops)."""
    vh = si.volume(dims) // 2
    t = time.time()
    flops = 0
    for nf, kw, ops in ((1, DEG, ((ASYM, 0), (SYM, 0))), (2, NDEG, ((ASYM, 0), (ASYM, 1)))):
        p = ora.params(dims, KAPPA, **kw)
        for typ, dagger in ops:
            ora.matpc(inp[nf], gauge[nf], p, typ, dagger)
            flops += op_flops((nf, 8, typ, dagger), vh)
    return time.time() - t, flops


def run_reference(args, log):
    """--impl reference: the oracle as it stands on the host cores, bounded sample = a 32^3 x 8 time slab."""
    import oracle as ora
    import synth_inputs as si
    dims = (32, 32, 32, 8)
    gauge = {1: si.gauge_field(dims, SEED_DEG, "haar"), 2: si.gauge_field(dims, SEED_NDEG, "near_identity")}
    inp = {nf: si.mask_parity(si.spinor_field(dims, nf, s), dims, 0) for nf, s in ((1, SEED_DEG), (2, SEED_NDEG))}
    sample = "32^3x8 time slab (1/8 of the 32^3x64 lattice), the step's 4 distinct operators (deg ASYM, SYM; ndeg ASYM, ASYM-dagger) once each in fp64"
    for _ in range(args.warmup):
        oracle_step(ora, si, dims, gauge, inp, sample)
    tot_s, tot_f = 0.0, 0
    for _ in range(args.steps):
        s, f = oracle_step(ora, si, dims, gauge, inp, sample)
        tot_s += s
        tot_f += f
    val = tot_f / tot_s / 1e9
    cores = ora.num_threads()
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": "GFLOPS", "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": WORKLOAD % (RECON, RECON), "sample": sample},
           "cpu_baseline": {"value": val, "unit": "GFLOPS", "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": "GFLOPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


METRIC = "twisted-mass dslash GFLOPS (even-odd preconditioned operators, Eq. 2.2/2.3, 32^3x64, fp64+fp32+half sweep)"
WORKLOAD = ("32^3x64: configs[2] degenerate (Haar links, %d-real, mu=0.0015) ASYM+SYM in fp64/fp32/half + configs[3] "
            "non-degenerate (exp(i0.3H) links, %d-real, mu=0.15, eps=0.19) ASYM plain+dagger in fp32/half")
# plain-ALU peak: 128 FP32 / 64 FP64 FMA lanes per SM, 148 SMs, 2 flop per FMA, at the SM clock under load
SMS, LANES = 148, {8: 64, 4: 128, 2: 128}


def run_ours(args, log):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_1311_4462_b200 as tm
    slab = None
    if args.sharded:
        from paper_1311_4462_b200 import sharded
        slab = sharded.Slab((DIMS[0], DIMS[1], DIMS[2], DIMS[3] * world), rank, world, local)
    w = Workload(local, log, slab)
    lat, vh = w.lat, w.vh
    tm.tm_set_path(lat.ctx, args.path)
    ops = step_ops()
    step_flops = sum(op_flops(o, vh) for o in ops)
    step_bytes = sum(op_bytes(o, vh) for o in ops)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, K timed steps, per-launch events inside the timed region
    phys = os.environ.get("CUDA_VISIBLE_DEVICES", "").split(",")
    smi_index = phys[local] if len(phys) > local and phys[local] else str(local)
    sampler = ClockSampler(smi_index)
    for _ in range(max(args.warmup, 3)):
        w.step()
    barrier()
    tm.tm_timing_enable(lat.ctx, 1)
    n0 = lat.launches()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    ev0.record()
    for _ in range(args.steps):
        w.step()
    ev1.record()
    barrier()
    t1 = time.time()
    ms_local = ev0.elapsed_time(ev1)
    launches = lat.launches() - n0
    records = tm.tm_timing_read(lat.ctx, 1 << 20)
    tm.tm_timing_enable(lat.ctx, 0)
    clocks = sampler.stop(t0, t1)
    ms = reduce_over_ranks(ms_local, world)
    ms_per_step = ms / args.steps
    value = world * step_flops / (ms_per_step * 1e-3) / 1e9

    # ---- per-kernel roofline from the events recorded inside the timed region
    peak, peak_src = measured_peak()
    step_kernels = [k for op in ops for k in op_kernels(op)]        # launch order inside one step
    assert len(records) == args.steps * len(step_kernels), (len(records), args.steps, len(step_kernels))
    per = {}
    for i, (name, t) in enumerate(records):
        a = per.setdefault(step_kernels[i % len(step_kernels)], [0.0, 0, name])
        a[0] += t
        a[1] += 1
        assert a[2] == name, (a[2], name)
    total_ms = sum(v[0] for v in per.values())
    kernels = []
    for (nf, prec, kt, dagger), (tot, cnt, name) in per.items():
        avg_ms = tot / cnt
        b = bytes_per_site(nf, prec, RECON, kt) * vh
        f = flops_per_site(nf, kt) * vh
        gbs = b / (avg_ms * 1e-3) / 1e9
        kernels.append({"kernel": name, "flavors": nf, "prec": PREC_NAME[prec], "type": KT_NAME[kt], "dagger": dagger,
                        "launches": cnt, "us": 1e3 * avg_ms, "gflops": f / (avg_ms * 1e-3) / 1e9,
                        "alg_gbs": gbs, "frac_of_measured_peak": gbs / peak, "frac_of_8TBs": gbs / 8000.0,
                        "bytes_per_site": bytes_per_site(nf, prec, RECON, kt), "flops_per_site": flops_per_site(nf, kt),
                        "share_of_step": tot / total_ms, "prec_bytes": prec})
    dom = max(kernels, key=lambda k: k["share_of_step"]) if kernels else None
    roofline = None
    if dom:
        roofline = {"bound": "hbm", "kernel": dom["kernel"], "achieved": dom["alg_gbs"], "peak": peak, "unit": "GB/s",
                    "frac": dom["alg_gbs"] / peak, "traffic": ncu_traffic(dom["kernel"]), "peak_source": peak_src,
                    "bytes_per_launch": dom["bytes_per_site"] * vh, "us_per_launch": dom["us"],
                    "step_alg_gbs": step_bytes / (ms_per_step * 1e-3) / 1e9,
                    "step_frac": step_bytes / (ms_per_step * 1e-3) / 1e9 / peak}

    # ---- end to end through the C-ABI with pinned HOST buffers (copies inside the timed region)
    w.make_pinned()
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    w.step_e2e()
    barrier()
    tw0 = time.time()
    ev0.record()
    for _ in range(e2e_steps):
        h2d, d2h = w.step_e2e()
    ev1.record()
    barrier()
    e2e_ms = reduce_over_ranks(max(ev0.elapsed_time(ev1), 1e3 * (time.time() - tw0)), world) / e2e_steps
    e2e = {"value": world * step_flops / (e2e_ms * 1e-3) / 1e9, "unit": "GFLOPS", "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms, "steps": e2e_steps,
           "note": "per composite: tm_field_upload_cb_async (pinned host, fp64 canonical) + tm_mat_pc + tm_field_download_cb_async, "
                   "tm_sync per step; copies in both directions overlap each other and the kernels"}

    # ---- CPU baseline: the oracle as it stands, on this box's host cores (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle as ora
        si = w.si
        inp = {nf: si.from_parity(w.host_in[nf], DIMS, 0) for nf in (1, 2)}
        sample = "one fp64 pass of the step's 4 distinct operators (deg ASYM, SYM; ndeg ASYM, ASYM-dagger) on the full 32^3x64 lattice"
        s, f = oracle_step(ora, si, DIMS, w.host_gauge, inp, sample)
        cpu = {"value": f / s / 1e9, "unit": "GFLOPS", "cores": ora.num_threads(), "kind": "oracle", "sample": sample,
               "seconds": s}

    # second roofline per kernel: useful flops against the plain-ALU peak at the clock seen under load
    sm_mhz = (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz") or 1965.0
    for k in kernels:
        alu_peak = SMS * LANES[k.pop("prec_bytes")] * 2 * sm_mhz * 1e-3      # GFLOPS
        k["alu_peak_gflops"] = alu_peak
        k["frac_of_alu_peak"] = k["gflops"] / alu_peak
        # the half kernels are limited by the FP32 pipe (ncu fma pipe 63-66 % busy, math-pipe throttle the top
        # stall, same run time with 32 % more link bytes); everything else by HBM
        k["bound"] = "alu" if k["prec"] == "half" else "hbm"
    if rank == 0:
        out = {"metric": METRIC, "value": value, "unit": "GFLOPS", "n_gpus": world, "steps": args.steps,
               "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
               "vs_baseline": None, "dtype": "f64+f32+i16/f32", "data": "synthetic",
               "config": {"workload": WORKLOAD % (RECON, RECON), "lattice": list(DIMS), "recon": RECON, "kappa": KAPPA,
                          "parallelism": ("time-direction slabs of a 32^3 x %d lattice, one per GPU, face exchange per dslash (--sharded)" % (DIMS[3] * world))
                          if args.sharded else ("replicas only (north_star: no sharding)" if world > 1 else "single GPU"),
                          "l2": "inputs larger than L2 (gauge fields 201-805 MB each, 2.3 GB touched per step)"},
               "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
               "step_flops": step_flops, "step_alg_bytes": step_bytes, "kernels": kernels,
               "paper_table1_gflops_12real": {"%s/%s" % ("deg" if k[0] == 1 else "ndeg", PREC_NAME[k[1]]): v
                                              for k, v in PAPER_GFLOPS.items()},
               "paper_table1_gflops_8real": {"%s/%s" % ("deg" if k[0] == 1 else "ndeg", PREC_NAME[k[1]]): v
                                             for k, v in PAPER_GFLOPS_8REAL.items()}}
        print(json.dumps(out))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--path", type=int, default=0, help="tm_set_path: 0 = default kernel selection, 1 = scalar kernels only")
    ap.add_argument("--sharded", action="store_true",
                    help="each rank holds a 32^3x64 slab of a 32^3 x (64 N) lattice: kernels with open time hops, face exchange over "
                         "torch.distributed, boundary completion (DESIGN.md section 9); default: N independent replicas")
    ap.add_argument("--recon", type=int, default=12, choices=[18, 12, 8],
                    help="reals stored per link (BASELINE.json configs[2], configs[3]: 12); 18 and 8 are the other rows of the paper's Table 1")
    args = ap.parse_args()
    global RECON
    RECON = args.recon
    rank = int(os.environ.get("RANK", "0"))

    def log(msg):
        if rank == 0:
            sys.stderr.write("[bench] %s\n" % msg)

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, log)
        return
    run_ours(args, log)


if __name__ == "__main__":
    main()
