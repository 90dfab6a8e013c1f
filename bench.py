#!/usr/bin/env python
"""bench.py -- throughput of the fused twisted-mass dslash hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--recon 18|12|8] [--sharded] [--no-extra]
    python bench.py --sass-mix | --import-ncu FILE.csv      (host only: refresh profiles/sass_mix.csv / profiles/traffic.csv)

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

--impl reference times the CPU oracle (oracle/, fp64, as it stands) on the host cores on the same full-lattice step.
The JSON line also carries `kernels` (every launch of the step, timed inside a repeat of the K-step loop with an event pair per launch) and `kernels_extra` (every kernel type x
precision x flavors x link compression of the library + the Wilson limit, each timed alone in the same run) and `cg`
(tm_invert_cg: iterations and ms per iteration, double / double-single / double-half, Eq. 2.2 against Eq. 2.3).
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
    """SM clock, throttle reasons and board power while the GPU is under load (B200_PROFILING.md clocks line), sampled through NVML
    every 2 ms from a thread (the power limiter of the board acts within tens of milliseconds: nvidia-smi's 20 ms loop sees 3-4
    samples of a 75 ms region and misses the dips); falls back to an `nvidia-smi -lms 20` subprocess when pynvml is missing."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    REASONS = ((0x8, "hw_slowdown"), (0x40, "hw_thermal_slowdown"), (0x20, "sw_thermal_slowdown"), (0x4, "sw_power_cap"),
               (0x80, "hw_power_brake_slowdown"))

    def __init__(self, index):
        self.rows, self.proc, self.nv, self.samples, self.halt = [], None, None, [], False
        try:
            import pynvml
            pynvml.nvmlInit()
            idx = str(index)
            self.h = pynvml.nvmlDeviceGetHandleByIndex(int(idx)) if idx.isdigit() else pynvml.nvmlDeviceGetHandleByUUID(idx)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            try:
                self.limit_w = pynvml.nvmlDeviceGetEnforcedPowerLimit(self.h) / 1e3
            except Exception:
                self.limit_w = None
            self.nv = pynvml
            self.th = threading.Thread(target=self._poll, daemon=True)
            self.th.start()
            return
        except Exception:
            self.nv = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _poll(self):
        nv = self.nv
        while not self.halt:
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                watts = nv.nvmlDeviceGetPowerUsage(self.h) / 1e3            # the driver's average over about 100 ms
                try:                                                        # the instantaneous figure shows the cap tens of ms earlier
                    inst = nv.nvmlDeviceGetFieldValues(self.h, [nv.NVML_FI_DEV_POWER_INSTANT])[0].value.uiVal / 1e3
                except Exception:
                    inst = None
                self.samples.append((time.time(), float(mhz), int(mask), watts, inst))
            except Exception:
                pass
            time.sleep(0.002)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.nv is not None:
            time.sleep(0.01)
            self.halt = True
            self.th.join(timeout=2)
            rows = [r for r in self.samples if t0 <= r[0] <= t1] or self.samples[-3:]
            if not rows:
                return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["no NVML samples"]}
            sm = [r[1] for r in rows]
            mask = 0
            for r in rows:
                mask |= r[2]
            return {"sm_mhz": float(np.median(sm)), "sm_min_mhz": min(sm), "sm_max_mhz": self.max_mhz,
                    "reasons": sorted(n for b, n in self.REASONS if mask & b), "samples": len(sm), "power_max_w": max(r[3] for r in rows),
                    "power_instant_max_w": max([r[4] for r in rows if r[4] is not None], default=None),
                    "power_limit_w": self.limit_w, "source": "NVML, 2 ms period"}
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
                "reasons": sorted(reasons), "samples": len(sm), "source": "nvidia-smi -lms 20"}


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


KERNEL_SOURCES = ("tm_dslash.cuh", "tm_dslash_f2.cuh", "tm_dslash_tile.cuh", "tm_layout.cuh", "tm_f2.cuh", "tm_stream.cuh")


def source_hash():
    """sha256 (12 hex digits) over the fused-dslash kernel sources: ties the stored ncu traffic / SASS mix to the kernels being timed."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_1311_4462_b200", "csrc")
    for name in KERNEL_SOURCES:
        h.update(name.encode())
        h.update(open(os.path.join(csrc, name), "rb").read())
    return h.hexdigest()[:12]


def read_profile_table(fname):
    """profiles/<fname> (or an absolute path): '# source_hash=<h> ...' header, then 'kernel;v1;v2...' rows -> (hash or None, {kernel: [floats]})."""
    path = fname if os.path.isabs(fname) else os.path.join(ROOT, "profiles", fname)
    rows, h = {}, None
    if not os.path.exists(path):
        return None, rows
    for line in open(path):
        if line.startswith("#"):
            for tok in line[1:].split():
                if tok.startswith("source_hash="):
                    h = tok.split("=", 1)[1]
            continue
        f = [c.strip() for c in line.split(";")]
        try:
            rows[f[0]] = [float(v) for v in f[1:]]
        except ValueError:
            continue
    return h, rows


def ncu_traffic(name):
    """DRAM read+write bytes per launch of kernel `name` from the committed ncu summary (profiles/traffic.csv, written by
    `bench.py --import-ncu`), or None when the kernel sources have changed since that capture (hash mismatch)."""
    h, rows = read_profile_table("traffic.csv")
    if h != source_hash() or name not in rows:
        return None
    return rows[name][0]


def sass_mix(name):
    """(packed FP32, integer-pipe, scalar FP32, all) instructions per thread of kernel `name` from profiles/sass_mix.csv
    (written by `bench.py --sass-mix` from cuobjdump -sass of the built objects), or None on a hash mismatch."""
    h, rows = read_profile_table("sass_mix.csv")
    if h != source_hash() or name not in rows:
        return None
    return rows[name]


PACKED_OPS = ("FFMA2", "FMUL2", "FADD2")
INT_OPS = ("PRMT", "IADD3", "IMAD", "SHF", "LOP3", "ISETP", "LEA", "SEL", "MOV", "VIADDMNMX", "IABS", "FMNMX3", "FMNMX", "FSEL", "FSETP", "PLOP3")
FP32_OPS = ("FFMA", "FMUL", "FADD")
FP64_OPS = ("DFMA", "DMUL", "DADD")


def write_sass_mix():
    """--sass-mix: opcode histogram of every fused-dslash kernel in the built objects -> profiles/sass_mix.csv (one row per
    kernel: packed FP32; integer pipe; scalar FP32; FP64; all) and profiles/r2_sass_histogram.md (the full histograms)."""
    import glob
    import re
    build = os.path.join(ROOT, "paper_1311_4462_b200", "csrc", "build")
    rows, md = [], []
    for obj in sorted(glob.glob(os.path.join(build, "tm_f2_*.o")) + glob.glob(os.path.join(build, "tm_generic_*.o")) + glob.glob(os.path.join(build, "tm_tile_*.o"))):
        txt = subprocess.run(["cuobjdump", "-sass", obj], capture_output=True, text=True).stdout
        for blk in txt.split("Function : ")[1:]:
            mangled = blk.split("\n", 1)[0].strip()
            m = re.match(r"_Z\d+tm_dslash_(f2|generic)ILi(\d)ELi(\d)ELi(\d+)ELi(\d)ELb([01])ELb([01])ELb([01])EE", mangled)
            mt = re.match(r"_Z\d+tm_dslash_(tile)ILi(\d)ELi(\d)ELi(\d+)ELi(\d)ELb([01])EE", mangled)
            if not m and not mt:
                continue
            fam, prec, nf, recon, kt, dag, stg, twin = m.groups() if m else mt.groups() + ("0", "0")
            name = "%s%s%s<%s,%s,%s,%s,%s>" % (fam, "_twin" if twin == "1" else "", "_staged" if stg == "1" else "", prec, nf, recon, kt,
                                              "dagger" if dag == "1" else "plain")
            hist = {}
            for line in blk.splitlines():
                mm = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\w+\s+)?([A-Z][A-Z0-9_]*)", line)
                if mm:
                    hist[mm.group(1)] = hist.get(mm.group(1), 0) + 1
            for k in ("NOP", "BRA", "EXIT"):
                hist.pop(k, None)
            tot = sum(hist.values())
            cnt = lambda ops: sum(hist.get(o, 0) for o in ops)
            rows.append((name, cnt(PACKED_OPS), cnt(INT_OPS), cnt(FP32_OPS), cnt(FP64_OPS), tot))
            md.append("| `%s` | %d | %s |" % (name, tot, " ".join("%s:%d" % kv for kv in sorted(hist.items(), key=lambda kv: -kv[1])[:18])))
    hsh = source_hash()
    commit = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
    with open(os.path.join(ROOT, "profiles", "sass_mix.csv"), "w") as f:
        f.write("# source_hash=%s parent_commit=%s  kernel ; packed FP32 (FFMA2/FMUL2/FADD2) ; integer pipe ; scalar FP32 ; FP64 ; all  "
                "(static instruction counts per thread, both sides of the few branches; written by `python bench.py --sass-mix`)\n" % (hsh, commit))
        for r in rows:
            f.write(";".join(str(v) for v in r) + "\n")
    with open(os.path.join(ROOT, "profiles", "r2_sass_histogram.md"), "w") as f:
        f.write("# r2: SASS opcode histogram of every fused dslash kernel\n\nCommand: `python -m paper_1311_4462_b200.build && python bench.py --sass-mix` "
                "(cuobjdump -sass of `paper_1311_4462_b200/csrc/build/*.o`; source_hash=%s, parent commit %s).\n"
                "Static counts per thread (NOP / BRA / EXIT dropped); the kernels are straight-line code, so static = executed up to the prefetch prologue.\n\n"
                "| kernel | instructions | top opcodes |\n|---|---|---|\n" % (hsh, commit))
        f.write("\n".join(md) + "\n")
    print("wrote profiles/sass_mix.csv (%d kernels), profiles/r2_sass_histogram.md" % len(rows))


def import_ncu(csv_path, out_path=None):
    """--import-ncu FILE: an `ncu --csv --page raw` export (metrics dram__bytes_read.sum, dram__bytes_write.sum) of THIS build
    -> profiles/traffic.csv with the source hash, mean per launch and kernel."""
    import csv
    import re
    acc = {}
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    with open(csv_path, newline="") as f:
        rows = list(csv.reader(f))
    hdr = next(r for r in rows if "Kernel Name" in r)
    units = dict(zip(hdr, rows[rows.index(hdr) + 1]))            # the line under the header carries the unit of every column
    for row in rows:
        if len(row) != len(hdr) or not row[0].isdigit():
            continue
        d = dict(zip(hdr, row))
        kn = d["Kernel Name"].replace("(int)", "").replace("(bool)", "")
        m = re.search(r"tm_dslash_(f2|generic)<(\d), (\d), (\d+), (\d), (\w+), (\w+)(?:, (\w+))?>", kn)
        mt = re.search(r"tm_dslash_(tile)<(\d), (\d), (\d+), (\d), (\w+)>", kn)
        if not m and not mt:
            continue
        fam, prec, nf, recon, kt, dag, stg, twin = m.groups() if m else mt.groups() + ("0", "0")
        name = "%s%s%s<%s,%s,%s,%s,%s>" % (fam, "_twin" if twin in ("1", "true") else "", "_staged" if stg in ("1", "true") else "", prec, nf, recon, kt,
                                          "dagger" if dag in ("1", "true") else "plain")
        try:
            b = sum(float(d[k].replace(",", "")) * scale[units[k]] for k in ("dram__bytes_read.sum", "dram__bytes_write.sum"))
        except (KeyError, ValueError):
            continue
        a = acc.setdefault(name, [0.0, 0])
        a[0] += b
        a[1] += 1
    commit = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
    with open(out_path or os.path.join(ROOT, "profiles", "traffic.csv"), "w") as f:
        f.write("# source_hash=%s parent_commit=%s  kernel ; DRAM bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum, mean over "
                "the captured launches; written by `python bench.py --import-ncu %s`)\n" % (source_hash(), commit, os.path.basename(csv_path)))
        for name, (tot, n) in sorted(acc.items()):
            f.write("%s;%d\n" % (name, round(tot / n)))
    print("wrote profiles/traffic.csv (%d kernels)" % len(acc))


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
        """Pinned host buffers in the precision a user of that field precision holds: double for fp64 fields, float for fp32 / half."""
        torch = self.torch
        self.pin_in, self.pin_out = {}, {}
        for nf in (1, 2):
            n = nf * self.vh * 24
            for dt, key in ((torch.float64, 8), (torch.float32, 4)):
                a = torch.empty(n, dtype=dt, pin_memory=True)
                a.numpy()[:] = self.host_in[nf].view(np.float64).reshape(-1)
                self.pin_in[(nf, key)] = a
                self.pin_out[(nf, key)] = torch.empty(n, dtype=dt, pin_memory=True)

    def step_e2e(self, sync=True):
        """The same step through the C-ABI with HOST buffers: upload in_e, tm_mat_pc, download out_e, per composite.
        The asynchronous entry points overlap the H2D copy of the next input, the kernels and the D2H copy of the
        previous result; tm_sync at the end of the step: every result of the step is on the host when it returns.
        fp64 fields travel as double arrays, fp32 and half fields as float arrays (tm_field_upload_cb_async_f32)."""
        tm = self.tm
        h2d = d2h = 0
        for nf, prec, typ, dagger in step_ops():
            key = (nf, prec)
            hk = (nf, 8 if prec == 8 else 4)
            up, down = (tm.tm_field_upload_cb_async, tm.tm_field_download_cb_async) if prec == 8 else \
                (tm.tm_field_upload_cb_async_f32, tm.tm_field_download_cb_async_f32)
            up(self.fin[key].h, 0, self.pin_in[hk].data_ptr())
            self.mat_pc(key, nf, typ, dagger)
            down(self.fout[key].h, 0, self.pin_out[hk].data_ptr())
            h2d += self.pin_in[hk].numel() * self.pin_in[hk].element_size()
            d2h += self.pin_out[hk].numel() * self.pin_out[hk].element_size()
        if sync:
            self.lat.sync()
        return h2d, d2h


def pcie_bandwidth(torch, nbytes=1 << 28, reps=6):
    """GB/s of pinned-host <-> device copies on this box: H2D alone, D2H alone, and each way with both directions at once (the e2e bound)."""
    h_in, h_out = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True), torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    d_in, d_out = torch.empty(nbytes, dtype=torch.uint8, device="cuda"), torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()

    def run(h2d, d2h):
        torch.cuda.synchronize()
        t = time.time()
        for _ in range(reps):
            if h2d:
                with torch.cuda.stream(s1):
                    d_in.copy_(h_in, non_blocking=True)
            if d2h:
                with torch.cuda.stream(s2):
                    h_out.copy_(d_out, non_blocking=True)
        torch.cuda.synchronize()
        return nbytes * reps / (time.time() - t) / 1e9
    run(1, 1)
    return {"h2d_gbs": run(1, 0), "d2h_gbs": run(0, 1), "both_gbs_each_way": run(1, 1)}


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
    """--impl reference: the oracle as it stands on the host cores, the SAME workload as our arm's step: one fp64 pass of the
    step's 4 distinct operators on the full 32^3x64 lattice per step (~1.6 s on 16 cores).  Steps are capped by --ref-steps
    (default 5) and warm-up by 1 so that the run ends within a few minutes; the caps are reported."""
    import oracle as ora
    import synth_inputs as si
    dims = DIMS
    t = time.time()
    gauge = {1: si.gauge_field(dims, SEED_DEG, "haar"), 2: si.gauge_field(dims, SEED_NDEG, "near_identity")}
    inp = {nf: si.mask_parity(si.spinor_field(dims, nf, s), dims, 0) for nf, s in ((1, SEED_DEG), (2, SEED_NDEG))}
    log("host inputs generated in %.1f s" % (time.time() - t))
    sample = ("full 32^3x64 lattice: the step's 4 distinct operators (deg ASYM, SYM; ndeg ASYM, ASYM-dagger) once each in fp64 per step "
              "(the oracle has one precision; our arm runs them in fp64 / fp32 / half)")
    steps, warm = max(1, min(args.steps, args.ref_steps)), min(args.warmup, 1)
    for _ in range(warm):
        oracle_step(ora, si, dims, gauge, inp, sample)
    tot_s, tot_f = 0.0, 0
    for _ in range(steps):
        s, f = oracle_step(ora, si, dims, gauge, inp, sample)
        tot_s += s
        tot_f += f
    val = tot_f / tot_s / 1e9
    cores = ora.num_threads()
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": "GFLOPS", "n_gpus": args.gpus, "steps": steps,
           "warmup": warm, "steps_requested": args.steps, "warmup_requested": args.warmup, "ms_per_step": 1e3 * tot_s / steps,
           "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": WORKLOAD % (RECON, RECON), "lattice": list(dims), "sample": sample},
           "cpu_baseline": {"value": val, "unit": "GFLOPS", "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": "GFLOPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


METRIC = "twisted-mass dslash GFLOPS (even-odd preconditioned operators, Eq. 2.2/2.3, 32^3x64, fp64+fp32+half sweep)"
WORKLOAD = ("32^3x64: configs[2] degenerate (Haar links, %d-real, mu=0.0015) ASYM+SYM in fp64/fp32/half + configs[3] "
            "non-degenerate (exp(i0.3H) links, %d-real, mu=0.15, eps=0.19) ASYM plain+dagger in fp32/half")
# plain-ALU peak: 128 FP32 / 64 FP64 FMA lanes per SM, 148 SMs, 2 flop per FMA, at the SM clock under load
SMS, LANES = 148, {8: 64, 4: 128, 2: 128}


SMSPS = 148 * 4
CYC = {"packed": 2.0, "int": 1.0, "fp32": 1.0, "fp64": 2.0}


def annotate_bound(k, vh, sm_mhz):
    """Adds the plain-ALU flop fraction and the datapath fraction (see run_ours) to a kernel record; names the bound."""
    pb = k.pop("prec_bytes")
    alu_peak = SMS * LANES[pb] * 2 * sm_mhz * 1e-3      # GFLOPS
    k["alu_peak_gflops"] = alu_peak
    k["frac_of_alu_peak"] = k["gflops"] / alu_peak
    mix = sass_mix(k["kernel"])
    k["frac_of_datapath"] = None
    if mix:
        packed, integer, fp32, fp64 = mix[0], mix[1], mix[2], mix[3]
        cyc = CYC["packed"] * packed + CYC["int"] * integer + CYC["fp32"] * fp32 + CYC["fp64"] * fp64
        floor_us = cyc * (vh / 32.0) / SMSPS / sm_mhz
        k["datapath_cycles_per_warp"] = cyc
        k["frac_of_datapath"] = floor_us / k["us"]
    k["bound"] = "alu" if (k["frac_of_datapath"] or 0.0) > k["frac_of_measured_peak"] else "hbm"


def time_alone(fn, sync, launches=20, reps=3):
    """Mean microseconds per launch of fn(), `launches` back to back between two CUDA events, best of `reps`."""
    import torch
    for _ in range(10):
        fn()
    sync()
    best = None
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(launches):
            fn()
        e1.record()
        torch.cuda.synchronize()
        t = e0.elapsed_time(e1) / launches * 1e3
        best = t if best is None else min(best, t)
    return best


def kernels_extra(w, args, sm_mhz, peak):
    """Every (kernel type x precision x flavors x link compression) of the library, each timed ALONE in this run (20 launches
    between two CUDA events, best of 3, 50 ms of idle before each kernel) at 32^3x64 through tm_dslash_apply -- outside `value`, whose step
    stays BASELINE.json's.
    Rows: 12- / 18- / 8-real x fp64 / fp32 / half x degenerate / doublet x A / A-xpay / B / REC, and the Wilson limit
    (mu = eps = 0: the paper's Table 1 Wilson column) of kernel A."""
    tm, lat, vh = w.tm, w.lat, w.vh
    out = []
    host_u = w.host_gauge[1]
    for _ in range(20):          # the GPU idled during the CPU baseline: bring the clocks back up before timing anything
        w.step()
    lat.sync()
    fields = {}
    for prec in (8, 4, 2):
        for nf in (1, 2):
            fin = w.fin.get((nf, prec)) or lat.field(prec, nf).upload_cb(0, w.host_in[nf])
            fx = lat.field(prec, nf).upload_cb(0, w.host_in[nf])
            fields[(prec, nf)] = (fin, fx, w.fout.get((nf, prec)) or lat.field(prec, nf))
    wilson = tm.params(KAPPA, mu=0.0, epsilon=0.0, twist_flavor=1)
    for recon in (12, 18, 8):
        for prec in (8, 4, 2):
            g = w.gauge.get((1, prec)) if recon == RECON else None
            g = g or lat.gauge(host_u, prec, recon)
            for nf in (1, 2):
                fin, fx, fout = fields[(prec, nf)]
                for kt, label in ((0, "A"), (1, "A-xpay"), (2, "B"), (3, "REC"), (0, "A wilson"), (6, "R^-1 D R^-1 (fused)")):
                    if label == "A wilson" and (nf == 2 or recon != 12):
                        continue
                    if kt == 6 and recon != 12:
                        continue
                    p = wilson if label == "A wilson" else w.params[nf]
                    time.sleep(0.05)         # "alone": not on top of the power / thermal state the previous kernel's launches left behind
                    us = time_alone(lambda: tm.dslash_apply(fout, fin, None if kt in (0, 6) else fx, g, p, 1, 0, kt), lat.sync)
                    # the fused D R^-1 form reads the whole neighbour site on the time hops: one spinor (+ norms) more than kernel A
                    b = (bytes_per_site(nf, prec, recon, 0 if kt == 6 else kt) + (nf * 12 * prec + (4 * nf if prec == 2 else 0) if kt == 6 else 0)) * vh
                    f = (flops_per_site(nf, 0 if kt == 6 else kt) + (8 * (48 + 24 if nf == 1 else 240) if kt == 6 else 0)) * vh
                    k = {"kernel": tm.tm_last_kernel_name(lat.ctx), "flavors": nf, "prec": PREC_NAME[prec], "type": label, "recon": recon,
                         "us": us, "gflops": f / us / 1e3, "alg_gbs": b / us / 1e3, "frac_of_measured_peak": b / us / 1e3 / peak,
                         "bytes_per_site": b // vh, "prec_bytes": prec}
                    annotate_bound(k, vh, sm_mhz)
                    out.append(k)
            del g
    return out


def cg_leg(w):
    """Mixed-precision CG (tm_invert_cg, reliable updates) on M^dag M x = b at 32^3x64, 12-real links: iterations and device time per
    iteration for double, double-single (DS) and double-half (DH), Eq. 2.2 (asym) against Eq. 2.3 (sym) preconditioning -- the
    comparison of the paper's Table 2 with its parameters kappa = 0.156361, mu = 0.0015 for the degenerate
    doublet and mu = 0.15, eps = 0.19 for the non-degenerate one, but on SYNTHETIC exp(i 0.3 H) links, which are far better
    conditioned than the paper's ensembles (tens of iterations, not thousands): context for the cost per iteration, not a target."""
    import torch
    tm, lat = w.tm, w.lat
    host_u = w.host_gauge[2]
    gauges = {prec: (w.gauge.get((2, prec)) or lat.gauge(host_u, prec, RECON)) for prec in (8, 4, 2)}
    out = []
    for nf, kw, label in ((1, dict(mu=0.0015, epsilon=0.0, twist_flavor=1), "degenerate"), (2, NDEG, "non-degenerate")):
        p = tm.params(0.156361, **kw)
        fb = lat.field(8, nf).upload_cb(0, w.host_in[nf])
        fx = lat.field(8, nf)
        for typ, tname in ((ASYM, "asym (Eq. 2.2)"), (SYM, "sym (Eq. 2.3)")):
            for ps, pname, delta in ((8, "double", 0.1), (4, "double-single", 0.1), (2, "double-half", 0.3)):
                kwargs = dict(tol=1e-8, max_iter=2000, sloppy_precision=ps, delta=delta)
                tm.invert_cg(fx, fb, gauges[8], None if ps == 8 else gauges[ps], p, typ, **kwargs)      # warm-up: work fields allocated
                lat.sync()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                info = tm.invert_cg(fx, fb, gauges[8], None if ps == 8 else gauges[ps], p, typ, **kwargs)
                e1.record()
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1)
                out.append({"doublet": label, "preconditioning": tname, "precision": pname, "iterations": info["iterations"],
                            "reliable_updates": info["restarts"], "converged": info["converged"], "residual": info["residual"],
                            "ms": ms, "ms_per_iteration": ms / max(info["iterations"], 1)})
        del fb, fx
    tm.tm_cg_release(lat.ctx)
    return out


def run_kernels(args, log):
    """--kernels PREC:NF:RECON:KT[,...] [--dims X,Y,Z,T] [--tune key=value,...]: single kernels timed alone (30 launches between two
    CUDA events, best of 3) through tm_dslash_apply -- the tuning runs of profiles/r2_tuning.md.  KT = tm_kernel_type (0..8).  Inputs: links drawn
    from a pool of 4096 Haar matrices (seed 3), Gaussian spinors: fast to generate at 48^3x96; the kernels have no data-dependent control flow."""
    import torch
    import paper_1311_4462_b200 as tm
    import synth_inputs as si
    dims = tuple(int(v) for v in args.dims.split(","))
    specs = [tuple(int(v) for v in a.split(":")) for a in args.kernels.split(",")]
    V = si.volume(dims)
    vh = V // 2
    rng = np.random.default_rng(7)
    U = si.haar_su3(4096, 3)[rng.integers(0, 4096, size=4 * V)].reshape(4, V, 3, 3)
    lat = tm.Lattice(dims, 0)
    for kv in [t for t in args.tune.split(",") if t]:
        k, v = kv.split("=")
        tm.tm_set_tuning(lat.ctx, k, int(v))
    peak, _ = measured_peak()
    gauges, fields, out = {}, {}, []
    for prec, nf, recon, kt in specs:
        if (prec, recon) not in gauges:
            gauges[(prec, recon)] = lat.gauge(U, prec, recon)
        if (prec, nf) not in fields:
            h = rng.standard_normal((nf, vh, 4, 3)) + 1j * rng.standard_normal((nf, vh, 4, 3))
            fields[(prec, nf)] = (lat.field(prec, nf).upload_cb(0, h), lat.field(prec, nf).upload_cb(0, h), lat.field(prec, nf))
    pd, pn = tm.params(KAPPA, **DEG), tm.params(KAPPA, **NDEG)
    for prec, nf, recon, kt in specs:
        fin, fx, fout = fields[(prec, nf)]
        g, p = gauges[(prec, recon)], (pd if nf == 1 else pn)
        no_x = kt in (0, 6)
        us = time_alone(lambda: tm.dslash_apply(fout, fin, None if no_x else fx, g, p, 1, 0, kt), lat.sync, launches=30)
        kcode = {4: 2, 5: 3, 6: 0, 7: 3, 8: 3}.get(kt, kt)
        b = (bytes_per_site(nf, prec, recon, kcode) + (nf * 12 * prec + (4 * nf if prec == 2 else 0) if kt >= 6 else 0)) * vh     # D R^-1: full time-hop sites
        out.append({"spec": "%d:%d:%d:%d" % (prec, nf, recon, kt), "kernel": tm.tm_last_kernel_name(lat.ctx), "us": us, "alg_gbs": b / us / 1e3,
                    "frac_of_measured_peak": b / us / 1e3 / peak})
        log("%-12s %-36s %8.1f us  %6.0f GB/s  frac %.3f" % (out[-1]["spec"], out[-1]["kernel"], us, b / us / 1e3, b / us / 1e3 / peak))
    print(json.dumps({"mode": "kernels", "dims": list(dims), "tune": args.tune, "kernels": out}))


def config5(log, fast_links):
    """BASELINE.json configs[4] -- 48^3x96 non-degenerate doublet, fp64, 18-real links, kappa = 0.1632, mu = 0.135, eps = 0.17, the
    symmetric-preconditioned Eq. 2.3 operator applied 100 times back to back in one timed region.  fast_links: the links are drawn from
    a pool of 4096 Haar matrices (seconds to generate) instead of the configuration's own 42 M Haar matrices (seed 5, a minute and 25 GB
    of host memory: `--config5`); the kernels have no data-dependent control flow."""
    import torch
    import paper_1311_4462_b200 as tm
    import synth_inputs as si
    dims = (48, 48, 48, 96)
    t = time.time()
    if fast_links:
        rng = np.random.default_rng(5)
        V = si.volume(dims)
        U = si.haar_su3(4096, 5)[rng.integers(0, 4096, size=4 * V)].reshape(4, V, 3, 3)
        psi = rng.standard_normal((2, V // 2, 4, 3)) + 1j * rng.standard_normal((2, V // 2, 4, 3))
    else:
        U = si.gauge_field(dims, 5, "haar")
        psi = si.to_parity(si.spinor_field(dims, 2, 5), dims, 0)
    log("48^3x96 host inputs generated in %.1f s" % (time.time() - t))
    lat = tm.Lattice(dims, torch.cuda.current_device())
    vh = lat.Vh
    g = lat.gauge(U, 8, 18)
    del U
    fin, ftmp, fout = lat.field(8, 2).upload_cb(0, psi), lat.field(8, 2), lat.field(8, 2)
    p = tm.params(KAPPA, mu=0.135, epsilon=0.17, twist_flavor=0)
    for _ in range(10):
        tm.mat_pc(fout, fin, ftmp, g, p, SYM, 0)
    lat.sync()
    tm.tm_timing_enable(lat.ctx, 1)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(100):
        tm.mat_pc(fout, fin, ftmp, g, p, SYM, 0)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    rec = tm.tm_timing_read(lat.ctx, 1 << 12)
    tm.tm_timing_enable(lat.ctx, 0)
    peak, peak_src = measured_peak()
    flops = (flops_per_site(2, 0) + flops_per_site(2, 1)) * vh * 100
    byts = (bytes_per_site(2, 8, 18, 0) + bytes_per_site(2, 8, 18, 1)) * vh * 100
    per = {}
    for name, tms in rec:
        a = per.setdefault(name, [0.0, 0])
        a[0] += tms
        a[1] += 1
    kern = []
    for kt, (name, (tot, cnt)) in zip((0, 1), per.items()):
        us = 1e3 * tot / cnt
        b = bytes_per_site(2, 8, 18, kt) * vh
        kern.append({"kernel": name, "type": KT_NAME[kt], "us": us, "alg_gbs": b / us / 1e3, "frac_of_measured_peak": b / us / 1e3 / peak})
    return {"metric": "twisted-mass dslash GFLOPS (Eq. 2.3 operator, 48^3x96 non-degenerate fp64, 100 applications back to back)",
            "value": flops / (ms * 1e-3) / 1e9, "unit": "GFLOPS", "n_gpus": 1, "steps": 100, "ms_total": ms, "ms_per_application": ms / 100,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[4]: 48^3x96 non-degenerate doublet, fp64, 18-real links, kappa=0.1632, mu=0.135, eps=0.17, "
                                   "SYM (Eq. 2.3) x 100", "lattice": list(dims), "recon": 18,
                       "links": "pool of 4096 Haar matrices (fast)" if fast_links else "Haar, seed 5 (the configuration's recipe)"},
            "alg_gbs": byts / (ms * 1e-3) / 1e9, "frac_of_measured_peak": byts / (ms * 1e-3) / 1e9 / peak, "peak_source": peak_src,
            "kernels": kern, "gpu_launches": 200}


def run_config5(args, log):
    """--config5: configs[4] with its own gauge configuration; prints its own JSON line."""
    import torch
    torch.cuda.set_device(0)
    print(json.dumps(config5(log, fast_links=False)))


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
        grid = tuple(int(v) for v in args.grid.split(",")) if args.grid else (1, 1, world)
        slab = sharded.Slab((DIMS[0], DIMS[1] * grid[0], DIMS[2] * grid[1], DIMS[3] * grid[2]), rank, world, local, grid=grid, peer=args.peer)
    w = Workload(local, log, slab)
    lat, vh = w.lat, w.vh
    tm.tm_set_path(lat.ctx, args.path)
    for kv in [t for t in args.tune.split(",") if t]:
        k, v = kv.split("=")
        tm.tm_set_tuning(lat.ctx, k, int(v))
    ops = step_ops()
    step_flops = sum(op_flops(o, vh) for o in ops)
    step_bytes = sum(op_bytes(o, vh) for o in ops)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, K timed steps; then the same K steps with per-launch events
    phys = os.environ.get("CUDA_VISIBLE_DEVICES", "").split(",")
    smi_index = phys[local] if len(phys) > local and phys[local] else str(local)
    sampler = ClockSampler(smi_index)
    for _ in range(max(args.warmup, 3)):
        w.step()
    barrier()
    # the timed region proper: K steps, nothing but the step's own launches on the stream
    n0 = lat.launches()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    ev0.record()
    for _ in range(args.steps):
        w.step()
    ev1.record()
    barrier()
    ms_local = ev0.elapsed_time(ev1)
    launches = lat.launches() - n0
    # the same K steps again with one CUDA event between consecutive launches (tm_timing_enable(ctx, 2): a launch's interval runs from
    # its predecessor's stop event to its own, so the per-kernel durations of the roofline tile the region without gaps and add up to
    # ms_per_step_with_launch_events).  An event record between two kernels still costs 1-2 us of front-end time (an event PAIR around
    # every launch cost 5 us), which is why the headline value is taken from the region without them; both are reported.
    # (a second of idle and the warm-up steps again first: the board grants its maximum clocks for about 50 ms after an idle before the
    # power limiter steps in (profiles/r2_tuning.md section 7), and the second region should start from the same state as the first,
    # not 90 ms into it; `sustained` below reports the other state)
    t1 = time.time()
    time.sleep(1.0)
    for _ in range(max(args.warmup, 3)):
        w.step()
    barrier()
    tm.tm_timing_enable(lat.ctx, 1 if args.sharded else 2)      # --sharded: halo kernels run between the dslash launches: event pairs
    ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev2.record()
    for _ in range(args.steps):
        w.step()
    ev3.record()
    barrier()
    ms_instr = reduce_over_ranks(ev2.elapsed_time(ev3), world) / args.steps
    records = tm.tm_timing_read(lat.ctx, 1 << 20)
    tm.tm_timing_enable(lat.ctx, 0)
    clocks = sampler.stop(t0, t1)
    # ---- the same step in the board's sustained state.  This step draws the board's full power limit (NVML instantaneous power at the
    # 1000 W limit): after an idle the board runs about 50 ms at its maximum clocks, then the limiter lowers the SM clock in two or three
    # stages to ~1.5 GHz (sw_power_cap; profiles/r2_tuning.md section 7).  The default K = 30 timed steps lie mostly inside that first window,
    # as the burst figure of MEASURED_PEAKS.json does; `sustained` reports what a long run gets: 60 untimed steps, then 100 timed ones.
    sustained = None
    if not args.no_sustained:
        for _ in range(60):
            w.step()
        barrier()
        s_sampler = ClockSampler(smi_index)
        ts0 = time.time()
        ev4, ev5 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev4.record()
        for _ in range(100):
            w.step()
        ev5.record()
        barrier()
        ts1 = time.time()
        s_ms = reduce_over_ranks(ev4.elapsed_time(ev5), world) / 100
        sustained = {"ms_per_step": s_ms, "value": world * step_flops / (s_ms * 1e-3) / 1e9, "unit": "GFLOPS", "steps": 100, "after_untimed_steps": 60,
                     "clocks": s_sampler.stop(ts0, ts1)}
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
                    "traffic_source": "committed ncu --set full summary of this build (profiles/traffic.csv, source hash %s); null when the "
                                      "kernel sources have changed since the capture" % source_hash(),
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
    # the same without the per-step tm_sync (a caller streaming many inputs through: the last downloads of a step overlap the first
    # uploads of the next; one synchronisation at the end of the region) -- reported beside the per-step figure, which stays `value`
    tw0 = time.time()
    ev0.record()
    for _ in range(e2e_steps):
        w.step_e2e(sync=False)
    lat.sync()
    ev1.record()
    barrier()
    e2e_ms_stream = reduce_over_ranks(max(ev0.elapsed_time(ev1), 1e3 * (time.time() - tw0)), world) / e2e_steps
    try:
        pcie = pcie_bandwidth(torch)          # the bound of the e2e leg, measured on this box: copies in both directions at once
    except Exception:
        pcie = None
    e2e = {"value": world * step_flops / (e2e_ms * 1e-3) / 1e9, "unit": "GFLOPS", "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms, "steps": e2e_steps,
           "ms_per_step_streamed": e2e_ms_stream, "value_streamed": world * step_flops / (e2e_ms_stream * 1e-3) / 1e9,
           "pcie": pcie, "frac_of_pcie": (max(h2d, d2h) / (e2e_ms * 1e-3) / 1e9 / pcie["both_gbs_each_way"]) if pcie else None,
           "frac_of_pcie_streamed": (max(h2d, d2h) / (e2e_ms_stream * 1e-3) / 1e9 / pcie["both_gbs_each_way"]) if pcie else None,
           "note": "per composite: tm_field_upload_cb_async (pinned host arrays: double for fp64 fields, float for fp32 / half fields) + tm_mat_pc + tm_field_download_cb_async, "
                   "tm_sync per step (value) or once at the end of the region (value_streamed); copies in both directions overlap each other and the kernels; "
                   "pcie = pinned-host copies of 256 MiB measured in this run, frac_of_pcie = bytes each way / time / both_gbs_each_way"}

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

    # second roofline per kernel (profiles/r2_pipes.md): the FP32 / integer datapath.  Executed instructions
    # per thread by class (profiles/sass_mix.csv, from cuobjdump of this build) x the LEAST each can cost per warp and sub-partition
    # (packed FP32 and FP64: 2 cycles of the 32- / 16-lane pipe; integer-pipe and scalar FP32: their issue slot, 1 cycle -- measured
    # 2.08 alone and 1.07-2.6 next to FFMA2) = cycles the datapath needs per warp; x warps per sub-partition / SM clock = a time below
    # which the kernel cannot run.  A conservative floor: bound = "alu" only when even this fraction exceeds the HBM fraction.
    sm_mhz = (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz") or 1965.0
    for k in kernels:
        annotate_bound(k, vh, sm_mhz)
    if roofline and dom:
        roofline["bound"] = dom["bound"]                    # derived (annotate_bound), not asserted
        roofline["frac_of_datapath"] = dom["frac_of_datapath"]
    extra = kernels_extra(w, args, sm_mhz, peak) if (rank == 0 and world == 1 and not args.no_extra) else None
    cg = cg_leg(w) if (rank == 0 and world == 1 and not args.no_extra and not args.sharded) else None
    c5 = None
    if rank == 0 and world == 1 and not args.no_extra and not args.sharded:
        w.gauge.clear(), w.fin.clear(), w.ftmp.clear(), w.fout.clear()          # 48^3x96 needs 6 GB of links + 6 GB of staging
        c5 = config5(log, fast_links=True)
    if rank == 0:
        out = {"metric": METRIC, "value": value, "unit": "GFLOPS", "n_gpus": world, "steps": args.steps,
               "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "ms_per_step_with_launch_events": ms_instr, "higher_is_better": True, "scaling": "weak",
               "vs_baseline": None, "dtype": "f64+f32+i16/f32", "data": "synthetic",
               "config": {"workload": WORKLOAD % (RECON, RECON), "lattice": list(DIMS), "recon": RECON, "kappa": KAPPA,
                          "parallelism": ("sub-lattices of 32^3 x 64 on a (y, z, t) process grid %s, one per GPU, face exchange per dslash through %s (--sharded)"
                                          % (args.grid or "1,1,%d" % world, "peer-mapped buffers + flag words" if args.peer else "torch.distributed send / recv"))
                          if args.sharded else ("replicas only (north_star: no sharding)" if world > 1 else "single GPU"),
                          "l2": "inputs larger than L2 (gauge fields 201-805 MB each, 2.3 GB touched per step)",
                          "tune": args.tune or "defaults"},
               "roofline": roofline, "sustained": sustained, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
               "step_flops": step_flops, "step_alg_bytes": step_bytes, "kernels": kernels, "kernels_extra": extra, "cg": cg, "config5": c5,
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
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--ref-steps", type=int, default=5, help="--impl reference: cap on the timed full-lattice oracle steps (1.6 s each)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernels", default="", help="time single kernels alone instead: PREC:NF:RECON:KT[,...] (tuning runs; see run_kernels)")
    ap.add_argument("--dims", default="32,32,32,64", help="--kernels: lattice extents")
    ap.add_argument("--tune", default="", help="tm_set_tuning overrides, key=value[,...] (non-default values are recorded in config.tune)")
    ap.add_argument("--config5", action="store_true", help="time BASELINE.json configs[4] instead (48^3x96 fp64 doublet, Eq. 2.3 operator x 100; ~25 GB of host memory)")
    ap.add_argument("--no-sustained", action="store_true", help="skip the `sustained` leg (100 timed steps in the board's power-limited state)")
    ap.add_argument("--no-extra", action="store_true", help="skip the kernels_extra table (every kernel type x precision x compression, timed alone)")
    ap.add_argument("--sass-mix", action="store_true", help="host only: write profiles/sass_mix.csv + profiles/r2_sass_histogram.md from the built objects")
    ap.add_argument("--import-ncu", metavar="CSV", help="host only: turn an `ncu --csv --page raw` export of this build into profiles/traffic.csv")
    ap.add_argument("--path", type=int, default=0, help="tm_set_path: 0 = default kernel selection, 1 = scalar kernels only")
    ap.add_argument("--sharded", action="store_true",
                    help="each rank holds a 32^3x64 slab of a 32^3 x (64 N) lattice: kernels with open time hops, face exchange over "
                         "torch.distributed, boundary completion (DESIGN.md section 9); default: N independent replicas")
    ap.add_argument("--grid", default="", help="--sharded: process grid PY,PZ,PT over the y, z, t directions (default 1,1,N: time slabs)")
    ap.add_argument("--peer", action="store_true", help="--sharded: faces through peer-mapped buffers and flag words (CUDA IPC) instead of NCCL send / recv")
    ap.add_argument("--recon", type=int, default=12, choices=[18, 12, 8],
                    help="reals stored per link (BASELINE.json configs[2], configs[3]: 12); 18 and 8 are the other rows of the paper's Table 1")
    args = ap.parse_args()
    global RECON
    RECON = args.recon
    if args.sass_mix:
        return write_sass_mix()
    if args.import_ncu:
        return import_ncu(args.import_ncu)
    # --gpus N: one process per GPU.  Under torch.distributed.run (WORLD_SIZE set) the count must agree; a plain
    # `python bench.py --gpus N` starts the N ranks itself by re-executing under torch.distributed.run on this node.
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is not None and int(world_env) != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%s" % (args.gpus, world_env))
    if world_env is None and args.gpus > 1:
        import socket
        s = socket.socket()
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
        s.close()
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    rank = int(os.environ.get("RANK", "0"))

    def log(msg):
        if rank == 0:
            sys.stderr.write("[bench] %s\n" % msg)

    if args.kernels:
        return run_kernels(args, log)
    if args.config5:
        return run_config5(args, log)
    if args.impl == "reference":
        if rank == 0:
            run_reference(args, log)
        return
    run_ours(args, log)


if __name__ == "__main__":
    main()
