#!/usr/bin/env python
"""bench.py -- joint log-likelihood evaluations / s on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (rows a0-a9: glad_joint_loglike_batch) over one batch of the
RXJ1131-shaped synthetic workload (BASELINE.json configs[1] = "C2": 1024 parameter vectors).
  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--impl ours|reference]
N > 1 is launched by torch.distributed.run; batch elements are independent, so every rank evaluates its
own full batch with no data-path collective ("weak" scaling); NCCL is used only for the barrier and the
max-over-ranks of the device time.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "joint_loglike_evals_per_s"
UNIT = "evals/s"
FP32_LANES_PER_SM = 128
# ncu --set full numbers (DRAM traffic, executed FP32 instructions) are NOT typed in here: they are read from the committed capture
# summaries that profiles/current_capture.txt lists, each with the sha256 of the kernel source it was taken from.  When the
# source has changed since, the capture is stale and the key is reported as null with the reason.
CAPTURE_INDEX = os.path.join(ROOT, "profiles", "current_capture.txt")
_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def load_capture(key: str) -> dict:
    """{'fresh': bool, 'file': csv path, 'metrics': {name: value (bytes for byte units)}, 'note': str}"""
    import hashlib
    out = {"fresh": False, "file": None, "metrics": {}, "note": "no capture listed in profiles/current_capture.txt"}
    if not os.path.exists(CAPTURE_INDEX):
        return out
    for line in open(CAPTURE_INDEX):
        f = line.split()
        if len(f) < 4 or f[0] != key:
            continue
        csv_path, src, sha = os.path.join(ROOT, f[1]), os.path.join(ROOT, f[2]), f[3]
        out["file"] = f[1]
        if not (os.path.exists(csv_path) and os.path.exists(src)):
            out["note"] = "capture file or kernel source missing"
            return out
        now = hashlib.sha256(open(src, "rb").read()).hexdigest()[:16]
        for row in open(csv_path).read().splitlines()[1:]:
            c = row.split(",")
            if len(c) >= 3:
                try:
                    out["metrics"][c[0]] = float(c[2]) * _UNIT.get(c[1], 1.0)
                except ValueError:
                    pass
        out["fresh"] = now == sha
        out["note"] = (f"{f[1]} (taken at sha256[:16] of {f[2]} = {sha}" + (")" if out["fresh"] else f"; the source is now {now}: STALE)"))
        return out
    return out


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def read_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p))
        except Exception:
            pass
    return {}


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc = index, [], None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([c.strip() for c in line.split(",")])
        except Exception:
            pass

    def stop(self) -> dict:
        if self.proc:
            self.proc.terminate()
        self.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def oracle_data_model():
    import oracle

    def dm(w):
        img = vr = None
        if w["lens"]:
            img = oracle.lens_image_batch(w["lens"]["params"], w["lens"]["grid"], w["lens"]["psf"])["images"][0]
        if w["dyn"]:
            d = w["dyn"]
            vr = oracle.jam_vrms_batch(d["params"], d["lum_mge"], d["mass_mge"], d["beta"], d["kin"])["vrms"][0]
        return img, vr
    return dm


def gpu_data_model(device):
    """Mock data from the library's own forward model at the truth vector (what a user does to make a mock)."""
    from paper_2504_01302_b200 import Glad

    def dm(w):
        g = Glad(device)
        img = vr = None
        if w["lens"]:
            g.set_image_data(w["lens"]["grid"], w["lens"]["psf"])
            img = g.lens_image_batch(w["lens"]["params"], want_chi2=False)["images"][0].cpu().numpy()
        if w["dyn"]:
            d = w["dyn"]
            kin = dict(d["kin"]); kin["vrms_obs"] = kin["vrms_ivar"] = None
            g.set_kin_data(kin)
            vr = g.jam_vrms_batch(d["params"], d["lum_mge"], d["mass_mge"], d["beta"], want_chi2=False)["vrms"][0].cpu().numpy()
        g.close()
        return img, vr
    return dm


def oracle_joint(wl):
    import oracle
    L, D = wl["lens"], wl["dyn"]
    B = wl["B"]
    c2l = oracle.lens_image_batch(L["params"], L["grid"], L["psf"], L["data"], L["ivar"], want_images=False)["chi2"] if L else np.zeros(B)
    c2d = oracle.jam_vrms_batch(D["params"], D["lum_mge"], D["mass_mge"], D["beta"], D["kin"])["chi2"] if D else np.zeros(B)
    return oracle.joint_loglike(c2l, c2d)            # a lens-only / dynamics-only config: the half that exists


def workload_terms(wl):
    """Contraction size of row a6 per vector: K = nu * (n_mass + BH) * n_lum."""
    D = wl["dyn"]
    nm = D["mass_mge"].shape[-2] + (D["params"][:, 2] > 0).astype(np.int64)
    return D["kin"]["u_nodes"].size * nm * D["lum_mge"].shape[-2]


def run_reference(args, rank):
    """--impl reference: the fp64 CPU oracle as it stands on the box's host cores, bounded sample per step."""
    if rank != 0:
        return
    import oracle
    import workloads
    oracle.build()
    n_sample = args.ref_sample
    wl = workloads.make_workload(args.config, oracle_data_model(), B=n_sample)
    for _ in range(args.warmup if args.warmup < 1 else 1):
        oracle_joint(workloads.subset(wl, [0]))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_joint(wl)
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    cores = oracle.num_threads()
    sample = f"{n_sample} seeded {args.config} vectors per step (element 0 = truth), OpenMP over the batch"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.config} ({'BASELINE.json configs[1], RXJ1131-shaped joint model' if args.config == 'C2' else 'BASELINE.json config'}), bounded sample"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_sweep(args):
    """--sweep: per-kernel device times of every BASELINE.json config on one GPU (C2/C4/C5 at a bounded batch, three
    C3 cells), one JSON line per config.  Not the bench line: context for profiles/*.md."""
    import torch
    import workloads
    from paper_2504_01302_b200 import Glad
    cases = [("C1", None), ("C2", None), ("C3-10-40-4096", None), ("C3-20-80-4096", None), ("C3-40-160-256", None),
             ("C4", 1024), ("C5", 296)]
    for name, B in cases:
        wl = workloads.make_workload(name, gpu_data_model(0), B=B)
        L, D = wl["lens"], wl["dyn"]
        g = Glad(0)
        if L:
            g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
        if D:
            g.set_kin_data(D["kin"])

        def step():
            if L and D:
                g.joint_loglike_batch(L["params"], D["params"], D["lum_mge"], D["mass_mge"], D["beta"])
            elif L:
                g.lens_image_batch(L["params"], want_images=False)
            else:
                g.jam_vrms_batch(D["params"], D["lum_mge"], D["mass_mge"], D["beta"])
        for _ in range(2):
            step()
        torch.cuda.synchronize()
        g.profile_enable(True)
        g.profile_read()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n = 3
        e0.record()
        for _ in range(n):
            step()
        e1.record()
        torch.cuda.synchronize()
        prof = g.profile_read()
        ms = e0.elapsed_time(e1) / n
        line = {"config": name, "batch": wl["B"], "ms_per_step": ms, "evals_per_s": wl["B"] / (ms * 1e-3),
                "kernel_ms": {k: round(v[0] / n, 4) for k, v in prof.items() if v[1]}}
        if D:
            nx, ny = D["kin"]["xs"].size, D["kin"]["ys"].size
            fl = 2.0 * ((nx + 1) // 2) * ((ny + 1) // 2) * float(workload_terms(wl).sum())
            q = prof["jam_quad"][0] / n
            line["jam_quad_alg_tflops"] = fl / (q * 1e-3) / 1e12
        print(json.dumps(line), flush=True)
        g.close()


def run_pixsrc_sweep(args):
    """--pixsrc-sweep: glad_pixsrc_evidence_batch over source-grid resolutions (the axis of the paper's Fig. 1: "various
    source resolutions commonly adopted in practice") on the C2 image data, one JSON line per resolution.  Context, not the
    bench line."""
    import torch
    import workloads
    from paper_2504_01302_b200 import Glad
    B = 296
    wl = workloads.make_workload("C2", gpu_data_model(0), B=B)
    L = wl["lens"]
    g = Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    npx = L["grid"]["nx"] * L["grid"]["ny"]
    for n_s in (16, 24, 32, 40, 48, 64):
        pin = workloads.pixsrc_inputs(wl, n_s, n_s)
        a = (torch.from_numpy(L["params"]).cuda(), torch.from_numpy(pin["src_grids"]).cuda(), torch.from_numpy(pin["lam"]).cuda(), n_s, n_s)
        out = g.pixsrc_evidence_batch(*a, want_source=False, want_model=False)
        torch.cuda.synchronize()
        g.profile_enable(True)
        g.profile_read()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n = 2
        e0.record()
        for _ in range(n):
            out = g.pixsrc_evidence_batch(*a, want_source=False, want_model=False)
        e1.record()
        torch.cuda.synchronize()
        prof = g.profile_read()
        ms = e0.elapsed_time(e1) / n
        print(json.dumps({"workload": "C2 image data", "N_d": npx, "N_s": n_s * n_s, "batch": B, "ms_per_call": ms,
                          "evidences_per_s": B / (ms * 1e-3), "ms_per_evidence": ms / B,
                          "finite": int(torch.isfinite(out["logev"]).sum().item()),
                          "kernel_ms": {k[7:]: round(v[0] / n, 3) for k, v in prof.items() if v[1] and k.startswith("pixsrc_")}}), flush=True)
    g.close()


NCU_KEEP = ("Kernel Name", "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "launch__", "sm__throughput",
            "sm__warps_active", "smsp__issue_active", "sm__inst_executed_pipe_", "sm__pipe_fma_cycles", "sm__pipe_fp64", "sm__pipe_tensor",
            "l1tex__throughput", "lts__throughput", "dram__throughput", "l1tex__data_pipe_", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
            "smsp__inst_executed.sum", "smsp__average_warp", "sm__cycles_elapsed", "smsp__sass_thread_inst_executed_op_")


def ncu_summary(args):
    """--ncu-summary REP: filter `ncu -i REP --page raw --csv` (run here, no GPU needed) down to the metrics the write-ups and this
    bench use, write it to --out (a .csv under profiles/) and record it in profiles/current_capture.txt with the sha256 of the
    kernel source, so that load_capture() can tell a fresh capture from a stale one."""
    import csv
    import hashlib
    import io
    raw = subprocess.run(["ncu", "-i", args.ncu_summary, "--page", "raw", "--csv"], check=True, capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    h, u = rows[0], rows[1]
    v = rows[2 + args.capture_row]
    with open(os.path.join(ROOT, args.out), "w") as f:
        f.write("metric,unit,value\n")
        for i, name in enumerate(h):
            if any(name.startswith(k) for k in NCU_KEEP) and not name.endswith("_not_issued.ratio"):
                f.write(f"{name},{u[i]},{v[i].replace(',', ' ')}\n")
    sha = hashlib.sha256(open(os.path.join(ROOT, args.capture_source), "rb").read()).hexdigest()[:16]
    lines = [l for l in (open(CAPTURE_INDEX).read().splitlines() if os.path.exists(CAPTURE_INDEX) else []) if l.split()[:1] != [args.capture_key]]
    lines.append(f"{args.capture_key} {args.out} {args.capture_source} {sha}")
    open(CAPTURE_INDEX, "w").write("\n".join(lines) + "\n")
    print(f"wrote {args.out}; {args.capture_key} -> sha {sha}")


SASS_OPS = ["UTCHMMA", "LDTM", "UTMALDG", "UBLKCP", "LDGSTS", "MUFU.EX2", "MUFU.LG2", "MUFU.RCP", "MUFU.RSQ", "FFMA", "FMUL2", "FFMA2", "FHFMA",
            "F2FP", "DFMA", "HMMA", "SYNCS", "BAR"]


def sass_counts():
    """--sass-counts: `cuobjdump -sass paper_2504_01302_b200/libglad.so | python bench.py --sass-counts` prints a markdown table of opcode
    counts per kernel (UTCHMMA = tcgen05.mma, LDTM = tcgen05.ld, UTMALDG / UBLKCP = TMA, LDGSTS = cp.async; B200_PROFILING.md)."""
    import collections
    import re
    cur, cnt, total = None, collections.defaultdict(collections.Counter), collections.Counter()
    for line in sys.stdin:
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            continue
        m = re.search(r"/\*[0-9a-f]{4,8}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m and cur:
            op = m.group(1)
            total[cur] += 1
            for o in SASS_OPS:
                if op == o or op.startswith(o + "."):
                    cnt[cur][o] += 1
    names = {k: subprocess.run(["c++filt", k], capture_output=True, text=True).stdout.strip().split("(")[0] for k in total}
    print("| kernel | SASS instructions | " + " | ".join(SASS_OPS) + " |")
    print("|---|---|" + "---|" * len(SASS_OPS))
    for k in sorted(total, key=lambda k: names[k]):
        print(f"| `{names[k]}` | {total[k]} | " + " | ".join(str(cnt[k].get(o, 0)) for o in SASS_OPS) + " |")


def peak_tf_of(dev, clocks):
    import torch
    peaks = read_peaks()
    sm_max = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    return torch.cuda.get_device_properties(dev).multi_processor_count * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12


def run_configs(args, device, peak_tf, clocks):
    """Every other BASELINE.json config at its FULL batch on one GPU (C1; two C3 cells; C4 at 8192; C5 at 4096): evals/s, the two
    stage kernels' ms per launch and their fractions.  Per-kernel times on one stream (glad_set_overlap(0)); the step time with the
    default two streams."""
    import torch
    import workloads
    from paper_2504_01302_b200 import Glad
    sm_max = float(read_peaks().get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    xu_peak = torch.cuda.get_device_properties(device).multi_processor_count * 16 * sm_max * 1e6
    rows = {}
    for name in ("C1", "C3-10-40-4096", "C3-40-160-256", "C4", "C5"):
        wl = workloads.make_workload(name, gpu_data_model(device))
        L, D, B = wl["lens"], wl["dyn"], wl["B"]
        g = Glad(device)
        if L:
            g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
        if D:
            g.set_kin_data(D["kin"])
        dev = torch.device("cuda", device)
        tt = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
        lp = tt(L["params"]) if L else None
        da = tuple(tt(D[k]) for k in ("params", "lum_mge", "mass_mge", "beta")) if D else None

        def step():
            if L and D:
                g.joint_loglike_batch(lp, *da)
            elif L:
                g.lens_image_batch(lp, want_images=False)
            else:
                g.jam_vrms_batch(*da)
        n = 3
        for _ in range(2):
            step()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            step()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / n
        g.set_overlap(False)
        step()
        torch.cuda.synchronize()
        g.profile_enable(True); g.profile_read()
        for _ in range(n):
            step()
        prof = g.profile_read(); g.profile_enable(False)
        row = {"batch": B, "ms_per_step": ms, "evals_per_s": B / (ms * 1e-3),
               "kernel_ms": {k: round(v[0] / n, 4) for k, v in prof.items() if v[1]}}
        if D:
            nx, ny = D["kin"]["xs"].size, D["kin"]["ys"].size
            nxf, nyf = (nx + 1) // 2, (ny + 1) // 2
            terms = float(workload_terms(wl).sum())
            q = prof["jam_quad"][0] / n
            row["jam_quad"] = {"ms_per_launch": q, "xu_frac": terms * (nxf + nyf) / (q * 1e-3) / xu_peak,
                               "fp32_equivalent_tflops": 2.0 * nxf * nyf * terms / (q * 1e-3) / 1e12,
                               "fp32_equivalent_frac": 2.0 * nxf * nyf * terms / (q * 1e-3) / 1e12 / peak_tf}
        if L:
            ss, kp, npx = L["grid"]["supersample"], L["psf"].shape[0], L["grid"]["nx"] * L["grid"]["ny"]
            alg = B * (npx * ss * ss * 235.0 + npx * 2.0 * kp * kp)
            li = prof["lens_image"][0] / n
            row["lens_image"] = {"ms_per_launch": li, "algorithmic_tflops": alg / (li * 1e-3) / 1e12, "frac_algorithmic": alg / (li * 1e-3) / 1e12 / peak_tf}
        rows[name] = row
        g.close()
        del g
        torch.cuda.empty_cache()
    return rows


def run_ours(args, rank, world, local_rank):
    import torch
    import workloads
    from paper_2504_01302_b200 import Glad

    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    wl = workloads.make_workload(args.config, gpu_data_model(local_rank), B=args.batch)
    L, D = wl["lens"], wl["dyn"]
    B = wl["B"]
    g = Glad(local_rank)
    if args.jam_path == "simt":
        g.set_jam_options(path="simt")
    if args.no_overlap:
        g.set_overlap(False)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_kin_data(D["kin"])
    dev = torch.device("cuda", local_rank)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32))
    host = {k: t(v).pin_memory() for k, v in (("lens", L["params"]), ("dyn", D["params"]), ("lum", D["lum_mge"]),
                                               ("mass", D["mass_mge"]), ("beta", D["beta"]))}
    d = {k: v.to(dev) for k, v in host.items()}
    out = {"loglike": torch.empty(B, device=dev), "chi2_lens": torch.empty(B, device=dev),
           "chi2_dyn": torch.empty(B, device=dev), "flags": torch.empty(B, dtype=torch.int32, device=dev)}
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)   # > 126 MB L2

    def step():
        g.joint_loglike_batch(d["lens"], d["dyn"], d["lum"], d["mass"], d["beta"], out=out)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.25)
    g.profile_enable(True)
    g.profile_read()
    n0 = g.launch_count
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    for (e0, e1) in evs:
        flush.zero_()                       # L2 flush between timed iterations (outside the per-step events)
        e0.record()
        step()
        e1.record()
    barrier()
    launches = g.launch_count - n0
    prof_timed = g.profile_read()          # per-kernel event times inside the headline region (two streams: see below)
    ms = float(sum(e0.elapsed_time(e1) for e0, e1 in evs))
    # Per-kernel durations for the roofline: the same K steps again on ONE stream (glad_set_overlap(0)), because with the
    # lens half on the side stream an event pair around lens_image also times its wait for SMs held by jam_quad.
    overlapped = not args.no_overlap
    if overlapped:
        g.set_overlap(False)
        step()
        torch.cuda.synchronize()
        g.profile_read()
        for _ in range(args.steps):
            flush.zero_()
            step()
        torch.cuda.synchronize()
        prof = g.profile_read()
        g.set_overlap(True)
    else:
        prof = prof_timed
    g.profile_enable(False)
    ms_serial = sum(v[0] for v in prof.values())

    # end to end through the host-buffer C entry point: H2D of every input + D2H of lnL inside the timed region
    h_out = torch.empty(B, dtype=torch.float32).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    g.joint_loglike_host(host["lens"], host["dyn"], host["lum"], host["mass"], host["beta"], h_out)
    barrier()
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a0.record()
    for _ in range(e2e_steps):
        g.joint_loglike_host(host["lens"], host["dyn"], host["lum"], host["mass"], host["beta"], h_out)
    a1.record()
    barrier()
    e2e_ms = a0.elapsed_time(a1)
    clocks = sampler.stop()

    # the self-consistent entry (lens vector + distances -> MGE tables on the device -> both halves);
    # reported beside the headline, not instead of it (the headline keeps BASELINE.json's table inputs)
    model = None
    if rank == 0:
        ddt = t(wl["ddt"]).to(dev)
        nlm, nmm = D["lum_mge"].shape[-2], D["mass_mge"].shape[-2]
        margs = (d["lens"], d["dyn"], ddt, wl["z_d"], nlm, (0.02, 10.0), nmm, (0.02, 50.0), d["beta"])
        for _ in range(3):
            g.joint_loglike_model_batch(*margs, out=out)
        torch.cuda.synchronize()
        g.profile_enable(True)
        g.profile_read()
        m_steps = max(3, min(args.steps, 10))
        m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        m0.record()
        for _ in range(m_steps):
            g.joint_loglike_model_batch(*margs, out=out)
        m1.record()
        torch.cuda.synchronize()
        mp = g.profile_read()
        g.profile_enable(False)
        m_ms = m0.elapsed_time(m1) / m_steps
        model = {"api": "glad_joint_loglike_model_batch", "value": B / (m_ms * 1e-3), "unit": UNIT, "ms_per_step": m_ms,
                 "mge_ms_per_step": mp["mge"][0] / m_steps, "mge_launches_per_step": mp["mge"][1] / m_steps,
                 "tables": f"{nlm} luminous (Sersic, 0.02-10 arcsec) + {nmm} mass (EPL, 0.02-50 arcsec) Gaussians per vector, Euler order 12",
                 "paper_context": "1-D MGE of one profile: ~2e-4 s on one A100 (P:356, Table 2)"}
        # SURVEY 8(f) rank 4 (quasar part): the same entry plus chi2_img + chi2_tmd (Eq. 35-36) = every term of Eq. 53
        g.set_quasar_data(workloads.quasar_data(args.config))
        fout = dict(out)
        for _ in range(3):
            g.joint_loglike_full_batch(*margs, out=fout)
        torch.cuda.synchronize()
        g.profile_enable(True)
        g.profile_read()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record()
        for _ in range(m_steps):
            g.joint_loglike_full_batch(*margs, out=fout)
        f1.record()
        torch.cuda.synchronize()
        fp = g.profile_read()
        g.profile_enable(False)
        f_ms = f0.elapsed_time(f1) / m_steps
        model["full_entry"] = {"api": "glad_joint_loglike_full_batch", "value": B / (f_ms * 1e-3), "unit": UNIT, "ms_per_step": f_ms,
                               "quasar_ms_per_step": fp["quasar"][0] / m_steps, "quasar_launches_per_step": fp["quasar"][1] / m_steps,
                               "quasar": "4 images, 3 delays, 12 Newton steps per image, fp64; runs on the lens half's stream",
                               "paper_context": "image-position and time-delay terms: < 0.1 s on one CPU core, kept on the CPU (P:265-267)"}

        # the paper's own extended-image likelihood (pixelated-source inversion, Eq. 37-43) on the same image
        # data: N_d = all image pixels, 32 x 32 source pixels (Table 1: N_d ~ 1e4, N_s ~ 1e3), 2 vectors per SM
        nsx = nsy = 32
        Bp = min(B, 2 * torch.cuda.get_device_properties(dev).multi_processor_count)
        pin = workloads.pixsrc_inputs(workloads.subset(wl, np.arange(Bp)), nsx, nsy)
        pa = (d["lens"][:Bp].contiguous(), t(pin["src_grids"]).to(dev), t(pin["lam"]).to(dev), nsx, nsy)
        for _ in range(2):
            po = g.pixsrc_evidence_batch(*pa, want_source=False, want_model=False)
        torch.cuda.synchronize()
        g.profile_enable(True)
        g.profile_read()
        p_steps = 3
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record()
        for _ in range(p_steps):
            po = g.pixsrc_evidence_batch(*pa, want_source=False, want_model=False)
        p1.record()
        torch.cuda.synchronize()
        pp = g.profile_read()
        g.profile_enable(False)
        p_ms = p0.elapsed_time(p1) / p_steps
        npx, nsrc = L["grid"]["nx"] * L["grid"]["ny"], nsx * nsy
        syrk_ms = pp["pixsrc_syrk"][0] / p_steps
        chol_ms = pp["pixsrc_chol"][0] / p_steps
        syrk_flops = Bp * float(npx) * nsrc * (nsrc + 1)             # dense lower triangle of F = f^T C_d^-1 f, 2 flops per term
        chol_flops = Bp * nsrc ** 3 / 3.0                             # fp64: N^3/3 (multiplies and adds) per factorisation
        model["pixsrc_entry"] = {
            "api": "glad_pixsrc_evidence_batch", "value": Bp / (p_ms * 1e-3), "unit": "evidences/s", "ms_per_step": p_ms, "batch": Bp,
            "sizes": f"N_d = {npx} image pixels, PSF {L['psf'].shape[0]} x {L['psf'].shape[0]}, N_s = {nsx} x {nsy} source pixels",
            "kernel_ms": {k[7:]: pp[k][0] / p_steps for k in pp if k.startswith("pixsrc_")},
            "finite": int(torch.isfinite(po["logev"]).sum().item()),
            "contraction": {"kernel": "pixsrc_syrk_tc_kernel", "ms_per_launch": syrk_ms, "dense_flops_per_launch": syrk_flops,
                            "dense_equivalent_tflops": syrk_flops / (syrk_ms * 1e-3) / 1e12,
                            "note": "tcgen05.mma on two-term fp16 operands (22 mantissa bits), three products per K-step, fp32 accumulation in TMEM "
                                    "flushed into registers every 512 pixels; D = f^T C_d^-1 d accumulated in fp64 on the diagonal tiles in the same pass; "
                                    "only the pixel rows whose f row touches both column blocks of a tile are contracted (about a third), so the "
                                    "dense-equivalent rate exceeds the executed one"},
            "cholesky": {"kernels": "chol_diag / chol_trsm / chol_update (three per 64-wide panel over the batch) + pixsrc_solve", "ms_per_factorisation_and_solve": chol_ms,
                         "fp64_gflops": chol_flops / (chol_ms * 1e-3) / 1e9},
            "paper_context": "extended-image step, one vector, 64 x 64 source grid, N_d ~ 1e4: 0.21 s on one A100 in fp64, 2 s with GLEE on one CPU core (Table 2 P:453-458); other hardware, context only"}
        # Eq. 43: the same chain with lambda_hat searched on the device (22 extra factorisations per vector)
        for _ in range(1):
            lo = g.pixsrc_lambda_opt_batch(pa[0], pa[1], (1e-3, 1e3), nsx, nsy, want_source=False, want_model=False)
        torch.cuda.synchronize()
        l0, l1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0.record()
        lo = g.pixsrc_lambda_opt_batch(pa[0], pa[1], (1e-3, 1e3), nsx, nsy, want_source=False, want_model=False)
        l1.record()
        torch.cuda.synchronize()
        model["pixsrc_entry"]["lambda_opt"] = {"api": "glad_pixsrc_lambda_opt_batch", "ms_per_step": l0.elapsed_time(l1), "batch": Bp,
                                               "value": Bp / (l0.elapsed_time(l1) * 1e-3), "unit": "optimised evidences/s",
                                               "lambda_range": [1e-3, 1e3], "finite": int(torch.isfinite(lo["logev"]).sum().item())}

    if rank == 0:
        # JAM_sph, the paper's own dynamics, on the same dynamics inputs with the paper's mesh (P:358-362:
        # 16 x 16 rectangles of 7 x 7 Kronrod nodes; 20 x 10 polar points)
        sph = workloads.jam_sph_rules(D["kin"], sigma_max=float(D["lum_mge"][..., 1].max()))
        g.set_jam_sph_rules(sph)
        sargs = (d["dyn"], d["lum"], d["mass"], d["beta"])
        for _ in range(2):
            g.jam_sph_vrms_batch(*sargs)
        torch.cuda.synchronize()
        g.profile_enable(True); g.profile_read()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s_steps = 3
        s0.record()
        for _ in range(s_steps):
            g.jam_sph_vrms_batch(*sargs)
        s1.record()
        torch.cuda.synchronize()
        sp = g.profile_read(); g.profile_enable(False)
        s_ms = s0.elapsed_time(s1) / s_steps
        i_ms = sp["jam_sph"][0] / s_steps
        npol, nt_, nu_ = sph["rgrid"].size * sph["thgrid"].size, sph["tau"].size, sph["un"].size
        nmj = D["mass_mge"].shape[-2] + (D["params"][:, 2] > 0).astype(np.int64)
        nlj = D["lum_mge"].shape[-2]
        groups = 1 if D["beta"].ndim == 1 else nlj
        ex2 = float(np.sum(groups * npol * nt_ * (nmj * nu_ + nlj) + npol * (nmj * nu_ + nlj)))
        xu_peak = torch.cuda.get_device_properties(dev).multi_processor_count * 16 * float(clocks.get("sm_max_mhz") or 1965.0) * 1e6
        model["jam_sph_entry"] = {
            "api": "glad_jam_sph_vrms_batch", "value": B / (s_ms * 1e-3), "unit": "dynamics evals/s", "ms_per_step": s_ms,
            "kernel_ms": {k: sp[k][0] / s_steps for k in ("jam_prep", "jam_sph", "jam_sph_los", "jam_post")},
            "sizes": f"{npol} polar points x {nt_} x {nu_} quadrature nodes, {nlj} luminous x {D['mass_mge'].shape[-2]}(+BH) mass Gaussians, one beta_ani per vector",
            "roofline": {"bound": "alu", "kernel": "jam_sph_intr_kernel", "unit": "Gex2/s", "achieved": ex2 / (i_ms * 1e-3) / 1e9, "peak": xu_peak / 1e9,
                         "frac": ex2 / (i_ms * 1e-3) / xu_peak, "ms_per_launch": i_ms, "algorithmic_ex2_per_launch": ex2,
                         "peak_source": "148 SM x 16 MUFU lanes/clk x sm_max MHz (XU pipe): one ex2 per (polar point, radial node, mass Gaussian, u node) "
                                        "+ one per luminous Gaussian -- the product form that one beta_ani allows (DESIGN.md)"},
            "paper_context": "intrinsic moments at > 200 polar points, 42 x 95 Gaussians, ONE parameter vector: 0.32 s on one A100 in fp64, 13 s with JamPy on a CPU "
                             "(Table 2 P:456-461); other hardware and table sizes, context only"}

    configs = None
    if rank == 0 and world == 1 and not args.no_configs:
        configs = run_configs(args, local_rank, peak_tf_of(dev, clocks), clocks)

    # Strong scaling of the lens-only large batch (BASELINE.json configs[3], 8192 vectors): ONE batch cut into contiguous chunks by
    # paper_2504_01302_b200.sharding, each rank evaluates its chunk, one all-gather of lnL (32 KB) -- the only exchange a sampler needs
    strong = None
    if not args.no_configs:
        from paper_2504_01302_b200.sharding import gather_loglike, shard_range
        w4 = workloads.make_workload("C4", gpu_data_model(local_rank))
        lo, hi = shard_range(w4["B"], rank, world)
        g4 = Glad(local_rank)
        g4.set_image_data(w4["lens"]["grid"], w4["lens"]["psf"], w4["lens"]["data"], w4["lens"]["ivar"])
        p4 = t(w4["lens"]["params"][lo:hi]).to(dev)

        def strong_step():
            c2 = g4.lens_image_batch(p4, want_images=False)["chi2"]
            return gather_loglike(-0.5 * c2, w4["B"], rank, world, dist)
        for _ in range(2):
            full = strong_step()
        barrier()
        q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        q0.record()
        for _ in range(3):
            full = strong_step()
        q1.record()
        barrier()
        q_ms4 = q0.elapsed_time(q1) / 3
        if dist is not None:
            tq = torch.tensor([q_ms4], device=dev, dtype=torch.float64)
            dist.all_reduce(tq, op=dist.ReduceOp.MAX)
            q_ms4 = float(tq[0])
        strong = {"workload": "C4 (BASELINE.json configs[3]): ONE batch of 8192 lens-only vectors", "scaling": "strong", "n_gpus": world,
                  "vectors_per_rank": hi - lo, "ms_per_step": q_ms4, "value": w4["B"] / (q_ms4 * 1e-3), "unit": "lens-only lnL evals/s",
                  "collective": "one all_gather of 8192 floats per step (sharding.gather_loglike)" if world > 1 else "none at N = 1",
                  "gathered_finite": int(torch.isfinite(full).sum().item())}
        g4.close()

    if dist is not None:
        tt = torch.tensor([ms, e2e_ms], device=dev, dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms, e2e_ms = float(tt[0]), float(tt[1])
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    ms_per_step = ms / args.steps
    value = world * B / (ms_per_step * 1e-3)
    e2e_value = world * B / (e2e_ms / e2e_steps * 1e-3)
    h2d = sum(v.numel() * 4 for v in host.values())
    # roofline of the dominant kernel (row a6, jam_quad): algorithmic flops = 2 per (folded pixel, contraction row)
    peaks = read_peaks()
    props = torch.cuda.get_device_properties(local_rank)
    sm_max = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    peak_tf = props.multi_processor_count * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    nx, ny = D["kin"]["xs"].size, D["kin"]["ys"].size
    npf = ((nx + 1) // 2) * ((ny + 1) // 2)           # the bench grids are mirror-symmetric in both axes
    flops_per_launch = 2.0 * npf * float(workload_terms(wl).sum())
    q_ms, q_n = prof["jam_quad"]
    q_avg = q_ms / max(q_n, 1)
    achieved = flops_per_launch / (q_avg * 1e-3) / 1e12 if q_n else None
    shares = {k: round(v[0] / ms_serial, 4) for k, v in prof.items() if v[1]}
    simt = args.jam_path == "simt"
    cap_q = load_capture("jam_quad_simt" if simt else "jam_quad_tc")
    traffic = (cap_q["metrics"].get("dram__bytes_read.sum", 0.0) + cap_q["metrics"].get("dram__bytes_write.sum", 0.0)) if cap_q["fresh"] else None
    roofline = {"bound": "alu", "kernel": "jam_quad_kernel" if simt else "jam_quad_tc_kernel", "achieved": achieved,
                "peak": peak_tf, "unit": "TFLOP/s", "frac": (achieved / peak_tf) if achieved else None,
                "traffic": traffic, "traffic_source": cap_q["note"],
                "peak_source": f"{props.multi_processor_count} SM x 128 FP32 lanes x 2 flop x {sm_max:.0f} MHz (DESIGN.md); "
                               "'achieved' counts the contraction's algorithmic fp32 flops (2 per folded pixel and "
                               "contraction row), the quantity BASELINE.json's '% FP32 peak per stage' is quoted on",
                "ms_per_launch": q_avg, "algorithmic_flops_per_launch": flops_per_launch, "kernel_share_of_step": shares,
                "timing": (f"per-kernel durations from {args.steps} more steps on one stream (glad_set_overlap(0), CUDA events, L2 flushed "
                           "between steps); the headline region runs the lens half on the context's side stream beside jam_quad, "
                           "where jam_quad took " + (f"{prof_timed['jam_quad'][0] / max(prof_timed['jam_quad'][1], 1):.4f} ms per launch" if overlapped else "the same")
                           + "; kernel_share_of_step = share of the summed one-stream kernel time"),
                "ms_per_step_one_stream_kernels": ms_serial / args.steps}
    if not simt and q_n:
        # The tcgen05 form moves the contraction to the tensor cores, so its FP32-peak-equivalent can exceed 1 and is not a
        # roofline any more.  What is left on the SM's own pipes is operand generation, whose tightest unit is the XU pipe
        # (one MUFU.EX2 per operand value; 16 lanes/clk/SM): that is the roofline reported as primary; the
        # FP32-equivalent (the quantity BASELINE.json's "% FP32 peak per stage" names) and the tensor fraction sit beside it.
        nterms = float(workload_terms(wl).sum())
        nxf, nyf = (nx + 1) // 2, (ny + 1) // 2
        ex2_per_launch = nterms * (nxf + nyf)
        xu_peak = props.multi_processor_count * 16 * sm_max * 1e6
        r8 = lambda v: (v + 7) // 8 * 8
        mma_flops = 2.0 * 128 * (2 * r8(nxf)) * nterms            # executed: M = 128 tile, N = 2 bf16 terms x padded columns
        bf16_peak = float(peaks.get("bf16_tflops") or 2250.0)
        fp32_equiv = {k: roofline[k] for k in ("achieved", "peak", "unit", "frac", "peak_source", "algorithmic_flops_per_launch")}
        roofline.update({"bound": "alu", "unit": "Gex2/s", "achieved": ex2_per_launch / (q_avg * 1e-3) / 1e9, "peak": xu_peak / 1e9,
                         "frac": ex2_per_launch / (q_avg * 1e-3) / xu_peak,
                         "peak_source": f"{props.multi_processor_count} SM x 16 MUFU lanes/clk x {sm_max:.0f} MHz (XU pipe; DESIGN.md): "
                                        "algorithmic ex2 = (nx_f + ny_f) per contraction row",
                         "algorithmic_ex2_per_launch": ex2_per_launch})
        del roofline["algorithmic_flops_per_launch"]
        roofline["fp32_equivalent"] = fp32_equiv
        roofline["tensor_pipe"] = {"bound": "tensor", "unit": "TFLOP/s", "achieved": mma_flops / (q_avg * 1e-3) / 1e12,
                                   "peak": bf16_peak, "frac": mma_flops / (q_avg * 1e-3) / 1e12 / bf16_peak,
                                   "peak_source": "MEASURED_PEAKS.json bf16_tflops (burst)" if peaks.get("bf16_tflops") else "nominal 2250 (no MEASURED_PEAKS.json)"}

    # BASELINE.json's metric asks for the % of FP32 peak per stage: the lensing stage (ray-shoot + bin-down + PSF + chi2)
    l_ms, l_n = prof["lens_image"]
    if l_n:
        cap_l = load_capture("lens_image")
        m = cap_l["metrics"]
        l_avg = l_ms / l_n
        ss, kp = L["grid"]["supersample"], L["psf"].shape[0]
        npx_img = L["grid"]["nx"] * L["grid"]["ny"]
        alg = B * (npx_img * ss * ss * 235.0 + npx_img * 2.0 * kp * kp)      # ~235 flop per ray + 2 K^2 per pixel
        roofline["lens_image"] = {"bound": "alu", "kernel": "lens_image_kernel", "unit": "TFLOP/s", "peak": peak_tf, "ms_per_launch": l_avg,
                                  "algorithmic_flops_per_launch": alg, "achieved_algorithmic": alg / (l_avg * 1e-3) / 1e12,
                                  "frac_algorithmic": alg / (l_avg * 1e-3) / 1e12 / peak_tf}
        k3 = ["smsp__sass_thread_inst_executed_op_%s_pred_on.sum" % o for o in ("ffma", "fmul", "fadd")]
        if not all(k in m for k in k3) and "sm__cycles_elapsed.avg" in m and all(k + ".per_cycle_elapsed" in m for k in k3):
            for k in k3:                         # the raw page lists these counters per elapsed cycle only
                m[k] = m[k + ".per_cycle_elapsed"] * m["sm__cycles_elapsed.avg"]
        if cap_l["fresh"] and args.config == "C2" and all(k in m for k in k3) and m.get("launch__grid_size") == B:
            lf = 2.0 * m[k3[0]] + m[k3[1]] + m[k3[2]]
            roofline["lens_image"].update({"flops_per_launch": lf, "achieved": lf / (l_avg * 1e-3) / 1e12, "frac": lf / (l_avg * 1e-3) / 1e12 / peak_tf,
                                           "flops_source": "executed FP32 flops (FFMA = 2, FMUL = FADD = 1) counted by ncu: " + cap_l["note"]})
        else:
            roofline["lens_image"].update({"flops_per_launch": None, "achieved": None, "frac": None,
                                           "flops_source": "no fresh ncu capture of the executed flops for this workload: " + cap_l["note"]})

    # the same contraction with three bf16 terms per operand (24 mantissa bits): the price of the wider arithmetic, beside the default
    if rank == 0 and not simt:
        g.set_jam_options(terms=3)
        jargs = (d["dyn"], d["lum"], d["mass"], d["beta"])
        g.jam_vrms_batch(*jargs)
        torch.cuda.synchronize()
        g.profile_enable(True); g.profile_read()
        for _ in range(3):
            g.jam_vrms_batch(*jargs)
        p3 = g.profile_read(); g.profile_enable(False)
        g.set_jam_options(terms=2)
        roofline["three_term_ms_per_launch"] = p3["jam_quad"][0] / max(p3["jam_quad"][1], 1)

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        ns = args.cpu_sample
        cwl = workloads.make_workload(args.config, oracle_data_model(), B=ns)
        t0 = time.perf_counter()
        oracle_joint(cwl)
        dt = time.perf_counter() - t0
        cpu = {"value": ns / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "cpu_model": cpu_model(), "nproc": os.cpu_count(),
               "seconds": dt, "sample": f"{ns} seeded {args.config} vectors (element 0 = truth), one pass, OpenMP over the batch"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 (fp64-prepared per-vector constants; row a6 contraction on 2-term split-bf16 tensor-core operands, fp32 accumulate)" if not simt else "f32",
            "data": "synthetic",
            "config": {"workload": f"{args.config} (BASELINE.json configs[1], RXJ1131-shaped joint model)", "batch_per_gpu": B,
                       "image": f"{L['grid']['nx']}x{L['grid']['ny']} s={L['grid']['supersample']} psf={L['psf'].shape[0]}",
                       "jam": f"{D['lum_mge'].shape[-2]}+{D['mass_mge'].shape[-2]}(+BH) Gaussians, {nx}x{ny} sky grid, "
                              f"{D['kin']['nbins']} bins, {D['kin']['u_nodes'].size} nodes",
                       "l2": "256 MiB buffer zeroed between timed steps (outside the per-step events)",
                       "parallelism": f"dp{world} (independent batches, no collective)"},
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": B * 4,
                    "steps": e2e_steps, "api": "glad_joint_loglike_host (pinned host buffers)"},
            "roofline": roofline, "cpu_baseline": cpu, "model_entry": model, "configs": configs, "strong_scaling_entry": strong}
    print(json.dumps(line), flush=True)
    g.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C2")
    ap.add_argument("--batch", type=int, default=None, help="override the per-GPU batch (default: the config's)")
    ap.add_argument("--ref-sample", type=int, default=16, help="vectors per oracle step of --impl reference (K steps must end within minutes)")
    ap.add_argument("--cpu-sample", type=int, default=64, help="vectors of the one oracle pass behind cpu_baseline (SURVEY 8(d): 64 for C2)")
    ap.add_argument("--jam-path", default="auto", choices=["auto", "simt"], help="row a6 kernel: tcgen05 where it fits (default) or the FP32 SIMT form")
    ap.add_argument("--no-overlap", action="store_true", help="keep both halves on one stream (glad_set_overlap(0))")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config block (C1, C3 cells, C4, C5)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--pixsrc-sweep", action="store_true", help="pixelated-source evidence over source-grid resolutions (context)")
    ap.add_argument("--sweep", action="store_true", help="per-kernel times of every BASELINE.json config (context, not the bench line)")
    ap.add_argument("--ncu-summary", default=None, help="an .ncu-rep to summarise into --out and register in profiles/current_capture.txt")
    ap.add_argument("--capture-key", default="jam_quad_tc")
    ap.add_argument("--capture-source", default="paper_2504_01302_b200/csrc/jam_quad_tc.cu")
    ap.add_argument("--capture-row", type=int, default=0, help="which profiled launch of the report")
    ap.add_argument("--out", default=None)
    ap.add_argument("--sass-counts", action="store_true", help="opcode counts per kernel from `cuobjdump -sass` on stdin")
    args = ap.parse_args()
    if args.sass_counts:
        sass_counts()
        return
    if args.ncu_summary:
        ncu_summary(args)
        return
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.pixsrc_sweep:
        run_pixsrc_sweep(args)
        return
    if args.sweep:
        run_sweep(args)
        return
    if world == 1 and args.gpus > 1:
        # convenience: re-launch under torch.distributed.run
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", "29531", os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
