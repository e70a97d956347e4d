"""bench.py -- MRCQR FP64 thin-QR benchmark (BASELINE.json metric: ms per factorization at m x n,
achieved HBM GB/s and FP64 TFLOP/s against the B200's measured peaks).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C3|C0|C1|C2|C4n<n>]

A "step" is one pass of the whole hot path (mrcqr_factor: draw, K1..K5) over one synthetic matrix already
resident in HBM.  The headline workload is BASELINE.json configs[3] (C3: m = 2^21, n = 256, FP64 sketch, s = 512):
north_star quotes its target at m = 2^21, n <= 256, and C3 is the largest fixed configuration.  The same JSON line
carries, under "points", C1, C2 and the six FP16-sketch points of the column sweep configs[4] (per point: ms,
per-stage ms, both floors, both fractions, the clocks seen).  `e2e` is the headline factorization through
mrcqr_factor_host with pinned HOST buffers (H2D of A, D2H of Q and R inside the timed region).  The path does not
shard ("replicas only"): with N > 1 every rank factors its own replica; the value stays ms per
factorization of the slowest rank and `factorizations_per_s` aggregates the ranks.
--impl reference times the CPU oracle (oracle/) on the host cores, rank 0 only.
Prints ONE JSON line on rank 0.
"""
import argparse
import glob
import hashlib
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "MRCQR FP64 thin-QR ms per factorization"
# FP64 peak: nominal 148 SMs x 64 FMA/clk x 2 x 1.965 GHz = 37.2 TFLOP/s, confirmed by a DMMA.8x8x4 issue probe on this
# pool (profiles/r01_peaks.md); MEASURED_PEAKS.json has no FP64 figure, and the guide's bf16-scaled rule
# (1608.8 x 40 / 2250 = 28.6) would flatter every fraction by 1.3x
FP64_DMMA_PEAK_TFLOPS = 37.2
HBM_FALLBACK_GBS = 6650.0         # /opt/skills/guides/B200_PROFILING.md fallback
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r02_traffic.json")
POINTS = ["C1", "C2", "C4n16", "C4n32", "C4n64", "C4n128", "C4n256", "C4n512"]


def source_sha16():
    """Identity of the kernels being timed: sha256 over csrc/*.cu, *.cuh (the GPU box has no .git)."""
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2606_18411_b200", "csrc", "*.cu*"))):
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(config, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the ncu --set full capture recorded in
    profiles/r02_traffic.json (written by --traffic-from), or None when the capture is of other sources / configs."""
    try:
        d = json.load(open(TRAFFIC_FILE))
        if d.get("src_sha16") != source_sha16():
            return None
        for name, rec in sorted(d["configs"][config].items()):      # names carry their template arguments: match the prefix
            if name == kernel or name.startswith(kernel + "<") or name.startswith(kernel):
                return rec["dram_bytes_per_launch"]
        return None
    except Exception:
        return None


def write_traffic(csv_path, config):
    """--traffic-from: reads `ncu -i <rep> --page raw --csv` output and records, per kernel name, the mean
    dram__bytes_read.sum + dram__bytes_write.sum per launch, keyed by config and the sha of the kernel sources."""
    import csv
    rows = list(csv.reader(open(csv_path)))
    hdr = rows[0]
    units = rows[1]
    kn, rd, wr = hdr.index("Kernel Name"), hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    acc = {}
    for r in rows[2:]:
        if len(r) <= max(kn, rd, wr):
            continue
        name = r[kn].split("(")[0].replace("void ", "").replace("mrcqr::", "").strip()
        b = float(r[rd].replace(",", "")) * scale[units[rd]] + float(r[wr].replace(",", "")) * scale[units[wr]]
        acc.setdefault(name, []).append(b)
    try:
        d = json.load(open(TRAFFIC_FILE))
    except Exception:
        d = {}
    if d.get("src_sha16") != source_sha16():
        d = {"src_sha16": source_sha16(), "configs": {}}
    d["configs"][config] = {k: {"dram_bytes_per_launch": sum(v) / len(v), "launches": len(v)} for k, v in acc.items()}
    json.dump(d, open(TRAFFIC_FILE, "w"), indent=1, sort_keys=True)
    print("wrote", TRAFFIC_FILE, "for", config, "sources", d["src_sha16"])


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback"


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region.  The timed region of one bench run is
    tens of milliseconds, so the sampler polls NVML in-process every 4 ms (pynvml, the same counters nvidia-smi
    prints); if NVML cannot be opened it falls back to an `nvidia-smi -lms 200` child process."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    REASONS = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20), ("sw_power_cap", 0x4))

    def __init__(self, gpu_index):
        self.idx, self.proc, self.thread, self.rows = gpu_index, None, None, []
        self.tmp = None

    def _physical_index(self):
        vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
        ids = [v.strip() for v in vis.split(",") if v.strip()]
        if ids and self.idx < len(ids) and ids[self.idx].isdigit():
            return int(ids[self.idx])
        return self.idx

    def _poll(self):
        nv, h = self.nv
        while True:
            try:
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                self.rows.append((float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)),
                                  float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)), int(mask)))
            except Exception:
                pass
            if self.halt.wait(0.004):
                return

    def start(self):
        try:
            import threading
            import pynvml as nv
            nv.nvmlInit()
            self.nv = (nv, nv.nvmlDeviceGetHandleByIndex(self._physical_index()))
            self.halt = threading.Event()
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.thread = None
        try:
            self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=self.tmp, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm, reasons = [], set()
        if self.thread is not None:
            self.halt.set()
            self.thread.join(timeout=2)
            for clk, mx, mask in self.rows:
                sm.append(clk); out["sm_max_mhz"] = mx
                for name, bit in self.REASONS:
                    if mask & bit:
                        reasons.add(name)
            out["source"] = "nvml, 4 ms"
        elif self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
            self.tmp.flush()
            rows = [l.strip().split(",") for l in open(self.tmp.name) if l.strip()]
            os.unlink(self.tmp.name)
            for r in rows:
                try:
                    r = [x.strip() for x in r]
                    sm.append(float(r[1])); out["sm_max_mhz"] = float(r[2])
                    for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                        if v.lower().startswith("active"):
                            reasons.add(name)
                except Exception:
                    pass
            out["source"] = "nvidia-smi -lms 200"
        if sm:
            sm.sort()
            out["sm_mhz"] = sm[len(sm) // 2]
        out["reasons"] = sorted(reasons)
        out["samples"] = len(sm)
        return out


def workload(name):
    from paper_2606_18411_b200 import inputs
    if name.startswith("C4n"):          # a point of the column sweep (configs[4]), FP16 sketch: "C4n16", "C4n32", ...
        cfg = inputs.sweep_config(int(name[3:]), 16)
    else:
        cfg = dict(inputs.CONFIGS[name])
    cfg["name"] = name
    return cfg


def config_json(cfg, extra=None):
    c = {"workload": "%s: m=%d n=%d s=%d sketch=fp%d kappa~1e%d, A=G*diag(sigma)*V^T seeds %d/%d/%d" % (
        cfg["name"], cfg["m"], cfg["n"], cfg["s"], cfg["prec"], cfg["exponent"],
        cfg["seed_G"], cfg["seed_V"], cfg["seed_draw"]),
        "m": cfg["m"], "n": cfg["n"], "s": cfg["s"], "sketch_prec": "fp%d" % cfg["prec"],
        "l2": "inputs larger than L2 (A = %.0f MB read 3x, Q = %.0f MB written per step)" % (
            8e-6 * cfg["m"] * cfg["n"], 8e-6 * cfg["m"] * cfg["n"]),
        "parallelism": "replicas only (path does not shard)"}
    if extra:
        c.update(extra)
    return c


def oracle_sample(cfg):
    """The bounded CPU sample: the whole factorization when it is seconds of work (C0, C1, C2), else
    the first 2^18 rows of the same matrix (the oracle's cost is linear in m, so ms scales by m/2^18)."""
    full_flops = 4.0 * cfg["m"] * cfg["n"] ** 2
    if full_flops <= 1.5e11:
        return cfg["m"], 1.0, "whole factorization (all %d rows)" % cfg["m"]
    rows = 1 << 18
    return rows, cfg["m"] / rows, "first 2^18 rows of A, time scaled by m/2^18 = %g" % (cfg["m"] / rows)


def time_oracle(cfg, A_np, steps, warmup):
    import oracle
    rows, scale, what = oracle_sample(cfg)
    A = A_np[:rows]
    s = cfg["s"]
    signs, idx = oracle.draw(rows, s, cfg["seed_draw"])
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        out = oracle.factor_from_draw(A, signs, idx)
        dt = time.perf_counter() - t0
        assert out["rc"] == 0
        if it >= warmup:
            times.append(dt * 1e3 * scale)
    ms = sum(times) / len(times)
    return ms, {"value": ms, "unit": "ms", "cores": oracle.num_threads(), "kind": "oracle", "sample": what}


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    from paper_2606_18411_b200 import inputs
    cfg = workload(args.config)
    AT = inputs.make_config(cfg, "cuda" if torch.cuda.is_available() else "cpu").cpu()
    A_np = AT.numpy().T
    steps, warmup = max(1, min(args.steps, 3)), min(args.warmup, 1)
    ms, cpu = time_oracle(cfg, A_np, steps, warmup)
    line = {"impl": "reference", "metric": METRIC, "value": ms, "unit": "ms", "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": ms, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_json(cfg), "cpu_baseline": cpu,
            "e2e": {"value": ms, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def max_over_ranks(value, device="cpu"):
    """The multi-GPU timing rule: every rank contributes its device-measured time, the MAX is the job's.
    No-op for a single process.  (Replicas only: this and the barrier are the only collectives bench.py uses.)"""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def stores_y(n):
    """The library's default form of stage 2 (include/mrcqr.h, mrcqr_set_store_y): Y stored from n16 = 48 on."""
    return (n + 15) // 16 * 16 >= 48


def syrk_form(n):
    """... and from n16 = 128 on the stored Y goes through the panel solves and the SYRK (below: K3 with a Y dump + K5)."""
    return (n + 15) // 16 * 16 >= 128


def floors(m, n, hbm_peak, store_y=None):
    """Algorithmic work of one factorization: 32 m n bytes (3 reads of A + 1 write of Q) for every n;
    4 m n^2 flops in the fused (recompute) form, 3 m n^2 in the store-Y form (its extra write + read of Y is
    traffic, not algorithm).  Returns (bytes, flops, hbm floor ms, fp64 floor ms)."""
    alg_bytes = 32.0 * m * n
    if store_y is None:
        store_y = stores_y(n)
    flops = (3.0 if store_y else 4.0) * m * n * n
    return alg_bytes, flops, alg_bytes / (hbm_peak * 1e9) * 1e3, flops / (FP64_DMMA_PEAK_TFLOPS * 1e12) * 1e3


def time_point(B, AT, QT, R, cfg, steps, warmup, stream, sampler=None, barrier=None):
    """warmup + steps factorizations timed with CUDA events on `stream`; then the same loop again with the library's
    per-kernel events (kept out of the first loop: the extra event records cost a few % of a 1 ms step).
    Returns (total ms of the K steps, launches, {stage: ms per step})."""
    import torch
    prec, s, seed = cfg["prec"], cfg["s"], cfg["seed_draw"]
    for _ in range(warmup):
        B.mrcqr_factor(AT, prec, s, seed, QT, R, stream)
    launches = 0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    if sampler:
        sampler.start()
    e0.record(stream)
    for _ in range(steps):
        B.mrcqr_factor(AT, prec, s, seed, QT, R, stream)
        launches += B.mrcqr_last_launch_count()
    e1.record(stream)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    total_ms = e0.elapsed_time(e1)
    B.mrcqr_set_timing(True)
    stage_sum = {k: 0.0 for k in B.STAGES}
    for _ in range(steps):
        B.mrcqr_factor(AT, prec, s, seed, QT, R, stream)
        for k, v in B.mrcqr_last_timing().items():
            stage_sum[k] += v
    B.mrcqr_set_timing(False)
    return total_ms, launches, {k: v / steps for k, v in stage_sum.items()}


def dominant_kernel(cfg, stages, hbm_peak, how):
    """The kernel with the largest share of the step and its roofline (DESIGN.md section 5 states the per-row figures).
    n16 < 128: K3 (8n bytes read (+ 8n written when Y is stored), 2n^2 flops per row) or K5 (16n bytes; 2n^2 flops per row
    in the fused form, n^2 when it solves a stored Y), one launch = all m rows.
    n16 >= 128: one triangular solve = one mrcqr_panel_fused launch over the full 64-column panels (+ one mrcqr_panel_pass
    launch for a ragged first panel; n^2 flops, 16n bytes per row) or the SYRK launch (n^2 flops, 8n bytes per row);
    `kernel_ms` is the duration of the stage."""
    m, n = cfg["m"], cfg["n"]
    if not syrk_form(n):
        sy = stores_y(n)
        cand = {"k3_gram": ("mrcqr_k3_gram", (16.0 if sy else 8.0) * m * n, 2.0 * m * n * n),
                "k5_form_q": ("mrcqr_k5_formq", 16.0 * m * n, (1.0 if sy else 2.0) * m * n * n)}
    else:
        ragged = ((n + 15) // 16 * 16) % 64 != 0
        tail = (lambda f: " + mrcqr_panel_pass<%d> for the ragged first panel" % f if ragged else "")
        cand = {"k3_gram": ("mrcqr_panel_fused<0> (solve with R_s, all full panels in one launch)" + tail(0), 16.0 * m * n, 1.0 * m * n * n),
                "gram_reduce": ("mrcqr_syrk", 8.0 * m * n, 1.0 * m * n * n),
                "k5_form_q": ("mrcqr_panel_fused<1> (solve with R_c, all full panels in one launch)" + tail(1), 16.0 * m * n, 1.0 * m * n * n)}
    stage = max(cand, key=lambda k: stages[k])
    kname, dom_bytes, dom_flops = cand[stage]
    dom_ms = stages[stage]
    t_hbm, t_f64 = dom_bytes / (hbm_peak * 1e9), dom_flops / (FP64_DMMA_PEAK_TFLOPS * 1e12)
    if t_f64 >= t_hbm:
        ach = dom_flops / (dom_ms * 1e-3) / 1e12
        roof = {"bound": "tensor", "achieved": ach, "peak": FP64_DMMA_PEAK_TFLOPS, "unit": "TFLOP/s",
                "frac": ach / FP64_DMMA_PEAK_TFLOPS,
                "peak_source": "FP64 DMMA (mma.sync m8n8k4 f64) peak: nominal 148 x 64 x 2 x 1.965 GHz, confirmed by probe "
                               "(profiles/r01_peaks.md); MEASURED_PEAKS.json has no FP64 figure"}
    else:
        ach = dom_bytes / (dom_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
                "peak_source": "MEASURED_PEAKS.json hbm_gbs (%s)" % how}
    tkey = {"mrcqr_k3_gram": "mrcqr_k3_gram", "mrcqr_k5_formq": "mrcqr_k5_formq", "mrcqr_syrk": "mrcqr_syrk"}.get(
        kname, "mrcqr_panel_fused<0" if stage == "k3_gram" else "mrcqr_panel_fused<1")
    traffic = ncu_traffic(cfg["name"], tkey)
    if traffic is not None and tkey.startswith("mrcqr_panel_fused") and ((n + 15) // 16 * 16) % 64 != 0:
        rest = ncu_traffic(cfg["name"], tkey.replace("fused", "pass"))      # the ragged first panel's own launch
        traffic = None if rest is None else traffic + rest
    roof.update({"traffic": traffic, "kernel": kname, "stage": stage, "kernel_ms": dom_ms, "algorithmic_bytes": dom_bytes,
                 "algorithmic_flops": dom_flops, "hbm_gbs_achieved": dom_bytes / (dom_ms * 1e-3) / 1e9,
                 "traffic_source": "profiles/r02_traffic.json (ncu --set full of these kernel sources)" if traffic is not None
                 else "no ncu capture of these kernel sources / this config on file"})
    return roof


def time_forms(B, AT, QT, R, cfg, steps, stream):
    """ms per factorization with stage 2 forced to each of its two forms (mrcqr_set_store_y 0 / 1); the library's default
    picks by n16 (store-Y from 112 on)."""
    import torch
    out = {}
    try:
        for key, mode in (("fused_ms", False), ("store_y_ms", True)):
            B.mrcqr_set_store_y(mode)
            for _ in range(3):
                B.mrcqr_factor(AT, cfg["prec"], cfg["s"], cfg["seed_draw"], QT, R, stream)
            v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            v0.record(stream)
            for _ in range(steps):
                B.mrcqr_factor(AT, cfg["prec"], cfg["s"], cfg["seed_draw"], QT, R, stream)
            v1.record(stream)
            torch.cuda.synchronize()
            out[key] = v0.elapsed_time(v1) / steps
    finally:
        B.mrcqr_set_store_y(None)
    out["default"] = "store_y" if stores_y(cfg["n"]) else "fused"
    out["note"] = ("fused: Y = A Rs^-1 kept on chip by stage 2a and recomputed by stage 2b (north_star's form: 4 passes, "
                   "4 m n^2 flops); store_y: also written to Q's buffer and solved in place by stage 2b (5 passes, 3 m n^2 "
                   "flops; n16 = 128: panel solves + SYRK); default: the faster one as measured, store_y from n16 = 48 on")
    return out


def time_in_flight(B, AT, QT, R, cfg, steps, stream, hbm_peak):
    """The same K factorizations enqueued with mrcqr_factor_async and ONE mrcqr_wait at the end (include/mrcqr.h, "calls
    in flight"): no host round trip between two factorizations, so the device runs them back to back.
    CUDA events on `stream` around the K calls and the wait's work."""
    import torch
    prec, s, seed = cfg["prec"], cfg["s"], cfg["seed_draw"]
    for _ in range(3):
        B.mrcqr_factor_async(AT, prec, s, seed, QT, R, stream)
    B.mrcqr_wait()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        B.mrcqr_factor_async(AT, prec, s, seed, QT, R, stream)
    e1.record(stream)
    B.mrcqr_wait()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    _, _, t_hbm, t_f64 = floors(cfg["m"], cfg["n"], hbm_peak)
    return {"ms": ms, "hbm_frac": t_hbm / ms, "fp64_frac": t_f64 / ms, "binding_frac": max(t_hbm, t_f64) / ms, "steps": steps,
            "api": "mrcqr_factor_async x steps + one mrcqr_wait (status of the calls in flight read once, at the end)"}


def point_json(cfg, ms, stages, hbm_peak, clocks=None):
    alg_bytes, flops, t_hbm, t_f64 = floors(cfg["m"], cfg["n"], hbm_peak)
    out = {"config": "%s: m=%d n=%d s=%d fp%d" % (cfg["name"], cfg["m"], cfg["n"], cfg["s"], cfg["prec"]),
           "ms": ms, "stage_ms": stages, "hbm_floor_ms": t_hbm, "fp64_floor_ms": t_f64,
           "hbm_frac": t_hbm / ms, "fp64_frac": t_f64 / ms, "binding_frac": max(t_hbm, t_f64) / ms,
           "hbm_gbs": alg_bytes / (ms * 1e-3) / 1e9, "fp64_tflops": flops / (ms * 1e-3) / 1e12,
           "flops_form": "3 m n^2 (Y stored)" if stores_y(cfg["n"]) else "4 m n^2 (fused)"}
    if stores_y(cfg["n"]) and cfg["n"] <= 128:       # where a form was CHOSEN: the fraction against the fused form's floors too
        _, _, th4, tf4 = floors(cfg["m"], cfg["n"], hbm_peak, store_y=False)
        out["binding_frac_vs_fused_form_floors"] = max(th4, tf4) / ms
    if clocks is not None:
        out["clocks"] = clocks
    return out


def time_batched(B, inputs, stream, hbm_peak, batch=1024):
    """mrcqr_factor_batched on `batch` problems of BASELINE.json configs[0]'s shape (m = 4096, n = 16, s = 32, FP32 sketch)
    against the same problems factored one mrcqr_factor call after the other."""
    import torch
    c0 = inputs.CONFIGS["C0"]
    m, n, s, prec = c0["m"], c0["n"], c0["s"], c0["prec"]
    G = inputs.gaussian_colmajor(m, n * batch, 7000, "cuda").view(batch, n, m)
    V = inputs.orthogonal_factor(n, 7001, "cuda")
    AB = torch.matmul((V * inputs.sigma_logspaced(n, c0["exponent"], "cuda").unsqueeze(0)).unsqueeze(0), G).contiguous()
    QB = torch.empty_like(AB)
    RB = torch.empty((batch, n, n), dtype=torch.float64, device="cuda")
    for _ in range(3):
        B.mrcqr_factor_batched(AB, prec, s, 1, QB, RB, stream)
    reps = 10
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(reps):
        B.mrcqr_factor_batched(AB, prec, s, 1, QB, RB, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    loop_n = 64
    R1 = torch.empty((n, n), dtype=torch.float64, device="cuda")
    for b in range(3):
        B.mrcqr_factor(AB[b], prec, s, 1 + b, QB[b], R1, stream)
    e0.record(stream)
    for b in range(loop_n):
        B.mrcqr_factor(AB[b], prec, s, 1 + b, QB[b], R1, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    loop_ms = e0.elapsed_time(e1) / loop_n
    e0.record(stream)
    for b in range(loop_n):
        B.mrcqr_factor_async(AB[b], prec, s, 1 + b, QB[b], R1, stream)
    e1.record(stream)
    B.mrcqr_wait()
    torch.cuda.synchronize()
    loop_async_ms = e0.elapsed_time(e1) / loop_n
    alg = 32.0 * m * n * batch
    return {"workload": "%d problems of the C0 shape (m=%d n=%d s=%d fp%d) in one mrcqr_factor_batched call" % (batch, m, n, s, prec),
            "ms": ms, "us_per_problem": ms * 1e3 / batch, "one_call_after_the_other_ms_per_problem": loop_ms,
            "calls_in_flight_ms_per_problem": loop_async_ms,
            "speedup_over_loop": loop_ms * batch / ms, "hbm_gbs": alg / (ms * 1e-3) / 1e9, "hbm_frac": alg / (ms * 1e-3) / 1e9 / hbm_peak}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_18411_b200 import binding as B
    from paper_2606_18411_b200 import inputs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()
    cfg = workload(args.config)
    m, n, s, prec, seed = cfg["m"], cfg["n"], cfg["s"], cfg["prec"], cfg["seed_draw"]
    AT = inputs.make_config(cfg, "cuda")
    QT = torch.empty_like(AT)
    R = torch.empty((n, n), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    total_ms, launches, stages = time_point(B, AT, QT, R, cfg, args.steps, args.warmup, stream, sampler, barrier)
    clocks = sampler.stop()
    total_ms = max_over_ranks(total_ms, "cuda")
    ms = total_ms / args.steps

    hbm_peak, how = measured_peaks()
    in_flight = time_in_flight(B, AT, QT, R, cfg, args.steps, stream, hbm_peak)

    # ---- both forms of stage 2 where the library chooses (n16 <= 128) ----
    variants = time_forms(B, AT, QT, R, cfg, args.steps, stream) if n <= 128 else None

    # ---- end to end: HOST buffers through mrcqr_factor_host (H2D + D2H inside the timed region) ----
    A_host = torch.empty((n, m), dtype=torch.float64, pin_memory=True)
    A_host.copy_(AT)
    Q_host = torch.empty((n, m), dtype=torch.float64, pin_memory=True)
    R_host = torch.empty((n, n), dtype=torch.float64, pin_memory=True)
    e2e_steps = max(1, min(args.steps, 5))
    B.mrcqr_factor_host(A_host, prec, s, seed, Q_host, R_host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        B.mrcqr_factor_host(A_host, prec, s, seed, Q_host, R_host)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
    e2e_ms = max_over_ranks(e2e_ms, "cuda")
    del A_host, Q_host

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        _, cpu = time_oracle(cfg, AT.cpu().numpy().T, 1, 0)

    # ---- the other configurations of BASELINE.json, same protocol, carried in the same line ----
    points = []
    if rank == 0 and world == 1 and not args.no_points:
        del AT, QT
        torch.cuda.empty_cache()
        for name in POINTS:
            if name == cfg["name"]:
                continue
            pc = workload(name)
            PA = inputs.make_config(pc, "cuda")
            PQ = torch.empty_like(PA)
            PR = torch.empty((pc["n"], pc["n"]), dtype=torch.float64, device="cuda")
            psamp = ClockSampler(local)
            psteps = max(1, min(args.steps, 10))
            ptot, _, pstages = time_point(B, PA, PQ, PR, pc, psteps, 3, stream, psamp)
            pj = point_json(pc, ptot / psteps, pstages, hbm_peak, psamp.stop())
            pj["in_flight"] = time_in_flight(B, PA, PQ, PR, pc, 2 * psteps, stream, hbm_peak)
            if pc["n"] <= 128:
                pj["forms"] = time_forms(B, PA, PQ, PR, pc, psteps, stream)
            points.append(pj)
            del PA, PQ
            torch.cuda.empty_cache()

    # ---- repeated-call mode: 1024 problems of the C0 shape in one call ----
    batched = None
    if rank == 0 and world == 1 and not args.no_points:
        batched = time_batched(B, inputs, stream, hbm_peak)

    if rank == 0:
        alg_bytes, flops, t_hbm, t_f64 = floors(m, n, hbm_peak)
        roof = dominant_kernel(cfg, stages, hbm_peak, how)
        line = {"metric": METRIC, "value": ms, "unit": "ms", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_json(cfg),
                "factorizations_per_s": world * 1e3 / ms,
                "pipeline": {"algorithmic_bytes": alg_bytes, "algorithmic_flops": flops,
                             "hbm_gbs": alg_bytes / (ms * 1e-3) / 1e9, "hbm_peak_gbs": hbm_peak,
                             "hbm_frac": alg_bytes / (ms * 1e-3) / 1e9 / hbm_peak,
                             "fp64_tflops": flops / (ms * 1e-3) / 1e12, "fp64_peak_tflops": FP64_DMMA_PEAK_TFLOPS,
                             "fp64_frac": flops / (ms * 1e-3) / 1e12 / FP64_DMMA_PEAK_TFLOPS,
                             "hbm_floor_ms": t_hbm, "fp64_floor_ms": t_f64, "binding_frac": max(t_hbm, t_f64) / ms,
                             "stage_ms": stages,
                             "extra_traffic": ("Y stored: +8 m n bytes beyond the 32 m n algorithmic bytes (written by stage 2a, "
                                               "read instead of A by stage 2b)" + ("; + 8 m n read by the SYRK" if syrk_form(n) else ""))
                             if stores_y(n) else None},
                "in_flight": in_flight, "variants": variants, "roofline": roof, "cpu_baseline": cpu,
                "e2e": {"value": e2e_ms, "unit": "ms", "h2d_bytes_per_step": 8 * m * n,
                        "d2h_bytes_per_step": 8 * m * n + 8 * n * n, "steps": e2e_steps},
                "gpu_launches": launches, "clocks": clocks, "points": points, "batched": batched, "src_sha16": source_sha16()}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# The paper's Table I: MRCQR on an H100 PCIe with cuFFT / cuBLAS / cuSOLVER, m = 2^20,
# c = 3n, mean of 5 trials, ms, by sketch precision (fp64, fp32, fp16).  Context only: another machine, another build.
PAPER_TABLE1 = {20: (2.60, 2.33, 2.19), 40: (5.22, 4.71, 4.46), 60: (7.84, 7.06, 6.67), 80: (10.80, 9.77, 9.26),
                100: (14.05, 12.75, 12.11), 120: (17.18, 15.62, 14.84), 140: (21.15, 19.32, 18.41), 160: (23.64, 21.56, 20.53),
                180: (27.48, 25.18, 24.00), 200: (31.43, 28.83, 27.50)}


def run_table1(args):
    """--table1: the shapes of the paper's Table I (m = 2^20, n = 20 .. 200, s = 3n, the three sketch precisions) on
    synthetic matrices of the BASELINE.json recipe (kappa ~ 1e4, seeds 60+n / 61+n / 62+n), ms per factorization
    (mrcqr_factor, CUDA events, 3 warm-ups + --steps timed), the paper's H100 figure beside each as context."""
    import torch
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import gpu_orth_error_fro
    from paper_2606_18411_b200 import binding as B
    from paper_2606_18411_b200 import inputs
    m = 1 << 20
    print("| n | s | fp64 sketch ms (paper, H100 PCIe) | fp32 sketch ms (paper) | fp16 sketch ms (paper) | orth (fp16) |")
    print("|---|---|---|---|---|---|")
    for n in sorted(PAPER_TABLE1):
        AT = inputs.make_A(m, n, 4, 60 + n, 61 + n, "cuda")
        QT = torch.empty_like(AT)
        R = torch.empty((n, n), dtype=torch.float64, device="cuda")
        cells = []
        for k, prec in enumerate((64, 32, 16)):
            for _ in range(3):
                B.mrcqr_factor(AT, prec, 3 * n, 62 + n, QT=QT, R=R)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(args.steps):
                B.mrcqr_factor(AT, prec, 3 * n, 62 + n, QT=QT, R=R)
            e1.record()
            torch.cuda.synchronize()
            cells.append("%.3f (%.2f)" % (e0.elapsed_time(e1) / args.steps, PAPER_TABLE1[n][k]))
        print("| %d | %d | %s | %s | %s | %.1e |" % (n, 3 * n, cells[0], cells[1], cells[2], gpu_orth_error_fro(QT)), flush=True)
        del AT, QT
    return 0


def run_sweep(args):
    """--sweep: BASELINE.json configs[0..3] and the column sweep configs[4] (m = 2^21, n in 16..512, three sketch
    precisions): per-stage CUDA-event times and both roofline floors, one markdown table row per point (not the
    bench contract's JSON line; used for profiles/ and DESIGN.md)."""
    import torch
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import gpu_orth_error_fro, gpu_residual_fro
    from paper_2606_18411_b200 import binding as B
    from paper_2606_18411_b200 import inputs
    hbm_peak, _ = measured_peaks()
    points = [(k, dict(inputs.CONFIGS[k])) for k in ("C0", "C1", "C2", "C3")]
    for n in (16, 32, 64, 128, 256, 512):
        for prec in (16, 32, 64):
            points.append(("C4 n=%d fp%d" % (n, prec), inputs.sweep_config(n, prec)))
    print("| config | m | n | sketch | total ms | K1 | K2 | K3 / solve | reduce+K4 (+SYRK) | K5 / solve | HBM floor | FP64 floor | orth | resid |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for name, cfg in points:
        AT = inputs.make_config(cfg, "cuda")
        n, m = AT.shape
        QT = torch.empty_like(AT)
        R = torch.empty((n, n), dtype=torch.float64, device="cuda")
        B.mrcqr_set_timing(True)
        acc = {}
        for it in range(3 + args.steps):
            B.mrcqr_factor(AT, cfg["prec"], cfg["s"], cfg["seed_draw"], QT=QT, R=R)
            if it >= 3:
                for k, v in B.mrcqr_last_timing().items():
                    acc[k] = acc.get(k, 0.0) + v / args.steps
        B.mrcqr_set_timing(False)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            B.mrcqr_factor(AT, cfg["prec"], cfg["s"], cfg["seed_draw"], QT=QT, R=R)
        e1.record()
        torch.cuda.synchronize()
        tot = e0.elapsed_time(e1) / args.steps
        flop = (3.0 if stores_y(n) else 4.0) * m * n * n
        print("| %s | %d | %d | fp%d | %.3f | %.3f | %.3f | %.3f | %.3f | %.3f | %.3f | %.3f | %.1e | %.1e |" % (
            name, m, n, cfg["prec"], tot, acc["k1_srtt"], acc["k2_sketch_qr"], acc["k3_gram"], acc["gram_reduce"] + acc["k4_chol"],
            acc["k5_form_q"], 32.0 * m * n / (hbm_peak * 1e9) * 1e3, flop / (FP64_DMMA_PEAK_TFLOPS * 1e12) * 1e3,
            gpu_orth_error_fro(QT), gpu_residual_fro(AT, QT, R)), flush=True)
        del AT, QT
        torch.cuda.empty_cache()


def run_stability(args):
    """--stability: the MRCQR curves of the paper's Fig. 1 on its own test matrices (eq. (3):
    A = U Sigma V^T, m = 2^17, n = 50, kappa = 1e2 .. 1e16, s = 3n): ||I - Q^T Q||_F and ||A - QR||_F / ||A||_F for the
    three sketch precisions, plus the self-correcting wrapper started at FP16.  Markdown table."""
    import torch
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import gpu_residual_fro
    from paper_2606_18411_b200 import binding as B
    from paper_2606_18411_b200 import inputs
    m, n = 1 << 17, 50
    print("| kappa | fp16 orth | fp16 resid | fp32 orth | fp32 resid | fp64 orth | fp64 resid | auto: precision used, orth |")
    print("|---|---|---|---|---|---|---|---|")
    for e in range(2, 17, 2):
        AT = inputs.make_paper_eq3(m, n, 10.0 ** e, 100 + e, 200 + e, "cuda")
        QT = torch.empty_like(AT)
        R = torch.empty((n, n), dtype=torch.float64, device="cuda")
        cells = []
        for prec in (16, 32, 64):
            rc = B.mrcqr_factor(AT, prec, 3 * n, 7, QT, R, check=False)
            if rc != 0:
                cells += ["code %d" % rc, "-"]
            else:
                cells += ["%.1e" % B.mrcqr_orth_error(QT), "%.1e" % gpu_residual_fro(AT, QT, R)]
        rc, used, orth = B.mrcqr_factor_auto(AT, 16, 3 * n, 7, 0.0, QT, R, check=False)
        cells.append("fp%d, %.1e%s" % (used, orth, "" if rc == 0 else " (code %d)" % rc))
        print("| 1e%d | %s |" % (e, " | ".join(cells)), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    def config_name(v):                  # BASELINE.json configs[0..3], or a point of the column sweep: C4n<any n in 1 .. 512>
        if v in ("C0", "C1", "C2", "C3") or (v.startswith("C4n") and v[3:].isdigit() and 1 <= int(v[3:]) <= 512):
            return v
        raise argparse.ArgumentTypeError("C0 | C1 | C2 | C3 | C4n<n>, 1 <= n <= 512")
    ap.add_argument("--config", default="C3", type=config_name)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-points", action="store_true", help="skip the other configurations carried under \"points\"")
    ap.add_argument("--traffic-from", default=None, help="ncu --page raw --csv file: record per-kernel DRAM bytes of --config in profiles/r02_traffic.json")
    ap.add_argument("--stability", action="store_true", help="orthogonality / residual vs kappa on the paper's eq.(3) matrices")
    ap.add_argument("--sweep", action="store_true", help="per-stage table over BASELINE.json configs 0-4 instead of the JSON line")
    ap.add_argument("--table1", action="store_true", help="the shapes of the paper's Table I (m = 2^20, n = 20..200, s = 3n), the paper's H100 figures beside as context")
    args = ap.parse_args()
    if args.traffic_from:
        return write_traffic(args.traffic_from, args.config)
    if args.stability:
        return run_stability(args)
    if args.table1:
        return run_table1(args)
    if args.sweep:
        args.steps = min(args.steps, 5)
        return run_sweep(args)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
