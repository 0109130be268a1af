#!/usr/bin/env python
"""bench.py -- one JSON line: log-likelihood evaluations / s of the batched lens likelihood.

A step = one lensed_loglike call on one batch of B synthetic parameter vectors: prep ->
fused ray-trace + surface brightness + quadrature -> PSF convolution + chi-square -> logL[B]
(all rows of SURVEY.md section 8(a)).  Workload at N = 1: BASELINE.json's largest config,
the Euclid-scale sweep (512x512 @ 0.1"/px, SIE + shear + Sersic source + Sersic lens light
+ sky, 31x31 Moffat PSF, 16-point sub4 rule) at its largest batch, B = 16384 -- the config
north_star quotes the roofline target on.  The same line carries, as extras, a short row for each
of the other configs (`per_config`: 0-3 and 5 = the paper's mock scenario; flushed, back-to-back
and CUDA-graph step times, tracer / convolution fraction of the FP32 roofline, the oracle beside
it), the Euclid batch sweep (`sweep`) and the likelihood rate inside the device-resident nested
sampler (`nested_sampling`).  `--config N --batch B` time one config alone.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

N > 1 (under torchrun): every rank holds a replica of the handle and its own B vectors
(batch sharding, no data-path collective; "weak" scaling); time = max over ranks.
--impl reference times the CPU oracle (oracle/, test infrastructure, as it stands) on the
host cores on a bounded sample of the same workload.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1505_07674_b200 import synth  # noqa: E402

METRIC = "loglike_evals_per_sec"
UNIT = "logL/s"
DEFAULT_CONFIG = 4
SM_COUNT, FP32_LANES, SM_MAX_MHZ = 148, 128, 1965.0
NOMINAL_FP32_TFLOPS = SM_COUNT * FP32_LANES * 2 * SM_MAX_MHZ * 1e6 / 1e12      # 74.45

# Algorithmic FP32 flops (FMA = 2), SURVEY.md section 8(d) / DESIGN.md "flop model"
FLOPS_RAY_POS, FLOPS_QUAD = 4, 2
FLOPS_MODEL = {"sie": 50, "sis": 10, "point": 10, "shear": 8, "src_sersic": 17, "fg_sersic": 17,
               "src_gauss": 16, "fg_gauss": 16, "sky": 0}
MUFU_MODEL = {"sie": 4, "sis": 1, "point": 1, "shear": 0, "src_sersic": 3, "fg_sersic": 3,
              "src_gauss": 1, "fg_gauss": 1, "sky": 0}


def flops_per_ray(models):
    return FLOPS_RAY_POS + FLOPS_QUAD + sum(FLOPS_MODEL[m] for m in models)


# "if the build uses a cheaper algorithm ... it counts that algorithm's flops".  The
# specialised tracers take a foreground Sersic's pixel integral from its moment expansion
# (DESIGN.md section 5): 25-70 flops per PIXEL instead of 17 per RAY, for all but the few pixels
# around the profile's centre.  The count of the algorithm that runs charges the expansion's
# fourth-order cost for every pixel, spread over the pixel's rays.  The pixels that still take the
# per-ray sum do more work than that, so this is a LOWER bound on the work required and on the
# fraction; the bench line's `frac` of a tracer-dominant config uses it.
FG_EXPANSION_FLOPS_PER_PIXEL = 70


def rule_is_symmetric(quad):
    """first and third moments of the rule vanish (the condition api.cu puts on the expansion)"""
    q = np.asarray(quad, dtype=np.float64).reshape(-1, 3)
    x, y, w = q[:, 0], q[:, 1], q[:, 2] / q[:, 2].sum()
    m = [w @ x, w @ y, w @ x ** 3, w @ (x * x * y), w @ (x * y * y), w @ y ** 3]
    return bool(max(abs(v) for v in m[:2]) < 1e-7 and max(abs(v) for v in m[2:]) < 1e-8)


def flops_per_ray_run(models, n_quad, expansion):
    """flops per ray of the algorithm in use: as flops_per_ray, foreground Sersics by expansion"""
    if not expansion:
        return float(flops_per_ray(models))
    n_fg = sum(1 for m in models if m == "fg_sersic")
    return flops_per_ray(models) - n_fg * FLOPS_MODEL["fg_sersic"] + n_fg * FG_EXPANSION_FLOPS_PER_PIXEL / n_quad


def flops_per_conv_pixel(cfg):
    taps = 1 if cfg.psf is None else cfg.psf.size
    return 2 * taps + 3


def workload_name(cfg, B):
    psf = "delta" if cfg.psf is None else "%dx%d" % cfg.psf.shape
    return "%s %dx%d @%.2f\"/px, %s, PSF %s, %d-point rule, B=%d" % (
        cfg.name, cfg.H, cfg.W, cfg.scale, "+".join(cfg.models), psf, len(cfg.quad), B)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons while the timed region runs (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [c.strip() for c in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for t, r in self.rows if t0 <= t <= t1] or [r for _, r in self.rows[-3:]]
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_problem(cfg, image, weight):
    """(callable params -> logL) on the CPU oracle; imported here only (cpu_baseline / reference)."""
    from oracle import lensed_oracle as orc
    kinds = synth.kind_ids(cfg.models)

    def f(params):
        return orc.loglike(cfg.H, cfg.W, cfg.scale, image, weight, cfg.mask, cfg.psf, cfg.quad, kinds,
                           params, zp=cfg.zp)
    return f, orc.threads()


def time_oracle(cfg, image, weight, params, budget_s):
    """Oracle logL/s on a bounded sample: 1 vector to size it, then about budget_s of work."""
    f, cores = oracle_problem(cfg, image, weight)
    t0 = time.perf_counter(); f(params[:1]); t1 = time.perf_counter() - t0
    n = int(max(1, min(len(params), budget_s / max(t1, 1e-6))))
    t0 = time.perf_counter(); f(params[:n]); dt = time.perf_counter() - t0
    return n / dt, cores, n, dt


def make_observation_cuda(cfg, device):
    """Observed image + weights: truth rendered by the CUDA library, seeded noise from synth."""
    import torch
    from paper_1505_07674_b200 import lensed
    kinds = synth.kind_ids(cfg.models)
    h = lensed.lensed_create(np.zeros((cfg.H, cfg.W), np.float32), np.ones((cfg.H, cfg.W), np.float32),
                             None, cfg.psf, cfg.quad, kinds, cfg.scale, cfg.zp, device)
    p = torch.from_numpy(cfg.truth.astype(np.float32)[None]).cuda(device)
    m = torch.empty((1, cfg.H, cfg.W), dtype=torch.float32, device=p.device)
    lensed.lensed_render(h, p, m)
    torch.cuda.synchronize(device)
    lensed.lensed_destroy(h)
    return cfg.observe(m[0].cpu().numpy())


def make_observation_oracle(cfg):
    from oracle import lensed_oracle as orc
    truth = orc.render(cfg.H, cfg.W, cfg.scale, cfg.psf, cfg.quad, synth.kind_ids(cfg.models),
                       cfg.truth.astype(np.float32), zp=cfg.zp)[0]
    return cfg.observe(truth)


def run_reference(args, cfg, B):
    """The reference arm of this tier: the CPU oracle, rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    image, weight = make_observation_oracle(cfg)
    params = cfg.batch(B)
    f, cores = oracle_problem(cfg, image, weight)
    t0 = time.perf_counter(); f(params[:1]); t1 = time.perf_counter() - t0
    total = max(1, args.steps + args.warmup)
    n = int(max(1, min(B, 120.0 / total / max(t1, 1e-6))))          # whole run within ~2 minutes
    for _ in range(args.warmup):
        f(params[:n])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        f(params[:n])
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    sample = "%d of the %d vectors per step, full image" % (n, B)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": workload_name(cfg, B), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))




class Bench:
    """One handle on one config with its device buffers; `run` times K steps of lensed_loglike."""

    def __init__(self, lensed, torch, index, B, local, rank, args=None):
        self.L, self.torch, self.index, self.B, self.local = lensed, torch, index, B, local
        self.cfg = cfg = synth.get_config(index)
        self.dev = torch.device("cuda", local)
        self.image, self.weight = make_observation_cuda(cfg, local)
        self.h = lensed.lensed_create(self.image, self.weight, cfg.mask, cfg.psf, cfg.quad,
                                      synth.kind_ids(cfg.models), cfg.scale, cfg.zp, local)
        if args is not None and args.interpreter:
            lensed.lensed_set_static_tracer(self.h, 0)
        if args is not None and args.conv_shape != "auto":
            lensed.lensed_set_conv_shape(self.h, lensed.CONV_SHAPES.index(args.conv_shape))
        self.tracer_kind = ("interpreter", "static", "jit")[lensed.lensed_get_static_tracer(self.h)]
        self.conv_shape = lensed.CONV_SHAPES[lensed.lensed_get_conv_shape(self.h)]
        # the foreground expansion runs in the specialised tracers on rules without odd moments
        self.fg_expansion = self.tracer_kind != "interpreter" and rule_is_symmetric(cfg.quad)
        self.flops_ray = flops_per_ray(cfg.models)                                          # SURVEY.md 8(d)'s count
        self.flops_ray_run = flops_per_ray_run(cfg.models, len(cfg.quad), self.fg_expansion)   # the algorithm in use
        self.n_traced = cfg.n_traced()                       # m_d, the required set
        assert self.n_traced <= lensed.lensed_num_traced(self.h)
        self.n_counted = int(cfg.H * cfg.W if cfg.mask is None else cfg.mask.sum())
        self.params = cfg.batch(B, stream=2 + rank)          # this rank's shard of the global batch
        self.p_dev = torch.from_numpy(self.params).to(self.dev)
        self.logl = torch.empty(B, dtype=torch.float32, device=self.dev)

    def close(self):
        self.L.lensed_destroy(self.h)

    def run(self, steps, warmup, flush, barrier=None):
        """-> (ms of every timed step, per-phase ms, per-phase launches, wall t0, t1)"""
        L, torch, h = self.L, self.torch, self.h
        stream = torch.cuda.current_stream()
        for _ in range(warmup):
            L.lensed_loglike(h, self.p_dev, self.logl)
        L.lensed_set_profiling(h, True)
        L.lensed_reset_profile(h)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        (barrier or torch.cuda.synchronize)()
        t0 = time.perf_counter()
        for a, b in ev:
            flush.zero_()                                    # L2 flush between timed iterations (untimed)
            a.record(stream)
            L.lensed_loglike(h, self.p_dev, self.logl)
            b.record(stream)
        (barrier or torch.cuda.synchronize)()
        t1 = time.perf_counter()
        ms = [a.elapsed_time(b) for a, b in ev]
        phase_ms, phase_n = L.lensed_get_profile(h)
        L.lensed_set_profiling(h, False)
        return ms, phase_ms, phase_n, t0, t1

    def back_to_back(self, n=30):
        """ms per step of n calls in a row with profiling off and no L2 flush -- how a sampler calls it --
        issued one by one, and replayed from a CUDA graph of one step"""
        L, torch = self.L, self.torch
        a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        L.lensed_loglike(self.h, self.p_dev, self.logl)
        torch.cuda.synchronize()
        a.record()
        for _ in range(n):
            L.lensed_loglike(self.h, self.p_dev, self.logl)
        e.record()
        torch.cuda.synchronize()
        plain = a.elapsed_time(e) / n
        try:                                                 # an extra: never take the bench line down with it
            s, g = torch.cuda.Stream(), torch.cuda.CUDAGraph()
            with torch.cuda.stream(s):
                L.lensed_loglike(self.h, self.p_dev, self.logl, stream=s)
                s.synchronize()
                with torch.cuda.graph(g, stream=s):
                    L.lensed_loglike(self.h, self.p_dev, self.logl, stream=torch.cuda.current_stream())
            torch.cuda.synchronize()
            a.record()
            for _ in range(n):
                g.replay()
            e.record()
            torch.cuda.synchronize()
            graph = a.elapsed_time(e) / n
        except Exception:                                    # noqa: BLE001
            torch.cuda.synchronize()
            graph = None
        return plain, graph

    def flop_model(self, steps, phase_n):
        """algorithmic flops of ONE launch of the tracer / the convolution, averaged over its launches"""
        cfg = self.cfg
        return {"trace": self.flops_ray_run * len(cfg.quad) * self.n_traced * self.B * steps / max(phase_n["trace"], 1),
                "conv": flops_per_conv_pixel(cfg) * self.n_counted * self.B * steps / max(phase_n["conv"], 1)}

    def kernels(self, steps, phase_ms, phase_n):
        per_launch = self.flop_model(steps, phase_n)
        out = {}
        for k in self.L.PHASES:
            tf = None
            if k in per_launch and phase_ms[k] > 0:
                tf = per_launch[k] * phase_n[k] / (phase_ms[k] * 1e-3) / 1e12
            out[k] = {"ms_per_step": phase_ms[k] / steps, "launches_per_step": phase_n[k] / steps, "tflops": tf,
                      "frac": tf / NOMINAL_FP32_TFLOPS if tf else None}
        return out

    def summary(self, steps, warmup, flush):
        """short row for the per-config table of the bench line"""
        ms, phase_ms, phase_n, _, _ = self.run(steps, warmup, flush)
        cfg = self.cfg
        value = self.B * steps / (sum(ms) * 1e-3)
        per_launch = self.flop_model(steps, phase_n)
        k = self.kernels(steps, phase_ms, phase_n)
        whole = (per_launch["trace"] * phase_n["trace"] + per_launch["conv"] * phase_n["conv"]) / (sum(ms) * 1e-3) / 1e12
        b2b, graph = self.back_to_back()
        return {"config": self.index, "ms_per_step_back_to_back": b2b, "ms_per_step_cuda_graph": graph,
                "logl_per_s_back_to_back": self.B / (b2b * 1e-3), "workload": workload_name(cfg, self.B), "logl_per_s": value,
                "rays_per_s": value * self.n_traced * len(cfg.quad), "ms_per_step": sum(ms) / steps, "steps": steps,
                "tracer": self.tracer_kind, "conv_shape": self.conv_shape,
                "trace_ms": k["trace"]["ms_per_step"], "trace_frac": k["trace"]["frac"],
                "trace_frac_survey_count": k["trace"]["frac"] * self.flops_ray / self.flops_ray_run if k["trace"]["frac"] else None,
                "flops_per_ray": self.flops_ray, "flops_per_ray_run": self.flops_ray_run,
                "conv_ms": k["conv"]["ms_per_step"], "conv_frac": k["conv"]["frac"],
                "other_ms": sum(k[p]["ms_per_step"] for p in ("prep", "refine", "final")),
                "whole_step_frac": whole / NOMINAL_FP32_TFLOPS}


def parity_sample(lensed, torch, bench, logl_dev, n):
    """SURVEY.md section 4 "max and 99.999th-percentile pixel error", at the scale the bench runs: n vectors
    spread evenly over the timed batch, logL (the values the timed region produced) and rendered pixels
    against the CPU oracle as checker, in chunks of 32 vectors.  Also the FP64-refined pixels per vector,
    so that the refinement threshold is looked at once at full batch size."""
    from oracle import lensed_oracle as orc
    cfg = bench.cfg
    idx = np.unique(np.linspace(0, bench.B - 1, min(n, bench.B)).astype(np.int64))
    kinds = synth.kind_ids(cfg.models)
    logl_g = logl_dev.cpu().numpy()[idx].astype(np.float64)
    el, ep, pix_all = [], [], []
    model = torch.empty((32, cfg.H, cfg.W), dtype=torch.float32, device=bench.dev)
    for c0 in range(0, len(idx), 32):
        sel = idx[c0:c0 + 32]
        p = bench.params[sel]
        lo, mo = orc.loglike(cfg.H, cfg.W, cfg.scale, bench.image, bench.weight, cfg.mask, cfg.psf, cfg.quad, kinds, p,
                             zp=cfg.zp, want_model=True)
        lensed.lensed_render(bench.h, torch.from_numpy(p).to(bench.dev), model[:len(sel)])
        torch.cuda.synchronize()
        mg = model[:len(sel)].cpu().numpy().astype(np.float64)
        el.extend(np.abs(logl_g[c0:c0 + 32] - lo) / np.maximum(np.abs(lo), 1e-300))
        for g, r in zip(mg, mo):
            big = np.abs(r) > 1e-3 * np.abs(r).max()
            e = np.abs(g[big] - r[big]) / np.abs(r[big])
            ep.append(e.max())
            pix_all.append(e)
    el, ep, pix_all = np.array(el), np.array(ep), np.concatenate(pix_all)
    lensed.lensed_reset_profile(bench.h)
    lensed.lensed_loglike(bench.h, bench.p_dev, bench.logl)
    refined = lensed.lensed_get_refined(bench.h)
    return {"vectors": int(len(idx)), "logl_tol": 1e-5, "pixel_tol": 1e-4,
            "logl_err_max": float(el.max()), "logl_err_p999": float(np.quantile(el, 0.999)), "logl_over_tol": int((el > 1e-5).sum()),
            "pixel_err_max": float(ep.max()), "pixel_err_p99999": float(np.quantile(pix_all, 0.99999)),
            "pixels_checked": int(pix_all.size), "vectors_with_a_pixel_over_tol": int((ep > 1e-4).sum()),
            "refined_pixels_per_vector": refined / bench.B}


def nested_row(lensed, torch, local, rounds=40, n_live=1024, batch=1024):
    """The batched likelihood inside its caller: a fixed number of rounds of the
    device-resident nested sampler on the HST config at full size, six free parameters in a box
    around the truth.  Likelihood evaluations per second of wall time, everything included
    (proposals, lensed_loglike, replacement, evidence); the call is synchronous."""
    b = Bench(lensed, torch, 1, 1, local, 0)
    t = b.cfg.truth.astype(np.float64)
    lo, hi = t.copy(), t.copy()
    lo[2], hi[2] = t[2] - 0.03, t[2] + 0.03                  # Einstein radius
    lo[3], hi[3] = t[3] - 0.05, t[3] + 0.05                  # lens axis ratio
    lo[7:9], hi[7:9] = t[7:9] - 0.03, t[7:9] + 0.03          # source position
    lo[9], hi[9] = 0.8 * t[9], 1.25 * t[9]                   # source radius
    lo[10], hi[10] = t[10] - 0.3, t[10] + 0.3                # source magnitude
    kw = dict(n_live=n_live, batch=batch, tol=1e-30, enlarge=1.2, seed=5)
    lensed.lensed_ns_run(b.h, lo, hi, max_rounds=3, **kw)    # warm-up: allocations, first launches
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    res = lensed.lensed_ns_run(b.h, lo, hi, max_rounds=rounds, **kw)
    dt = time.perf_counter() - t0
    b.close()
    return {"workload": workload_name(b.cfg, batch) + ", %d live points, 6 free parameters" % n_live,
            "rounds": int(res["n_rounds"]), "likelihood_calls": int(res["n_likelihood"]),
            "likelihood_per_s": res["n_likelihood"] / dt, "rounds_per_s": res["n_rounds"] / dt,
            "dead_points": int(res["n_dead"]), "wall_s": dt, "timing": "host wall clock around the synchronous call"}


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` with no launcher around it: start the N ranks ourselves, the
    way the driver's torchrun line does (one process per GPU, NCCL rendezvous on 127.0.0.1)."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG)
    ap.add_argument("--batch", type=int, default=0, help="vectors per GPU per step (0 = the config's)")
    ap.add_argument("--no-sweep", action="store_true", help="skip the batch sweep of the Euclid config")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the per-config rows (configs 0-3, 5, 6) and the nested-sampling row")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--conv-shape", default="auto", choices=("auto", "wide", "narrow", "strip", "half"),
                    help="convolution shape (include/lensed.h); auto = what lensed_create picks")
    ap.add_argument("--parity-sample", type=int, default=0, metavar="N",
                    help="extra, outside the timed region: N vectors spread over the batch against the CPU oracle "
                         "(logL and rendered pixels), max and 99.9th-percentile error; Euclid: ~0.06 s of oracle per vector")
    ap.add_argument("--interpreter", action="store_true",
                    help="run the interpreting tracer instead of the compile-time specialised one")
    args = ap.parse_args()
    cfg = synth.get_config(args.config)
    B = args.batch or cfg.B
    if args.impl == "reference":
        return run_reference(args, cfg, B)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return respawn_under_torchrun(args)

    import torch
    import torch.distributed as dist
    from paper_1505_07674_b200 import lensed

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device: the library has no CPU fallback")
    if local >= torch.cuda.device_count():
        raise SystemExit("bench.py --gpus %d: rank %d has no GPU (%d visible)" % (world, local, torch.cuda.device_count()))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2
    bench = Bench(lensed, torch, args.config, B, local, rank, args)
    h, params, logl = bench.h, bench.params, bench.logl
    n_traced = bench.n_traced

    # ---------------------------------------------------------------- device-resident timing
    clocks = ClockSampler(local)
    ms_steps, phase_ms, phase_n, t_wall0, t_wall1 = bench.run(args.steps, args.warmup, flush, barrier)
    clock_info = clocks.stop(t_wall0, t_wall1)
    total_ms = max_over_ranks(sum(ms_steps))
    value = world * B * args.steps / (total_ms * 1e-3)
    rays_per_s = value * n_traced * len(cfg.quad)

    # ------------------------------------------------------------- end to end, host buffers
    p_host = torch.from_numpy(params).pin_memory()
    l_host = torch.empty(B, dtype=torch.float32).pin_memory()
    lensed.lensed_loglike_host(h, p_host, l_host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        lensed.lensed_loglike_host(h, p_host, l_host)       # H2D + path + D2H + stream sync, every step
    e2e_value = world * B * args.steps / max_over_ranks(time.perf_counter() - t0)
    assert np.array_equal(l_host.numpy(), logl.cpu().numpy())

    # ------------------------------------------------------------------------------ roofline
    per_launch = bench.flop_model(args.steps, phase_n)
    kern = bench.kernels(args.steps, phase_ms, phase_n)
    dom = max(("trace", "conv"), key=lambda k: phase_ms[k])
    avg_ms = phase_ms[dom] / max(phase_n[dom], 1)
    achieved = per_launch[dom] / (avg_ms * 1e-3) / 1e12
    try:
        measured_ffma = lensed.lensed_fma_peak(local, 2048)
    except lensed.LensedError:
        measured_ffma = None
    traffic = traffic_src = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")   # dram bytes per vector from the ncu capture
    if os.path.exists(tpath):
        with open(tpath) as fh:
            t = json.load(fh).get("%s:%d" % (dom, args.config))
            if t:                                            # per vector in the capture -> per launch of this run
                traffic = int(t["bytes_per_vector"] * B * args.steps / max(phase_n[dom], 1))
                traffic_src = t["capture"]
    roofline = {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": NOMINAL_FP32_TFLOPS,
                "unit": "TFLOP/s", "frac": achieved / NOMINAL_FP32_TFLOPS, "traffic": traffic,
                "traffic_source": traffic_src,
                "peak_source": "nominal 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md)",
                "measured_ffma_tflops": measured_ffma,
                "frac_of_measured_ffma": achieved / measured_ffma if measured_ffma else None,
                "whole_step_tflops": (per_launch["trace"] * phase_n["trace"] + per_launch["conv"] * phase_n["conv"])
                / (total_ms * 1e-3) / 1e12 if world == 1 else None,
                "flops_per_ray": bench.flops_ray, "flops_per_ray_run": bench.flops_ray_run,
                "flop_count": "flops_per_ray_run: SURVEY 8(d)'s per-ray counts with each foreground Sersic charged its "
                              "moment expansion (70 flops per pixel / n_quad per ray) where the specialised tracer uses it -- "
                              "a lower bound on the work required; every tflops / frac here uses it",
                "fg_expansion": bench.fg_expansion,
                "flops_per_conv_pixel": flops_per_conv_pixel(cfg),
                "kernels": kern}
    if kern["trace"]["frac"]:
        roofline["trace_frac"] = kern["trace"]["frac"]
        roofline["trace_frac_survey_count"] = kern["trace"]["frac"] * bench.flops_ray / bench.flops_ray_run
    if roofline["whole_step_tflops"]:
        roofline["whole_step_frac"] = roofline["whole_step_tflops"] / NOMINAL_FP32_TFLOPS
    if traffic:
        # algorithmic bytes of the dominant kernel per launch: the convolution reads each padded frame once (4 B per
        # pixel; d, w and the taps are amortised over the batch), the tracer writes it once
        alg = 4.0 * cfg.H * cfg.W * B * args.steps / max(phase_n[dom], 1)
        roofline["traffic_over_algorithmic_bytes"] = traffic / alg
        roofline["traffic_note"] = ("not measured in this run: dram bytes per vector of the committed ncu capture (traffic_source), "
                                    "scaled to this launch; above 1 = halo re-reads across tiles, harmless on an ALU-bound kernel")

    # -------------------------------------------------------------- batch sweep (config 4 only)
    sweep = None
    stream = torch.cuda.current_stream()
    if args.config == 4 and not args.no_sweep and world == 1:
        sweep = []
        for Bs in (256, 1024, 4096, 16384):
            ps = torch.from_numpy(cfg.batch(Bs)).to(dev)
            ls = torch.empty(Bs, dtype=torch.float32, device=dev)
            lensed.lensed_loglike(h, ps, ls)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            flush.zero_()
            a.record(stream); lensed.lensed_loglike(h, ps, ls); b.record(stream)
            torch.cuda.synchronize()
            v = Bs / (a.elapsed_time(b) * 1e-3)
            sweep.append({"B": Bs, "logl_per_s": v, "rays_per_s": v * n_traced * len(cfg.quad)})

    # ---------------------------------------------------------------------------- cpu baseline
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, cores, n, dt = time_oracle(cfg, bench.image, bench.weight, params, 15.0)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "%d of the %d vectors, full image, %.1f s" % (n, B, dt)}
    gpu_launches = int(sum(phase_n.values()))
    parity = None
    if rank == 0 and world == 1 and args.parity_sample > 0:
        try:
            parity = parity_sample(lensed, torch, bench, logl, args.parity_sample)
        except Exception as ex:                              # noqa: BLE001 -- an extra: the bench line stands without it
            parity = {"error": str(ex)[:200]}
    bench.close()

    # ------------------------------- the other configs and the sampler row (short, rank 0, N = 1)
    per_config = nested = None
    if args.config == DEFAULT_CONFIG and not args.no_extras and world == 1 and not args.batch:
        per_config = []
        for c, steps in ((0, 20), (1, 20), (2, 10), (3, 5), (5, 10), (6, 10)):
            try:
                b = Bench(lensed, torch, c, synth.get_config(c).B, local, rank, args)
                row = b.summary(steps, 3, flush)
                if not args.no_cpu_baseline:                 # the oracle beside every row, ~3 s each
                    v, cores, n, dt = time_oracle(b.cfg, b.image, b.weight, b.params, 3.0)
                    row["cpu_oracle"] = {"logl_per_s": v, "cores": cores, "sample": "%d vectors, %.1f s" % (n, dt)}
                b.close()
            except Exception as ex:                          # noqa: BLE001 -- an extra: the bench line stands without it
                row = {"config": c, "error": str(ex)[:200]}
            per_config.append(row)
        try:
            nested = nested_row(lensed, torch, local)
        except Exception as ex:                              # noqa: BLE001 -- an extra, see above
            nested = {"error": str(ex)[:200]}

    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(cfg, B), "batch_per_gpu": B, "global_batch": B * world,
                       "traced_pixels": n_traced, "rays_per_step": B * world * n_traced * len(cfg.quad),
                       "parallelism": "batch-sharded x%d, no collective" % world,
                       "tracer": bench.tracer_kind, "conv_shape": bench.conv_shape,
                       "timing": "CUDA events per step, L2 flushed (256 MB write) between steps, max over ranks"},
            "rays_per_sec": rays_per_s,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(params.nbytes),
                    "d2h_bytes_per_step": int(B * 4)},
            "gpu_launches": gpu_launches,
            "clocks": clock_info, "roofline": roofline, "cpu_baseline": cpu,
        }
        if parity is not None:
            out["parity_sample"] = parity
        if sweep is not None:
            out["sweep"] = sweep
        if per_config is not None:
            out["per_config"] = per_config
            out["nested_sampling"] = nested
        print(json.dumps(out, default=lambda o: o.item() if hasattr(o, "item") else str(o)))   # numpy scalars
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
