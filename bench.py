#!/usr/bin/env python
"""bench.py — whole-hot-path throughput of the GA inversion (ga_invert) on synthetic SOLIS/VSM-shaped maps.

A "step" is one pass of the whole hot path over one batch: one `ga_invert` call (observation staging, generation 0,
G generations of select/crossover/mutate/evaluate, output) over the map of the chosen workload.
    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config3|config1|config4|config0|config2] [--impl reference]
Default workload: config3, the north_star target (2048 x 2048 full-disc map, 3.14 M on-disc pixels, 200 generations; one step
takes about a minute on a B200).  config2 times me_synth (forward synthesis of 1e6 prior draws) as the step.
One JSON line on stdout (rank 0).  See DESIGN.md "Measurement" for every field.
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

from paper_1208_0302_b200 import workloads as W  # noqa: E402

# The EXECUTED FP32 work per wavelength point, the FMA-pipe busy fraction and the DRAM bytes per pixel of the kernel
# come from profiles/r*_counters.json, written from an ncu capture by `python -m paper_1208_0302_b200.counters` together with
# a hash of the csrc/ sources that capture ran.  Nothing of that kind is typed in here: a
# workload without a capture, or a capture of other sources, gives `frac: null` and says why.
SM_COUNT, FP32_LANES_PER_SM = 148, 128


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="config3", choices=["config0", "config1", "config2", "config3", "config4"])
    ap.add_argument("--budget-s", type=float, default=1500.0,
                    help="wall-clock budget of the GPU legs: the end-to-end leg is shortened, then dropped, before the timed "
                         "steps are touched; the line says what was done")
    ap.add_argument("--n-side", type=int, default=0, help="override the map side (config1: 256, config3: 2048, config4: 512)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--lines", type=int, default=0, choices=[0, 3],
                    help="3: add a synthetic third line (Fe I 6302.5's pattern at 6302.0 A, as in the parity tests) to exercise the "
                         "run-time-sized multi-line kernels; a measured variant, not a BASELINE config")
    ap.add_argument("--pop", type=int, default=0, help="override the GA population of the workload (a measured variant, not a BASELINE config)")
    ap.add_argument("--generations", type=int, default=-1, help="override the number of generations (likewise)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--aux", action="store_true", help="also run the auxiliary me_synth (config2) legs and saturation trace inside this run")
    ap.add_argument("--no-aux", action="store_true", help="accepted for old command lines; the auxiliary legs are off unless --aux")
    ap.add_argument("--vectors", type=int, default=1_000_000, help="config2: parameter vectors per step")
    ap.add_argument("--chi2-only", action="store_true", help="config2: no [P,4,L] output, chi2 against the fixed profile only")
    ap.add_argument("--zeeman", default="triplets", choices=["triplets", "full"],
                    help="full = LS-coupling Zeeman patterns (12 + 3 components, PAPER.md:351) instead of effective triplets; "
                         "a measured variant, not the headline configuration")
    return ap.parse_args()


def workload(args):
    c, n, side = _workload(args)
    if getattr(args, "zeeman", "triplets") == "full":
        c = dict(c, triplets=False)
    if getattr(args, "lines", 0) == 3:
        c = dict(c, name=c["name"] + "_3lines", lines=list(c["lines"]) + [dict(W.FE_6302, lambda0=6302.0)])
    pop, gens = getattr(args, "pop", 0), getattr(args, "generations", -1)
    if pop > 0 or gens >= 0:            # same box, weights and noise; the name changes so that no counters entry is mistaken for it
        ga = c["ga"]
        pop, gens = pop or ga["pop"], gens if gens >= 0 else ga["generations"]
        c = dict(c, name="%s_pop%d_g%d" % (c["name"], pop, gens),
                 ga=W.ga_config(pop, gens, sigma=c["sigma"], b_lo=c["b_range"][0], b_hi=c["b_range"][1], npar=c.get("npar", 9)))
    return c, n, side


def _workload(args):
    if args.workload == "config2":
        c = W.config2(args.vectors)
        return c, args.vectors, None
    if args.workload == "config0":
        c = W.config0()
        return c, c["n_pixels"], None
    if args.workload == "config1":
        side = args.n_side or 256
        c = W.config1(side)
        return c, side * side, None
    if args.workload == "config4":
        side = args.n_side or 512
        c = W.config4(side)
        return c, side * side, None
    side = args.n_side or 2048
    c = W.config3(side)
    return c, side * side, side


def roofline_from_counters(key, kernel, points_per_launch, units_per_launch, launch_s, peak, sm_max, clocks, probe, algorithmic_bytes):
    """`roofline` for an ALU-bound kernel from the committed ncu counters of `key` (= "<workload>/<triplets|full>").
    frac is null, with the reason in `counters.note`, when there is no capture for this key or the capture ran other sources."""
    from paper_1208_0302_b200 import counters as C
    table, path = C.load()
    ent, now = table.get(key), C.csrc_sha()
    info = {"file": path, "key": key, "csrc_sha_now": now, "csrc_sha_capture": ent["csrc_sha"] if ent else None,
            "stale": bool(ent) and ent["csrc_sha"] != now, "command": ent.get("command") if ent else None}
    r = {"bound": "alu", "achieved": None, "peak": peak, "unit": "TFLOP/s", "frac": None, "traffic": None,
         "algorithmic_bytes": algorithmic_bytes, "kernel": kernel, "counters": info,
         "peak_measured_ffma_tflops": probe["ffma"]["tflops"], "mufu_per_s_measured": probe["mufu"]["thread_inst_per_s"],
         "peak_basis": "148 SM x 128 FP32 lanes x 2 flop x %.0f MHz (max SM clock)" % sm_max}
    if not ent:
        info["note"] = "no ncu capture of this workload in %s: executed flop per wavelength point unknown, frac not reported" % path
        return r
    flop_pt, mufu_pt = ent["flop_per_lambda_point"], ent["mufu_per_lambda_point"]
    achieved = flop_pt * points_per_launch / launch_s / 1e12
    r.update({"flop_per_lambda_point": flop_pt, "fma_pipe_busy_ncu": ent["fma_pipe_busy_elapsed"],
              "sfu": {"mufu_per_lambda_point": mufu_pt, "achieved_per_s": mufu_pt * points_per_launch / launch_s,
                      "peak_per_s_measured": probe["mufu"]["thread_inst_per_s"],
                      "frac": mufu_pt * points_per_launch / launch_s / probe["mufu"]["thread_inst_per_s"]}})
    if info["stale"]:
        info["note"] = "the capture ran other csrc/ sources than this run: its count is not this kernel's; frac not reported"
        r["frac_with_stale_count"] = achieved / peak
        return r
    r["achieved"], r["frac"] = achieved, achieved / peak
    r["frac_at_sampled_clock"] = (achieved / (peak * clocks["sm_mhz"] / sm_max)) if clocks.get("sm_mhz") else None
    if ent.get("dram_bytes_per_pixel") is not None:          # measured bytes per unit of the capture x units of this launch
        r["traffic"] = ent["dram_bytes_per_pixel"] * units_per_launch
    return r


def syntheses_per_pixel(ga):
    return ga["pop"] + ga["generations"] * (ga["pop"] - 1)


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons while the timed region runs."""

    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc is not None:
            time.sleep(0.25)
            self.proc.terminate()
            self.thr.join(timeout=2)

    def summary(self):
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "power_w_max": float(max(pw)), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------ oracle legs
def oracle_lines_for(cfg):
    from oracle import api as orc
    lines = []
    for l in cfg["lines"]:
        if cfg["triplets"]:
            sh, we, ki = [0.0, -l["g_eff"], l["g_eff"]], [1, 1, 1], [0, -1, 1]
        else:
            sh, we, ki = orc.zeeman_pattern(l["lower"], l["upper"])
        lines.append(dict(lambda0=l["lambda0"], strength=l["strength"], shift=sh, weight=we, kind=ki))
    return orc.Lines(lines, W.LAMBDA_REF)


_FULLDISC = {}


def oracle_sample(cfg, n, stream=0):
    """n pixels of the workload, observations synthesised by the oracle itself (+ seeded noise, rounded to f32).
    config3: pixels OF the full-disc map (80 % quiet / 20 % active region, mu per pixel) under their global ids.
    Returns (lines, obs, nm_profile, mu or None, ids or None)."""
    from oracle import api as orc
    ln = oracle_lines_for(cfg)
    npar = cfg.get("npar", 9)
    mu = ids = None
    if "n_side" in cfg:
        key = (cfg["n_side"], cfg["radius"])
        if key not in _FULLDISC:
            _FULLDISC[key] = W.fulldisc_truth(cfg["n_side"], cfg["radius"])
        mask, mu_all, truth_all, active = _FULLDISC[key]
        on = mask.astype(bool)
        q, ac = np.flatnonzero(on & ~active), np.flatnonzero(on & active)
        nq = n - n // 5
        pick = lambda a, m: a[(stream * 7919 + np.arange(m) * max(1, a.size // max(m, 1))) % a.size]
        ids = np.concatenate([pick(q, nq), pick(ac, n - nq)])
        truth, mu = truth_all[ids], mu_all[ids]
    else:
        truth = W.draw_truth(n, seed=W.SEED_TRUTH, b_lo=cfg["b_range"][0], b_hi=cfg["b_range"][1], stream=100 + stream, npar=npar)
    nm = orc.synth(W.NM_PARAMS[None, :], cfg["lam"], ln)[0, 0] if npar == 11 else None
    clean = orc.synth(truth, cfg["lam"], ln, mu=mu, threads=orc.hardware_threads(), nm_profile=nm)
    obs = (clean + W.draw_noise(clean.shape, cfg["sigma"], stream=100 + stream)).astype(np.float32).astype(np.float64)
    return ln, obs, nm, mu, ids


def bounded_oracle_cfg(cfg, core_seconds_per_pixel=12.0):
    """The oracle needs ~2 us per wavelength point per core (x2 for the 11-parameter model).  Where one pixel of the
    workload would take much longer than the budget (config4: ~150 core-s), the sample runs the SAME pixel problem for
    fewer generations and the result is reported in pixel-equivalents: pixels x (syntheses done / syntheses of a full
    inversion).  Returns (cfg for the oracle, that fraction, a note for the sample text)."""
    ga = cfg["ga"]
    per_synth = 2.0e-6 * cfg["lam"].size * (2 if cfg.get("npar", 9) == 11 else 1) * len(cfg["lines"]) / 2.0
    full = syntheses_per_pixel(ga)
    if full * per_synth <= 2.5 * core_seconds_per_pixel:
        return cfg, 1.0, ""
    g = max(1, int((core_seconds_per_pixel / per_synth - ga["pop"]) / (ga["pop"] - 1)))
    ga2 = dict(ga, generations=g, mut_scale=ga["mut_scale"][:g + 1])
    frac = (ga["pop"] + g * (ga["pop"] - 1)) / full
    return dict(cfg, ga=ga2), frac, " cut to %d of %d generations (value in pixel-equivalents by syntheses)" % (g, ga["generations"])


def time_oracle(cfg, n, stream=0):
    from oracle import api as orc
    ln, obs, nm, mu, ids = oracle_sample(cfg, n, stream)
    cores = orc.hardware_threads()
    t0 = time.perf_counter()
    if ids is None:
        orc.ga_invert(obs, cfg["lam"], ln, cfg["ga"], seed=W.SEED_GA, threads=cores, nm_profile=nm)
    else:                                     # scattered global ids: one oracle call per pixel, spread over the cores
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(cores) as ex:         # ctypes releases the GIL
            list(ex.map(lambda k: orc.ga_invert(obs[k:k + 1], cfg["lam"], ln, cfg["ga"], seed=W.SEED_GA, mu=mu[k:k + 1],
                                                pixel_base=int(ids[k]), threads=1), range(n)))
    return time.perf_counter() - t0, cores


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the same workload per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import api as orc
    cfg, n_pixels, _ = workload(args)
    cores = orc.hardware_threads()
    if args.workload == "config2":            # the step is forward synthesis: the oracle's synth on a bounded batch per step
        n, ln = 2000 * cores, oracle_lines_for(cfg)
        t = 0.0
        for k in range(args.warmup + args.steps):
            truth = W.draw_truth(n, seed=W.SEED_TRUTH, stream=7 + k)
            t0 = time.perf_counter(); orc.synth(truth, cfg["lam"], ln, threads=cores); dt = time.perf_counter() - t0
            t += dt if k >= args.warmup else 0.0
        val = n * args.steps / t
        sample = "%d vectors of %s per step, all %d host threads" % (n, cfg["name"], cores)
        print(json.dumps({"impl": "reference", "metric": "ME syntheses/s", "value": val, "unit": "syntheses/s", "n_gpus": args.gpus,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                          "config": {"workload": cfg["name"], "vectors_per_step": n, "L": int(cfg["lam"].size), "lines": 2},
                          "cpu_baseline": {"value": val, "unit": "syntheses/s", "cores": cores, "kind": "oracle", "sample": sample},
                          "e2e": {"value": val, "unit": "syntheses/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                          "gpu_launches": 0}), flush=True)
        return
    ocfg, frac, note = bounded_oracle_cfg(cfg, core_seconds_per_pixel=6.0)
    per_pixel_points = syntheses_per_pixel(ocfg["ga"]) * cfg["lam"].size * sum(3 for _ in cfg["lines"])
    n = max(cores, int(cores * max(1.0, 2.0e7 / per_pixel_points)))      # ~ a few seconds of work per core per step
    n = min(n, n_pixels)
    for w in range(args.warmup):
        time_oracle(ocfg, n, stream=w)
    t = 0.0
    for k in range(args.steps):
        dt, _ = time_oracle(ocfg, n, stream=args.warmup + k)
        t += dt
    val = n * frac * args.steps / t
    sample = "%d pixels of %s%s per step (%soracle-synthesised obs), all %d host threads" % (
        n, cfg["name"], note, "map pixels stratified 80/20 quiet/active with their mu and global ids, " if "n_side" in cfg else "", cores)
    line = {"impl": "reference", "metric": "pixel-inversions/s", "value": val, "unit": "pixels/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "pixels_per_step": n, "L": int(cfg["lam"].size), "pop": cfg["ga"]["pop"],
                       "generations": cfg["ga"]["generations"], "lines": len(cfg["lines"])},
            "syntheses_per_s": val * syntheses_per_pixel(cfg["ga"]),
            "cpu_baseline": {"value": val, "unit": "pixels/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "pixels/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------ GPU leg
def build_inputs(cfg, n_pixels, side, rank, torch, B):
    """Synthetic observation cube resident in HBM: truth -> me_synth (this library) -> + Gaussian noise (device RNG)."""
    dev = torch.device("cuda")
    npar = cfg.get("npar", 9)
    if side is None:
        truth = W.draw_truth(n_pixels, seed=W.SEED_TRUTH, b_lo=cfg["b_range"][0], b_hi=cfg["b_range"][1], stream=rank, npar=npar)
        mask_t = mu_t = None
        n_active = n_pixels
    else:
        mask, mu, truth, _ = W.fulldisc_truth(cfg["n_side"], cfg["radius"], seed=W.SEED_TRUTH + rank)
        mask_t = torch.from_numpy(mask).to(dev)
        mu_t = torch.from_numpy(mu.astype(np.float32)).to(dev)
        n_active = int(mask.sum())
    ld = B.line_data_from_workload(cfg["lines"], cfg["triplets"])
    if npar == 11:        # reading F13: I_fixed = the B = 0 profile of workloads.NM_PARAMS, synthesised by this library
        nm, _ = B.me_synth(torch.from_numpy(W.NM_PARAMS[None, :].astype(np.float32)).to(dev), cfg["lam"], ld)
        ld = B.line_data_from_workload(cfg["lines"], cfg["triplets"], n_params=11, nm_profile=nm[0, 0].contiguous())
    truth_t = torch.from_numpy(truth.astype(np.float32)).to(dev)
    obs, _ = B.me_synth(truth_t, cfg["lam"], ld, mu=mu_t)
    gen = torch.Generator(device=dev)
    gen.manual_seed(W.SEED_NOISE + 1000 * rank)
    chunk = 1 << 18
    for s in range(0, n_pixels, chunk):                       # in place, bounded temporaries
        o = obs[s:s + chunk]
        o.add_(torch.randn(o.shape, generator=gen, device=dev, dtype=torch.float32), alpha=float(cfg["sigma"]))
    torch.cuda.synchronize()
    return ld, obs, mask_t, mu_t, n_active, truth


def bench_me_synth(torch, B, peaks, P=1_000_000, chi2_only=True):
    """BASELINE config 2: forward synthesis of P prior draws on the two-line 128-point grid, IQUV output + chi2 against
    one fixed profile (and chi2 only, to separate ALU from the store stream).  Not the headline metric: reported beside it."""
    c2 = W.config2(P)
    lam, ld = c2["lam"], B.line_data_from_workload(c2["lines"], True)
    L = int(lam.size)
    params = torch.from_numpy(W.draw_truth(P, seed=W.SEED_TRUTH, stream=7).astype(np.float32)).cuda()
    obs_ref, _ = B.me_synth(params[:1].contiguous(), lam, ld)
    obs_ref = obs_ref[0].contiguous()
    wos = c2["ga"]["stokes_weight"] / c2["ga"]["sigma"]
    out = torch.empty((P, 4, L), dtype=torch.float32, device="cuda")
    chi = torch.empty((P,), dtype=torch.float32, device="cuda")
    res = {}
    legs = [("stokes_and_chi2", dict(out_stokes=out, out_chi2=chi))]
    if chi2_only:
        legs.append(("chi2_only", dict(out_chi2=chi, want_stokes=False)))
    for name, kw in legs:
        for _ in range(3):
            B.me_synth(params, lam, ld, obs_ref=obs_ref, w_over_sigma=wos, **kw)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 5
        e0.record()
        for _ in range(reps):
            B.me_synth(params, lam, ld, obs_ref=obs_ref, w_over_sigma=wos, **kw)
        e1.record()
        torch.cuda.synchronize()
        sec = e0.elapsed_time(e1) * 1e-3 / reps
        nbytes = P * (36 + 4 + (16 * L if name == "stokes_and_chi2" else 0))
        res[name] = {"syntheses_per_s": P / sec, "ms": sec * 1e3, "hbm_gbs": nbytes / sec / 1e9,
                     "hbm_frac_of_measured": nbytes / sec / 1e9 / float(peaks.get("hbm_gbs", 6650.0))}
    res["P"] = P
    res["L"] = L
    return res


def run_b200(args):
    import torch
    from paper_1208_0302_b200 import binding as B, build as mebuild
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if rank == 0:
        mebuild.build()
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()
    B.lib()
    cfg, n_pixels, side = workload(args)
    ld, obs, mask_t, mu_t, n_active, _ = build_inputs(cfg, n_pixels, side, rank, torch, B)
    ga, lam = cfg["ga"], cfg["lam"]
    base = rank * n_pixels                                    # shards keyed by global pixel id (no data-path collective)
    out_p = torch.empty((n_pixels, cfg.get("npar", 9)), dtype=torch.float32, device="cuda")
    out_c = torch.empty((n_pixels,), dtype=torch.float32, device="cuda")

    def step():
        B.ga_invert(obs, lam, ld, ga, W.SEED_GA, mask=mask_t, mu=mu_t, pixel_id_base=base, out_params=out_p, out_chi2=out_c)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    # Wall-clock budget (--budget-s): one step of config3 takes about a minute, and the driver asks for 5 + 20 of them.
    # The first warm-up step is timed on the host; if warm-up + K steps + the end-to-end leg would not fit, the end-to-end
    # leg is cut to one step without its own warm-up, then dropped; K is reduced only if the steps alone do not fit, and
    # the line then carries the K that was timed and says so.
    t_wall0 = time.perf_counter()
    notes = []
    steps = args.steps
    t_step = None
    for w in range(args.warmup):
        t0 = time.perf_counter()
        step()
        if w == 0:
            torch.cuda.synchronize()
            t_step = time.perf_counter() - t0
    barrier()
    if t_step is None:
        t0 = time.perf_counter(); step(); torch.cuda.synchronize(); t_step = time.perf_counter() - t0
        notes.append("warmup 0 requested: one untimed step was run to size the budget")
    left = args.budget_s - (time.perf_counter() - t_wall0)
    e2e_plan = 0 if args.no_e2e else (3 if t_step < 20.0 else 1)          # e2e steps incl. its warm-up (none when a step is long)
    if not args.no_e2e and (steps + e2e_plan) * t_step > left:
        e2e_plan = 1 if (steps + 1) * t_step <= left else 0
        notes.append("end-to-end leg %s to fit --budget-s %.0f" % ("cut to one step" if e2e_plan else "dropped", args.budget_s))
    if steps * t_step > left:
        steps = max(1, int(left / t_step))
        notes.append("TIMED %d OF THE %d STEPS ASKED FOR: %d x %.1f s does not fit --budget-s %.0f" % (steps, args.steps, args.steps, t_step, args.budget_s))
    if world > 1:                                                          # every rank must run the same plan
        plan = torch.tensor([steps, e2e_plan], device="cuda"); dist.all_reduce(plan, op=dist.ReduceOp.MIN)
        steps, e2e_plan = int(plan[0].item()), int(plan[1].item())
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        ev0.record()
        for _ in range(steps):
            step()
        ev1.record()
        barrier()
    ms = ev0.elapsed_time(ev1)
    if dist is not None:
        t = torch.tensor([ms], device="cuda"); dist.all_reduce(t, op=dist.ReduceOp.MAX); ms = float(t.item())
    med_chi2 = float(out_c[~torch.isnan(out_c)].median().item())

    # end to end through the C ABI from HOST buffers: pinned obs -> H2D -> ga_invert -> D2H of params + chi2
    e2e = None
    if e2e_plan > 0:
        h_obs = torch.empty(obs.shape, dtype=torch.float32, pin_memory=True); h_obs.copy_(obs)
        h_p = torch.empty(out_p.shape, dtype=torch.float32, pin_memory=True)
        h_c = torch.empty(out_c.shape, dtype=torch.float32, pin_memory=True)
        d_obs = torch.empty_like(obs)
        h2d = h_obs.numel() * 4
        d2h = (h_p.numel() + h_c.numel()) * 4

        def e2e_step():
            d_obs.copy_(h_obs, non_blocking=True)
            B.ga_invert(d_obs, lam, ld, ga, W.SEED_GA, mask=mask_t, mu=mu_t, pixel_id_base=base, out_params=out_p, out_chi2=out_c)
            h_p.copy_(out_p, non_blocking=True); h_c.copy_(out_c, non_blocking=True)

        if e2e_plan > 1:
            e2e_step()                                   # its own warm-up (the kernel itself is warm either way)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_e2e = max(1, min(steps, e2e_plan - 1)) if e2e_plan > 1 else 1
        e0.record()
        for _ in range(n_e2e):
            e2e_step()
        e1.record(); barrier()
        ems = e0.elapsed_time(e1)
        if dist is not None:
            t = torch.tensor([ems], device="cuda"); dist.all_reduce(t, op=dist.ReduceOp.MAX); ems = float(t.item())
        e2e = {"value": world * n_active * n_e2e / (ems * 1e-3), "unit": "pixels/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": n_e2e}
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    sec = ms * 1e-3
    value = world * n_active * steps / sec
    syn = syntheses_per_pixel(ga)
    L = int(lam.size)
    points_per_launch = n_active * syn * L
    launch_s = sec / steps
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    peak = SM_COUNT * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    clocks = clk.summary()
    # the FP32 FMA rate this box actually sustains (scalar FFMA probe of the library, 8 resident CTAs/SM), for context
    from paper_1208_0302_b200 import peaks as mepeaks, counters as mecounters
    probe = mepeaks.measure(iters=2048, kinds=(0, 3))["probes"]
    key = "%s/%s" % (cfg["name"], "triplets" if cfg["triplets"] else "full")
    roof = roofline_from_counters(key, "ga_invert_kernel", points_per_launch, n_active, launch_s, peak, sm_max, clocks, probe,
                                  (16 * L + 40) * n_active)
    line = {"metric": "pixel-inversions/s", "value": value, "unit": "pixels/s", "n_gpus": world, "steps": steps,
            "warmup": args.warmup, "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg["name"], "pixels_per_gpu": n_pixels, "active_pixels_per_gpu": n_active, "L": L,
                       "pop": ga["pop"], "generations": ga["generations"], "lines": len(cfg["lines"]),
                       "zeeman": "effective triplets" if cfg["triplets"] else "full LS patterns", "parallelism": "pixel shards x%d" % world,
                       "l2": "obs cube %.0f MB per step (> 126 MB L2 for config1/3); path is ALU-bound" % (obs.numel() * 4 / 1e6)},
            "syntheses_per_s": value * syn, "median_chi2": med_chi2, "roofline": roof,
            "clocks": clocks, "gpu_launches": steps, "e2e": e2e, "csrc_sha": mecounters.csrc_sha()}
    if steps != args.steps:
        line["steps_requested"] = args.steps
    if notes:
        line["notes"] = notes
    if args.aux:
        line["me_synth_config2"] = bench_me_synth(torch, B, peaks)
        # BASELINE config 2's saturation trace: P = 1e4 .. 1e7 with the full [P,4,L] output (20.5 GB at 1e7)
        line["me_synth_config2"]["saturation"] = {
            str(P): round(bench_me_synth(torch, B, peaks, P=P, chi2_only=False)["stokes_and_chi2"]["syntheses_per_s"])
            for P in (10_000, 100_000, 10_000_000)}
        torch.cuda.empty_cache()
    if not args.no_cpu_baseline:
        from oracle import api as orc
        cores = orc.hardware_threads()
        ocfg, frac, note = bounded_oracle_cfg(cfg)
        n = min(n_pixels, (4 if frac == 1.0 else 1) * cores)        # ~10-30 s on the box's cores; BASELINE.md says why not more
        dt, cores = time_oracle(ocfg, n)
        line["cpu_baseline"] = {"value": n * frac / dt, "unit": "pixels/s", "cores": cores, "kind": "oracle",
                                "sample": "%d pixels of %s%s, oracle-synthesised obs, %.1f s" % (n, cfg["name"], note, dt)}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_config2(args):
    """BASELINE config 2 as the step: me_synth over `--vectors` iid prior draws on the two-line 128-point grid, [P,4,L] output
    + chi2 against one fixed profile (or --chi2-only).  Single GPU; the ordering workspace is allocated ONCE by the caller
    (me_synth_ws), so the timed region holds the library's launches only."""
    import torch
    from paper_1208_0302_b200 import binding as B, build as mebuild, peaks as mepeaks, counters as mecounters
    if int(os.environ.get("RANK", "0")) != 0:
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    mebuild.build(); B.lib()
    P = args.vectors
    c2 = W.config2(P)
    lam, ld, L = c2["lam"], B.line_data_from_workload(c2["lines"], True), int(c2["lam"].size)
    params = torch.from_numpy(W.draw_truth(P, seed=W.SEED_TRUTH, stream=7).astype(np.float32)).cuda()
    obs_ref = B.me_synth(params[:1].contiguous(), lam, ld)[0][0].contiguous()
    wos = c2["ga"]["stokes_weight"] / c2["ga"]["sigma"]
    out = None if args.chi2_only else torch.empty((P, 4, L), dtype=torch.float32, device="cuda")
    chi = torch.empty((P,), dtype=torch.float32, device="cuda")
    need = B.me_synth_workspace_bytes(P)
    ws = torch.empty((need,), dtype=torch.uint8, device="cuda") if need else False

    def step():
        B.me_synth(params, lam, ld, out_stokes=out, obs_ref=obs_ref, w_over_sigma=wos, out_chi2=chi, want_stokes=not args.chi2_only, workspace=ws)

    for _ in range(max(args.warmup, 1)):
        step()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(0) as clk:
        ev0.record()
        for _ in range(args.steps):
            step()
        ev1.record()
        torch.cuda.synchronize()
    sec = ev0.elapsed_time(ev1) * 1e-3
    launch_s = sec / args.steps
    e2e = None
    if not args.no_e2e:                      # host params -> H2D -> me_synth -> D2H of chi2 (and of the cube when it is produced)
        h_p = torch.empty(params.shape, dtype=torch.float32, pin_memory=True); h_p.copy_(params)
        h_c = torch.empty(chi.shape, dtype=torch.float32, pin_memory=True)
        h_o = None if out is None else torch.empty(out.shape, dtype=torch.float32, pin_memory=True)
        d_p = torch.empty_like(params)

        def e2e_step():
            d_p.copy_(h_p, non_blocking=True)
            B.me_synth(d_p, lam, ld, out_stokes=out, obs_ref=obs_ref, w_over_sigma=wos, out_chi2=chi, want_stokes=not args.chi2_only, workspace=ws)
            h_c.copy_(chi, non_blocking=True)
            if h_o is not None:
                h_o.copy_(out, non_blocking=True)
        e2e_step(); torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            e2e_step()
        e1.record(); torch.cuda.synchronize()
        e2e = {"value": P * args.steps / (e0.elapsed_time(e1) * 1e-3), "unit": "syntheses/s", "h2d_bytes_per_step": h_p.numel() * 4,
               "d2h_bytes_per_step": (h_c.numel() + (h_o.numel() if h_o is not None else 0)) * 4, "steps": args.steps}
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    peak = SM_COUNT * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    clocks = clk.summary()
    probe = mepeaks.measure(iters=2048, kinds=(0, 3))["probes"]
    nbytes = P * (36 + 4 + (0 if args.chi2_only else 16 * L))
    key = "config2_synth_sweep/%s" % ("chi2_only" if args.chi2_only else "stokes")
    roof = roofline_from_counters(key, "me_synth_kernel", P * L, P, launch_s, peak, sm_max, clocks, probe, nbytes)
    roof["hbm"] = {"achieved_gbs": nbytes / launch_s / 1e9, "peak_gbs_measured": float(peaks.get("hbm_gbs", 0.0)) or None,
                   "frac": (nbytes / launch_s / 1e9 / float(peaks["hbm_gbs"])) if peaks.get("hbm_gbs") else None}
    n_launch = (3 if need else 1)    # kernels per me_synth_ws call: histogram + scan, scatter, synthesis (plus one cudaMemsetAsync of 128 KB)
    line = {"metric": "ME syntheses/s", "value": P / launch_s, "unit": "syntheses/s", "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 1), "ms_per_step": launch_s * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": c2["name"], "vectors": P, "L": L, "lines": 2, "zeeman": "effective triplets",
                       "output": "chi2 only" if args.chi2_only else "[P,4,L] Stokes + chi2",
                       "l2": "output %.0f MB per step (> 126 MB L2)" % (nbytes / 1e6) if not args.chi2_only else "inputs 40 MB per step; path is ALU-bound",
                       "ordered_visit": bool(need)},
            "roofline": roof, "clocks": clocks, "gpu_launches": args.steps * n_launch, "e2e": e2e, "csrc_sha": mecounters.csrc_sha()}
    if not args.no_cpu_baseline:
        from oracle import api as orc
        cores = orc.hardware_threads()
        n = 2000 * cores
        truth = W.draw_truth(n, seed=W.SEED_TRUTH, stream=7)
        ln = oracle_lines_for(c2)
        t0 = time.perf_counter(); orc.synth(truth, lam, ln, threads=cores); dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": n / dt, "unit": "syntheses/s", "cores": cores, "kind": "oracle",
                                "sample": "%d vectors of %s, %.1f s" % (n, c2["name"], dt)}
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    elif a.workload == "config2":
        run_config2(a)
    else:
        run_b200(a)
