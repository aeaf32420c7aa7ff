"""bench.py -- log-posterior + gradient particle-evaluations per second (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--impl ours|reference]

A "step" is one pass of the whole hot path (unpack/prior, ray-trace, paint, PSF+bin, chi^2,
adjoint) over one batch of synthetic particles: one gl_logpost_grad call on the full batch of the chosen config.
BASELINE.json's `metric` names no config, so the default is the LARGEST single-GPU configuration, config 5
(configs[4]: 200x200 pixels, supersample 4 = 640,000 rays, 41x41 PSF, EPL + shear + multipoles, Sersic + shapelets
n_max 10, two lens Sersics, 100 parameters, 2048 particles); the default run also times configs 2-4 in fp64 and
config 5 in fp32 for a few steps each and reports them in `all_configs` / `f32` (compact records, same process).
`value` times that call with the particles already resident in HBM; `e2e` times gl_logpost_grad_host, i.e. the
same work plus the host->device copy of the particles from pinned memory and the device->host copy of logp and
the gradient, every step.  N > 1 runs N replicas (the path does not shard further: SURVEY 8(e)), one process per
GPU, no data-path collective; `value` = N * P / max-over-ranks time.

--impl reference times the fp64 CPU oracle (oracle/) as it stands on the host cores, on a bounded sample.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "log-posterior+grad particle-evals/sec"
UNIT = "particle-evals/s"
WORKLOAD_NAMES = {1: "cfg1 tiny SIE 40x40 s2 K11 P64", 2: "cfg2 DESI-Legacy-like EPL+shear 60x60 s4 K21 Moffat P4096",
                  3: "cfg3 HST-like EPL+shear+shapelets(6) 100x100 s2 K31 P8192",
                  4: "cfg4 100-system ensemble 60x60 s4 K21 P102400", 5: "cfg5 EPL+multipoles+shapelets(10) 200x200 s4 K41 P2048",
                  6: "cfg6 (not in BASELINE.json) real-system component list: EPL+shear, 3 lens Sersic, 2 source Sersic, 60x60 s4 K21 P4096"}

# ALU peaks of one B200 from unit counts and clocks: 148 SMs x 128 FP32 lanes (64 FP64 lanes)
# x sm_max_mhz; an FMA counts as ONE lane-operation.
N_SM, FP32_LANES, FP64_LANES = 148, 128, 64


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            mp = json.load(f)
        return float(mp.get("sm_max_mhz", 1965.0)), "MEASURED_PEAKS.json sm_max_mhz"
    except Exception:
        return 1965.0, "fallback clocks.max.sm 1965 MHz (B200_PROFILING.md)"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--no-all-configs", action="store_true",
                    help="skip the short runs of the other configs and of the fp32 mode (all_configs / f32 records)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"],
                    help="arithmetic of the CUDA path: f64 = GL_PRECISION_F64 (default; strict parity), f32 = GL_PRECISION_F32")
    ap.add_argument("--stage", default="grad", choices=["grad", "map", "svi", "svi_score", "hmc"],
                    help="grad: one gl_logpost_grad call per step (the headline); map / svi / hmc: one fused gl_map_step (Adam), "
                         "gl_svi_step (AdaBelief) or gl_hmc_step (4 leapfrog steps) per step; svi_score: gl_svi_step_score, the "
                         "score-function iteration of the paper's Eq. 3 (forward pass only; the metric then counts log-posterior "
                         "evaluations WITHOUT gradient)")
    ap.add_argument("--amplitudes", default="sampled", choices=["sampled", "solved"],
                    help="solved: backward modelling (amplitude_mode 1, DESIGN.md section 16); a diagnostic line, no cpu_baseline")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def ncu_traffic(k, precision, stage):
    """DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of ONE launch of the kernel of `stage`, from the committed
    `ncu --set full` captures: profiles/ncu_traffic.json, written by `python -m paper_2606_30633_b200.ncu_traffic` from the
    raw-page CSV exports (bench.py cannot run a profiler).  None where no capture exists."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            tab = json.load(f)
        return tab["cfg%d_%s" % (k, precision)][stage]["dram_bytes_per_launch"]
    except Exception:
        return None


# ----------------------------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index, period=0.01):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.sm, self.mask, self.max_mhz, self.stop_flag, self.ok = [], 0, None, False, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        while not self.stop_flag:
            try:
                self.sm.append(int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
            except Exception:
                try:
                    self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                except Exception:
                    pass
            time.sleep(self.period)

    def summary(self):
        if not self.ok or not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml_unavailable"]}
        reasons = [n for b, n in self.REASONS.items() if (self.mask & b) and n != "gpu_idle"]
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples": len(self.sm)}


# ----------------------------------------------------------------------------------------------- oracle legs
def oracle_rate(k, seconds, log=None):
    """Time the fp64 oracle (as it stands, OpenMP over particles on every host core) on a bounded prefix of the
    config-k batch sized for about `seconds` of CPU wall time.  Returns (evals/s, threads, sample description)."""
    import oracle
    import workloads as W
    P_full = W.FULL_PARTICLES[k]
    probe_n = min(P_full, max(2 * oracle.n_threads(), 16))
    wl = W.make_workload(k, n_particles=probe_n) if k != 4 else W.make_workload(4, per_system=1)
    sp = wl.spec
    sid_sys = np.arange(sp.n_systems, dtype=np.int32) if sp.n_systems > 1 else None
    truth = oracle.model_image(sp, wl.psf.astype(np.float64), wl.truth_theta, system_id=sid_sys)
    obs, sig = W.finish_observation(wl, truth)
    z = wl.params[:probe_n].astype(np.float64)
    sid = wl.system_id[:probe_n] if wl.system_id is not None else None
    t0 = time.perf_counter()
    oracle.logpost_grad(sp, obs, sig, wl.psf, z, sid)
    dt = time.perf_counter() - t0
    n = int(max(probe_n, min(P_full, probe_n * seconds / max(dt, 1e-6))))
    n = max(oracle.n_threads(), (n // oracle.n_threads()) * oracle.n_threads())
    if n > probe_n:
        wl = W.make_workload(k, n_particles=n) if k != 4 else W.make_workload(4, per_system=max(1, (n + 99) // 100))
        z = wl.params[:n].astype(np.float64)
        sid = wl.system_id[:n] if wl.system_id is not None else None
        n = z.shape[0]
        t0 = time.perf_counter()
        oracle.logpost_grad(sp, obs, sig, wl.psf, z, sid)
        dt = time.perf_counter() - t0
    else:
        n = probe_n
    return n / dt, oracle.n_threads(), "first %d particles of %s, one oracle.logpost_grad call, %.1f s" % (
        n, WORKLOAD_NAMES[k], dt), (sp, obs, sig, wl)


def run_reference(a):
    """--impl reference: the oracle on the host cores; each step = one bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    import workloads as W
    k = a.config
    rate, cores, sample, (sp, obs, sig, wl) = oracle_rate(k, 2.0)
    n = int(max(cores, min(W.FULL_PARTICLES[k], rate * 1.5)))          # ~1.5 s per step
    n = max(cores, n // cores * cores)
    wl = W.make_workload(k, n_particles=n) if k != 4 else W.make_workload(4, per_system=max(1, n // 100))
    z = wl.params.astype(np.float64)[:n] if k != 4 else wl.params.astype(np.float64)
    sid = wl.system_id if wl.system_id is not None else None
    n = z.shape[0]
    for _ in range(a.warmup):
        oracle.logpost_grad(sp, obs, sig, wl.psf, z, sid)
    t0 = time.perf_counter()
    for _ in range(a.steps):
        oracle.logpost_grad(sp, obs, sig, wl.psf, z, sid)
    dt = (time.perf_counter() - t0) / a.steps
    v = n / dt
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_NAMES[k], "sample": "%d particles per step" % n},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "%d particles per step of %s" % (n, WORKLOAD_NAMES[k])},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ----------------------------------------------------------------------------------------------- multi-rank host logic
def max_over_ranks(values, device="cpu"):
    """Max over ranks of each entry of `values` (device seconds).  Replicas exchange nothing else;
    works on any initialised backend (nccl on the box, gloo in tests/test_bench_host.py)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_rate(world, particles_per_rank, steps, seconds):
    """Replicas: every rank evaluates its own full batch, so the job processed world * P * steps evaluations."""
    return world * particles_per_rank * steps / seconds




# ----------------------------------------------------------------------------------------------- GPU arm: helpers
def _peak(precision, mhz):
    lanes = FP64_LANES if precision == "f64" else FP32_LANES
    return N_SM * lanes * mhz * 1e6 / 1e12, lanes                     # T lane-op/s


def make_model(gl, W, torch, k, precision, dev, amplitudes="sampled"):
    """Workload k on the device: (wl, spec, LensModel).  The observation is the truth rendered by THIS side
    (gl_model_image) + the seeded noise (workloads docstring)."""
    wl = W.make_workload(k)
    sp = wl.spec
    sp.precision = 0 if precision == "f64" else 1
    N = sp.n_pix
    zeros = np.zeros((sp.n_systems, N, N), np.float32)
    m0 = gl.LensModel(sp, zeros, zeros + 1, wl.psf, device=dev)
    sid_sys = np.arange(sp.n_systems, dtype=np.int32) if sp.n_systems > 1 else None
    truth = m0.model_image(torch.from_numpy(wl.truth_z).to(dev), sid_sys).cpu().numpy()
    m0.close()
    obs, sig = W.finish_observation(wl, truth)
    if amplitudes == "solved":
        sp.amplitude_mode = 1
    return wl, sp, gl.LensModel(sp, obs, sig, wl.psf, device=dev)


def band_means(gl, torch, m, ws, P):
    """(mean M1, mean M2, particles read) of the series precision bands step A chose (csrc/gl_ray.cuh knuth_banded), over
    the valid particles of the LAST chunk of the most recent call, read from the workspace (gl_workspace_layout)."""
    if m.spec.mass_model != 1:
        return None
    lay = gl.gl_workspace_layout(m.h, P)
    n = min(lay["chunk"], P - lay["last_chunk_first"])
    dt = torch.float64 if lay["elem_bytes"] == 8 else torch.float32
    nb = n * lay["pb_stride"] * lay["elem_bytes"]
    pb = ws[lay["off_pb"]:lay["off_pb"] + nb].view(dt).view(n, lay["pb_stride"])
    ok = pb[:, lay["idx_valid"]] != 0
    if int(ok.sum()) == 0:
        return None
    return float(pb[ok, lay["idx_m1"]].double().mean()), float(pb[ok, lay["idx_m2"]].double().mean()), int(ok.sum())


def stage_profile(gl, step, flush, reps):
    """Per-stage device time of one step from the library's own CUDA events on the launching stream (mean over reps)."""
    gl.gl_stage_timing_enable(True)
    stage_ms, stage_n = {}, {}
    for _ in range(reps):
        flush.zero_()
        step()
        for name, (ms, cnt) in gl.gl_stage_times().items():
            stage_ms[name] = stage_ms.get(name, 0.0) + ms / reps
            stage_n[name] = cnt
    gl.gl_stage_timing_enable(False)
    return stage_ms, stage_n


def roofline_record(workmodel, sp, k, precision, P, evals_per_particle, stage_ms, stage_n, ms_per_step, bands, mhz_max,
                    peak_src, sm_mhz=None, evals_in_stage_times=None, forward_only=False):
    """The `roofline` object of the contract for the dominant kernel of a measured step.
    frac          executed-band work: only the series steps that run in the arithmetic type are credited (bands)
    frac_fixed30  the fixed 30-term formulation (every term credited to the arithmetic type's pipe): the round-1 figure
    fp32_cofrac   fp64 mode: the series steps run in fp32, as a fraction of the FP32 pipe's peak (same kernel, same time)
    step_frac     one forward + one reverse sweep credited over the whole step (executed-band), step_frac_fixed30 likewise"""
    peak, lanes = _peak(precision, mhz_max)
    pipe = "FP64" if precision == "f64" else "FP32"
    wm30 = workmodel.per_eval(sp, precision)
    wmb = workmodel.per_eval(sp, precision, bands[:2]) if bands else wm30
    if forward_only:                     # a step that runs steps A-E only (gl_logpost): credit one forward sweep
        wm30 = dict(wm30, total_fwd_grad=wm30["total_fwd"]); wmb = dict(wmb, total_fwd_grad=wmb["total_fwd"])
    dom = max(stage_ms, key=stage_ms.get)
    dom_t = stage_ms[dom] * 1e-3
    # the stage timer holds the LAST gl_logpost_grad of a step (an HMC transition makes several: one of them is timed)
    n_st = evals_per_particle if evals_in_stage_times is None else evals_in_stage_times
    rate = lambda ops: ops * P * n_st / dom_t / 1e12 if dom_t > 0 else 0.0
    achieved = rate(wmb.get(dom, 0))
    t_step = ms_per_step * 1e-3
    r = {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "T %s lane-op/s (FMA=1)" % pipe,
         "frac": achieved / peak, "frac_fixed30": rate(wm30.get(dom, 0)) / peak,
         "traffic": ncu_traffic(k, precision, dom),
         "peak_source": "148 SM x %d %s lanes x %g MHz (%s)" % (lanes, pipe, mhz_max, peak_src),
         "kernel_ms_per_launch": stage_ms[dom] / max(stage_n[dom], 1), "kernel_launches_per_step": stage_n[dom],
         "algorithmic_laneops_per_eval": wmb.get(dom, 0), "algorithmic_laneops_per_eval_fixed30": wm30.get(dom, 0),
         "series_bands": ({"mean_m1": round(bands[0], 3), "mean_m2": round(bands[1], 3), "particles": bands[2],
                           "meaning": "4*m1 recurrence steps in %s, 4*m2 in fp32, rest skipped (of 28)" % pipe.lower()}
                          if bands else None),
         "stage_ms": {s: round(v, 4) for s, v in stage_ms.items()},
         "stage_share": {s: round(v / max(sum(stage_ms.values()), 1e-12), 4) for s, v in stage_ms.items()},
         "step_frac": wmb["total_fwd_grad"] * P * evals_per_particle / t_step / 1e12 / peak,
         "step_frac_fixed30": wm30["total_fwd_grad"] * P * evals_per_particle / t_step / 1e12 / peak,
         "step_algorithmic_laneops_per_eval": wmb["total_fwd_grad"],
         "per_stage_frac": {s: round(wmb[s] * P * n_st / (stage_ms[s] * 1e-3) / 1e12 / peak, 4)
                            for s in ("ray_fwd", "conv_chi2", "conv_transpose", "ray_adjoint")
                            if s in wmb and stage_ms.get(s, 0) > 0}}
    if precision == "f64":
        p32, _ = _peak("f32", mhz_max)
        r["fp32_cofrac"] = rate(wmb.get(dom + "_fp32band", 0)) / p32
        r["step_frac_of_fp32_peak"] = r["step_frac"] * peak / p32     # the pipe BASELINE.json's metric names
    else:
        r["mufu_T_ops_per_s"] = wmb["total_fwd_grad_mufu"] * P * evals_per_particle / t_step / 1e12
    if sm_mhz:
        r["frac_at_measured_clock"] = achieved / _peak(precision, sm_mhz)[0]
    return r


def short_run(gl, W, torch, workmodel, k, precision, dev, flush, steps, warmup, mhz_max, peak_src):
    """A compact record of config k in `precision`: a few gl_logpost_grad steps on the full batch, CUDA events."""
    wl, sp, m = make_model(gl, W, torch, k, precision, dev)
    P, n_p = wl.params.shape[0], sp.n_params
    z = torch.from_numpy(wl.params).to(dev)
    sid = torch.from_numpy(wl.system_id).to(dev) if wl.system_id is not None else None
    lp = torch.empty(P, dtype=torch.float32, device=dev); g = torch.empty((P, n_p), dtype=torch.float32, device=dev)
    ws = m.workspace(P)
    step = lambda: gl.gl_logpost_grad(m.h, m.obs, m.noise_sigma, m.psf, z, sid, lp, g, ws)
    for _ in range(max(warmup, 3)):
        step()
    launches = int(gl.gl_last_launch_count())
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for e0, e1 in ev:
        flush.zero_()
        e0.record(); step(); e1.record()
    torch.cuda.synchronize()
    ms = sum(e0.elapsed_time(e1) for e0, e1 in ev) / steps
    bands = band_means(gl, torch, m, ws, P)
    stage_ms, stage_n = stage_profile(gl, step, flush, min(steps, 3))
    roof = roofline_record(workmodel, sp, k, precision, P, 1, stage_ms, stage_n, ms, bands, mhz_max, peak_src)
    rec = {"cfg": k, "workload": WORKLOAD_NAMES[k], "dtype": precision, "value": P / (ms * 1e-3), "unit": UNIT,
           "ms_per_step": ms, "steps": steps, "n_particles": P, "gpu_launches_per_step": launches,
           "finite_fraction": float(torch.isfinite(lp).float().mean()),
           "kernel": roof["kernel"], "frac": roof["frac"], "frac_fixed30": roof["frac_fixed30"],
           "step_frac": roof["step_frac"], "step_frac_fixed30": roof["step_frac_fixed30"],
           "per_stage_frac": roof["per_stage_frac"], "stage_ms": roof["stage_ms"], "traffic": roof["traffic"]}
    for key in ("fp32_cofrac", "step_frac_of_fp32_peak", "mufu_T_ops_per_s", "series_bands"):
        if key in roof:
            rec[key] = roof[key]
    m.close()
    del ws, z, lp, g, m
    torch.cuda.empty_cache()
    return rec


# ----------------------------------------------------------------------------------------------- GPU arm
def run_ours(a):
    import torch
    import torch.distributed as dist
    import workloads as W
    import paper_2606_30633_b200 as gl
    from paper_2606_30633_b200 import workmodel

    gl.lib()                                             # fail loudly if libgigalens.so is missing: no fallback
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (libgigalens has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    k = a.config
    if a.amplitudes == "solved":
        a.no_cpu_baseline = True
    wl, sp, m = make_model(gl, W, torch, k, a.precision, dev, a.amplitudes)
    P, n_p = wl.params.shape[0], sp.n_params
    z = torch.from_numpy(wl.params).to(dev)
    sid = torch.from_numpy(wl.system_id).to(dev) if wl.system_id is not None else None
    lp = torch.empty(P, dtype=torch.float32, device=dev)
    g = torch.empty((P, n_p), dtype=torch.float32, device=dev)
    ws = m.workspace(P, host=True)
    ws_bytes = gl.gl_workspace_bytes(m.h, P)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # 256 MiB > 126 MB L2

    # ---- the timed call of each stage (device-resident inputs) and its host-buffer form (pinned copies inside)
    evals_per_particle = 1
    extra_launches = 0                                       # kernels launched per step outside the last counted API call
    pin = lambda t: t.cpu().pin_memory()
    if a.stage == "grad":
        zh = torch.from_numpy(wl.params).pin_memory()
        lph = torch.empty(P, dtype=torch.float32).pin_memory()
        gh = torch.empty((P, n_p), dtype=torch.float32).pin_memory()
        h2d_bytes, d2h_bytes = zh.numel() * 4, (lph.numel() + gh.numel()) * 4

        def step():
            gl.gl_logpost_grad(m.h, m.obs, m.noise_sigma, m.psf, z, sid, lp, g, ws)

        def step_host():
            gl.gl_logpost_grad_host(m.h, m.obs, m.noise_sigma, m.psf, zh, sid, lph, gh, ws)
    elif a.stage == "map":                                   # NEXT-1: fused gradient + Adam update; logp read back
        zm, om, ov = z.clone(), torch.zeros_like(z), torch.zeros_like(z)
        adam = dict(kind=gl.GL_OPT_ADAM, lr=1e-3, b1=0.9, b2=0.999, eps=1e-8, eps_root=0.0)
        tstep = [0]
        lph = torch.empty(P, dtype=torch.float32).pin_memory()
        h2d_bytes, d2h_bytes = 0, lph.numel() * 4

        def step():
            tstep[0] += 1
            gl.gl_map_step(m.h, adam, m.obs, m.noise_sigma, m.psf, zm, sid, om, ov, tstep[0], lp, g, ws)

        def step_host():
            step(); lph.copy_(lp, non_blocking=True)
    elif a.stage in ("svi", "svi_score"):                    # NEXT-2: P draws of one surrogate; xi in, loss out
        if sp.n_systems != 1:
            raise SystemExit("--stage svi needs a single-system config")
        nt = n_p * (n_p + 1) // 2
        mu = torch.from_numpy(wl.truth_z[0].copy()).to(dev)
        lt = torch.zeros(nt, device=dev); lt[torch.arange(n_p, device=dev) * (torch.arange(n_p, device=dev) + 3) // 2] = 0.01
        sm, sv, stats = torch.zeros(n_p + nt, device=dev), torch.zeros(n_p + nt, device=dev), torch.zeros(2, device=dev)
        xi = torch.randn((P, n_p), device=dev, generator=torch.Generator(device=dev).manual_seed(1))
        xih, statsh = pin(xi), torch.empty(2).pin_memory()
        belief = dict(kind=gl.GL_OPT_ADABELIEF, lr=1e-4, b1=0.95, b2=0.99, eps=1e-16, eps_root=1e-16)
        ws = torch.empty(gl.gl_svi_workspace_bytes(m.h, P), dtype=torch.uint8, device=dev)
        tstep = [0]
        h2d_bytes, d2h_bytes = xih.numel() * 4, 8

        extra_launches = 1

        def svi_call(t):
            if a.stage == "svi":
                gl.gl_svi_step(m.h, belief, m.obs, m.noise_sigma, m.psf, mu, lt, xi, sid, sm, sv, t, stats, ws)
            else:                                            # Eq. 3 as printed + leave-one-out baseline: gl_logpost only
                gl.gl_svi_step_score(m.h, belief, m.obs, m.noise_sigma, m.psf, mu, lt, xi, sid, sm, sv, t, 1, stats, ws)

        def step():                                          # fresh draws on the device every iteration (reading S22)
            tstep[0] += 1
            gl.gl_draw_normal(2026, tstep[0], 0, xi)
            svi_call(tstep[0])

        def step_host():                                     # host-made draws through a pinned buffer
            tstep[0] += 1
            xi.copy_(xih, non_blocking=True)
            svi_call(tstep[0])
            statsh.copy_(stats, non_blocking=True)
    else:                                                    # NEXT-3: P chains, one transition of 4 leapfrog steps
        n_leap = 4
        evals_per_particle = n_leap
        zc = z.clone()
        gl.gl_logpost_grad(m.h, m.obs, m.noise_sigma, m.psf, zc, sid, lp, g, ws)
        lpc, gc = lp.clone(), g.clone()
        gen = torch.Generator(device=dev).manual_seed(2)
        xi = torch.randn((P, n_p), device=dev, generator=gen)
        lu = torch.log(torch.rand(P, device=dev, generator=gen))
        acc, dh = torch.zeros(P, dtype=torch.int32, device=dev), torch.zeros(P, device=dev)
        xih, luh, acch = pin(xi), pin(lu), torch.empty(P, dtype=torch.int32).pin_memory()
        ws = torch.empty(gl.gl_hmc_workspace_bytes(m.h, P), dtype=torch.uint8, device=dev)
        h2d_bytes, d2h_bytes = (xih.numel() + luh.numel()) * 4, acch.numel() * 4

        tstep = [0]
        extra_launches = 2

        def hmc():
            gl.gl_hmc_step(m.h, m.obs, m.noise_sigma, m.psf, zc, lpc, gc, None, xi, lu, sid, 2e-5, n_leap, acc, dh, ws)

        def step():                                          # momenta and acceptance uniforms drawn on the device (S22)
            tstep[0] += 1
            gl.gl_draw_normal(2026, tstep[0], 1, xi); gl.gl_draw_log_uniform(2026, tstep[0], 2, lu)
            hmc()

        def step_host():                                     # host-made draws through pinned buffers
            xi.copy_(xih, non_blocking=True); lu.copy_(luh, non_blocking=True); hmc(); acch.copy_(acc, non_blocking=True)

    for _ in range(max(a.warmup, 3)):
        step()
    launches_per_step = int(gl.gl_last_launch_count()) + extra_launches
    sampler = ClockSampler(local)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(a.steps)]
    barrier()
    sampler.start()
    for e0, e1 in ev:
        flush.zero_()                                    # evict L2 between timed iterations (outside the event pair)
        e0.record(); step(); e1.record()
    barrier()
    t_steps = [e0.elapsed_time(e1) for e0, e1 in ev]        # per-step device times (ms): median and min go into the line
    t_dev = sum(t_steps) * 1e-3
    # e2e: host buffers (pinned), copies inside the timed region
    for _ in range(3):
        step_host()
    barrier()
    ev2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(a.steps)]
    for e0, e1 in ev2:
        flush.zero_()
        e0.record(); step_host(); e1.record()
    barrier()
    sampler.stop_flag = True
    sampler.join(timeout=2)
    t_e2e = sum(e0.elapsed_time(e1) for e0, e1 in ev2) * 1e-3
    if a.stage == "grad":
        assert torch.equal(lph, lp.cpu()) and torch.equal(gh, g.cpu()), "host-buffer path disagrees with the device path"
    fwd_only = None
    if a.stage == "grad" and a.amplitudes == "sampled":
        # SURVEY 8(d) timing protocol: gl_logpost (steps A-E, no adjoint) timed separately, same batch, same L2 flush
        nf = max(3, min(a.steps, 5))
        for _ in range(3):
            gl.gl_logpost(m.h, m.obs, m.noise_sigma, m.psf, z, sid, lp, ws)
        ev3 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nf)]
        for e0, e1 in ev3:
            flush.zero_()
            e0.record(); gl.gl_logpost(m.h, m.obs, m.noise_sigma, m.psf, z, sid, lp, ws); e1.record()
        torch.cuda.synchronize()
        tf = sorted(e0.elapsed_time(e1) for e0, e1 in ev3)
        fwd_only = {"call": "gl_logpost", "value": P / (float(np.median(tf)) * 1e-3), "unit": UNIT, "steps": nf,
                    "ms_per_step_median": float(np.median(tf)), "ms_per_step_min": tf[0]}
        gl.gl_logpost_grad(m.h, m.obs, m.noise_sigma, m.psf, z, sid, lp, g, ws)      # lp, g of the gradient call again
    if a.stage == "hmc":
        lp = lpc
    finite = float(torch.isfinite(lp).float().mean())

    # dominant-kernel roofline: per-stage device time from the library's own CUDA events on the launching stream
    bands = band_means(gl, torch, m, ws, P) if a.stage in ("grad", "map") else None
    stage_ms, stage_n = stage_profile(gl, step, flush, max(3, min(a.steps, 10)))

    t_dev, t_e2e = max_over_ranks([t_dev, t_e2e], dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    mhz_max, peak_src = _peaks()
    clocks = sampler.summary()
    roof = roofline_record(workmodel, sp, k, a.precision, P, evals_per_particle, stage_ms, stage_n, t_dev / a.steps * 1e3, bands,
                           mhz_max, peak_src, clocks.get("sm_mhz"), evals_in_stage_times=1 if a.stage == "hmc" else None,
                           forward_only=a.stage == "svi_score")
    probe = {}
    for kind, name in ((0, "fp32_fma"), (1, "fp64_fma"), (2, "mufu_ex2"), (4, "fp64_fma_distinct_operands"),
                       (5, "fp64_mma_m8n8k4"), (6, "fp64_mma_plus_fma"),
                       (7, "fp64_fma_two_vector_one_uniform_operand"), (8, "fp64_fma_three_vector_operands_one_shared")):
        try:
            probe[name] = round(gl.gl_probe_pipe(kind, 256)[0], 3)
        except Exception:                                             # measurement utility only
            probe[name] = None
    roof["probe_T_laneops_per_s"] = probe
    wm = workmodel.per_eval(sp, a.precision)
    out = {"metric": METRIC, "value": whole_job_rate(world, P * evals_per_particle, a.steps, t_dev), "unit": UNIT, "n_gpus": world, "steps": a.steps,
           "warmup": max(a.warmup, 3), "ms_per_step": t_dev / a.steps * 1e3, "ms_per_step_median": float(np.median(t_steps)),
           "ms_per_step_min": float(min(t_steps)), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": a.precision, "data": "synthetic",
           "config": {"workload": WORKLOAD_NAMES[k], "n_particles_per_gpu": P, "n_params": n_p,
                      "rays_per_particle": wm["rays"], "parallelism": "replicas x%d" % world, "stage": a.stage,
                      "l2": "256 MiB flush write between timed iterations; workspace %.0f MB" % (ws_bytes / 1e6),
                      "finite_fraction": finite, "amplitudes": a.amplitudes},
           "e2e": {"value": whole_job_rate(world, P * evals_per_particle, a.steps, t_e2e), "unit": UNIT, "h2d_bytes_per_step": int(h2d_bytes),
                   "d2h_bytes_per_step": int(d2h_bytes), "ms_per_step": t_e2e / a.steps * 1e3},
           "gpu_launches": launches_per_step * a.steps, "clocks": clocks, "roofline": roof}
    if fwd_only is not None:
        out["forward_only"] = fwd_only
    if a.stage == "grad" and a.amplitudes == "sampled" and world == 1 and not a.no_all_configs:
        # free this config's buffers, then a few steps of every other BASELINE.json config (fp64) and of this one in fp32
        m.close()
        m._ws = None
        del ws
        torch.cuda.empty_cache()
        short = max(3, min(a.steps, 5))
        recs = [{"cfg": k, "workload": WORKLOAD_NAMES[k], "dtype": a.precision, "value": out["value"], "unit": UNIT,
                 "ms_per_step": out["ms_per_step"], "steps": a.steps, "n_particles": P, "kernel": roof["kernel"],
                 "frac": roof["frac"], "frac_fixed30": roof["frac_fixed30"], "step_frac": roof["step_frac"],
                 "step_frac_fixed30": roof["step_frac_fixed30"], "per_stage_frac": roof["per_stage_frac"],
                 "stage_ms": roof["stage_ms"], "traffic": roof["traffic"]}]
        for kk in (2, 3, 4, 5):
            if kk != k:
                recs.append(short_run(gl, W, torch, workmodel, kk, a.precision, dev, flush, short, 3, mhz_max, peak_src))
        out["all_configs"] = sorted(recs, key=lambda r: r["cfg"])
        other = "f32" if a.precision == "f64" else "f64"
        out[other] = short_run(gl, W, torch, workmodel, k, other, dev, flush, short, 3, mhz_max, peak_src)
    if not a.no_cpu_baseline:
        rate, cores, sample, _ = oracle_rate(k, a.cpu_seconds)
        out["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    print(json.dumps(out))
    m.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)
