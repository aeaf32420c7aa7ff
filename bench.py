"""bench.py -- log-posterior + gradient particle-evaluations per second (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--impl ours|reference]

A "step" is one pass of the whole hot path (unpack/prior, ray-trace, paint, PSF+bin, chi^2,
adjoint) over one batch of synthetic particles: one gl_logpost_grad call on the full batch of the chosen config
(default config 2 = BASELINE.json configs[1], the DESI-Legacy-like multi-start MAP batch of 4096 particles).
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
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"],
                    help="arithmetic of the CUDA path: f64 = GL_PRECISION_F64 (default; strict parity), f32 = GL_PRECISION_F32")
    ap.add_argument("--stage", default="grad", choices=["grad", "map", "svi", "hmc"],
                    help="grad: one gl_logpost_grad call per step (the headline); map / svi / hmc: one fused gl_map_step (Adam), "
                         "gl_svi_step (AdaBelief) or gl_hmc_step (4 leapfrog steps) per step")
    ap.add_argument("--amplitudes", default="sampled", choices=["sampled", "solved"],
                    help="solved: backward modelling (amplitude_mode 1, DESIGN.md section 16); a diagnostic line, no cpu_baseline")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of ONE launch of the dominant kernel at the default
# workload, from the committed `ncu --set full` capture profiles/r1c_cfg2_f64.md (bench.py cannot run a profiler):
# keyed by (config, precision, stage).  None elsewhere.
NCU_TRAFFIC_BYTES = {(2, "f64", "ray_adjoint"): 2.153155e9 + 0.035220e9}


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
    wl = W.make_workload(k)
    sp = wl.spec
    sp.precision = 0 if a.precision == "f64" else 1
    P, n_p, N = wl.params.shape[0], sp.n_params, sp.n_pix
    # observation: truth rendered by THIS side (gl_model_image), noise from the seeded stream (workloads docstring)
    zeros = np.zeros((sp.n_systems, N, N), np.float32)
    m0 = gl.LensModel(sp, zeros, zeros + 1, wl.psf, device=dev)
    sid_sys = np.arange(sp.n_systems, dtype=np.int32) if sp.n_systems > 1 else None
    truth = m0.model_image(torch.from_numpy(wl.truth_z).to(dev), sid_sys).cpu().numpy()
    m0.close()
    obs, sig = W.finish_observation(wl, truth)
    if a.amplitudes == "solved":
        sp.amplitude_mode = 1
        a.no_cpu_baseline = True
    m = gl.LensModel(sp, obs, sig, wl.psf, device=dev)
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
    elif a.stage == "svi":                                   # NEXT-2: P draws of one surrogate; xi in, loss out
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

        def step():                                          # fresh draws on the device every iteration (reading S22)
            tstep[0] += 1
            gl.gl_draw_normal(2026, tstep[0], 0, xi)
            gl.gl_svi_step(m.h, belief, m.obs, m.noise_sigma, m.psf, mu, lt, xi, sid, sm, sv, tstep[0], stats, ws)

        def step_host():                                     # host-made draws through a pinned buffer
            tstep[0] += 1
            xi.copy_(xih, non_blocking=True)
            gl.gl_svi_step(m.h, belief, m.obs, m.noise_sigma, m.psf, mu, lt, xi, sid, sm, sv, tstep[0], stats, ws)
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
    t_dev = sum(e0.elapsed_time(e1) for e0, e1 in ev) * 1e-3
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
    if a.stage == "hmc":
        lp = lpc
    finite = float(torch.isfinite(lp).float().mean())

    # dominant-kernel roofline: per-stage device time from the library's own CUDA events on the launching stream
    gl.gl_stage_timing_enable(True)
    stage_ms, stage_n = {}, {}
    reps = max(3, min(a.steps, 10))
    for _ in range(reps):
        flush.zero_()
        step()
        for name, (ms, cnt) in gl.gl_stage_times().items():
            stage_ms[name] = stage_ms.get(name, 0.0) + ms / reps
            stage_n[name] = cnt
    gl.gl_stage_timing_enable(False)

    t_dev, t_e2e = max_over_ranks([t_dev, t_e2e], dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    mhz_max, peak_src = _peaks()
    lanes = FP64_LANES if a.precision == "f64" else FP32_LANES
    pipe = "FP64" if a.precision == "f64" else "FP32"
    peak = N_SM * lanes * mhz_max * 1e6 / 1e12                        # T lane-op/s
    wm = workmodel.per_eval(sp, a.precision)
    probe = {}
    for kind, name in ((0, "fp32_fma"), (1, "fp64_fma"), (2, "mufu_ex2"), (4, "fp64_fma_distinct_operands")):
        try:
            probe[name] = round(gl.gl_probe_pipe(kind, 256)[0], 3)
        except Exception as e:                                        # measurement utility only
            probe[name] = None
    dom = max(stage_ms, key=stage_ms.get)
    dom_ops = wm.get(dom, 0) * P
    dom_t = stage_ms[dom] * 1e-3
    achieved = dom_ops / dom_t / 1e12 if dom_t > 0 else 0.0
    clocks = sampler.summary()
    roof = {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "T %s lane-op/s (FMA=1)" % pipe,
            "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES.get((k, a.precision, dom)),
            "peak_source": "148 SM x %d %s lanes x %g MHz (%s)" % (lanes, pipe, mhz_max, peak_src),
            "probe_T_laneops_per_s": probe,
            "kernel_ms_per_launch": stage_ms[dom] / max(stage_n[dom], 1), "kernel_launches_per_step": stage_n[dom],
            "algorithmic_laneops_per_eval": wm.get(dom, 0),
            "stage_ms": {s: round(v, 4) for s, v in stage_ms.items()},
            "stage_share": {s: round(v / max(sum(stage_ms.values()), 1e-12), 4) for s, v in stage_ms.items()},
            "step_frac": wm["total_fwd_grad"] * P * evals_per_particle * a.steps / t_dev / 1e12 / peak,
            "step_algorithmic_laneops_per_eval": wm["total_fwd_grad"]}
    if clocks.get("sm_mhz"):
        roof["frac_at_measured_clock"] = achieved / (N_SM * lanes * clocks["sm_mhz"] * 1e6 / 1e12)
    out = {"metric": METRIC, "value": whole_job_rate(world, P * evals_per_particle, a.steps, t_dev), "unit": UNIT, "n_gpus": world, "steps": a.steps,
           "warmup": max(a.warmup, 3), "ms_per_step": t_dev / a.steps * 1e3, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": a.precision, "data": "synthetic",
           "config": {"workload": WORKLOAD_NAMES[k], "n_particles_per_gpu": P, "n_params": n_p,
                      "rays_per_particle": wm["rays"], "parallelism": "replicas x%d" % world, "stage": a.stage,
                      "l2": "256 MiB flush write between timed iterations; workspace %.0f MB" % (ws_bytes / 1e6),
                      "finite_fraction": finite, "amplitudes": a.amplitudes},
           "e2e": {"value": whole_job_rate(world, P * evals_per_particle, a.steps, t_e2e), "unit": UNIT, "h2d_bytes_per_step": int(h2d_bytes),
                   "d2h_bytes_per_step": int(d2h_bytes), "ms_per_step": t_e2e / a.steps * 1e3},
           "gpu_launches": launches_per_step * a.steps, "clocks": clocks, "roofline": roof}
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
