#!/usr/bin/env python
"""bench.py -- throughput of the RGF hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One "step" = one pass of the whole hot path (lead decimation A2, sweep A3-A5 over all L slices,
trace A6) over the headline batch: BASELINE.json configs[2], M=244, L=8000, 512 energies in
[-1, 1] eV, Anderson disorder +-0.1 eV (seed 5300), complex128, synthetic seeded input.
Metric: RGF slice-steps/s (slice-step = one (seed, energy, slice) triple).

  value      inputs resident in HBM (energies / T_out are device tensors, ribbon already set)
  e2e        the same through the C ABI with HOST buffers: rgf_set_device(host onsite) +
             rgf_transmission(host energies -> host T) inside the timed region
  roofline   dominant kernel = half_sweep_kernel (FP64 DMMA): algorithmic flops per launch divided
             by its mean CUDA-event duration inside the timed region, against the FP64 tensor
             ceiling measured live on the same GPU (rgf_fp64_peak_tflops)
  cpu_baseline  the oracle (oracle/rgf_oracle.c, naive LU, OpenMP over energies) on a bounded sample

--impl reference times the CPU oracle alone (there is no reference implementation to install:
/root/reference holds only the paper's text).
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

from paper_1107_5300_b200 import inputs  # noqa: E402

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel at the headline launch configuration: it
# cannot be measured inside a timed run, so it is READ from the committed ncu --set full summary (its `dram_bytes_per_launch:` line)
TRAFFIC_PROFILE = os.path.join("profiles", "ncu_r02_half_sweep.md")


def traffic_from_profile():
    try:
        for line in open(os.path.join(ROOT, TRAFFIC_PROFILE)):
            if line.startswith("dram_bytes_per_launch:"):
                return float(line.split(":")[1])
    except OSError:
        pass
    return None

METRIC = "rgf_slice_steps_per_s"
UNIT = "slice-steps/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    # exploration knobs (the driver never passes them; defaults = the headline workload)
    ap.add_argument("--M", type=int, default=244)
    ap.add_argument("--L", type=int, default=8000)
    ap.add_argument("--n-E", type=int, default=512)
    ap.add_argument("--cohort", type=int, default=0)
    ap.add_argument("--form", default="half", choices=["half", "dense"], help="formulation of the sweep (include/rgf.h)")
    ap.add_argument("--no-guard", action="store_true", help="switch the near-neutrality guard off (rgf_set_guard 0)")
    ap.add_argument("--ldos", action="store_true", help="time the second workload instead (rgf_ldos, SURVEY.md 8(f) F-4): M, L as given, n-E energies")
    ap.add_argument("--workload", default="", choices=["", "configs[3]-clean", "configs[3]", "configs[4]"],
                    help="time another BASELINE.json config instead of the headline (one compact JSON line, no e2e / cpu legs)")
    ap.add_argument("--precision", default="c128", choices=["c128", "c64"], help="with --workload: arithmetic of the sweep")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def workload(a, world, rank):
    """Headline ribbon; with N GPUs the global grid has 512*N energies and rank r takes E[r::N] (weak scaling)."""
    from paper_1107_5300_b200 import binding as rgf
    w = inputs.config2(M=a.M, L=a.L, n_E=a.n_E * world)
    E = np.empty(rgf.rgf_shard_count(w.n_E, world, rank))
    rgf.rgf_shard_energies(w.energies, w.n_E, world, rank, E)          # the library's round-robin split (include/rgf.h)
    return w, E


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index):
        self.rows, self.proc, self.thread = [], None, None
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + q, "--format=csv,noheader,nounits",
                                          "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def update_flops_per_inverse(n, B=32):
    """Algorithmic real flops of the gj_update launches of one n x n inverse (8 per complex MAC)."""
    tot, launches = 0, 0
    for k0 in range(0, n, B):
        bw = min(B, n - k0)
        if n > B:
            tot += 8 * n * (n - bw) * bw
            launches += 1
    return tot, launches


def cpu_baseline(a, repeats=1):
    """Oracle steady-state sweep rate on all host cores, as it stands (oracle/ is not tuned for this).

    The oracle has no entry point without the lead decimation (2 leads x 37 iterations, ~20 s per energy at M = 244), so the
    rate is a difference: one untimed warm-up call (thread pool, page faults), one call at L1 slices, then `repeats` calls
    at L2 slices on the same energies; rate_k = n_E (L2 - L1) / (t2_k - t1).  L2 - L1 is chosen so that the sweep difference
    (~25 s) is larger than the lead time it cancels, which is what makes the number reproducible (481 ... 1459
    with a 72-slice difference).  value = median of the repeats; the spread is printed in `sample`.
    """
    from oracle import rgf_oracle as orc
    w = inputs.config2(M=a.M, L=max(a.L, 512), n_E=a.n_E)
    nthr = orc.num_threads()
    idx = np.linspace(0, w.n_E - 1, nthr).astype(int)
    E = w.energies[idx]
    per_step = 2.4e-9 * 2.4 * a.M ** 3                     # s per slice-step per core, naive LU + matmul
    L1 = int(min(max(4, 2.5 / per_step), 32))
    L2 = int(min(L1 + max(16, 25.0 / per_step), w.L))

    def run(Lx, Ex):
        ws = inputs.truncate(w, Lx)
        t0 = time.perf_counter()
        orc.transmission_batch(ws.onsite[0], None, ws.t, Ex, ws.eta, method=orc.LEAD_BLOCK, nthreads=nthr)
        return time.perf_counter() - t0

    run(1, E[:1])                                          # untimed warm-up (one energy, one slice)
    t1 = run(L1, E)
    t2 = [run(L2, E) for _ in range(max(1, repeats))]
    rates = [len(E) * (L2 - L1) / max(t - t1, 1e-9) for t in t2]
    return {"value": float(np.median(rates)), "unit": UNIT, "cores": nthr, "kind": "oracle",
            "sample": "%d energies x (%d - %d) slices of the M=%d headline ribbon after one warm-up call; t(L1) = %.1f s, t(L2) = %s s "
                      "(both include the lead decimation, which cancels); rates %s"
                      % (len(E), L2, L1, a.M, t1, "/".join("%.1f" % t for t in t2), "/".join("%.0f" % r for r in rates)),
            "seconds": t1 + sum(t2)}


def run_reference(a):
    """--impl reference: the oracle alone on the host cores.  A step = one oracle call at L2 slices (a bounded sample of the
    workload); as many of the K requested steps are timed as fit in about four minutes of wall time, and `steps` reports
    the number really timed.  The warm-up is one small untimed call plus the L1 call that cancels the lead time."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    t0 = time.perf_counter()
    probe = cpu_baseline(a, repeats=1)
    per = probe["seconds"]
    extra = int(max(0, min(a.steps - 1, (240.0 - per) // max(per * 0.6, 1.0))))
    base = cpu_baseline(a, repeats=extra) if extra >= 2 else probe
    steps = max(1, extra) if extra >= 2 else 1
    wall = time.perf_counter() - t0
    val = base["value"]
    line = {"metric": METRIC, "value": val, "unit": UNIT, "n_gpus": a.gpus, "steps": steps, "warmup": 1,
            "ms_per_step": 1e3 * base["seconds"] / (steps + 1), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": "configs[2] M=%d L=%d n_E=%d complex128 (bounded sample, see cpu_baseline.sample)" % (a.M, a.L, a.n_E),
                       "steps_requested": a.steps, "warmup_requested": a.warmup, "wall_s": wall},
            "cpu_baseline": base, "gpu_launches": 0,
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def run_ldos(a):
    """Second workload (not the headline line): LDOS of the connected device, three batched M x M inverses per slice."""
    import torch
    from paper_1107_5300_b200 import binding as rgf
    w = inputs.config2(M=a.M, L=a.L, n_E=a.n_E)
    plan = rgf.rgf_plan_create(0, torch.cuda.current_stream().cuda_stream)
    peak = rgf.rgf_fp64_peak_tflops(plan)
    rgf.rgf_set_device(plan, w.M, w.L, np.ascontiguousarray(w.onsite[0]), w.t, None)
    E = torch.from_numpy(w.energies).cuda()
    out = torch.empty((1, w.n_E, w.L, w.M), dtype=torch.float64, device="cuda")
    eta = 2.0 / w.n_E
    for _ in range(max(1, a.warmup)):
        rgf.rgf_ldos(plan, E, w.n_E, eta, out)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(a.steps):
        rgf.rgf_ldos(plan, E, w.n_E, eta, out)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / a.steps
    st = rgf.rgf_get_stats(plan)
    flops = 3 * 8.0 * w.M ** 3 * w.n_E * w.L
    print(json.dumps({"metric": "rgf_ldos_slice_steps_per_s", "value": w.n_E * w.L / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "steps": a.steps,
                      "config": {"workload": "LDOS of the configs[2] ribbon, M=%d L=%d n_E=%d, eta=%.3g eV, complex128" % (w.M, w.L, w.n_E, eta), "chunk": st["cohort"]},
                      "tflops_executed": flops / (ms * 1e-3) * 1e-12, "frac_of_fp64_tensor_peak": flops / (ms * 1e-3) * 1e-12 / peak, "peak": peak,
                      "gpu_launches": st["launches"], "dtype": "f64", "data": "synthetic"}))
    rgf.rgf_destroy(plan)


def run_other(a):
    """The other BASELINE.json configs (not the headline line): one rgf_transmission call per step on the config's own
    arrays (vacancies included), inputs resident in HBM, CUDA events around the timed steps."""
    import torch
    from paper_1107_5300_b200 import binding as rgf
    w = {"configs[3]-clean": lambda: inputs.config3(disordered=False), "configs[3]": lambda: inputs.config3(disordered=True),
         "configs[4]": inputs.config4}[a.workload]()
    c64 = a.precision == "c64"
    plan = rgf.rgf_plan_create(0, torch.cuda.current_stream().cuda_stream)
    peak = rgf.rgf_fp64_peak_tflops(plan)
    vac = None if w.vacancy is None else np.ascontiguousarray(w.vacancy[0])
    rgf.rgf_set_device(plan, w.M, w.L, np.ascontiguousarray(w.onsite[0]), w.t, vac)
    E = torch.from_numpy(w.energies).cuda()
    T = torch.empty(w.n_E, dtype=torch.float64, device="cuda")
    ok = (rgf.RGF_ESINGULAR,) if c64 else ()             # complex64 overflows in and next to the gap: NaN + ESINGULAR
    prec = rgf.RGF_C64 if c64 else rgf.RGF_C128
    for _ in range(max(1, a.warmup)):
        rgf.rgf_transmission(plan, E, w.n_E, w.eta, prec, T, ok)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(a.steps):
        rgf.rgf_transmission(plan, E, w.n_E, w.eta, prec, T, ok)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / a.steps
    st = rgf.rgf_get_stats(plan)
    n = w.M // 2
    flops = w.n_E * w.L * 2 * 16.0 * n ** 3               # executed: per half-step an (M/2) inverse + the (M/2)^3 propagator product
    tf = flops / (ms * 1e-3) * 1e-12
    fp32_peak = 148 * 128 * 2 * 1.965e-3                  # TFLOP/s, FFMA lanes x clock
    print(json.dumps({"metric": METRIC, "value": w.n_E * w.L / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "steps": a.steps, "warmup": a.warmup,
                      "config": {"workload": w.name, "precision": a.precision, "formulation": "half"},
                      "tflops_executed": tf, "roofline": {"bound": "alu" if c64 else "tensor", "achieved": tf, "peak": fp32_peak if c64 else peak,
                                                          "unit": "TFLOP/s", "frac": tf / (fp32_peak if c64 else peak),
                                                          "note": "whole call (all kernels), executed flops 2 x 16 (M/2)^3 per slice"},
                      "phase_ms_last_step": {k: st[k] for k in ("ms_total", "ms_leads", "ms_sweep", "ms_trace", "ms_guard")},
                      "guard_redone_energies": st["guard_redone"], "gpu_launches": st["launches"],
                      "dtype": "f32" if c64 else "f64", "data": "synthetic"}))
    rgf.rgf_destroy(plan)


def main():
    a = parse()
    if a.impl == "reference":
        return run_reference(a)
    if a.ldos:
        return run_ldos(a)
    if a.workload:
        return run_other(a)
    import torch
    from paper_1107_5300_b200 import binding as rgf     # fails loudly if the CUDA library is missing

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    w, E_host = workload(a, world, rank)
    n_E = len(E_host)
    onsite = np.ascontiguousarray(w.onsite[0])
    stream = torch.cuda.current_stream()
    plan = rgf.rgf_plan_create(local, stream.cuda_stream)
    if a.cohort:
        rgf.rgf_set_cohort(plan, a.cohort)
    rgf.rgf_set_formulation(plan, rgf.RGF_FORM_HALF if a.form == "half" else rgf.RGF_FORM_DENSE)
    if a.no_guard:
        rgf.rgf_set_guard(plan, 0.0)
    peak = rgf.rgf_fp64_peak_tflops(plan)
    rgf.rgf_set_device(plan, w.M, w.L, onsite, w.t, None)
    E_dev = torch.from_numpy(E_host).to(dev)
    T_dev = torch.empty(n_E, dtype=torch.float64, device=dev)
    rgf.rgf_set_profiling(plan, 1)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    def step_resident():
        rgf.rgf_transmission(plan, E_dev, n_E, w.eta, rgf.RGF_C128, T_dev)

    for _ in range(a.warmup):
        step_resident()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches, ms_upd, n_upd, stats = 0, 0.0, 0, None
    e0.record()
    for _ in range(a.steps):
        step_resident()
        stats = rgf.rgf_get_stats(plan)
        launches += stats["launches"]; ms_upd += stats["ms_inverse_update"]; n_upd += stats["launches_inverse_update"]
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if sampler else None
    T_first = T_dev.cpu().numpy().copy()

    # ---- e2e: host buffers, set_device + transmission inside the timed region
    e2e = None
    if not a.no_e2e:
        rgf.rgf_set_profiling(plan, 0)
        E_pin = torch.from_numpy(E_host.copy()).pin_memory()
        on_pin = torch.from_numpy(onsite.copy()).pin_memory()
        T_pin = torch.empty(n_E, dtype=torch.float64).pin_memory()
        e2e_steps = max(1, min(a.steps, 1 if ms / a.steps > 20000 else a.steps))
        barrier()
        e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e2.record()
        for _ in range(e2e_steps):
            rgf.rgf_set_device(plan, w.M, w.L, on_pin.numpy(), w.t, None)
            rgf.rgf_transmission(plan, E_pin.numpy(), n_E, w.eta, rgf.RGF_C128, T_pin.numpy())
        e3.record()
        barrier()
        ms_e2e = e2.elapsed_time(e3)
        assert np.allclose(T_pin.numpy(), T_first, rtol=0, atol=1e-9, equal_nan=True)
        e2e = (ms_e2e, e2e_steps)

    tmax = torch.tensor([ms, e2e[0] if e2e else 0.0], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    ms_max, ms_e2e_max = float(tmax[0]), float(tmax[1])
    units_step = world * n_E * w.L                        # slice-steps per step over all ranks
    if rank == 0:
        value = units_step * a.steps / (ms_max * 1e-3)
        fused = a.form == "half" and (w.M + 1) // 2 <= 128          # the fused half_sweep_kernel runs the whole sweep
        n_inv = w.M // 2 if a.form == "half" else w.M          # matrix size of the inverses (M even at the headline)
        avg_ms = ms_upd / max(n_upd, 1)
        if fused:
            # algorithmic flops of one half-step: n^3 complex MACs for the in-place Gauss-Jordan inverse + n^2 nc for the
            # propagator columns that ride along as right-hand sides (8 real flops per complex MAC); 2 half-steps per slice
            flops_step = n_E * w.L * 2 * (8.0 * n_inv ** 3 + 8.0 * n_inv ** 2 * (w.M // 2))
            flops_per_launch = flops_step * a.steps / max(n_upd, 1)
            kernel_name = "half_sweep_kernel (fused assembly + augmented Gauss-Jordan [A | C P], FP64 DMMA.8x8x4)"
        else:
            fl_inv, l_inv = update_flops_per_inverse(n_inv)
            flops_per_launch = fl_inv / max(l_inv, 1) * stats["cohort"]
            kernel_name = "gj32_update_kernel (FP64 DMMA.8x8x4)"
            if n_inv > 256:      # generic path: its update launches are not event-timed (use --workload 'configs[4]' for the whole-call figure)
                kernel_name = "gj_update_kernel<B> (n > 256: rank-B ping-pong update, not event-timed in this mode)"
            if a.form == "half":
                flops_step = n_E * w.L * 2 * (8.0 * n_inv ** 3 + 8.0 * n_inv ** 3)     # executed: 2 x ((M/2) inverse + (M/2)^3 GEMM)
            else:
                flops_step = n_E * w.L * (8.0 * w.M ** 3 + 8.0 * (w.M / 2) ** 3)      # executed: dense inverse + compact propagator
        achieved = flops_per_launch / (avg_ms * 1e-3) * 1e-12 if avg_ms > 0 else 0.0
        state_bytes = 4 * (n_inv + (n_inv & 1)) ** 2 * 16 if fused else w.M * w.M * 16
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
            "ms_per_step": ms_max / a.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[2] armchair ribbon M=%d L=%d n_E=%d per GPU, Anderson +-0.1 eV seed 5300, complex128" % (w.M, w.L, n_E),
                       "eta": w.eta, "t": w.t, "cohort": stats["cohort"], "formulation": a.form,
                       "l2_policy": "inputs larger than L2 (%.0f MB of per-matrix state streamed every slice)" % (stats["cohort"] * state_bytes / 1e6)},
            "energies_per_s": world * n_E * a.steps / (ms_max * 1e-3),
            "tflops_executed": flops_step * world * a.steps / (ms_max * 1e-3) * 1e-12,
            "tflops_dense_equivalent": 16.0 * w.M ** 3 * units_step * a.steps / (ms_max * 1e-3) * 1e-12,
            "phase_ms_last_step": {k: stats[k] for k in ("ms_total", "ms_leads", "ms_sweep", "ms_trace", "ms_inverse_update", "ms_guard")},
            "lead_iterations": stats["lead_iterations"],
            "guard_redone_energies": stats["guard_redone"],
            "gpu_launches": launches,
            "clocks": clocks,
            "roofline": {"bound": "tensor", "kernel": kernel_name, "achieved": achieved, "peak": peak,
                         "unit": "TFLOP/s", "frac": achieved / peak if peak else None, "traffic": traffic_from_profile() if (a.form, w.M, w.L, n_E) == ("half", 244, 8000, 512) else None,
                         "traffic_source": "ncu dram__bytes_read.sum + dram__bytes_write.sum of one launch, " + TRAFFIC_PROFILE,
                         "peak_source": "measured live: rgf_fp64_peak_tflops (DMMA issue rate, this GPU)",
                         "launches_timed": n_upd, "share_of_step": ms_upd / ms if ms else None},
        }
        if e2e:
            line["e2e"] = {"value": units_step * e2e[1] / (ms_e2e_max * 1e-3), "unit": UNIT, "steps": e2e[1],
                           "h2d_bytes_per_step": int(onsite.nbytes + E_host.nbytes), "d2h_bytes_per_step": int(T_first.nbytes)}
        if not a.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(a)
        elif world > 1:
            line["cpu_baseline"] = None
        print(json.dumps(line))
    rgf.rgf_destroy(plan)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
