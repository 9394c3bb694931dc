#!/usr/bin/env python
"""bench.py -- env x taxel updates/s and step latency of the fused tactile readout (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 5] [--envs E]

A "step" is one ts_step() = the whole hot path (transform, geometry query, depth,
contact, force/torque, marker dilation, proximity march, noise chain) over E envs x T taxel slots.
Workload at N=1: BASELINE.json configs[4] ("paper-scale stress case", 20,480 envs x 1,000 taxels,
mixed primitives + 8 SDFs at 96^3, all outputs, full noise), the configuration the metric is quoted
on; synthetic seeded inputs (paper_2606_22332_b200.workloads, recipe in DESIGN.md).  N>1: one
process per GPU, each rank its own 20,480-env shard (weak scaling, no collective on the data path:
environments are independent); rank r uses env_id_base = r*E so Philox streams differ.

`value`      device-timed: inputs of all timed steps already resident in HBM, K steps between two
             CUDA events on the launch stream, barrier + synchronize on both sides, max over ranks.
`e2e`        the same metric through ts_step_host(): pinned HOST inputs and outputs, H2D + kernel +
             D2H of every requested output inside the timed region.
`roofline`   the step's kernels (ts_frames_kernel + ts_step_kernel): algorithmic bytes (DESIGN.md, 169 B per
             env-taxel with ASYM hysteresis) / mean duration of ALL kernels of a step from CUDA events recorded
             around every launch inside ts_step (a second pass over the same steps with recording on), vs
             MEASURED_PEAKS.json hbm_gbs; per-step median / p10 / p90, per-kernel means and the kernels' own
             %globaltimer span (first block start to last block end) are reported beside it.
`cpu_baseline` the oracle (oracle/, as it stands) on this box's host cores over the 16-env parity
             subset of the same workload; a reported baseline, not the target.
--impl reference: the oracle arm (this tier has no reference implementation): each step is the
             16-env sample, same metric/unit.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "env_taxel_updates_per_sec"
UNIT = "env*taxel/s"
# SURVEY 8d / DESIGN.md "algorithmic bytes": per (env, taxel) per step, everything on.
# ncu --set full capture of ts_step_kernel at this workload: DRAM bytes per launch and L2 hit rate, copied from the
# committed capture summary named in the file (a profile run, never measured inside this benchmark).
NCU_FILE = os.path.join(ROOT, "profiles", "ncu_config%d.txt")


def algorithmic_bytes_per_taxel(w, T, L, K, M):
    b = (L + K) * 13 * 4.0 / T                     # poses + velocities in
    outs = set(w.outputs)
    b += 1.0 * ("contact" in outs) + 4.0 * ("depth" in outs) + 24.0 * ("ft" in outs) + 4.0 * ("prox" in outs)
    b += (M * 12.0 / T) * ("marker" in outs)
    b += 2.0                                        # contact-bit / dead flag state read + write
    if w.noise:
        b += 24.0 * ("ft_noisy" in outs) + 1.0 * ("dead" in outs)
        b += 48.0                                   # drift state read + write
        hm = w.noise.get("hyst_mode", "off")
        b += {"asym": 48.0, "maxwell": 96.0}.get(hm, 0.0)
    return b


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def recorded_ncu(config):
    """{traffic_bytes_per_launch, lts_hit_rate_pct, l1_hit_rate_pct, source} from the committed ncu --set full capture
    of this config's step kernel (profiles/ncu_config<N>.txt), or {} if none is committed."""
    out = {}
    try:
        with open(NCU_FILE % config) as f:
            for line in f:
                if line.startswith("#") or not line.strip():
                    continue
                k, v = line.split(None, 1)
                out[k] = v.strip()
    except OSError:
        pass
    return out


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 6:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for n, v in zip(names, c[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


def oracle_arm(w, ids, steps, warmup, threads):
    """Times the oracle as it stands on `ids` (a bounded sample of the workload); returns (updates/s, ms/step)."""
    from oracle import oracle as O
    o = O.Oracle(w.patches, w.T, w.L, w.K, ids, physics=w.physics, noise=w.noise, threads=threads)
    o.set_geometry(w.types[ids], w.params[ids], w.bank, w.voxel)
    inps = [w.subset(w.inputs(s), ids) for s in range(warmup + steps)]
    for s in range(warmup):
        o.step(inps[s], want=w.outputs, aux=False)
    t0 = time.perf_counter()
    for s in range(warmup, warmup + steps):
        o.step(inps[s], want=w.outputs, aux=False)
    dt = time.perf_counter() - t0
    o.close()
    return len(ids) * w.T * steps / dt, 1e3 * dt / steps


def time_extras(W, TactileSim, torch, dev, n_envs=4096, steps=20):
    """Device time per step (CUDA events on the launch stream, mean of `steps` after 3 warm-up steps) of the SURVEY 8(f)
    sensor kernels: a context that asks for the extra output next to `depth`, minus the same context without it.
    Workload: config 4 (8 star objects, 1,000 taxels) at 4,096 envs; tracked clouds of 5,000 surface points (the
    shear kernel also with 1,000) and 1,280-triangle meshes per object."""
    w = W.config(4, n_envs=n_envs)
    stream = torch.cuda.current_stream(dev)
    inputs = None

    def run(outs, physics=None, noise=None, setup=None):
        nonlocal inputs
        sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=physics or w.physics, noise=noise, outputs=outs)
        sim.set_geometry(w.types, w.params, w.bank, w.voxel)
        if setup:
            setup(sim)
        if inputs is None:
            inputs = [sim.upload(w.inputs(s)) for s in range(8)]
        out = sim.alloc_outputs()
        for s in range(3):
            sim.step(inputs[s % 8], out)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        e0.record(stream)
        for s in range(steps):
            sim.step(inputs[s % 8], out)
        e1.record(stream)
        torch.cuda.synchronize(dev)
        sim.close()
        return e0.elapsed_time(e1) / steps

    res = {"workload": "config4 noise: %d envs x %d taxels, %d markers" % (w.E, w.T, 980)}
    base = run(("depth",))
    base_m = run(("depth", "marker"))
    pts5, cid = W.point_cloud_bank(w, 5000)
    pts1, _ = W.point_cloud_bank(w, 1000)
    meshes, mid = W.mesh_bank(w, 3)
    res["base_depth_only_ms"] = base
    res["proxpc_ms"] = run(("depth", "proxpc"), setup=lambda s: s.set_pointclouds(pts5, cid)) - base
    res["raycast_ms"] = run(("depth", "depth_rc", "nrm_rc"), setup=lambda s: s.set_meshes(meshes, mid)) - base
    res["shear_ms"] = run(("depth", "marker"), physics=dict(w.physics, shear_enable=1), setup=lambda s: s.set_pointclouds(pts5, cid)) - base_m
    res["shear_1000pts_ms"] = run(("depth", "marker"), physics=dict(w.physics, shear_enable=1), setup=lambda s: s.set_pointclouds(pts1, cid)) - base_m
    t12 = dict(w.noise, sigma_white_depth=2e-4, sigma_white_prox=1e-2, sigma_rw_prox=1e-3, quant_prox=1e-2, sigma_white_marker=1e-4,
               sigma_rw_marker=1e-5, quant_marker=1e-4, gain_min=0.85, gain_max=1.15)
    full = tuple(w.outputs)
    res["scalar_noise_ms"] = run(full + ("depth_noisy", "prox_noisy", "marker_noisy"), noise=t12) - run(full, noise=t12)
    n = float(w.E) * w.T
    res["env_taxel_per_s"] = {k[:-3]: n / (v * 1e-3) for k, v in res.items() if k.endswith("_ms") and k != "base_depth_only_ms" and v > 0}
    # What bounds them (profiles/r02_other_configs.md): the scalar-noise kernel streams its state:
    # per taxel clean depth + prox 8 B, flags 1 B, state 24 B read + 24 B written, outputs 8 B; per marker 12 B in, 36 B
    # of state read + 36 B written, 12 B out.  The other three move little and wait on dependent loads.
    b = (8 + 1 + 48 + 8) + (12 + 72 + 12) * 980.0 / w.T
    peak, src = hbm_peak()
    ach = b * n / (res["scalar_noise_ms"] * 1e-3) / 1e9 if res["scalar_noise_ms"] > 0 else 0.0
    res["roofline"] = {"scalar_noise": {"bound": "hbm", "bytes_per_env_taxel": b, "achieved": ach, "peak": peak, "unit": "GB/s",
                                        "frac": ach / peak, "peak_source": src},
                       "proxpc": {"bound": "latency (dependent loads: run bounds -> points)", "frac": None},
                       "raycast": {"bound": "latency (BVH node -> children / triangles)", "frac": None},
                       "shear": {"bound": "latency (per-pad phases: flag scan -> anchored points -> prism rows -> candidates)", "frac": None}}
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--envs", type=int, default=0, help="override the env count (debugging only; 0 = BASELINE size)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="budget of the cpu_baseline leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--extras", action="store_true", help="also time the SURVEY 8(f) sensor kernels (noisy scalar readouts, "
                    "point-cloud ProximityTaxel, shear history, raycast depth) on a 4,096-env config-4 scene; adds an "
                    "`extras` object to the line")
    ap.add_argument("--noise-knobs", default="", help="profiling aid, not the headline workload: extra App. A.8 knobs "
                    "as k=v,k=v (e.g. bias_force=0.02,read_delay=2); named in config.workload")
    a = ap.parse_args()
    K, Wm = a.steps, max(a.warmup, 0)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    from paper_2606_22332_b200 import workloads as W

    # ------------------------------------------------------------------ reference arm = the oracle
    if a.impl == "reference":
        if rank != 0:
            return 0
        w = W.config(a.config, n_envs=a.envs or None)
        ids = w.parity_envs()[:16]
        threads = os.cpu_count() or 1
        val, ms = oracle_arm(w, ids, K, Wm, threads)
        wl = "config%d %s: %d envs x %d taxels" % (a.config, w.name, w.E, w.T)
        sample = "%d envs %s x %d taxels per step, %d steps (oracle, OpenMP over envs)" % (len(ids), ids.tolist(), w.T, K)
        print(json.dumps({
            "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": a.gpus, "steps": K, "warmup": Wm,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": wl, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}))
        return 0

    # ------------------------------------------------------------------ our arm
    import torch
    import torch.distributed as dist
    from paper_2606_22332_b200.binding import TactileSim, IN_KEYS
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w = W.config(a.config, n_envs=a.envs or None, seed=rank)
    if a.noise_knobs:
        assert w.noise, "--noise-knobs needs a config with the noise model on (4 or 5)"
        extra = {k: (int(v) if k.startswith("read_") else (v if k == "hyst_mode" else float(v)))
                 for k, v in (kv.split("=") for kv in a.noise_knobs.split(","))}
        w.noise = dict(w.noise, **extra)
    sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=w.physics, noise=w.noise, outputs=w.outputs,
                     env_id_base=rank * w.E, device=local)
    sim.set_geometry(w.types, w.params, w.bank, w.voxel)
    E, T, M = w.E, sim.T, sim.M
    n_in = Wm + K
    period = W.T_PERIOD if a.config >= 4 else n_in          # configs 4-5 are 40-step periodic trajectories
    n_distinct = min(n_in, period)
    dev_in = [sim.upload(w.inputs(s)) for s in range(n_distinct)]   # resident in HBM before the timed region
    out = sim.alloc_outputs()
    stream = torch.cuda.current_stream(dev)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    clocks = ClockSampler(local)                           # nvidia-smi needs ~1 s to start: sample from warm-up on
    for s in range(Wm):
        sim.step(dev_in[s % n_distinct], out)
    barrier()
    t_spin = time.perf_counter()                           # keep the GPU under the same load until the sampler is live
    while time.perf_counter() - t_spin < 1.5:
        for s in range(8):
            sim.step(dev_in[s % n_distinct], out)
        torch.cuda.synchronize(dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record(stream)
    for s in range(Wm, Wm + K):
        sim.step(dev_in[s % n_distinct], out)
    ev1.record(stream)
    barrier()
    total_ms = ev0.elapsed_time(ev1)
    # second pass over the same K steps with per-launch recording on (CUDA events around every kernel inside ts_step,
    # on the step's stream, plus the kernels' own %globaltimer stamps): the per-kernel numbers behind `roofline`
    sim.kernel_time_ms(1)                                  # one pair of events around the kernels of each step
    for s in range(Wm, Wm + K):
        sim.step(dev_in[s % n_distinct], out)
    barrier()
    clk = clocks.stop()
    whole = sim.kernel_times_ms()                          # [K, 4]: column 1 = all kernels of the step, 3 = device-side clock
    kern_ms, kern_n = sim.kernel_time_ms(2)                # third pass: events between the kernels too (per-kernel split)
    for s in range(Wm, Wm + K):
        sim.step(dev_in[s % n_distinct], out)
    barrier()
    per_step = sim.kernel_times_ms()                       # [K, 4]: frames, step, noise kernel; device-side clock span
    sim.kernel_time_ms(False)
    first_ms = sim.first_kernel_time_ms()
    launches = K * sim.launches_per_step()
    # how much contact / march work the scene carries (last timed step, this rank): belongs next to the timing
    act_n = max(int((sim.layout.view()["radius"] > 0).sum()) * E, 1)
    scene = {k2: round(float(fn(out[k1]).sum().item()) / act_n, 4) for k1, k2, fn in
             (("depth", "frac_depth_gt0", lambda x: x > 0), ("contact", "frac_contact", lambda x: x > 0),
              ("prox", "frac_prox_gt0", lambda x: x > 0), ("dead", "frac_dead", lambda x: x > 0)) if k1 in out}

    # ---- e2e: ts_step_host on pinned host buffers (H2D + kernel + D2H inside the timed region)
    Ke = max(1, min(a.e2e_steps, K))
    host_in = [{k: v.cpu().pin_memory() for k, v in dev_in[s % n_distinct].items()} for s in range(min(Ke + 1, n_distinct))]
    host_out = sim.alloc_outputs(pinned_host=True)
    h2d = sum(v.numel() * v.element_size() for v in host_in[0].values())
    d2h = sum(v.numel() * v.element_size() for v in host_out.values())
    sim.step_host(host_in[0], host_out)                    # warm-up (allocates the staging buffers)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for s in range(Ke):
        sim.step_host(host_in[(s + 1) % len(host_in)], host_out)
    e1.record(stream)
    barrier()
    e2e_ms = e0.elapsed_time(e1)

    t = torch.tensor([total_ms, e2e_ms, kern_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms, e2e_ms, kern_ms = [float(x) for x in t.tolist()]
    units = float(E) * T * world
    value = units * K / (total_ms * 1e-3)
    e2e_value = units * Ke / (e2e_ms * 1e-3)

    bpt = algorithmic_bytes_per_taxel(w, T, w.L, w.K, M)
    peak, peak_src = hbm_peak()
    achieved = bpt * E * T / (kern_ms * 1e-3) / 1e9 if kern_ms > 0 else 0.0
    ncu = recorded_ncu(a.config) if not a.noise_knobs and not a.envs else {}
    tot = whole[:, 1] if len(whole) else np.zeros(1)
    pct = lambda v: {"median": float(np.median(v)), "p10": float(np.percentile(v, 10)), "p90": float(np.percentile(v, 90))}
    # `achieved` divides the step's algorithmic bytes by the duration of ALL kernels of the step (frames kernel + step
    # kernel [+ noise kernel]): the frames kernel's intermediate bytes count as time, not as useful bytes.
    roof = {"bound": "hbm", "kernel": "ts_frames_kernel + ts_step_kernel" + (" + ts_noise_kernel" if sim.launches_per_step() == 3 else ""),
            "achieved": achieved, "peak": peak, "unit": "GB/s",
            "frac": achieved / peak,
            "traffic": float(ncu["traffic_bytes_per_launch"]) if "traffic_bytes_per_launch" in ncu else None,
            "traffic_source": ncu.get("source"),
            "l2_hit_rate_pct": float(ncu["lts_hit_rate_pct"]) if "lts_hit_rate_pct" in ncu else None,
            "algorithmic_bytes_per_launch": bpt * E * T,
            "bytes_per_env_taxel": bpt, "kernel_ms": kern_ms, "kernel_ms_stats": pct(tot),
            "kernels_ms_mean": {"ts_frames_kernel": float(per_step[:, 0].mean()) if len(per_step) else None,
                                "ts_step_kernel": float(per_step[:, 1].mean()) if len(per_step) else None,
                                **({"ts_noise_kernel": float(per_step[:, 2].mean())}
                                   if len(per_step) and sim.launches_per_step() == 3 else {})},
            "device_clock_ms_stats": pct(whole[:, 3]) if len(whole) else None,
            "kernel_launches_timed": kern_n, "peak_source": peak_src,
            "frac_of_nominal_8TBs": achieved / 8000.0}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": "config%d %s: %d envs x %d taxels per GPU, %d links, %d markers, outputs=%s, noise=%s"
                                   % (a.config, w.name, E, T, w.L, M, "+".join(w.outputs),
                                      ((w.noise or {}).get("hyst_mode", "off") if w.noise else "off")
                                      + ("+" + a.noise_knobs if a.noise_knobs else "")),
                       "n_envs_per_gpu": E, "n_taxels": T, "scene": scene, "parallelism": "env-shard x%d, no collective" % world,
                       "l2": ("per-step working set %.2f GB >> 126 MB L2 (state + outputs stream through); no explicit flush"
                              if bpt * E * T > 4 * 126e6 else
                              "per-step working set %.2f GB is NOT well above the 126 MB L2 and is not flushed: part of it stays "
                              "L2-resident between steps (parity-size config, not the headline line)") % (bpt * E * T / 1e9),
                       "precision": "fp32 I/O and state; relative pose, first query, force/torque and marker sums in fp64 (DESIGN.md section 5)"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms / Ke, "steps": Ke},
            "gpu_launches": launches, "clocks": clk, "roofline": roof}

    if rank == 0 and world == 1 and not a.no_cpu_baseline:
        ids = w.parity_envs()[:16]
        threads = os.cpu_count() or 1
        # size the sample to ~cpu_seconds from one probe step
        v1, ms1 = oracle_arm(w, ids, 1, 1, threads)
        n = int(max(2, min(200, a.cpu_seconds * 1e3 / max(ms1, 1e-3))))
        v, ms = oracle_arm(w, ids, n, 1, threads)
        n1 = int(max(1, min(50, 0.25 * a.cpu_seconds * 1e3 / max(ms1 * threads, 1e-3))))
        v_st, ms_st = oracle_arm(w, ids, n1, 1, 1)             # the same oracle on ONE thread (SURVEY 8d asks for both)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                                "sample": "%d envs %s x %d taxels, %d steps, OpenMP over envs; %.1f ms per 16-env step "
                                          "(x%d envs/16 = %.0f ms per full step, linear extrapolation)"
                                          % (len(ids), ids.tolist(), T, n, ms, E, ms * E / len(ids)),
                                "single_thread": {"value": v_st, "unit": UNIT, "cores": 1, "steps": n1, "ms_per_16env_step": ms_st}}
    if a.extras and rank == 0 and world == 1:
        line["extras"] = time_extras(W, TactileSim, torch, dev)
    if rank == 0:
        print(json.dumps(line))
    sim.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
