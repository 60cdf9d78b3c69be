#!/usr/bin/env python
"""bench.py — throughput of the Diffusion Restore hot path on B200 (BASELINE.json metric).

A "step" is one frame of BASELINE.json configs[3] (the 1024x576 'transparent machines' scene, 589 824 chains,
one chain per pixel): dr_step(1 iteration) + dr_resolve_image, i.e. every row a1-a12 of SURVEY.md section 8(a).
Prints ONE JSON line (see the contract in the task statement).  `--impl reference` times the CPU oracle instead.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "chain mutations/s at 1024x576 (Diffusion Restore, transparent-machines scene)"
UNIT = "mutations/s"
# Algorithmic FLOPs of the path evaluation: one BVH8 node visit = 8 slab tests of
# 6 FMA + 12 min/max = 192 FLOP; one Moeller-Trumbore test = 50 FLOP.  The shading that k_wave also does is not counted.
F_NODE, F_TRI = 192.0, 50.0
# Algorithmic bytes per mutation of the state-streaming kernels (propose + decide + scan + scatter), d = 2L:
# read x, score (2 * 4d) + write x, score (2 * 4d) + p, f/p_hat, pixel, flags read and written (2 * 21).
def stream_bytes_per_mutation(d, grad):
    return (4 if grad else 2) * 4 * d + 42


def make_desc(name, nee=False):
    from dr_inputs import scenes as S
    d = {"machines": S.machines, "cornell": S.cornell, "caustic": S.caustic, "furnace": S.furnace,
         "mini_machines": S.mini_machines}[name]()
    d.nee = bool(nee)          # next-event estimation + MIS (Q21): four PSS coordinates per vertex
    return d


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.gpu)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for t, line in self.rows:
            f = [c.strip() for c in line.split(",")]
            if len(f) < 9 or not (t0 - 0.05 <= t <= t1 + 0.15):
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no sample inside the timed region"], samples=0)
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(np.max(mx)), reasons=sorted(reasons), samples=len(sm))


def cpu_baseline(desc, method, n_chains, iterations, seed):
    """The oracle as it stands on the host cores, on a bounded sample of the same workload."""
    from oracle import oracle as O
    sc = O.Scene(desc, O.F32)
    ch = O.Chains(sc, method, n_chains, seed=seed)
    ch.init(0)
    r0 = ch.stats()["rays"]
    t = time.perf_counter()
    ch.step(iterations)
    dt = time.perf_counter() - t
    st = ch.stats()
    return dict(value=n_chains * iterations / dt, unit=UNIT, cores=O.max_threads(), kind="oracle",
                sample=f"{desc.name}: {n_chains} chains x {iterations} iterations after init, {method}, fp32 oracle, OpenMP",
                mrays_per_s=(st["rays"] - r0) / dt / 1e6, seconds=dt)


def run_reference(args):
    """--impl reference: the CPU oracle, one bounded step = 8192 chains x 1 iteration of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    desc = make_desc(args.scene, args.nee)
    n = 8192
    sc = O.Scene(desc, O.F32)
    ch = O.Chains(sc, args.method, n, seed=4)
    ch.init(0)
    ch.step(args.warmup)
    r0 = ch.stats()["rays"]
    t = time.perf_counter()
    ch.step(args.steps)
    dt = time.perf_counter() - t
    val = n * args.steps / dt
    sample = f"{desc.name}: {n} chains x 1 iteration per step, {args.method}, fp32 oracle, OpenMP"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"configs[3] {desc.name} {desc.width}x{desc.height}, {desc.n_tris} triangles, L={desc.max_path_len}",
                   "method": args.method, "chains_per_step": n,
                   "path_construction": "direction sampling + next-event estimation with MIS (Q21)" if args.nee else "direction sampling only (Q5)"},
        "mrays_per_s": (ch.stats()["rays"] - r0) / dt / 1e6,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": O.max_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def second_reading(dr, torch, args, n_local):
    """The same scene, method and ensemble with next-event estimation + MIS (Q21): the paper does not say which path
    construction it uses, and under Q21 the Langevin step, the score and the race do real work.  A short
    run of the same frame loop: its numbers go into the JSON line beside the headline ones (`python bench.py --nee` is the full run)."""
    desc = make_desc(args.scene, True)
    chains = dr.Chains(dr.Scene(desc), args.method, n_local, seed=4)
    stream = torch.cuda.current_stream()
    steps, warm = min(args.steps, 60), max(args.warmup, 3)
    chains.init(0)
    for _ in range(warm):
        chains.step(1); chains.resolve()
    torch.cuda.synchronize()
    st0 = chains.stats()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        chains.step(1); chains.resolve()
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    st1 = chains.stats()
    pf = min(steps, 8)
    chains.profile_enable(True)
    for _ in range(pf):
        chains.step(1); chains.resolve()
    prof = chains.profile_read()
    chains.profile_enable(False)
    return {"path_construction": "direction sampling + next-event estimation with MIS (Q21)", "steps": steps, "warmup": warm,
            "ms_per_step": ms / steps, "value": n_local * steps / (ms * 1e-3), "unit": UNIT,
            "mrays_per_s": (st1["rays"] - st0["rays"]) / (ms * 1e-3) / 1e6,
            "rays_per_mutation": (st1["rays"] - st0["rays"]) / (n_local * steps),
            "kernels_ms_per_frame": {k: v["ms"] / pf for k, v in prof.items()},
            "kernel_launches_per_frame": sum(v["launches"] for v in prof.values()) / pf,
            "kill_fraction_last": st1["kills_last_step"] / n_local,
            "zeta_lit_fraction_of_uniform_samples": st1["lit_init"] / n_local,
            "grad_list_share_of_evaluations": (st1["grad_states"] - st0["grad_states"]) / (n_local * steps)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=120)       # configs[3]: 120 frames after init
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--method", default="diffusion_restore")
    ap.add_argument("--scene", default="machines")
    ap.add_argument("--chains", type=int, default=0, help="chains per GPU (default: one per pixel)")
    ap.add_argument("--nee", action="store_true", help="path construction with next-event estimation + MIS (second reading, DESIGN.md Q21)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-second-reading", action="store_true", help="skip the short run of the other path construction (N = 1 only)")
    ap.add_argument("--e2e-steps", type=int, default=10)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2605_08916_b200 import build as gpu_build
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if rank == 0:
        gpu_build.build()
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()
    import paper_2605_08916_b200 as dr
    from paper_2605_08916_b200 import sharding

    desc = make_desc(args.scene, args.nee)
    scene = dr.Scene(desc)
    n_local = args.chains or desc.width * desc.height            # weak scaling: every GPU runs one chain per pixel
    offset = sharding.shard_offset(n_local, rank)
    # sharded runs need the same p_lambda on every shard: fix it from a rank-0 bootstrap
    p_override = 0.0
    if world > 1:
        probe = dr.Chains(scene, args.method, n_local, seed=4, chain_offset=0)
        probe.init(0)
        t = torch.tensor([probe.stats()["p_lambda"]], device="cuda")
        dist.broadcast(t, 0)
        p_override = float(t.item())
        del probe
    chains = dr.Chains(scene, args.method, n_local, seed=4, chain_offset=offset, p_lambda_override=p_override)
    stream = torch.cuda.current_stream()

    def frame():
        chains.step(1)
        if world > 1:
            sharding.resolve_frame(chains)
        else:
            chains.resolve()

    ev = lambda: torch.cuda.Event(enable_timing=True)
    e0, e1 = ev(), ev()
    e0.record(stream); chains.init(0); e1.record(stream); torch.cuda.synchronize()
    init_ms = e0.elapsed_time(e1)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(args.warmup):
        frame()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    st0 = chains.stats()
    per = [(ev(), ev()) for _ in range(args.steps)]
    torch.cuda.synchronize()
    t_wall0 = time.time()
    e0.record(stream)
    for a, b in per:
        a.record(stream); frame(); b.record(stream)
    e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t_wall1 = time.time()
    total_ms = e0.elapsed_time(e1)
    if world > 1:
        t = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    st1 = chains.stats()
    frame_ms = sorted(a.elapsed_time(b) for a, b in per)
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    # per-kernel device times: a second, untimed pass with an event pair around every launch
    prof_frames = min(args.steps, 16)
    chains.profile_enable(True)
    for _ in range(prof_frames):
        frame()
    prof = chains.profile_read()
    chains.profile_enable(False)
    st2 = chains.stats()
    work = chains.work_stats()

    rays_local = st1["rays"] - st0["rays"]
    rays_total = rays_local
    if world > 1:
        t = torch.tensor([rays_local], device="cuda", dtype=torch.int64)
        dist.all_reduce(t)
        rays_total = int(t.item())
    mutations = n_local * world * args.steps
    value = mutations / (total_ms * 1e-3)

    # ---- end to end (1): host owns the chain state; every step uploads it from pinned host memory, steps, resolves, and
    # reads image + state back into pinned host memory (dr_chains_upload / dr_chains_download: DMA + transposition kernels)
    e2e = None
    if rank == 0:
        names = ("x", "p", "fop", "pix", "killed", "g", "sig")
        st = chains.download()
        host = {k: torch.from_numpy(np.ascontiguousarray(st[k])).pin_memory() for k in names}
        views = {k: host[k].numpy() for k in names}
        img_host = torch.empty(desc.height, desc.width, 3, dtype=torch.float32).pin_memory()
        h2d = sum(host[k].numel() * host[k].element_size() for k in names)
        d2h = h2d + img_host.numel() * 4
        it = st1["iteration"]
        for k in range(2):                                   # warm-up: staging buffers are allocated on first use
            chains.upload(views, it)
            chains.download(views)
        torch.cuda.synchronize()
        e0.record(stream)
        for k in range(args.e2e_steps):
            chains.upload(views, it + k)
            chains.step(1)
            img, _ = chains.resolve()
            img_host.copy_(img, non_blocking=True)
            chains.download(views)
        e1.record(stream)
        torch.cuda.synchronize()
        e2e_ms = e0.elapsed_time(e1)
        # ---- end to end (2): the renderer's own per-frame boundary (chains persist across frames on the device):
        # dr_step(1) + dr_resolve_image, image read back to pinned host memory every frame
        e0.record(stream)
        for k in range(args.e2e_steps):
            chains.step(1)
            img, _ = chains.resolve()
            img_host.copy_(img, non_blocking=True)
            stream.synchronize()                             # the host has the frame
        e1.record(stream)
        torch.cuda.synchronize()
        res_ms = e0.elapsed_time(e1)
        e2e = {"value": n_local * args.e2e_steps / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms / args.e2e_steps, "steps": args.e2e_steps,
               "what": "host-owned chain state: dr_chains_upload (pinned host -> device) + dr_step(1) + dr_resolve_image + "
                       "image and dr_chains_download back to pinned host memory, every step, N = 1 GPU",
               "resident_state_frame": {"value": n_local * args.e2e_steps / (res_ms * 1e-3), "unit": UNIT,
                                        "ms_per_step": res_ms / args.e2e_steps, "h2d_bytes_per_step": 0,
                                        "d2h_bytes_per_step": int(img_host.numel() * 4),
                                        "what": "chain state resident on the device (PAPER.md L482): dr_step(1) + "
                                                "dr_resolve_image + image to pinned host memory, host waits for every frame"}}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    pk = peaks()
    nodes_per_ray = work["node_visits"] / max(work["rays"], 1)
    tris_per_ray = work["tri_tests"] / max(work["rays"], 1)
    flop_per_ray = F_NODE * nodes_per_ray + F_TRI * tris_per_ray
    trace_launches = max(prof["trace"]["launches"], 1)
    trace_ms = prof["trace"]["ms"] / trace_launches
    rays_per_launch = (st2["rays"] - st1["rays"]) / trace_launches
    alu_peak = 148 * 128 * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
    achieved = flop_per_ray * rays_per_launch / (trace_ms * 1e-3) / 1e12
    grad = args.method in ("mala", "mala_restore", "diffusion_restore")
    stream_ms = sum(prof[k]["ms"] for k in ("propose", "decide", "scan", "scatter")) / prof_frames
    stream_gbs = stream_bytes_per_mutation(desc.dim, grad) * n_local / (stream_ms * 1e-3) / 1e9
    launches_per_frame = sum(v["launches"] for v in prof.values()) / prof_frames
    # evaluations below 2^21 states run traversal + shading of all segments as one persistent kernel (k_wave, one launch per
    # frame); larger ones the per-segment loop (k_trace + k_shade, L launches each per frame)
    wave = prof["shade"]["launches"] == 0
    cap = {}                                                      # counters of the last ncu --set full capture of that kernel
    tp = os.path.join(ROOT, "profiles", "trace_traffic.txt")
    if os.path.exists(tp):
        for line in open(tp):
            f = line.split()
            if len(f) == 2 and f[0].endswith("_k_wave" if wave else "_k_trace"):
                cap[f[0].rsplit("_k_", 1)[0]] = float(f[1])
    traffic = int(cap["dram_bytes_per_launch"]) if "dram_bytes_per_launch" in cap else None
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"configs[3] {desc.name} {desc.width}x{desc.height}, {desc.n_tris} triangles, L={desc.max_path_len} (d={desc.dim})",
                   "method": args.method, "chains_per_gpu": n_local, "iterations_per_frame": 1,
                   "path_construction": "direction sampling + next-event estimation with MIS (Q21)" if args.nee else "direction sampling only (Q5)",
                   "l2": "chain state (%.0f MB) larger than L2; no flush" % (chains.state.numel() / 1e6),
                   "seed": 4, "stddev": float(chains.cfg.stddev), "c_tilde": float(chains.cfg.c_tilde), "dt": float(chains.cfg.dt),
                   "m": float(chains.cfg.m)},
        "mrays_per_s": rays_total / (total_ms * 1e-3) / 1e6,
        "ms_per_frame": {"mean": total_ms / args.steps, "median": frame_ms[len(frame_ms) // 2], "min": frame_ms[0], "max": frame_ms[-1]},
        "init_ms": init_ms,
        "workload_stats": {"rays_per_mutation": rays_local / (n_local * args.steps), "nodes_per_ray": nodes_per_ray,
                           "tris_per_ray": tris_per_ray, "kill_fraction_last": st1["kills_last_step"] / n_local,
                           "tours": st1["tours"], "p_lambda": st1["p_lambda"], "nonfinite": st1["nonfinite"],
                           "zeta_lit_fraction_of_uniform_samples": st1["lit_init"] / n_local,
                           "mh_acceptance_rate": (st1["mh_accepts"] - st0["mh_accepts"]) / (n_local * args.steps) if args.method in ("metropolis", "mala", "metropolis_restore", "mala_restore") else None,
                           "grad_list_share_of_evaluations": (st1["grad_states"] - st0["grad_states"]) / (n_local * args.steps)},
        "kernels_ms_per_frame": {k: v["ms"] / prof_frames for k, v in prof.items()},
        "kernel_launches_per_frame": launches_per_frame,
        "gpu_launches": int(round(launches_per_frame * args.steps)),
        "clocks": clocks,
        "roofline": {"kernel": "k_wave" if wave else "k_trace", "bound": "alu", "achieved": achieved, "peak": alu_peak,
                     "unit": "TFLOP/s", "frac": achieved / alu_peak, "traffic": traffic,
                     "traffic_source": "ncu --set full capture, profiles/trace_traffic.txt (not measured in this run)",
                     "ncu_capture": {k: v for k, v in cap.items() if k != "dram_bytes_per_launch"},
                     "peak_source": f"148 SM x 128 FP32 lanes x 2 x {pk['sm_max_mhz']:.0f} MHz ({pk['source']} sm_max_mhz)",
                     "flop_per_ray": flop_per_ray, "rays_per_launch": rays_per_launch, "launch_ms": trace_ms,
                     "grays_per_s_in_kernel": rays_per_launch / (trace_ms * 1e-3) / 1e9},
        "roofline_streaming": {"kernels": "k_propose+k_decide+k_scan+k_scatter", "bound": "hbm", "achieved": stream_gbs,
                               "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": stream_gbs / pk["hbm_gbs"],
                               "bytes_per_mutation": stream_bytes_per_mutation(desc.dim, grad), "ms_per_frame": stream_ms,
                               "peak_source": pk["source"]},
        "e2e": e2e,
    }
    if world == 1 and not args.nee and not args.no_second_reading:
        del chains
        out["second_reading"] = second_reading(dr, torch, args, n_local)
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(desc, args.method, 32768, 6, 4)
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
