#!/usr/bin/env python
"""bench_sweep.py — the measurements of SURVEY.md section 8(d) beyond bench.py's one line (BASELINE.json configs[4]):

  sweep   throughput of every sampler at 2^14 .. 2^22 chains on the configs[3] scene and on the caustic scene (Q19):
          mutations/s, Mrays/s, ms/frame, per-kernel time, traversal FLOP/s and streaming GB/s against their peaks, workload
          statistics; plus relMSE of the GPU image against the oracle's for N <= 2^18 (same seeds, same iterations)
  oracle  the oracle timed on the host cores: configs[1] in full and configs[3] at 2^16 chains x 8 iterations (section 8d)
  curves  equal-spp / equal-time error curves of path tracing and the five samplers against a long path-tracing reference
          (MAE, MSE, MRSE, MAPE, the shape of its Tables A.1 / B.1 on the synthetic scenes; row f2)

Everything is synthetic and seeded (dr_inputs/); output is markdown on stdout (the files under profiles/ are copies).
Only `sweep --relmse` and `oracle` execute oracle/ (test infrastructure, as bench.py's cpu_baseline leg does).
"""
import argparse
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

SAMPLERS = ["metropolis", "mala", "metropolis_restore", "mala_restore", "diffusion_restore"]
F_NODE, F_TRI = 192.0, 50.0        # algorithmic FLOPs per BVH8 node test / triangle test


def make(scene, nee):
    from dr_inputs import scenes as S
    d = getattr(S, scene)()
    d.nee = bool(nee)
    return d


def peaks():
    import json
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    d = json.load(open(p)) if os.path.exists(p) else {}
    return float(d.get("hbm_gbs", 6650.0)), 148 * 128 * 2 * float(d.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12


def timed_run(dr, torch, scene, method, n, warm, iters, seed=4):
    ch = dr.Chains(scene, method, n, seed=seed)
    ch.init(0)
    for _ in range(warm):
        ch.step(1); ch.resolve()
    st0 = ch.stats()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(iters):
        ch.step(1); ch.resolve()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    st1 = ch.stats()
    ch.profile_enable(True)
    pf = min(iters, 8)
    for _ in range(pf):
        ch.step(1); ch.resolve()
    prof = ch.profile_read()
    ch.profile_enable(False)
    work = ch.work_stats()
    return ch, ms, st0, st1, {k: v["ms"] / pf for k, v in prof.items()}, work


def cmd_sweep(args):
    import torch
    import paper_2605_08916_b200 as dr
    hbm, alu = peaks()
    print(f"| scene | sampler | chains | mutations/s | Mrays/s | ms/frame | rays/mut | kernel ms/frame: eval (trace+shade) / grad / propose+decide+scan+scatter | "
          f"traversal TFLOP/s (% of {alu:.1f}) | streaming GB/s (% of {hbm:.0f}) | kill frac | MH accept | grad share |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for scene_name in args.scenes:
        desc = make(scene_name, args.nee)
        scene = dr.Scene(desc)
        for method in args.methods:
            for n in args.chains:
                ch, ms, st0, st1, k, work = timed_run(dr, torch, scene, method, n, args.warmup, args.iters)
                rays = st1["rays"] - st0["rays"]
                npr, tpr = work["node_visits"] / max(work["rays"], 1), work["tri_tests"] / max(work["rays"], 1)
                ev = k["trace"] + k["shade"] + k["raygen"]
                tf = (F_NODE * npr + F_TRI * tpr) * (rays / args.iters) / (max(k["trace"], 1e-9) * 1e-3) / 1e12
                grad = method in ("mala", "mala_restore", "diffusion_restore")
                sb = (4 if grad else 2) * 4 * desc.dim + 42
                sms = k["propose"] + k["decide"] + k["scan"] + k["scatter"]
                gbs = sb * n / (sms * 1e-3) / 1e9
                acc = (st1["mh_accepts"] - st0["mh_accepts"]) / (n * args.iters) if method != "diffusion_restore" else float("nan")
                print(f"| {desc.name}{'+nee' if args.nee else ''} | {method} | {n} | {n * args.iters / (ms * 1e-3):.3g} | {rays / (ms * 1e-3) / 1e6:.0f} | "
                      f"{ms / args.iters:.3f} | {rays / (n * args.iters):.2f} | {ev:.3f} / {k['grad']:.3f} / {sms:.3f} | {tf:.2f} ({100 * tf / alu:.1f} %) | "
                      f"{gbs:.0f} ({100 * gbs / hbm:.0f} %) | {st1['kills_last_step'] / n:.3f} | {acc:.3f} | "
                      f"{(st1['grad_states'] - st0['grad_states']) / (n * args.iters):.4f} |", flush=True)
                del ch
                torch.cuda.empty_cache()
    if args.relmse:
        from oracle import oracle as O
        print(f"\n| scene | sampler | chains | iterations | relMSE GPU vs oracle | oracle s ({O.max_threads()} threads) |")
        print("|---|---|---|---|---|---|")
        for scene_name in args.scenes:
            desc = make(scene_name, args.nee)
            scene, osc = dr.Scene(desc), O.Scene(desc, O.F32)
            for method in args.methods:
                for n in [c for c in args.chains if c <= (1 << 18)]:
                    g = dr.Chains(scene, method, n, seed=4)
                    g.init(0); g.step(args.relmse)
                    gimg = g.resolve()[0].cpu().numpy()
                    t = time.perf_counter()
                    o = O.Chains(osc, method, n, seed=4)
                    o.init(0); o.step(args.relmse)
                    oimg = o.resolve()[0]
                    dt = time.perf_counter() - t
                    print(f"| {desc.name} | {method} | {n} | {args.relmse} | {O.rel_mse(gimg, oimg):.2e} | {dt:.1f} |", flush=True)
                    del g, o


def cmd_oracle(args):
    from oracle import oracle as O
    print(f"| workload | sampler | chains x iterations | seconds | mutations/s | Mrays/s | threads |")
    print("|---|---|---|---|---|---|---|")
    for scene_name, n, iters, seed in (("cornell", 65536, 256, 2), ("machines", 65536, 8, 4)):
        desc = make(scene_name, False)
        sc = O.Scene(desc, O.F32)
        for method in (["diffusion_restore", "metropolis_restore"] if scene_name == "cornell" else ["diffusion_restore"]):
            ch = O.Chains(sc, method, n, seed=seed)
            t = time.perf_counter()
            ch.init(0)
            ch.step(iters)
            dt = time.perf_counter() - t
            st = ch.stats()
            print(f"| configs[{1 if scene_name == 'cornell' else 3}] {desc.name} | {method} | {n} x {iters} (+ init) | {dt:.1f} | {st['mutations'] / dt:.3g} | "
                  f"{st['rays'] / dt / 1e6:.2f} | {O.max_threads()} |", flush=True)


def metrics(a, b):
    """MAE, MSE, MRSE, MAPE of image a against reference b (relative forms with 1e-2 in the denominator)."""
    d = a - b
    return np.mean(np.abs(d)), np.mean(d * d), np.mean(d * d / (b * b + 1e-2)), np.mean(np.abs(d) / (np.abs(b) + 1e-2))


def cmd_curves(args):
    import torch
    import paper_2605_08916_b200 as dr
    for scene_name in args.scenes:
        desc = make(scene_name, args.nee)
        scene = dr.Scene(desc)
        n = desc.width * desc.height
        ref = dr.Chains(scene, "path_tracing", n, seed=999)
        ref.init(0); ref.step(args.ref_spp - 1)
        rimg = ref.resolve()[0].cpu().numpy().astype(np.float64)
        del ref
        print(f"\n### {desc.name}{'+nee' if args.nee else ''} {desc.width}x{desc.height}, L = {desc.max_path_len}, {n} chains, reference: path tracing {args.ref_spp} spp "
              f"(mean radiance {rimg.mean():.4f}), {args.seeds} seeds per method\n")
        print("| method | spp | ms (device) | MAE | MSE | MRSE | MAPE |")
        print("|---|---|---|---|---|---|---|")
        marks = [2 ** k for k in range(0, int(np.log2(args.max_spp)) + 1, 2)]
        for method in ["path_tracing"] + SAMPLERS:
            acc = {m: [] for m in marks}
            for seed in range(args.seeds):
                ch = dr.Chains(scene, method, n, seed=100 + seed)
                e0 = torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                ch.init(0)
                spp = 1
                for m in marks:
                    if m > spp:
                        ch.step(m - spp); spp = m
                    img = ch.resolve()[0]
                    e1 = torch.cuda.Event(enable_timing=True)
                    e1.record(); torch.cuda.synchronize()
                    acc[m].append((e0.elapsed_time(e1),) + metrics(img.cpu().numpy().astype(np.float64), rimg))
                del ch
            for m in marks:
                v = np.mean(np.array(acc[m]), axis=0)
                print(f"| {method} | {m} | {v[0]:.2f} | {v[1]:.4g} | {v[2]:.4g} | {v[3]:.4g} | {v[4]:.4g} |", flush=True)


def main():
    ap = argparse.ArgumentParser()
    sub = ap.add_subparsers(dest="cmd", required=True)
    s = sub.add_parser("sweep")
    s.add_argument("--scenes", nargs="+", default=["machines", "caustic"])
    s.add_argument("--methods", nargs="+", default=SAMPLERS)
    s.add_argument("--chains", nargs="+", type=int, default=[1 << 14, 1 << 16, 1 << 18, 1 << 20, 1 << 22])
    s.add_argument("--warmup", type=int, default=64)
    s.add_argument("--iters", type=int, default=64)
    s.add_argument("--relmse", type=int, default=0, help="iterations of the GPU-vs-oracle image comparison (0 = skip)")
    s.add_argument("--nee", action="store_true")
    o = sub.add_parser("oracle")
    c = sub.add_parser("curves")
    c.add_argument("--scenes", nargs="+", default=["cornell", "caustic", "machines"])
    c.add_argument("--ref-spp", type=int, default=4096)
    c.add_argument("--max-spp", type=int, default=1024)
    c.add_argument("--seeds", type=int, default=4)
    c.add_argument("--nee", action="store_true")
    args = ap.parse_args()
    from paper_2605_08916_b200 import build
    if args.cmd != "oracle":
        build.build()
    {"sweep": cmd_sweep, "oracle": cmd_oracle, "curves": cmd_curves}[args.cmd](args)


if __name__ == "__main__":
    main()
