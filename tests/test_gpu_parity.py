"""GPU-vs-oracle parity through the C-ABI (every test here needs a B200)."""
import numpy as np
import pytest

from dr_inputs import scenes as S

pytestmark = pytest.mark.gpu

from gpu_util import METHODS, compare_states, min_image  # noqa: E402


@pytest.fixture(scope="module")
def dr():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2605_08916_b200 import build
    build.build()
    import paper_2605_08916_b200 as dr_
    return dr_


@pytest.fixture(scope="module")
def torch_():
    import torch
    return torch


# ---- a1: RNG ---------------------------------------------------------------------------------------------------
def test_philox_bit_exact(dr, oracle, torch_):
    rng = np.random.default_rng(0)
    ctr = rng.integers(0, 2**32, size=(5000, 4), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0
    ctr[1] = 0xFFFFFFFF
    for seed in (0, 0xFFFFFFFFFFFFFFFF, 0x0123456789ABCDEF):
        got = dr.philox_blocks(seed, torch_.from_numpy(ctr.view(np.int32)).cuda()).cpu().numpy().view(np.uint32)
        for k in range(0, 5000, 7):
            want = oracle.philox([seed & 0xFFFFFFFF, seed >> 32], ctr[k])
            assert (got[k] == want).all()
    # three-way: cuRAND's own Philox4x32-10 is checked against the same words in test_gpu_curand.py if nvcc is present


def test_rng_transforms(dr, oracle, torch_):
    rng = np.random.default_rng(1)
    words = rng.integers(0, 2**32, size=(4000, 2), dtype=np.uint64).astype(np.uint32)
    words[0] = (0, 0)
    words[1] = (0xFFFFFFFF, 0xFFFFFFFF)
    got = dr.rng_transforms(torch_.from_numpy(words.view(np.int32)).cuda()).cpu().numpy()
    for k in range(4000):
        want = oracle.rng_transforms(int(words[k, 0]), int(words[k, 1]), oracle.F32)
        assert got[k, 0] == want[0] and got[k, 1] == want[1]                   # uniforms: bit-exact
        assert np.allclose(got[k, 2:], want[2:], rtol=1e-6, atol=2e-6), (k, got[k], want)   # libm vs CUDA ulps


# ---- a4: closest hit ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scene", ["furnace", "cornell", "mini_machines", "caustic"])
def test_trace_matches_oracle(dr, oracle, torch_, scene):
    desc = {"furnace": S.furnace, "cornell": S.cornell, "mini_machines": S.mini_machines, "caustic": S.caustic}[scene]()
    gsc = dr.Scene(desc)
    osc = oracle.Scene(desc, oracle.F32)
    n = 20011                                   # several blocks and a ragged tail
    o, d = S.seeded_rays(desc, n, 5)
    t, prim = gsc.trace_rays(torch_.from_numpy(o).cuda(), torch_.from_numpy(d).cuda())
    t, prim = t.cpu().numpy(), prim.cpu().numpy()
    brute = desc.n_tris <= 6000
    ot, otri = osc.trace(o, d, brute=brute)
    mism = prim != otri
    assert mism.mean() < 1e-4, mism.sum()        # edge-grazing rays may pick the neighbour: counted
    hit = (~mism) & (otri >= 0)
    assert hit.sum() > 1000
    diag = float(np.linalg.norm(desc.vertices.max(0) - desc.vertices.min(0)))
    assert np.all(np.abs(t[hit] - ot[hit]) <= 1e-5 * np.maximum(np.abs(ot[hit]), 0.25 * diag))   # fp32 Moeller-Trumbore on both sides
    assert np.all(t[(~mism) & (otri < 0)] == -1.0)
    info = gsc.info()
    assert info["n_tris"] == desc.n_tris and info["n_nodes"] >= 1 and info["smem_nodes"] <= 585


def test_trace_degenerate_rays(dr, oracle, torch_):
    desc = S.cornell()
    gsc = dr.Scene(desc)
    o = np.array([[0.5, 0.5, -1.0], [0.5, 0.5, 0.5], [0.5, 0.5, 0.5], [5, 5, 5]], dtype=np.float32)
    d = np.array([[0, 0, 1], [1, 0, 0], [0, -1, 0], [1, 0, 0]], dtype=np.float32)   # axis-aligned: zero components
    t, prim = gsc.trace_rays(torch_.from_numpy(o).cuda(), torch_.from_numpy(d).cuda())
    t, prim = t.cpu().numpy(), prim.cpu().numpy()
    ot, otri = oracle.Scene(desc, oracle.F32).trace(o, d, brute=True)
    assert (prim == otri).all() and np.allclose(t, ot, rtol=1e-6)
    assert np.isclose(t[1], 0.5) and np.isclose(t[2], 0.5) and t[3] == -1.0     # walls at x = 1 and y = 0
    t0, _ = gsc.trace_rays(torch_.zeros(0, 3, device="cuda"), torch_.zeros(0, 3, device="cuda"))    # empty input
    assert t0.numel() == 0


# ---- a3, a5, a6: target evaluation --------------------------------------------------------------------------------
@pytest.mark.parametrize("scene", ["furnace", "cornell", "mini_machines", "ggx_room", "closed_furnace", "mixture3"])
def test_eval_matches_oracle(dr, oracle, torch_, scene):
    desc = {"furnace": S.furnace, "cornell": lambda: S.cornell(width=64, height=64), "mini_machines": S.mini_machines,
            "ggx_room": S.ggx_room, "closed_furnace": S.closed_furnace, "mixture3": S.mixture3}[scene]()
    gsc = dr.Scene(desc)
    osc = oracle.Scene(desc, oracle.F32)
    n = 30011
    x = S.seeded_states(n, desc.dim, 3)
    g = gsc.eval_states(torch_.from_numpy(x).cuda(), want_score=True)
    g = {k: v.cpu().numpy() for k, v in g.items()}
    e = osc.eval(x, True)
    assert (g["pix"].view(np.uint32) == e["pix"]).all()                         # splat pixel indices: bit-exact
    div = (g["sig"].view(np.uint32) != e["sig"])
    assert div.mean() < 1e-3, div.sum()                                         # near-threshold decisions: counted
    ok = ~div
    assert (g["nrays"][ok] == e["nrays"][ok]).all()
    rel = np.abs(g["p"][ok] - e["p"][ok]) / np.maximum(e["p"][ok], 1e-8)
    assert rel.max() <= 1e-4, rel.max()
    relf = np.abs(g["f"][ok] - e["f"][ok]) / np.maximum(np.abs(e["f"][ok]), 1e-8)
    assert relf.max() <= 1e-4
    stddev = 5e-3
    tol = 1e-4 * np.abs(e["g"][ok]) + 2e-4 / stddev
    assert (np.abs(g["g"][ok] - e["g"][ok]) <= tol).all()
    if scene in ("mini_machines", "ggx_room"):
        assert (np.abs(e["g"][ok]).max(1) > 0).sum() > 20                       # the score path is exercised
    # without the score the value outputs are identical
    g2 = gsc.eval_states(torch_.from_numpy(x).cuda(), want_score=False)
    assert np.allclose(g2["p"].cpu().numpy(), g["p"], rtol=1e-6, atol=0) and (g2["sig"].cpu().numpy() == g["sig"]).all()


def test_furnace_states_hit_the_closed_form_exactly(dr, torch_):
    desc = S.furnace()
    gsc = dr.Scene(desc)
    x = S.seeded_states(100000, desc.dim, 9)
    g = gsc.eval_states(torch_.from_numpy(x).cuda(), want_score=True)
    f, nr = g["f"].cpu().numpy(), g["nrays"].cpu().numpy()
    assert ((f == 0.5) | (f == 1.0)).all()
    assert (f[nr == 2] == 0.5).all() and (f[nr == 1] == 1.0).all()
    assert (g["g"].cpu().numpy() == 0).all()
    r = np.hypot(x[:, 0] * 64 - 32, x[:, 1] * 64 - 32)
    clear = np.abs(r - 22.7007) > 0.05
    assert ((nr == 2)[clear] == (r[clear] < 22.7007)).all()


# ---- the five samplers: init + teacher-forced steps ------------------------------------------------------------------
CASES = [("furnace", S.furnace, 4096), ("mini_machines", S.mini_machines, 5000), ("ggx_room", S.ggx_room, 3001),
         ("mixture3", S.mixture3, 4097)]


@pytest.mark.parametrize("method", METHODS)
@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_teacher_forced_parity(dr, oracle, torch_, method, case):
    name, make, N = case
    desc = make()
    seed = 0 if name == "furnace" else 3
    gsc = dr.Scene(desc)
    osc = oracle.Scene(desc, oracle.F32)
    gch = dr.Chains(gsc, method, N, seed=seed)
    och = oracle.Chains(osc, method, N, seed=seed)
    stddev = float(gch.cfg.stddev)
    # --- init (Alg. 1) from the same seed: states are exact uniforms on both sides
    gch.init(2)
    och.init(2)
    gs, os_ = gch.download(), och.state()
    assert (gs["x"].astype(np.float64) == os_["x"]).all()                       # RNG streams: bit-exact
    gst, ost = gch.stats(), och.stats()
    assert np.isclose(gst["p_lambda"], ost["p_lambda"], rtol=2e-6) and np.isclose(gst["kappa0"], ost["kappa0"], rtol=2e-6)
    assert gst["mutations"] == ost["mutations"] == N and gst["rays"] == ost["rays"] or name != "furnace"
    div, rep = compare_states(gs, os_, gch.last_step(), och.last(), stddev)
    assert div.mean() < 1e-3, rep
    if not div.any():
        assert (gch.queue() == och.queue()).all()                               # regeneration queue: bit-exact
        assert gst["tours"] == ost["tours"]
    worst = rep["frac"]
    # --- teacher-forced steps at several points of a run (Q15)
    for burst in (0, 3, 12):
        och.step(burst)                       # let the oracle run on to a later point
        n0 = och.stats()["iteration"]
        st = och.state()
        gch.upload(st, n0)
        gch.accum.zero_()
        och.zero_accum()
        t0g, t0o = gch.stats()["tours"], och.stats()["tours"]
        gch.step(1)
        och.step(1)
        gs, os_ = gch.download(), och.state()
        div, rep = compare_states(gs, os_, gch.last_step(), och.last(), stddev)
        worst = max(worst, rep["frac"])
        assert div.mean() < 1e-3, (method, name, burst, rep)
        if not div.any():
            assert (gch.queue() == och.queue()).all()
            assert gch.stats()["tours"] - t0g == och.stats()["tours"] - t0o
            ga, oa = gch.accum.cpu().numpy().astype(np.float64), och.accum()
            scale = np.abs(oa).max() + 1e-30
            assert np.abs(ga - oa).max() <= 2e-5 * scale + 1e-4 * np.abs(oa).max(), (method, name)
        assert (gs["x"] >= 0).all() and (gs["x"] < 1).all()
    print(f"{method}/{name}: worst per-step diverged fraction {worst:.2e}")


@pytest.mark.parametrize("method", METHODS)
def test_furnace_config0(dr, oracle, torch_, method):
    """BASELINE.json configs[0]: 4096 chains, 64 iterations, seed 0.  Gates of DESIGN.md Q12."""
    desc = S.furnace()
    gsc, osc = dr.Scene(desc), oracle.Scene(desc, oracle.F32)
    gch, och = dr.Chains(gsc, method, 4096, seed=0), oracle.Chains(osc, method, 4096, seed=0)
    gch.init(0)
    och.init(0)
    gch.step(64)
    och.step(64)
    acc = gch.accum.cpu().numpy().astype(np.float64)
    with np.errstate(invalid="ignore", divide="ignore"):
        ratio = acc[:, 0] / acc[:, 3]
    yy, xx = np.mgrid[0:64, 0:64]
    corners = [np.hypot(xx + a - 32, yy + b - 32) for a in (0, 1) for b in (0, 1)]
    inside = (np.max(corners, axis=0) < 22.7007 - 0.05).ravel()
    outside = (np.min(corners, axis=0) > 22.7007 + 0.05).ravel()
    seen = acc[:, 3] > 0
    assert seen.mean() > 0.9
    assert np.abs(ratio[inside & seen] - 0.5).max() <= 1e-5                     # closed form, 1e-5 (B: north_star)
    assert np.abs(ratio[outside & seen] - 1.0).max() <= 1e-5
    gimg, st = gch.resolve()
    oimg, _ = och.resolve()
    assert st == 0
    assert oracle.rel_mse(gimg.cpu().numpy(), oimg) <= 1e-3                       # image-level GPU vs oracle
    gs, os_ = gch.stats(), och.stats()
    assert gs["mutations"] == os_["mutations"] == 4096 * 65
    assert abs(gs["tours"] - os_["tours"]) <= 3 and abs(gs["rays"] - os_["rays"]) <= 50


def test_free_running_image_matches_oracle(dr, oracle, torch_):
    desc = S.cornell(width=32, height=32, max_path_len=5)
    gsc, osc = dr.Scene(desc), oracle.Scene(desc, oracle.F32)
    for method in ("metropolis_restore", "diffusion_restore"):
        gch, och = dr.Chains(gsc, method, 20000, seed=1), oracle.Chains(osc, method, 20000, seed=1)
        gch.init(0)
        och.init(0)
        gch.step(40)
        och.step(40)
        gimg, _ = gch.resolve()
        oimg, _ = och.resolve()
        assert oracle.rel_mse(gimg.cpu().numpy(), oimg) <= 1e-3


# ---- edge cases and the boundary's error behaviour ----------------------------------------------------------------------
def test_edge_cases(dr, torch_):
    desc = S.furnace()
    gsc = dr.Scene(desc)
    for N in (1, 31, 257):                                                      # ragged and tiny chain counts
        ch = dr.Chains(gsc, "diffusion_restore", N, seed=1)
        ch.init(0)
        ch.step(3)
        s = ch.stats()
        assert s["mutations"] == 4 * N and s["iteration"] == 3
        x = ch.download()["x"]
        assert np.isfinite(x).all() and (x >= 0).all() and (x < 1).all()
    # resolve before any tour: warning + zero image
    ch = dr.Chains(gsc, "diffusion_restore", 4, seed=1, m=1e9)
    ch.init(0)
    img, status = ch.resolve()
    assert status == dr.DR_WARN_NO_TOURS and float(img.abs().max()) == 0.0
    # wrong method in dr_step, invalid configs
    with pytest.raises(dr.DrError):
        dr.binding._check(dr.lib.dr_step(ch.h, 0, 1, None))
    for bad in (dict(stddev=0.0), dict(dt=-1.0), dict(m=0.0), dict(large_step_prob=1.5), dict(stddev=float("nan"))):
        with pytest.raises(dr.DrError):
            dr.Chains(gsc, "metropolis", 16, **bad)
    bad_desc = S.furnace()
    bad_desc.vertices = bad_desc.vertices.copy()
    bad_desc.vertices[0, 0] = np.inf
    with pytest.raises(dr.DrError) as ei:
        dr.Scene(bad_desc)
    assert ei.value.status == dr.DR_ERR_NONFINITE
    bad_desc = S.furnace()
    bad_desc.max_path_len = 17
    with pytest.raises(dr.DrError):
        dr.Scene(bad_desc)
    # L = 1 (camera ray only) and an odd L (padded plane)
    for L in (1, 3):
        d1 = S.furnace(max_path_len=L)
        ch = dr.Chains(dr.Scene(d1), "mala_restore", 300, seed=2)
        ch.init(0)
        ch.step(2)
        assert ch.stats()["nonfinite"] == 0


def test_sharded_chains_reproduce_the_unsharded_run(dr, torch_):
    """chains keyed by global id -> two half-size shards == one full run (states bit-identical)."""
    desc = S.mini_machines()
    gsc = dr.Scene(desc)
    full = dr.Chains(gsc, "diffusion_restore", 2000, seed=4, p_lambda_override=0.05)
    full.init(0)
    full.step(4)
    xs = full.download()
    parts = []
    for off in (0, 1000):
        ch = dr.Chains(gsc, "diffusion_restore", 1000, seed=4, p_lambda_override=0.05, chain_offset=off)
        ch.init(0)
        ch.step(4)
        parts.append((ch.download(), ch.accum.clone(), ch.stats()["tours"]))
    assert (np.concatenate([p[0]["x"] for p in parts]) == xs["x"]).all()
    assert (np.concatenate([p[0]["killed"] for p in parts]) == xs["killed"]).all()
    assert parts[0][2] + parts[1][2] == full.stats()["tours"]
    summed = (parts[0][1] + parts[1][1]).cpu().numpy()
    assert np.allclose(summed, full.accum.cpu().numpy(), rtol=1e-4, atol=1e-7)


# ---- BASELINE.json full sizes, in the launch configuration bench.py times ------------------------------------------------
FULL = [("cornell", S.cornell, 65536, 2), ("caustic", S.caustic, 262144, 3), ("machines", S.machines, 589824, 4)]


@pytest.mark.parametrize("case", FULL, ids=[c[0] for c in FULL])
def test_full_size_configs(dr, oracle, torch_, case):
    """configs[1..3] at their full chain counts: bit-exact RNG / queue / counters, and sampled states re-evaluated
    one by one by the oracle (the stored (f/p_hat, p, pixel, score, signature) of a chain is the evaluation of its x)."""
    name, make, N, seed = case
    desc = make()
    gsc, osc = dr.Scene(desc), oracle.Scene(desc, oracle.F32)
    method = "diffusion_restore"
    gch = dr.Chains(gsc, method, N, seed=seed)
    gch.init(0)
    rng = np.random.default_rng(7)
    ids = np.unique(np.concatenate([rng.integers(0, N, 3000), [0, 1, 255, 256, N - 257, N - 1]]))
    gs = gch.download()
    # init states are the Philox uniforms of (chain, iteration 0, slot, REGEN_U, epoch 0): bit-exact
    for i in ids[:200]:
        for j in range(desc.dim // 4):
            w = oracle.stream_block(seed, int(i), 0, j, 0, 0)
            want = (w >> 8).astype(np.float64) * 2.0 ** -24
            assert (gs["x"][i, 4 * j:4 * j + 4].astype(np.float64) == want).all()

    def check_sample(gs):
        e = osc.eval(np.ascontiguousarray(gs["x"][ids]), True)
        assert (gs["pix"][ids] == e["pix"]).all()                                # splat pixel indices: bit-exact
        ok = gs["sig"][ids] == e["sig"]
        # Whole-path signatures (up to 16 hit triangles and lobes each): a path that grazes a triangle edge within
        # fp32 rounding continues from the neighbour on one side.  Counted; bound 1e-3 per path, 5e-3 for the
        # machines scene (14 segments per path over 0.01-0.2 wide facets, specular chains; Q15).
        assert (~ok).mean() < (5e-3 if name == "machines" else 1e-3), (~ok).sum()
        p, fop = gs["p"][ids][ok].astype(np.float64), gs["fop"][ids][ok].astype(np.float64)
        assert (np.abs(p - e["p"][ok]) <= 1e-4 * np.maximum(e["p"][ok], 1e-8)).all()
        want = e["f"][ok] / (e["p"][ok][:, None] + 1e-8)
        assert (np.abs(fop - want) <= 1e-4 * np.maximum(np.abs(want), 1e-8)).all()
        tol = 1e-4 * np.abs(e["g"][ok]) + 2e-4 / 5e-3
        assert (np.abs(gs["g"][ids][ok] - e["g"][ok]) <= tol).all()

    check_sample(gs)
    kills = int(gs["killed"].sum())
    for it in range(1, 3):
        gch.step(1)
        gs = gch.download()
        st = gch.stats()
        assert st["mutations"] == N * (it + 1) and st["iteration"] == it and st["nonfinite"] == 0
        assert (gs["x"] >= 0).all() and (gs["x"] < 1).all()
        q = gch.queue()
        assert (q == np.flatnonzero(gs["killed"])).all()                        # regeneration queue: bit-exact, ascending
        kills += len(q)
        assert st["tours"] == kills and st["kills_last_step"] == len(q)
        check_sample(gs)
    if name != "machines":      # the oracle runs these two in full in seconds: whole-ensemble teacher-forced step
        och = oracle.Chains(osc, method, N, seed=seed)
        och.init(0)
        och.step(2)
        gch.upload(och.state(), 2)
        gch.step(1)
        och.step(1)
        div, rep = compare_states(gch.download(), och.state(), gch.last_step(), och.last(), float(gch.cfg.stddev))
        assert div.mean() < 1e-3, rep
        if not div.any():
            assert (gch.queue() == och.queue()).all()


# ---- the two forms of the evaluation (k_wave vs per-segment loop) -------------------------------------------------
_EVAL_SNIPPET = """
import sys, numpy as np, torch
sys.path.insert(0, {root!r})
import paper_2605_08916_b200 as dr
from dr_inputs import scenes as S
desc = getattr(S, {scene!r})()
x = torch.from_numpy(S.seeded_states({n}, desc.dim, 11)).cuda()
e = dr.Scene(desc).eval_states(x, True)
torch.cuda.synchronize()
np.savez({out!r}, **{{k: v.cpu().numpy() for k, v in e.items()}})
"""


@pytest.mark.parametrize("scene", ["mini_machines", "ggx_room"])
def test_wave_kernel_equals_segment_loop(dr, torch_, tmp_path, scene):
    """2^18 states evaluated by k_wave (one persistent kernel, dr_wave.cuh) and, in a second process with DR_WAVE=0, by
    the per-segment loop k_trace / k_shade: both run the same shade_vertex on the same closest hits, so f, p, pixel,
    rays per path, signature and score must be identical bit for bit -- anything else is a ray lost, duplicated or
    read before it was written in the ring.  (The small parity scenes above never reach k_wave: it starts at 2^18.)"""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    n = 1 << 18
    res = {}
    for mode in ("1", "0"):
        out = str(tmp_path / f"eval_{mode}.npz")
        env = dict(os.environ, DR_WAVE=mode)
        subprocess.run([sys.executable, "-c", _EVAL_SNIPPET.format(root=root, scene=scene, n=n, out=out)], check=True, env=env,
                       timeout=600)
        res[mode] = np.load(out)
    a, b = res["1"], res["0"]
    assert int(a["nrays"].sum()) == int(b["nrays"].sum()) and a["nrays"].sum() > n      # paths do bounce
    for k in ("f", "p", "pix", "nrays", "sig", "g"):
        assert np.array_equal(a[k].view(np.uint32), b[k].view(np.uint32)), k
