"""GPU-vs-oracle parity through the C-ABI (every test here needs a B200)."""
import numpy as np
import pytest

from dr_inputs import scenes as S

pytestmark = pytest.mark.gpu

from gpu_util import METHODS, compare_bulk, compare_states, min_image, three_way  # noqa: E402


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


def test_philox_three_way_with_curand(dr, oracle, torch_, tmp_path):
    """SURVEY.md 8c pin: the kernels' generator, the oracle's and cuRAND's own device function (curand_philox4x32_x.h,
    compiled here into a test-only library) give the same words for the same (key, counter)."""
    import ctypes
    import os
    import shutil
    import subprocess
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    assert os.path.exists(nvcc), "nvcc is part of the image"
    so = str(tmp_path / "curand_check.so")
    src = os.path.join(os.path.dirname(os.path.abspath(__file__)), "curand_check.cu")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-shared", "-Xcompiler", "-fPIC", "-o", so, src], check=True)
    lib = ctypes.CDLL(so)
    lib.curand_philox_blocks.argtypes = [ctypes.c_uint64, ctypes.c_void_p, ctypes.c_uint32, ctypes.c_void_p]
    rng = np.random.default_rng(5)
    ctr = rng.integers(0, 2**32, size=(4096, 4), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0
    ctr[1] = 0xFFFFFFFF
    dctr = torch_.from_numpy(ctr.view(np.int32)).cuda()
    for seed in (0, 0xFFFFFFFFFFFFFFFF, 0x0123456789ABCDEF):
        ours = dr.philox_blocks(seed, dctr).cpu().numpy().view(np.uint32)
        theirs = torch_.empty_like(dctr)
        assert lib.curand_philox_blocks(seed, dctr.data_ptr(), len(ctr), theirs.data_ptr()) == 0
        theirs = theirs.cpu().numpy().view(np.uint32)
        assert np.array_equal(ours, theirs)
        for k in range(0, len(ctr), 97):
            assert (theirs[k] == oracle.philox([seed & 0xFFFFFFFF, seed >> 32], ctr[k])).all()


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
    # fp32 Moeller-Trumbore on both sides: its error scales with the scene extent, not with t (Q8, measured fp32-vs-fp64 numbers there)
    assert np.all(np.abs(t[hit] - ot[hit]) <= 1e-5 * np.maximum(np.abs(ot[hit]), 0.25 * diag))
    assert np.all(t[(~mism) & (otri < 0)] == -1.0)
    info = gsc.info()
    assert info["n_tris"] == desc.n_tris and info["n_nodes"] >= 1 and info["smem_nodes"] == 0


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


def _tri_soup(n, seed):
    rng = np.random.default_rng(seed)
    c = rng.uniform(0, 4, size=(n, 1, 3))
    v = (c + rng.uniform(-0.4, 0.4, size=(n, 3, 3))).astype(np.float32)
    return v


def test_tie_rule_coincident_triangles(dr, oracle, torch_):
    """Q8: equal t -> smaller triangle index.  Every triangle of a soup exists twice (ids i and a shuffled partner): the
    two copies give bit-identical t on either side, so the winner is decided by the tie rule alone, and the oracle's
    brute force names it."""
    n = 600
    v = _tri_soup(n, 1)
    perm = np.random.default_rng(2).permutation(n)
    verts = np.concatenate([v, v[perm]]).reshape(-1, 3)                 # ids n + j duplicate id perm[j]
    idx = np.arange(6 * n, dtype=np.uint32).reshape(-1, 3)
    desc = S.SceneDesc(verts, idx, np.zeros(2 * n, np.uint32), np.stack([S.material(S.MAT_LAMBERT, (0.5,) * 3)]), max_path_len=2)
    o, d = S.seeded_rays(desc, 40000, 3)
    t, prim = dr.Scene(desc).trace_rays(torch_.from_numpy(o).cuda(), torch_.from_numpy(d).cuda())
    t, prim = t.cpu().numpy(), prim.cpu().numpy()
    ot, otri = oracle.Scene(desc, oracle.F32).trace(o, d, brute=True)
    assert (otri[otri >= 0] < n).all()                                  # the oracle follows the rule
    hit = otri >= 0
    assert hit.sum() > 5000
    assert (prim[hit] < n).all()                                        # never the duplicate with the larger id
    mism = prim != otri
    assert mism.mean() < 1e-4, mism.sum()
    ok = ~mism & hit
    assert np.all(np.abs(t[ok] - ot[ok]) <= 1e-5 * np.maximum(np.abs(ot[ok]), 1.0))     # scene extent 4


def test_tie_rule_coplanar_box_on_floor(dr, oracle, torch_):
    """A box standing on the floor: its bottom face is coplanar with the floor (the configuration commit 6a75dbf took
    out of ggx_room).  Different triangles in one plane give t that differ by rounding, so either may win; what must
    hold: same t as the oracle to 1e-5, and where the triangle differs both are faces of that plane."""
    mesh = S._Mesh()
    mesh.quad((0, 0, 0), (0, 0, 4), (4, 0, 4), (4, 0, 0), 0, div=2)     # floor, 8 triangles (ids 0-7)
    S._box_faces(mesh, (2.0, 0.5, 2.0), (0.75, 0.5, 0.75), np.eye(3), 0)  # ids 8-19; face k = ids 8 + 2k, 9 + 2k; k = 3 is -y
    v, i, m = mesh.finish()
    desc = S.SceneDesc(v, i, m, np.stack([S.material(S.MAT_LAMBERT, (0.5,) * 3)]), max_path_len=2)
    rng = np.random.default_rng(4)
    n = 30000
    o = np.stack([rng.uniform(0.5, 3.5, n), rng.uniform(-3, -0.5, n), rng.uniform(0.5, 3.5, n)], 1).astype(np.float32)   # from below
    tgt = np.stack([rng.uniform(1.3, 2.7, n), np.zeros(n), rng.uniform(1.3, 2.7, n)], 1)
    d = tgt - o
    d = (d / np.linalg.norm(d, axis=1, keepdims=True)).astype(np.float32)
    t, prim = dr.Scene(desc).trace_rays(torch_.from_numpy(o).cuda(), torch_.from_numpy(d).cuda())
    t, prim = t.cpu().numpy(), prim.cpu().numpy()
    ot, otri = oracle.Scene(desc, oracle.F32).trace(o, d, brute=True)
    plane = lambda a: (a < 8) | (a == 14) | (a == 15)
    assert plane(otri).all() and plane(prim).all()
    assert np.all(np.abs(t - ot) <= 1e-5 * np.abs(ot))
    both = np.isin(otri, [14, 15]).mean()
    assert 0.05 < both < 0.95                                           # both outcomes occur: the tie path is exercised


# ---- a3, a5, a6: target evaluation --------------------------------------------------------------------------------
def _nee(desc):
    import copy
    d = copy.copy(desc)
    d.nee = True
    d.name = desc.name + "_nee"
    return d


EVAL_SCENES = {"furnace": S.furnace, "cornell": lambda: S.cornell(width=64, height=64), "mini_machines": S.mini_machines,
               "ggx_room": S.ggx_room, "closed_furnace": S.closed_furnace, "mixture3": S.mixture3,
               # next-event estimation + MIS (Q21): four coordinates per vertex, shadow rays, position-dependent score
               "cornell_nee": lambda: _nee(S.cornell(width=64, height=64)), "mini_machines_nee": lambda: _nee(S.mini_machines()),
               "ggx_room_nee": lambda: _nee(S.ggx_room()), "closed_furnace_nee": lambda: _nee(S.closed_furnace())}


@pytest.mark.parametrize("scene", list(EVAL_SCENES))
def test_eval_matches_oracle(dr, oracle, torch_, scene):
    desc = EVAL_SCENES[scene]()
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
    stddev = 5e-3
    relp = np.abs(g["p"] - e["p"]) / np.maximum(e["p"], 1e-8)
    relf = (np.abs(g["f"] - e["f"]) / np.maximum(np.abs(e["f"]), 1e-8)).max(1)
    badg = (np.abs(g["g"] - e["g"]) > 1e-4 * np.abs(e["g"]) + 2e-4 / stddev).any(1)
    if scene.endswith("_nee"):
        # a connection that grazes the emitter (cos_l -> 0) or is very short divides by a cancelled quantity: fp32 on either
        # side then carries a relative error far above its usual 1e-7.  Every state whose values differ is judged against the
        # fp64 oracle (gpu_util.three_way): ill-conditioned or on a decision boundary of the fp64 path -> counted; else a defect.
        idx = np.flatnonzero(ok & ((relp > 1e-4) | (relf > 1e-4) | badg))
        if len(idx):
            ill, other, e_gpu, e_orc, sens = three_way(oracle.Scene(desc, oracle.F64), dict(g, x=x), dict(e, x=x.astype(np.float64)), idx, stddev)
            defect = ~(ill | other)
            print(f"{scene}: {int(div.sum())} discrete, {int(ill.sum())} ill-conditioned, {int(other.sum())} on an fp64 decision boundary")
            assert not defect.any(), (idx[defect][:8], e_gpu[defect][:8], e_orc[defect][:8], sens[defect][:8])
        assert div.sum() + len(idx) < 1e-3 * n, (div.sum(), len(idx))
        ok[idx] = False
    assert relp[ok].max() <= 1e-4, relp[ok].max()
    assert relf[ok].max() <= 1e-4
    assert not badg[ok].any(), (int(badg[ok].sum()), float(np.abs(g["g"][ok] - e["g"][ok]).max()))
    if scene in ("mini_machines", "ggx_room") or scene.endswith("_nee"):
        assert (np.abs(e["g"][ok]).max(1) > 0).sum() > 20                       # the score path is exercised
    if scene.endswith("_nee"):
        assert (e["p"] > 0).mean() > 0.2 and (e["nrays"] > desc.max_path_len).any()   # connections are live, shadow rays counted
    # without the score the value outputs are identical
    g2 = gsc.eval_states(torch_.from_numpy(x).cuda(), want_score=False)
    assert np.allclose(g2["p"].cpu().numpy(), g["p"], rtol=1e-6, atol=0) and (g2["sig"].cpu().numpy() == g["sig"]).all()


def test_furnace_states_hit_the_closed_form_exactly(dr, oracle, torch_):
    desc = S.furnace()
    gsc = dr.Scene(desc)
    x = S.seeded_states(100000, desc.dim, 9)
    g = gsc.eval_states(torch_.from_numpy(x).cuda(), want_score=True)
    f, nr = g["f"].cpu().numpy(), g["nrays"].cpu().numpy()
    # The fp32 Moeller-Trumbore test of Q8 is not watertight: about one ray in 1e5 slips between two facets of the
    # sphere (u < 0 on one side of the shared edge, u + v > 1 on the other) and is then trapped inside -- in the
    # oracle's fp32 evaluation as well (state 61404 of this set).  Counted, at most 3; every other state is exact.
    e = oracle.Scene(desc, oracle.F32).eval(x, False)
    leak = ~(((f == 0.5) | (f == 1.0)).all(1))
    leak_o = ~(((e["f"] == 0.5) | (e["f"] == 1.0)).all(1))
    assert leak.sum() <= 3 and leak_o.sum() <= 3, (leak.sum(), leak_o.sum())
    both = ~leak & ~leak_o
    assert np.array_equal(f[both].astype(np.float64), e["f"][both]) and np.array_equal(nr[both], e["nrays"][both])
    f, nr, x = f[~leak], nr[~leak], x[~leak]
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
    _teacher_forced(dr, oracle, torch_, method, case)


CASES_NEE = [("cornell_nee", lambda: _nee(S.cornell(width=64, height=64, max_path_len=5)), 6000),
             ("mini_machines_nee", lambda: _nee(S.mini_machines()), 5000), ("ggx_room_nee", lambda: _nee(S.ggx_room()), 3001)]


@pytest.mark.parametrize("method", METHODS + ["path_tracing"])
@pytest.mark.parametrize("case", CASES_NEE, ids=[c[0] for c in CASES_NEE])
def test_teacher_forced_parity_with_nee(dr, oracle, torch_, method, case):
    """every sampler on scenes with next-event estimation + MIS, same protocol."""
    _teacher_forced(dr, oracle, torch_, method, case)


def test_an_emitter_without_area_is_never_sampled_on_the_gpu(dr, oracle, torch_):
    """DESIGN.md Q21: zero-area emitters are not on the emitter list (the oracle's pin: test_oracle_nee.py).  Appending one
    changes no evaluation, bit for bit; when it is the only emitter the scene is lit by the environment alone, no vertex
    makes a connection, and the evaluation matches the oracle's like any other."""
    import copy
    from test_oracle_nee import degenerate_emitter_appended
    base = _nee(S.cornell(width=32, height=32, max_path_len=4))
    plus = degenerate_emitter_appended(base)
    x = S.seeded_states(4000, base.dim, 21)
    x[:2000, 6::4] = np.float32(1.0 - 2.0 ** -24)
    xg = torch_.from_numpy(x).cuda()
    a, b = dr.Scene(base).eval_states(xg, True), dr.Scene(plus).eval_states(xg, True)
    for k in ("f", "p", "pix", "nrays", "sig", "g"):
        assert torch_.equal(a[k], b[k]), k
    assert int((a["p"][:2000] > 0).sum()) > 200
    dark = copy.copy(plus)
    dark.tri_material = plus.tri_material.copy()
    dark.tri_material[:-1][plus.tri_material[:-1] == plus.tri_material[-1]] = 0
    dark.env_radiance = (1.0, 0.5, 0.25)
    g = dr.Scene(dark).eval_states(xg, True)
    o = oracle.Scene(dark, oracle.F32).eval(x.astype(np.float64), True)
    gf, gp, gg = g["f"].cpu().numpy(), g["p"].cpu().numpy(), g["g"].cpu().numpy()
    assert np.isfinite(gf).all() and np.isfinite(gg).all() and not o["nonfinite"].any()
    same = g["sig"].cpu().numpy().view(np.uint32) == o["sig"]
    assert same.mean() > 0.999 and (gp[same] > 0).mean() > 0.3
    assert np.array_equal(g["pix"].cpu().numpy()[same], o["pix"][same])
    assert np.allclose(gf[same], o["f"][same], rtol=1e-4, atol=1e-6) and np.allclose(gp[same], o["p"][same], rtol=1e-4, atol=1e-6)
    assert not gg.reshape(len(x), -1, 4)[:, :, 2:].any()     # no connection anywhere: the emitter coordinates carry no score


# ---- Q18: non-finite f or score -> zero-contribution state, counted -------------------------------------------------------
def test_q18_overflowing_f_is_zeroed_on_the_same_states(dr, oracle, torch_):
    """DESIGN.md Q18.  The oracle's branch is pinned by fp64 in test_oracle_q18.py; here the kernels
    (finish_path, k_grad) against it on the closed box with albedo 2 and a 1e38 emitter: the same states are zeroed, with and
    without the score, and the chain counters agree."""
    from test_oracle_q18 import overflow_box
    desc = overflow_box()
    gsc, osc = dr.Scene(desc), oracle.Scene(desc, oracle.F32)
    x = S.seeded_states(4000, desc.dim, 31)
    for want_score in (False, True):
        g = gsc.eval_states(torch_.from_numpy(x).cuda(), want_score)
        o = osc.eval(x.astype(np.float64), want_score)
        same = g["sig"].cpu().numpy().view(np.uint32) == o["sig"]
        assert same.mean() > 0.999
        gf, gp = g["f"].cpu().numpy(), g["p"].cpu().numpy()
        flagged = o["nonfinite"].astype(bool)
        assert flagged[same].sum() > 500
        assert not gf[same & flagged].any() and not gp[same & flagged].any()               # zeroed where the oracle zeroes
        keep = same & ~flagged
        assert np.array_equal(gp[keep] > 0, o["p"][keep] > 0) and (gp[keep] > 0).sum() > 300  # and nowhere else
        assert np.allclose(gf[keep], o["f"][keep], rtol=1e-4) and np.isfinite(gf).all()
        if want_score:
            gg = g["g"].cpu().numpy()
            assert not gg[same & flagged].any() and np.isfinite(gg).all()
    # counters and one step of plain Metropolis with fresh uniform proposals: same decisions
    N = 3000
    kw = dict(seed=5, large_step_prob=1.0)
    for method in ("metropolis", "mala"):
        gch, och = dr.Chains(gsc, method, N, **kw), oracle.Chains(osc, method, N, **kw)
        gch.init(1)
        och.init(1)
        gst, ost = gch.stats(), och.stats()
        assert gst["nonfinite"] == ost["nonfinite"] > 500
        assert np.isclose(gst["p_lambda"], ost["p_lambda"], rtol=2e-6)
        gch.step(1)
        och.step(1)
        gs, os_ = gch.download(), och.state()
        assert gch.stats()["nonfinite"] == och.stats()["nonfinite"] > ost["nonfinite"]
        assert (gs["x"].astype(np.float64) == os_["x"]).all()                                # large steps only: the states are exact uniforms
        assert np.array_equal(gch.last_step()[0].astype(bool), och.last()[0].astype(bool))
        assert np.allclose(gs["p"], os_["p"], rtol=1e-5)
        assert np.isfinite(gch.accum.cpu().numpy()).all()


def test_q18_overflowing_score_is_zeroed_like_the_oracle(dr, oracle, torch_):
    """Only the score overflows (GGX room, 1e38 emitters).  The oracle differentiates forwards, k_grad backwards, so fp32 leaves
    its range at slightly different points of the two computations: the states are compared by what fp64 says about them.  Both
    sides zero every state whose |grad p| exceeds FLT_MAX by a factor 16 and none below FLT_MAX / 16; in between either may."""
    from test_oracle_q18 import FLT_MAX, bright_ggx_room
    desc = bright_ggx_room()
    gsc, o32, o64 = dr.Scene(desc), oracle.Scene(desc, oracle.F32), oracle.Scene(desc, oracle.F64)
    x = S.seeded_states(60000, desc.dim, 32)
    g = gsc.eval_states(torch_.from_numpy(x).cuda(), True)
    a, b = o32.eval(x.astype(np.float64), True), o64.eval(x.astype(np.float64), True)
    gf, gp, gg = g["f"].cpu().numpy(), g["p"].cpu().numpy(), g["g"].cpu().numpy()
    assert np.isfinite(gf).all() and np.isfinite(gg).all()
    same = (g["sig"].cpu().numpy().view(np.uint32) == b["sig"]) & (a["sig"] == b["sig"])
    grad_p = np.abs(b["g"]).max(1) * (b["p"] + 1e-8)
    lit = same & (b["p"] > 0)
    g_flag, o_flag = lit & (gp == 0), lit & a["nonfinite"].astype(bool)
    must, must_not = lit & (grad_p > 16 * FLT_MAX), lit & (grad_p < FLT_MAX / 16)
    print(f"Q18 score overflow: gpu zeroed {g_flag.sum()}, oracle zeroed {o_flag.sum()}, both {(g_flag & o_flag).sum()}, "
          f"|grad p| > 16 FLT_MAX: {must.sum()}, in between: {(lit & ~must & ~must_not).sum()}")
    assert g_flag[must].all() and o_flag[must].all() and not g_flag[must_not].any() and not o_flag[must_not].any()
    assert must_not.sum() > 1000 and (g_flag | o_flag).sum() >= 10
    assert not gf[g_flag].any() and not gg[g_flag].any()
    keep = lit & ~g_flag & ~o_flag
    assert np.allclose(gf[keep], a["f"][keep], rtol=1e-4)


EXTRA = [("path_tracing", {}), ("metropolis_restore", dict(rao_blackwell=True)), ("mala_restore", dict(rao_blackwell=True)),
         ("diffusion_restore", dict(rao_blackwell=True))]


@pytest.mark.parametrize("variant", EXTRA, ids=[m + ("-rao_blackwell" if kw else "") for m, kw in EXTRA])
@pytest.mark.parametrize("case", CASES[:2] + CASES[3:], ids=[c[0] for c in CASES[:2] + CASES[3:]])
def test_teacher_forced_parity_pt_and_rao_blackwell(dr, oracle, torch_, variant, case):
    """SURVEY 8f rows f2 (path tracing as a sixth method) and f3 (Rao-Blackwellised Accumulate), same protocol."""
    _teacher_forced(dr, oracle, torch_, variant[0], case, **variant[1])


def _rho(grid, seed):
    w = np.random.default_rng(seed).uniform(0.2, 3.0, size=(grid, grid))
    return (w / w.sum()).astype(np.float32)


F4 = [("diffusion_restore", dict(a_mode=1)), ("diffusion_restore", dict(rho=_rho(4, 1))), ("metropolis_restore", dict(rho=_rho(7, 2))),
      ("mala_restore", dict(rho=_rho(3, 3), rao_blackwell=True)), ("diffusion_restore", dict(a_mode=1, rho=_rho(16, 4))), ("metropolis", dict(rho=_rho(5, 5)))]


@pytest.mark.parametrize("variant", F4, ids=[f"{m}-{'-'.join(sorted(kw))}" for m, kw in F4])
@pytest.mark.parametrize("case", [CASES[1], CASES[3], CASES_NEE[1]], ids=["mini_machines", "mixture3", "mini_machines_nee"])
def test_teacher_forced_parity_f4(dr, oracle, torch_, variant, case):
    """regeneration from a density rho on film tiles with the killing rate (rho / rho_lambda) kappa0 / p_hat
    (PAPER.md L443-L445), and a second antisymmetric pattern of the Langevin drift (L567, L822); same protocol: bit-exact
    regenerated states, decisions, queue, tourCount, buffer against the oracle."""
    _teacher_forced(dr, oracle, torch_, variant[0], case, **variant[1])


def test_packed_frame_equals_plain_resolve(dr, torch_):
    """a sharded frame is dr_pack_frame -> ONE all-reduce -> dr_resolve_image_packed.  With one shard the
    all-reduce is the identity: the packed path must give the image of dr_resolve_image, the tail must hold the counters as
    16-bit limbs, and two shards' buffers added together must resolve to the image of the unsharded run."""
    from paper_2605_08916_b200 import sharding
    desc = S.mini_machines()
    gsc = dr.Scene(desc)
    for method in ("diffusion_restore", "metropolis"):
        ch = dr.Chains(gsc, method, 3000, seed=6, p_lambda_override=0.05)
        ch.init(0)
        ch.step(5)
        want = ch.resolve()[0].clone()
        buf = ch.pack_frame()
        st = ch.stats()
        tail = buf[-8:].cpu().numpy()
        assert list(tail[:4]) == sharding.limbs(st["tours"]) and list(tail[4:]) == sharding.limbs(st["mutations"])
        assert torch_.equal(buf[:-8].view(-1, 4), ch.accum)
        got = sharding.resolve_frame(ch)
        assert torch_.equal(got, want)
    full = dr.Chains(gsc, "diffusion_restore", 2000, seed=4, p_lambda_override=0.05)
    full.init(0); full.step(4)
    want = full.resolve()[0].clone()
    shards = [dr.Chains(gsc, "diffusion_restore", 1000, seed=4, p_lambda_override=0.05, chain_offset=off) for off in (0, 1000)]
    total = None
    for ch in shards:
        ch.init(0); ch.step(4)
        b = ch.pack_frame().clone()
        total = b if total is None else total + b              # what the all-reduce(sum) does
    got = shards[0].resolve_packed(total)
    assert torch_.allclose(got, want, rtol=1e-4, atol=1e-7)


def test_sharded_chains_against_the_oracle(dr, oracle, torch_):
    """a shard (global chain ids 1000 .. 1999 of a 2000-chain run) against the oracle's shard with the same
    chain_offset, teacher-forced like everything else: the RNG streams are keyed by global chain id on both sides."""
    _teacher_forced(dr, oracle, torch_, "diffusion_restore", ("mini_machines", S.mini_machines, 1000), chain_offset=1000, p_lambda_override=0.05)
    _teacher_forced(dr, oracle, torch_, "metropolis", ("ggx_room", S.ggx_room, 999), chain_offset=12345)


def test_scene_change_reinitialises_everything(dr, oracle, torch_):
    """when the scene changes (camera, geometry) all accumulated samples are invalid and the whole stateBuffer
    is initialised again (Alg. 1).  As a call sequence: new dr_scene, dr_chains_create on the SAME caller-owned memory,
    dr_chains_init(frame_index): states are the Philox uniforms of that frame's epoch, buffer and counters start from zero,
    and the result equals a run that never saw the first scene."""
    d1, d2 = S.mini_machines(), S.mini_machines(seed=8)                          # "the geometry changed"
    N = 4096
    a = dr.Chains(dr.Scene(d1), "diffusion_restore", N, seed=9)
    a.init(0)
    a.step(5)
    a.resolve()
    assert a.stats()["tours"] > 0 and float(a.accum.abs().sum()) > 0
    sc2 = dr.Scene(d2)
    b = dr.Chains(sc2, "diffusion_restore", N, seed=9)
    b.state, b.accum = a.state, a.accum                                         # reuse the memory of the old ensemble
    import ctypes as C
    h = C.c_void_p()
    dr.binding._check(dr.lib.dr_chains_create(sc2.h, C.byref(b.cfg), C.c_void_p(a.state.data_ptr()), a.state.numel(),
                                              C.c_void_p(a.accum.data_ptr()), C.byref(h)))
    dr.lib.dr_chains_destroy(b.h)
    b.h = h
    b.init(7)                                                                   # frame 7: a new epoch of every stream
    fresh = dr.Chains(dr.Scene(d2), "diffusion_restore", N, seed=9)
    fresh.init(7)
    sb, sf = b.download(), fresh.download()
    for k in sb:
        assert np.array_equal(sb[k].view(np.uint8), sf[k].view(np.uint8)), k
    stb, stf = b.stats(), fresh.stats()
    assert stb["mutations"] == stf["mutations"] == N and stb["tours"] == stf["tours"] and stb["iteration"] == 0
    assert torch_.allclose(b.accum, fresh.accum, rtol=1e-5, atol=1e-9)             # float atomics: order of the addends
    och = oracle.Chains(oracle.Scene(d2, oracle.F32), "diffusion_restore", N, seed=9)
    och.init(7)
    assert (sb["x"].astype(np.float64) == och.state()["x"]).all()                # the epoch-7 uniforms, bit-exact
    b.step(3); fresh.step(3)
    assert np.array_equal(b.download()["x"], fresh.download()["x"])


def _teacher_forced(dr, oracle, torch_, method, case, **kw):
    name, make, N = case
    desc = make()
    seed = 0 if name == "furnace" else 3
    gsc = dr.Scene(desc)
    osc = oracle.Scene(desc, oracle.F32)
    gch = dr.Chains(gsc, method, N, seed=seed, **kw)
    och = oracle.Chains(osc, method, N, seed=seed, **kw)
    stddev = float(gch.cfg.stddev)
    # --- init (Alg. 1) from the same seed: states are exact uniforms on both sides
    gch.init(2)
    och.init(2)
    gs, os_ = gch.download(), och.state()
    assert (gs["x"].astype(np.float64) == os_["x"]).all()                       # RNG streams: bit-exact
    gst, ost = gch.stats(), och.stats()
    assert np.isclose(gst["p_lambda"], ost["p_lambda"], rtol=2e-6) and np.isclose(gst["kappa0"], ost["kappa0"], rtol=2e-6)
    assert gst["mutations"] == ost["mutations"] == N
    g_last, o_last = gch.last_step(), och.last()
    osc64 = oracle.Scene(desc, oracle.F64) if getattr(desc, "nee", False) else None   # judges value differences three ways (gpu_util.three_way)
    div, rep = compare_states(gs, os_, g_last, o_last, stddev, osc64=osc64)
    assert div.mean() < 1e-3, rep
    nr_g, nr_o = gsc.eval_states(torch_.from_numpy(gs["x"]).cuda(), False)["nrays"].cpu().numpy(), osc.eval(os_["x"], False)["nrays"]
    assert gst["rays"] == int(nr_g.sum()) and ost["rays"] == int(nr_o.sum()) and (nr_g[~div] == nr_o[~div]).all()   # closest-hit queries: counted exactly
    compare_bulk(gch, och, gs, os_, g_last, o_last, div, gst["tours"], ost["tours"])
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
        g_last, o_last = gch.last_step(), och.last()
        div, rep = compare_states(gs, os_, g_last, o_last, stddev, osc64=osc64)
        worst = max(worst, rep["frac"])
        assert div.mean() < 1e-3, (method, name, burst, rep)
        compare_bulk(gch, och, gs, os_, g_last, o_last, div, gch.stats()["tours"] - t0g, och.stats()["tours"] - t0o)
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
    assert ch.stats()["status"] == dr.DR_OK
    img, _ = ch.resolve()
    st = ch.stats()
    assert st["status"] == dr.DR_WARN_NO_TOURS and st["no_tour_resolves"] == 1 and float(img.abs().max()) == 0.0
    # wrong method in dr_step, invalid configs
    with pytest.raises(dr.DrError):
        dr.binding._check(dr.lib.dr_step(ch.h, 0, 1, None))
    for bad in (dict(stddev=0.0), dict(dt=-1.0), dict(m=0.0), dict(large_step_prob=1.5), dict(stddev=float("nan")), dict(a_mode=2),
                dict(rho=np.full((3, 3), 0.2, np.float32)), dict(rho=np.array([[0.5, 0.5], [0.0, 0.0]], np.float32))):
        with pytest.raises(dr.DrError):
            dr.Chains(gsc, "metropolis", 16, **bad)
    with pytest.raises(dr.DrError):          # path tracing has no regeneration density (include/dr.h rho_grid)
        dr.Chains(gsc, "path_tracing", 16, rho=np.full((2, 2), 0.25, np.float32))
    with pytest.raises(ValueError):          # not G x G values: refused before dr_chains_create reads past the array
        dr.Chains(gsc, "metropolis_restore", 16, rho=np.full(6, 1.0 / 6.0, np.float32))
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
_SCENES = {}


def _full_scene(dr, oracle, name, make):
    """One scene build per module: the 539 k-triangle BVHs take seconds on either side."""
    if name not in _SCENES:
        desc = make()
        _SCENES[name] = (desc, dr.Scene(desc), oracle.Scene(desc, oracle.F32))
    return _SCENES[name]


@pytest.mark.parametrize("case", FULL, ids=[c[0] for c in FULL])
def test_full_size_configs(dr, oracle, torch_, case):
    """configs[1..3] at their full chain counts: bit-exact RNG / queue / counters, and sampled states re-evaluated
    one by one by the oracle (the stored (f/p_hat, p, pixel, score, signature) of a chain is the evaluation of its x)."""
    name, make, N, seed = case
    desc, gsc, osc = _full_scene(dr, oracle, name, make)
    method = "diffusion_restore"
    gch = dr.Chains(gsc, method, N, seed=seed)
    gch.init(0)
    rng = np.random.default_rng(7)
    ids = np.unique(np.concatenate([rng.integers(0, N, 40000), [0, 1, 255, 256, N - 257, N - 1]]))
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
        # fp32 rounding continues from the neighbour on one side.  Counted; < 1e-3 of the paths (Q15).
        assert (~ok).mean() < 1e-3, (~ok).sum()
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
        assert (q == np.flatnonzero(gs["killed"])).all()                        # regeneration queue: ascending killed ids
        kills += len(q)
        assert st["tours"] == kills and st["kills_last_step"] == len(q)
        check_sample(gs)


WHOLE = [("cornell", S.cornell, 65536, 2, m) for m in METHODS] + [("caustic", S.caustic, 262144, 3, m) for m in METHODS] + \
        [("machines", S.machines, 589824, 4, m) for m in ("metropolis_restore", "diffusion_restore")] + \
        [("machines_nee", lambda: _nee(S.machines()), 131072, 4, m) for m in ("mala", "diffusion_restore")]   # Q21 at the scene's full geometry


@pytest.mark.parametrize("case", WHOLE, ids=[f"{c[0]}-{c[4]}" for c in WHOLE])
def test_whole_ensemble_teacher_forced_step(dr, oracle, torch_, case):
    """Every chain of the full-size ensemble, every sampler: the oracle runs init + 2 iterations, its state is uploaded,
    both sides take one step (through k_wave<GRAD> for the Langevin-based samplers, k_wave<false> for the others), and
    states, decisions, queue, tourCount and accumulation buffer are compared with the oracle's (Q15)."""
    name, make, N, seed, method = case
    desc, gsc, osc = _full_scene(dr, oracle, name, make)
    och = oracle.Chains(osc, method, N, seed=seed)
    och.init(0)
    # Teacher forcing covers the run's constants too: kappa0 = p_lambda / (m dt) comes from the bootstrap over the init states, and
    # the handful of init states that diverge or are ill-conditioned move the GPU's own p_lambda by 3e-5 .. 6e-5 relative, which
    # then sits in EVERY weight of the step (measured with next-event estimation: dw = dp + 3.08e-5 on all chains).  The bootstrap itself is compared below
    # and, at 2e-6, in _teacher_forced; the step under test takes the oracle's p_lambda like it takes the oracle's state.
    own = dr.Chains(gsc, method, N, seed=seed)
    own.init(0)
    p_lambda = och.stats()["p_lambda"]
    assert np.isclose(own.stats()["p_lambda"], p_lambda, rtol=1e-4)   # a mean over every init state, the few diverged ones included (Cornell box: 6e-5)
    del own
    gch = dr.Chains(gsc, method, N, seed=seed, p_lambda_override=p_lambda)
    gch.init(0)
    assert np.isclose(gch.stats()["kappa0"], och.stats()["kappa0"], rtol=1e-6)
    och.step(2)
    gch.upload(och.state(), 2)
    gch.accum.zero_()
    och.zero_accum()
    t0g, t0o = gch.stats()["tours"], och.stats()["tours"]
    gch.step(1)
    och.step(1)
    gs, os_ = gch.download(), och.state()
    g_last, o_last = gch.last_step(), och.last()
    osc64 = oracle.Scene(desc, oracle.F64) if name.endswith("_nee") else None
    div, rep = compare_states(gs, os_, g_last, o_last, float(gch.cfg.stddev), osc64=osc64)
    print(f"{name}/{method}: {rep}")
    # < 0.1 % of the chains per step take other discrete decisions (B: north_star), every case.  With next-event estimation the
    # states whose values differ are judged against fp64 one by one (gpu_util.three_way: a defect fails inside compare_states);
    # the ill-conditioned ones and those on a decision boundary of the fp64 path are counted apart, each under 0.1 % too.
    assert rep["discrete_frac"] < 1e-3 and rep["ill_frac"] < 1e-3 and rep["fp64_other_path"] < 1e-3 * N, rep
    compare_bulk(gch, och, gs, os_, g_last, o_last, div, gch.stats()["tours"] - t0g, och.stats()["tours"] - t0o)


# ---- the two forms of the evaluation (k_wave vs per-segment loop) -------------------------------------------------
def _same_eval(a, b):
    for k in ("f", "p", "pix", "nrays", "sig", "g"):
        if a[k] is None:
            assert b[k] is None
            continue
        x, y = a[k].cpu().numpy(), b[k].cpu().numpy()
        assert np.array_equal(x.view(np.uint32), y.view(np.uint32)), k


WAVE = [("mini_machines", S.mini_machines, 1 << 18), ("ggx_room", S.ggx_room, 1 << 18), ("mini_machines", S.mini_machines, 4999),
        ("ggx_room", S.ggx_room, 33), ("caustic", S.caustic, 262144), ("machines", S.machines, 589824)]


@pytest.mark.parametrize("score", [True, False], ids=["grad", "nograd"])
@pytest.mark.parametrize("case", WAVE, ids=[f"{c[0]}-{c[2]}" for c in WAVE])
def test_wave_kernel_equals_segment_loop(dr, oracle, torch_, case, score):
    """The same states evaluated by k_wave (one persistent kernel, dr_wave.cuh; both instantiations) and by the
    per-segment loop k_trace / k_shade: both run the same shade_vertex on the same closest hits, so f, p, pixel, rays per
    path, signature and score must be identical bit for bit -- anything else is a ray lost, duplicated or read before it
    was written.  Sizes from 33 states (most warps idle) to the bench configuration (machines, one state per pixel)."""
    name, make, n = case
    desc, gsc, _ = _full_scene(dr, oracle, name, make) if name in ("caustic", "machines") else (make(), None, None)
    gsc = gsc or dr.Scene(desc)
    x = torch_.from_numpy(S.seeded_states(n, desc.dim, 11)).cuda()
    a = gsc.eval_states(x, score, form=2)                                        # the block shape chosen by the size
    b = gsc.eval_states(x, score, form=1)
    assert int(a["nrays"].sum()) > n                                             # paths do bounce
    _same_eval(a, b)
    for form in (3, 4):                                                          # both block shapes (640 threads and two triangle
        c = gsc.eval_states(x, score, form=form)                                 # slots per lane; 768 and one), each a further
        _same_eval(a, c)                                                         # launch on fresh memory


def test_chains_run_identically_in_both_forms(dr, torch_):
    """dr_step through k_wave and through the loop: same states, flags and counters after 6 iterations, for a sampler
    of each kind (the queue memory is reused by successive evaluations: tags, not clearing, tell them apart)."""
    desc = S.mini_machines()
    gsc = dr.Scene(desc)
    for method in ("metropolis", "mala_restore", "diffusion_restore"):
        out = []
        for form in (2, 1, 4):
            ch = dr.Chains(gsc, method, 20000, seed=5)
            ch.set_eval_form(form)
            ch.init(1)
            ch.step(6)
            out.append((ch.download(), ch.stats()))
        (sa, ta) = out[0]
        for sb, tb in out[1:]:
            for k in sa:
                assert np.array_equal(sa[k].view(np.uint8), sb[k].view(np.uint8)), (method, k)
            assert ta["tours"] == tb["tours"] and ta["rays"] == tb["rays"] and ta["mh_accepts"] == tb["mh_accepts"]


def test_chains_with_nee_run_identically_in_both_block_shapes(dr, torch_):
    """Next-event estimation has no per-segment loop: the two block shapes of k_wave (640 threads with two triangle slots per lane
    and three shade warps, 768 with one and five) check each other, through the whole step of a gradient sampler -- shading with
    shadow rays, vertex records, the reverse sweep per vertex index, MH decision -- bit for bit after 5 iterations."""
    desc = S.mini_machines()
    desc.nee = True
    gsc = dr.Scene(desc)
    for method in ("mala", "diffusion_restore"):
        out = []
        for form in (3, 4):
            ch = dr.Chains(gsc, method, 30000, seed=6)
            ch.set_eval_form(form)
            ch.init(2)
            ch.step(5)
            out.append((ch.download(), ch.stats()))
        (sa, ta), (sb, tb) = out
        for k in sa:
            assert np.array_equal(sa[k].view(np.uint8), sb[k].view(np.uint8)), (method, k)
        assert ta["tours"] == tb["tours"] and ta["rays"] == tb["rays"] and ta["grad_states"] == tb["grad_states"] > 0


def test_profile_counts_every_kernel_launch(dr, torch_):
    """dr_profile_read: 8 launches per frame without, 8 + L with next-event estimation and a score (the reverse sweep is an init
    launch, one launch per vertex index and a finish launch); bench.py's gpu_launches is this count."""
    for nee, want in ((False, 8), (True, None)):
        desc = S.mini_machines()
        desc.nee = nee
        ch = dr.Chains(dr.Scene(desc), "diffusion_restore", 4096, seed=3)
        ch.init(0)
        ch.profile_enable(True)
        ch.step(3)
        ch.resolve()
        prof = ch.profile_read()
        ch.profile_enable(False)
        n = sum(v["launches"] for v in prof.values())
        per_step = 7 + (desc.max_path_len + 1 if nee else 1) - 1      # propose, raygen, k_wave, score, decide, scan, scatter
        assert n == 3 * per_step + 1, (nee, n, prof)                  # + one resolve


_STALL_SNIPPET = """
import sys, numpy as np, torch
sys.path.insert(0, {root!r})
import paper_2605_08916_b200 as dr
from dr_inputs import scenes as S
desc = S.mini_machines()
x = torch.from_numpy(S.seeded_states({n}, desc.dim, 11)).cuda()
e = dr.Scene(desc).eval_states(x, True, form=2)
torch.cuda.synchronize()
np.savez({out!r}, **{{k: v.cpu().numpy() for k, v in e.items()}})
"""


def test_wave_kernel_with_stalled_consumers(dr, torch_, tmp_path):
    """A build in which every trace warp sleeps 1 ms between claiming queue entries and reading them
    (-DDR_WAVE_STALL_NS=1000000): the results must not change.  The queue protocol of dr_wave.cuh does not rely on
    entries being read soon after they were claimed (round 1's ring did, and lost rays under such a stall)."""
    import os
    import subprocess
    import sys
    from paper_2605_08916_b200 import build
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    lib = build.build_variant("stall", ["-DDR_WAVE_STALL_NS=1000000"])
    n = 100003
    out = str(tmp_path / "stall.npz")
    subprocess.run([sys.executable, "-c", _STALL_SNIPPET.format(root=root, n=n, out=out)], check=True, env=dict(os.environ, DR_LIB=lib),
                   timeout=900)
    a = np.load(out)
    desc = S.mini_machines()
    b = dr.Scene(desc).eval_states(torch_.from_numpy(S.seeded_states(n, desc.dim, 11)).cuda(), True, form=1)
    for k in ("f", "p", "pix", "nrays", "sig", "g"):
        assert np.array_equal(a[k].view(np.uint32), b[k].cpu().numpy().view(np.uint32)), k


def test_small_run_under_the_checked_build(dr, tmp_path):
    """compute-sanitizer is closed on this pool (profiles/r02_sanitizer.md), so the queue protocol of k_wave is checked by
    a build with device-side assertions instead (-DDR_CHECKS=1, csrc/dr_wave.cuh): indices inside the queue, records owned by
    the state that the entry names, every segment of a state shaded exactly once and in order, the block's ring never
    overwriting an unread entry, every path finished.  Run on the stalled-consumer timing as well."""
    import os
    import subprocess
    import sys
    from paper_2605_08916_b200 import build
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for name, flags in (("checked", ["-DDR_CHECKS=1"]), ("checked_stall", ["-DDR_CHECKS=1", "-DDR_WAVE_STALL_NS=300000"])):
        lib = build.build_variant(name, flags)
        r = subprocess.run([sys.executable, os.path.join(root, "tests", "sanitizer", "small_run.py")], env=dict(os.environ, DR_LIB=lib),
                           capture_output=True, text=True, timeout=900)
        assert r.returncode == 0 and "small_run ok" in r.stdout, r.stdout + r.stderr


def test_bias_field_matches_oracle(dr, oracle, torch_):
    """Appendix C: the bias field L^* p_hat / p_hat of the Alg. 4 dynamics on the analytic target,
    dr_bias_field against the oracle's quadrature (both in double), at the paper's dt = 1e-5 and at a coarse one."""
    desc = S.mixture3()
    gsc, osc = dr.Scene(desc), oracle.Scene(desc, oracle.F64)
    for sigma, dt in ((0.5, 1e-5), (0.5, 1e-3), (2.0, 1e-4)):
        s, ct = sigma * np.sqrt(dt), 0.5 * sigma * sigma * dt
        g = gsc.bias_field(s, ct, dt, G=24, M=256).cpu().numpy()
        o = osc.bias_field(s, ct, dt, G=24, M=256)
        # single-precision mixture parameters on the device side, double arithmetic on both: agreement to rounding of the sums
        assert np.abs(g - o).max() <= 1e-6 * np.abs(o).max() + 1e-7 / dt * 1e-2, (sigma, dt, np.abs(g - o).max(), np.abs(o).max())
    with pytest.raises(dr.DrError):
        dr.Scene(S.furnace()).bias_field(0.01, 0.0, 1e-3)


_LOST_RAY_SNIPPET = """
import sys, torch
sys.path.insert(0, {root!r})
import paper_2605_08916_b200 as dr
from dr_inputs import scenes as S
ch = dr.Chains(dr.Scene(S.closed_furnace()), "metropolis_restore", 64, seed=1)
ch.init(0)
torch.cuda.synchronize()
try:
    ch.stats()
    print("no error")
except dr.DrError as e:
    print("DrError", e.status, ch.lib_stats_timeouts() if hasattr(ch, "lib_stats_timeouts") else "")
# the evaluation hook and the counting pass report the watchdog as well (no partial result returned as DR_OK)
desc = S.closed_furnace()
x = torch.from_numpy(S.seeded_states(64, desc.dim, 3)).cuda()
try:
    dr.Scene(desc).eval_states(x, False, form=2)
    print("eval: no error")
except dr.DrError as e:
    print("eval DrError", e.status)
"""


def test_a_lost_ray_ends_in_an_error_not_in_a_hang(dr, tmp_path):
    """'if a path is lost ... every warp spins forever.  There is no watchdog, so the GPU hangs.'  The queue cannot
    lose a ray any more, but the kernel does not rely on that to terminate: a build that drops one ray on purpose
    (-DDR_WAVE_LOSE_RAY=1, idle limit lowered to milliseconds) ends, and dr_chains_stats reports DR_ERR_CUDA."""
    import os
    import subprocess
    import sys
    from paper_2605_08916_b200 import build
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    lib = build.build_variant("lose_ray", ["-DDR_WAVE_LOSE_RAY=1", "-DDR_WAVE_IDLE_LIMIT=4096"])
    r = subprocess.run([sys.executable, "-c", _LOST_RAY_SNIPPET.format(root=root)], env=dict(os.environ, DR_LIB=lib), capture_output=True,
                       text=True, timeout=120)
    assert r.returncode == 0 and f"DrError {dr.DR_ERR_CUDA}" in r.stdout, r.stdout + r.stderr
    assert f"eval DrError {dr.DR_ERR_CUDA}" in r.stdout, r.stdout + r.stderr
