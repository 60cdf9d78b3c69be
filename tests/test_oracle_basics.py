"""Golden worked values for torus ops, rates and resolve (tests/golden/*.txt, each line cited)."""
import os

import numpy as np

from dr_inputs import scenes as S

G = os.path.join(os.path.dirname(__file__), "golden")


def rows(name):
    for line in open(os.path.join(G, name)):
        line = line.split("#")[0].strip()
        if line:
            yield line.split()


def uniform_scene():
    """Environment-only scene: f = p = 1 for every x (one far-away triangle behind the camera)."""
    v = np.array([[100, 100, -50], [101, 100, -50], [100, 101, -50]], dtype=np.float32)
    return S.SceneDesc(v, np.array([[0, 1, 2]], dtype=np.uint32), np.zeros(1, dtype=np.uint32),
                       np.stack([S.material(S.MAT_LAMBERT, (0.5, 0.5, 0.5))]), env_radiance=(1, 1, 1), cam_pos=(0, 0, 0),
                       cam_look=(0, 0, 1), width=4, height=4, max_path_len=2, name="uniform")


def test_torus_ops(oracle):
    for r in rows("torus_ops.txt"):
        if r[0] == "wrap":
            for prec in (oracle.F64, oracle.F32):
                assert oracle.wrap(float(r[1]), prec) == float(r[2])
        elif r[0] == "wrap_lt1":
            for prec in (oracle.F64, oracle.F32):
                w = oracle.wrap(float(r[1]), prec)
                assert 0.0 <= w < 1.0
        elif r[0] == "min_image":
            assert np.isclose(oracle.min_image(float(r[1])), float(r[2]), atol=1e-15)
    # properties
    rng = np.random.default_rng(0)
    for v in rng.uniform(-5, 5, size=200):
        w = oracle.wrap(v)
        assert 0 <= w < 1 and np.isclose(oracle.wrap(w + 3), w, atol=1e-12)
        dl = oracle.min_image(v)
        assert -0.5 <= dl < 0.5 and np.isclose((dl - v) % 1.0, 0, atol=1e-12) or np.isclose((dl - v) % 1.0, 1, atol=1e-12)


def test_rotate_convention(oracle):
    """Alg. 4: x += (s^2/2) g + c~ (g2, -g1) + s xi.  One Diffusion-Restore step on an analytic target:
    what is left of the move after removing drift and noise must be c~ (g2, -g1)  (golden: S:L190)."""
    r = next(x for x in rows("torus_ops.txt") if x[0] == "rotate")
    ct, v1, v2, e1, e2 = map(float, r[1:])
    assert (ct * v2, -ct * v1) == (e1, e2)          # the fixture itself states the convention
    sc = oracle.Scene(S.single_mode(0.15), oracle.F64)
    s, ctil = 1e-3, 7e-4
    ch = oracle.Chains(sc, "diffusion_restore", 64, stddev=s, c_tilde=ctil, seed=5, p_lambda_override=1.0)
    ch.init(0)
    st0 = ch.state()
    ch.step(1)
    st1 = ch.state()
    moved = 0
    for i in range(64):
        if st0["killed"][i]:
            continue
        w = oracle.stream_block(5, i, 1, 0, 1, 0)
        z = oracle.rng_transforms(int(w[0]), int(w[1]), oracle.F64)[2:]
        g = st0["g"][i]
        resid = np.array([oracle.min_image(st1["x"][i, k] - st0["x"][i, k] - 0.5 * s * s * g[k] - s * z[k]) for k in range(2)])
        assert np.allclose(resid, [ctil * g[1], -ctil * g[0]], atol=1e-13)
        assert np.dot(resid, g) == 0 or abs(np.dot(resid, g)) < 1e-12 * np.dot(g, g)   # rotate(v).v = 0
        moved += 1
    assert moved > 50


def test_rates_and_resolve(oracle):
    sc = oracle.Scene(uniform_scene(), oracle.F64)
    for r in rows("rates.txt"):
        if r[0] == "lambda":
            ch = oracle.Chains(sc, "diffusion_restore", 4, dt=float(r[1]), p_lambda_override=1.0)
            ch.init(0)
            assert np.isclose(ch.stats()["lambda"], float(r[2]), rtol=1e-12)
        elif r[0] == "kappa0":
            ch = oracle.Chains(sc, "diffusion_restore", 4, dt=float(r[3]), m=float(r[2]), p_lambda_override=float(r[1]))
            ch.init(0)
            assert np.isclose(ch.stats()["kappa0"], float(r[4]), rtol=1e-12)
        elif r[0] == "resolve":
            # kappa0 = 2 (p_lambda = 2, m = 1, lambda == 1 for Metropolis-Restore); force tours and buffer via a run:
            # resolve is linear, so check out = npix * kappa0 / tours * accum on whatever the run produced
            ch = oracle.Chains(sc, "metropolis_restore", 256, m=1.0, p_lambda_override=float(r[1]), seed=1)
            ch.init(0)
            ch.step(5)
            img, status = ch.resolve()
            st = ch.stats()
            assert status == 0 and np.isclose(st["kappa0"], float(r[1]))
            want = sc.npix * st["kappa0"] / st["tours"] * ch.accum()[:, :3]
            assert np.allclose(img.reshape(-1, 3), want, rtol=1e-14)
            # the fixture's arithmetic: kappa0 / tours * buffer
            assert float(r[1]) / float(r[2]) * float(r[3]) == float(r[4])


def test_kill_probability_law(oracle):
    """Race of Alg. 1: P(killed) = kappa / (lambda + kappa).  Uniform target, kappa0 = p_lambda/(m dt)
    => 1/(m+1) per event (golden); also a non-trivial ratio with kappa = 4 lambda."""
    sc = oracle.Scene(uniform_scene(), oracle.F64)
    (m_gold, p_gold), = [(float(r[1]), float(r[2])) for r in rows("rates.txt") if r[0] == "kill_prob_uniform"]
    assert m_gold == 64.0 and abs(p_gold - 1 / 65) < 1e-15
    for meth, m, want in [("diffusion_restore", m_gold, p_gold), ("metropolis_restore", m_gold, p_gold),
                          ("mala_restore", 0.25, 0.8), ("diffusion_restore", 1.0, 0.5)]:
        ch = oracle.Chains(sc, meth, 20000, m=m, seed=11)
        ch.init(0)
        ch.step(9)
        st = ch.stats()
        assert abs(st["p_lambda"] - (1 + 1e-8)) < 1e-12          # bootstrap on f = 1
        n = st["mutations"]
        assert n == 20000 * 10
        frac = st["tours"] / n
        assert abs(frac - want) < 5 * np.sqrt(want * (1 - want) / n), (meth, frac, want)


def test_killing_rate_is_kappa0_over_p_hat(oracle):
    """kappa = kappa0 / p_hat for uniform rho; golden row S:L279: kappa0 = 4, p = 2 -> kappa = 2.  On a constant
    target of luminance p with lambda = 1 (Metropolis-Restore) the race of Alg. 1 kills with probability
    kappa / (1 + kappa), which the tour count of a run shows."""
    (kappa0, p, kappa), = [tuple(float(v) for v in r[1:]) for r in rows("rates.txt") if r[0] == "kappa"]
    assert kappa0 / p == kappa
    desc = uniform_scene()
    desc.env_radiance = (p, p, p)
    sc = oracle.Scene(desc, oracle.F64)
    ch = oracle.Chains(sc, "metropolis_restore", 20000, m=1.0, p_lambda_override=kappa0, seed=13)   # kappa0 = p_lambda / (m dt), dt := 1
    ch.init(0)
    assert np.allclose(ch.state()["p"], p, rtol=1e-12)
    ch.step(9)
    st = ch.stats()
    assert np.isclose(st["kappa0"], kappa0, rtol=1e-12) and st["lambda"] == 1.0
    n, want = st["mutations"], kappa / (1.0 + kappa)
    assert abs(st["tours"] / n - want) < 5 * np.sqrt(want * (1 - want) / n), (st["tours"] / n, want)
    # and the sampled weights: E[dtau] = 1 / (lambda + kappa), so sum w / p_hat over the run = n / ((1 + kappa) p) within 5 s.e.
    acc = ch.accum()[:, 3].sum()
    assert abs(acc / n * (1.0 + kappa) * p - 1.0) < 5 / np.sqrt(n), acc


def test_uniform_target_resolves_to_one_and_tours_are_geometric(oracle):
    """f = p = 1: image == 1 in expectation, events per tour geometric with mean m + 1."""
    sc = oracle.Scene(uniform_scene(), oracle.F64)
    m = 8.0
    ch = oracle.Chains(sc, "diffusion_restore", 4000, m=m, seed=2)
    ch.init(0)
    lengths, cur, start = [], np.ones(4000, dtype=np.int64), np.zeros(4000, dtype=np.int64)
    for it in range(260):
        k = ch.state()["killed"].astype(bool)
        lengths += [l for l, s0 in zip(cur[k], start[k]) if s0 < 100]   # tours started early: none is censored
        cur[k] = 0
        start[k] = it + 1
        ch.step(1)
        cur += 1
    lengths = np.array(lengths)
    assert abs(lengths.mean() - (m + 1)) < 5 * np.sqrt(m * (m + 1) / len(lengths))
    # geometric law: P(len = k) = q (1-q)^(k-1), q = 1/(m+1)
    q = 1 / (m + 1)
    for k in (1, 2, 5):
        want = q * (1 - q) ** (k - 1)
        assert abs((lengths == k).mean() - want) < 5 * np.sqrt(want / len(lengths))
    img, _ = ch.resolve()
    st = ch.stats()
    # memoryless tours: E[accum]/E[tours] exact; MC error ~ 1/sqrt(tours)
    assert abs(img.mean() - 1.0) < 5 / np.sqrt(st["tours"])
    # plain MH on the same target: every f/p_hat = 1/(1+eps) -> image == p_lambda/(1+eps) == 1 exactly
    ch = oracle.Chains(sc, "metropolis", 512, seed=2)
    ch.init(0)
    ch.step(3)
    img, _ = ch.resolve()
    assert np.allclose(img.mean(), 1.0, rtol=1e-12)
    assert ch.stats()["mh_accepts"] == 512 * 3     # flat density: every proposal accepted


def test_resolve_without_tours_warns(oracle):
    sc = oracle.Scene(uniform_scene(), oracle.F64)
    ch = oracle.Chains(sc, "diffusion_restore", 1, m=1e9, seed=0)
    ch.init(0)
    img, status = ch.resolve()
    assert status == 1 and (img == 0).all()
