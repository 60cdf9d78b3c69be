"""Pins for the oracle's target evaluation: furnace closed form, material closed forms, score vs finite differences."""
import os

import numpy as np

from dr_inputs import scenes as S

G = os.path.join(os.path.dirname(__file__), "golden")
GOLD = {r.split()[0]: float(r.split()[1]) for r in open(os.path.join(G, "furnace.txt")) if r.strip() and not r.startswith("#")}


def test_white_furnace_closed_form(oracle):
    """BASELINE.json configs[0]; closed form derived in tests/golden/furnace.txt."""
    desc = S.furnace()
    sc = oracle.Scene(desc, oracle.F64)
    x = S.seeded_states(200000, desc.dim, 1)
    e = sc.eval(x, True)
    # every state's f is exactly its class value (Q12 (i))
    inside = e["nrays"] == 2
    assert ((e["nrays"] == 1) | inside).all()
    assert (e["f"][inside] == GOLD["f_inside"]).all() and (e["f"][~inside] == GOLD["f_outside"]).all()
    # class membership = silhouette disc of radius r_px around the film centre
    r = np.hypot(x[:, 0] * 64 - 32, x[:, 1] * 64 - 32)
    clear = np.abs(r - GOLD["r_px"]) > 0.05          # level-4 icosphere moves the silhouette by < 0.02 px
    assert (inside[clear] == (r[clear] < GOLD["r_px"])).all()
    # p_lambda closed form within MC error (binomial)
    frac = np.pi * GOLD["r_px"] ** 2 / 4096
    assert abs(e["p"].mean() - GOLD["p_lambda"]) < 5 * 0.5 * np.sqrt(frac * (1 - frac) / len(x))
    # Lambert-only scene: score == 0 exactly (weights do not depend on x under Q5-Q7)
    assert (e["g"] == 0).all()
    # PT image: fully-inside pixels 0.5, fully-outside 1.0, in expectation; check class means
    img = sc.pt_render(400000, seed=3)[..., 0]
    yy, xx = np.mgrid[0:64, 0:64]
    corners = [np.hypot(xx + a - 32, yy + b - 32) for a in (0, 1) for b in (0, 1)]
    inside_px = np.max(corners, axis=0) < GOLD["r_px"]
    outside_px = np.min(corners, axis=0) > GOLD["r_px"]
    assert inside_px.sum() == 1528 and outside_px.sum() == 2388     # pixel classes for r_px = 22.70
    inside_px = np.max(corners, axis=0) < GOLD["r_px"] - 0.05      # margin for the faceted silhouette
    outside_px = np.min(corners, axis=0) > GOLD["r_px"] + 0.05
    assert abs(img[inside_px].mean() - 0.5) < 0.01 and abs(img[outside_px].mean() - 1.0) < 0.01
    assert abs(img.mean() - GOLD["p_lambda"]) < 0.01


def test_closed_box_values_are_powers_of_albedo(oracle):
    """Closed Lambert box with an emitting ceiling: f in {a^k E, k < L} or 0, never anything else."""
    a, E, L = 0.5, 2.0, 6
    desc = S.closed_furnace(albedo=a, emission=E, max_path_len=L)
    sc = oracle.Scene(desc, oracle.F64)
    e = sc.eval(S.seeded_states(50000, desc.dim, 4), True)
    allowed = np.array([0.0] + [a ** k * E for k in range(L)])
    assert np.isin(e["f"][:, 0], allowed).all()
    k = e["nrays"] - 1
    lit = e["f"][:, 0] > 0
    assert (e["f"][lit, 0] == a ** k[lit] * E).all()
    assert (e["nrays"][~lit] == L).all()            # closed room, no roulette: unlit paths run to the cap
    assert (e["g"] == 0).all()


def glass_slab(theta_deg, strip_lo, strip_hi, ior=1.5, L=3):
    """Camera looks at a glass interface (plane y=0, normal +y) under incidence angle theta; an up-facing strip
    emitter at y=-1 spans x in [strip_lo, strip_hi]; environment above is black."""
    mesh = S._Mesh()
    B = 50.0
    mesh.quad((-B, 0, -B), (-B, 0, B), (B, 0, B), (B, 0, -B), 0)               # +y normal
    mesh.quad((strip_lo, -1, -B), (strip_lo, -1, B), (strip_hi, -1, B), (strip_hi, -1, -B), 1)   # +y normal
    v, i, m = mesh.finish()
    th = np.deg2rad(theta_deg)
    pos = (-np.sin(th), np.cos(th), 0.0)
    mats = np.stack([S.material(S.MAT_DIELECTRIC, ior=ior), S.material(S.MAT_EMITTER, le=(1, 1, 1))])
    return S.SceneDesc(v, i, m, mats, cam_pos=pos, cam_look=(0, 0, 0), cam_up=(0, 0, 1), vfov_deg=1.0, width=1, height=1,
                       max_path_len=L)


def test_dielectric_fresnel_and_snell(oracle):
    """Textbook closed forms: F(0) = ((n-1)/(n+1))^2; unpolarised Fresnel at angle; Snell sin(t) = sin(i)/n."""
    n = 1.5
    for theta in (0.0, 30.0, 56.30993247, 75.0):       # 56.3 deg = Brewster angle atan(1.5)
        ci = np.cos(np.deg2rad(theta))
        st = np.sin(np.deg2rad(theta)) / n
        ct = np.sqrt(1 - st * st)
        rs = ((ci - n * ct) / (ci + n * ct)) ** 2
        rp = ((n * ci - ct) / (n * ci + ct)) ** 2
        F = 0.5 * (rs + rp)
        if theta == 0.0:
            assert np.isclose(F, ((n - 1) / (n + 1)) ** 2)
        x_hit = st / ct                                 # refracted ray reaches y=-1 at x = tan(theta_t)
        desc = glass_slab(theta, x_hit - 0.01, x_hit + 0.01)
        sc = oracle.Scene(desc, oracle.F64)
        x = np.full((4001, desc.dim), 0.5)
        x[:, 2] = (np.arange(4001) + 0.5) / 4001        # u1 decides reflect (u1 < F) or refract
        e = sc.eval(x, False)
        lit = e["p"] > 0                                # refracted -> hits the strip; reflected -> black sky
        assert abs((~lit).mean() - F) < 1.0 / 4001 + 1e-9, (theta, (~lit).mean(), F)
        assert (lit == (x[:, 2] >= F)).all()
        assert (e["f"][lit] == 1.0).all()               # weight 1 on both lobes (Q7)
        # Snell: moving the strip away by 0.05 loses the refracted ray
        desc2 = glass_slab(theta, x_hit + 0.04, x_hit + 0.06)
        assert (oracle.Scene(desc2, oracle.F64).eval(x, False)["p"] == 0).all()
    # total internal reflection from inside: camera below the interface looking up at 60 deg > asin(1/1.5) = 41.8 deg
    mesh = S._Mesh()
    mesh.quad((-50, 0, -50), (-50, 0, 50), (50, 0, 50), (50, 0, -50), 0)
    v, i, m = mesh.finish()
    th = np.deg2rad(60)
    desc = S.SceneDesc(v, i, m, np.stack([S.material(S.MAT_DIELECTRIC, ior=n)]), env_radiance=(1, 1, 1),
                       cam_pos=(-np.sin(th), -np.cos(th), 0), cam_look=(0, 0, 0), cam_up=(0, 0, 1), vfov_deg=1.0, width=1,
                       height=1, max_path_len=2)
    x = np.full((101, 4), 0.5)
    x[:, 2] = (np.arange(101) + 0.5) / 101
    e = oracle.Scene(desc, oracle.F64).eval(x, False)
    assert (e["sig"] == e["sig"][0]).all()              # always the reflect lobe, whatever u1


def ggx_plane(alpha, f0, theta_deg, L=2):
    mesh = S._Mesh()
    mesh.quad((-50, 0, -50), (-50, 0, 50), (50, 0, 50), (50, 0, -50), 0)
    v, i, m = mesh.finish()
    th = np.deg2rad(theta_deg)
    return S.SceneDesc(v, i, m, np.stack([S.material(S.MAT_GGX, f0, rough=alpha)]), env_radiance=(1, 1, 1),
                       cam_pos=(-np.sin(th), np.cos(th), 0), cam_look=(0, 0, 0), cam_up=(0, 0, 1), vfov_deg=1.0, width=1,
                       height=1, max_path_len=L)


def test_ggx_limits_and_energy(oracle):
    f0 = (0.9, 0.6, 0.3)
    # alpha -> 0: mirror; weight -> Schlick F(cos theta) G1 -> F
    for theta in (0.0, 40.0, 70.0):
        desc = ggx_plane(1e-5, f0, theta)
        x = S.seeded_states(200, 4, 1).astype(np.float64)
        x[:, :2] = 0.5                                   # film centre: incidence angle is exactly theta
        e = oracle.Scene(desc, oracle.F64).eval(x, False)
        c = np.cos(np.deg2rad(theta))
        want = np.array(f0) + (1 - np.array(f0)) * (1 - c) ** 5
        assert np.allclose(e["f"], want[None, :], rtol=1e-3)
    # F0 = 1 (white conductor): weight = G1(w_i) in (0, 1]; mean weight = directional albedo <= 1 and
    # >= 0.5 for moderate roughness at near-normal incidence (single-scattering energy loss is small)
    for alpha, theta in ((0.3, 10.0), (0.5, 50.0)):
        desc = ggx_plane(alpha, (1, 1, 1), theta)
        e = oracle.Scene(desc, oracle.F64).eval(S.seeded_states(40000, 4, 2), False)
        w = e["f"][:, 0]
        assert (w >= 0).all() and (w <= 1 + 1e-12).all()
        assert 0.5 < w.mean() <= 1.0
    # visible-normal sampling: with F0 = 1 the estimator E[G1(w_i)] equals the textbook integral
    #   int D(h) G1(w_o) G1(w_i) / (4 cos_o) dw_i  evaluated by brute-force quadrature over the hemisphere
    alpha, theta = 0.4, 35.0
    desc = ggx_plane(alpha, (1, 1, 1), theta)
    e = oracle.Scene(desc, oracle.F64).eval(S.seeded_states(400000, 4, 3), False)
    th = np.deg2rad(theta)
    wo = np.array([np.sin(th), 0.0, np.cos(th)])      # local frame: any azimuth (isotropic)
    n = 1500
    mu = (np.arange(n) + 0.5) / n                      # cos(theta_i)
    ph = (np.arange(2 * n) + 0.5) / (2 * n) * 2 * np.pi
    MU, PH = np.meshgrid(mu, ph, indexing="ij")
    sn = np.sqrt(1 - MU * MU)
    wi = np.stack([sn * np.cos(PH), sn * np.sin(PH), MU], -1)
    h = wi + wo
    h /= np.linalg.norm(h, axis=-1, keepdims=True)
    D = alpha ** 2 / (np.pi * ((h[..., 2] ** 2) * (alpha ** 2 - 1) + 1) ** 2)
    G1 = lambda w: 2 * w[..., 2] / (w[..., 2] + np.sqrt(alpha ** 2 * (w[..., 0] ** 2 + w[..., 1] ** 2) + w[..., 2] ** 2))
    integrand = D * G1(wo) * G1(wi) / (4 * wo[2])
    want = integrand.sum() * (1.0 / n) * (2 * np.pi / (2 * n))
    got = e["f"][:, 0].mean()
    assert abs(got - want) < 5 * e["f"][:, 0].std() / np.sqrt(len(e["p"])) + 2e-4, (got, want)


def test_score_matches_finite_differences(oracle):
    """score = grad ln(p + eps): dual numbers vs central differences in fp64, h = 1e-6,
    at states whose discrete decisions are constant over the stencil."""
    for desc, nstates in ((S.ggx_room(), 6000), (S.mini_machines(max_path_len=6), 60000)):
        sc = oracle.Scene(desc, oracle.F64)
        x = S.seeded_states(nstates, desc.dim, 7).astype(np.float64)
        e = sc.eval(x, True)
        cand = np.where((e["p"] > 0) & (np.abs(e["g"]).max(1) > 0))[0][:60]
        assert len(cand) >= 25
        h, checked = 1e-6, 0
        for i in cand:
            xs = np.repeat(x[i][None, :], 2 * desc.dim, 0)
            for j in range(desc.dim):
                xs[2 * j, j] += h
                xs[2 * j + 1, j] -= h
            ee = sc.eval(xs, False)
            if not (ee["sig"] == e["sig"][i]).all():
                continue
            lp = np.log(ee["p"] + 1e-8)
            fd = (lp[0::2] - lp[1::2]) / (2 * h)
            scale = np.abs(e["g"][i]).max()
            assert np.allclose(e["g"][i], fd, rtol=2e-5, atol=2e-6 * max(scale, 1.0)), (i, e["g"][i], fd)
            checked += 1
        assert checked >= 15
    # a path without a GGX vertex has score == 0 exactly
    desc = S.cornell(width=16, height=16, max_path_len=5)
    e = oracle.Scene(desc, oracle.F64).eval(S.seeded_states(20000, desc.dim, 1), True)
    assert (e["p"] > 0).sum() > 100 and (e["g"] == 0).all()


def test_analytic_target(oracle):
    desc = S.mixture3()
    sc = oracle.Scene(desc, oracle.F64)
    # normalisation = sum of weights (wrapped Gaussians integrate to 1): 256^2 midpoint quadrature
    n = 256
    c = (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(c, c)
    pts = np.stack([X.ravel(), Y.ravel()], 1)
    e = sc.eval(pts, True)
    assert abs(e["p"].mean() - 1.0) < 1e-6      # float32-rounded weights sum to 1 within 1e-7
    # closed form at a point: direct evaluation of the definition with 5 images per axis
    x = np.array([0.31, 0.72])
    want = 0.0
    for w, mu, s in zip(desc.weights.astype(np.float64), desc.means.astype(np.float64), desc.stddevs.astype(np.float64)):
        term = w
        for k in range(2):
            dl = (x[k] - mu[k] + 0.5) % 1.0 - 0.5
            term *= sum(np.exp(-0.5 * ((dl + j) / s) ** 2) / (s * np.sqrt(2 * np.pi)) for j in range(-2, 3))
        want += term
    got = sc.eval(x[None, :], True)
    assert np.isclose(got["p"][0], want, rtol=1e-12)
    assert (got["f"][0] == got["p"][0]).all()
    # score vs finite differences; periodicity
    h = 1e-6
    for k in range(2):
        xp, xm = x.copy(), x.copy()
        xp[k] += h
        xm[k] -= h
        fd = (np.log(sc.eval(xp[None], False)["p"][0] + 1e-8) - np.log(sc.eval(xm[None], False)["p"][0] + 1e-8)) / (2 * h)
        assert np.isclose(got["g"][0, k], fd, rtol=1e-6)
    assert np.isclose(sc.eval(np.array([[0.0, 0.3]]), False)["p"][0], sc.eval(np.array([[1 - 1e-15, 0.3]]), False)["p"][0], rtol=1e-9)


def test_bias_field_closed_form_single_gaussian(oracle):
    """Appendix C: b = L^* p / p for the Alg. 4 dynamics.  For one isotropic Gaussian mode of width tau
    the Euler-Maruyama step is linear, x' - mu = A (x - mu) + s xi with A = (1 - s^2 / (2 tau^2)) I + (c~ / tau^2) J, so the
    pushed-forward density is Gaussian with variance v' = tau^2 ((1 - a)^2 + b^2) + s^2 and
    b(y) = (N(y; mu, v') / N(y; mu, tau^2) - 1) / dt in closed form.  Also: the integral of L^* p vanishes, and at fixed
    sigma (s^2 = sigma^2 dt) the field shrinks with dt (the vanishing bias the appendix shows)."""
    tau = 0.05
    sc = oracle.Scene(S.single_mode(s=tau), oracle.F64)
    G = 32
    c = (np.arange(G) + 0.5) / G
    X, Y = np.meshgrid(c, c)
    r2 = (X - 0.5) ** 2 + (Y - 0.5) ** 2
    N = lambda r2, var: np.exp(-r2 / (2 * var)) / (2 * np.pi * var)
    near = r2 < (3 * tau) ** 2
    for s, ct, dt in ((0.01, 2e-5, 1e-2), (0.005, 0.0, 1e-3), (0.02, -1e-4, 1.0)):
        b = sc.bias_field(s, ct, dt, G=G, M=512)
        a, bb = s * s / (2 * tau * tau), ct / (tau * tau)
        v = tau * tau * ((1 - a) ** 2 + bb * bb) + s * s
        want = (N(r2, v) / N(r2, tau * tau) - 1) / dt
        assert np.abs(b - want)[near].max() <= 1e-5 * np.abs(want[near]).max() + 1e-9, (s, ct, dt)
        p = sc.eval(np.stack([X.ravel(), Y.ravel()], 1), False)["p"].reshape(G, G)
        assert abs((b * p).mean()) < 1e-6 * np.abs(b * p).max() * G                # mass is conserved: integral of L^* p = 0
    # separated modes (the appendix' left panel): the field shrinks like dt at fixed sigma
    sc3 = oracle.Scene(S.mixture3(), oracle.F64)
    sigma = 0.5
    c = (np.arange(24) + 0.5) / 24
    X, Y = np.meshgrid(c, c)
    p3 = sc3.eval(np.stack([X.ravel(), Y.ravel()], 1), False)["p"].reshape(24, 24)
    bulk = p3 > 0.05 * p3.max()                                                     # away from the tails, where 1 / p explodes
    m = [np.abs(sc3.bias_field(sigma * np.sqrt(dt), 0.5 * sigma ** 2 * dt, dt, G=24, M=384))[bulk].max() for dt in (4e-4, 1e-4)]
    assert 3.0 < m[0] / m[1] < 5.0, m
