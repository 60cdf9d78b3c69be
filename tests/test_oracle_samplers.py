"""Pins for the oracle's five samplers and estimator (Alg. 1-4).

Main pin: BRUTE FORCE ON A TINY INPUT.  On a smooth 2-D analytic target the state space
is discretised into a G x G grid and the printed algorithm is propagated EXACTLY as a
finite Markov chain (dense transition matrix, no sampling): initial law nu, per-event
expected accumulation E[dtau f/p_hat] = f/(p_hat (lambda+kappa)), kill probability
kappa/(lambda+kappa), regeneration, local kernel (Metropolis / MALA / unadjusted
nonreversible Langevin).  That gives the exact expected accumulation buffer and
tourCount of Alg. 1-3 after T iterations, transient included, for every sampler; the
oracle's Monte-Carlo averages over many chains must match it within their standard
error.  The grid model is written here from the paper's formulas with numpy only.
"""
import numpy as np
import pytest

from dr_inputs import scenes as S

EPS = 1e-8
G, W = 40, 8            # grid cells per axis, image pixels per axis (G is a multiple of W)
T = 10                  # iterations after init


def target():
    return S.Analytic2DDesc(np.array([0.65, 0.35], dtype=np.float32), np.array([[0.3, 0.4], [0.72, 0.62]], dtype=np.float32),
                            np.array([0.13, 0.16], dtype=np.float32), W, W, "two_modes")


def grid_model(oracle):
    sc = oracle.Scene(target(), oracle.F64)
    c = (np.arange(G) + 0.5) / G
    X, Y = np.meshgrid(c, c)                      # row = y index, col = x index
    pts = np.stack([X.ravel(), Y.ravel()], 1)
    e = sc.eval(pts, True)                        # target values are pinned separately (test_oracle_target.py)
    pix = (np.floor(pts[:, 1] * W) * W + np.floor(pts[:, 0] * W)).astype(int)
    return sc, pts, e["p"], e["g"], pix


def wrapped_gauss_rows(mean, pts, s):
    """Row-normalised probabilities of landing in each grid cell for y = wrap(mean + s xi)."""
    out = np.ones((len(mean), len(pts)))
    for k in range(2):
        dl = pts[None, :, k] - mean[:, None, k]
        w = sum(np.exp(-0.5 * ((dl + j) / s) ** 2) for j in range(-3, 4))
        out *= w
    return out / out.sum(1, keepdims=True)


def min_image(v):
    return v - np.floor(v + 0.5)


def local_kernel(method, pts, p, g, s, ct):
    """Transition matrix of the local dynamics on the grid."""
    n = len(pts)
    ph = p + EPS
    h = 0.5 * s * s
    if method in ("metropolis", "metropolis_restore"):
        q = wrapped_gauss_rows(pts, pts, s)
        acc = np.minimum(1.0, ph[None, :] / ph[:, None])
    elif method in ("mala", "mala_restore"):
        mean = pts + h * g
        q = wrapped_gauss_rows(mean, pts, s)
        # ln q(a -> b) with the minimal-image difference (Q11)
        lq = np.zeros((n, n))
        for k in range(2):
            lq += min_image(pts[None, :, k] - mean[:, None, k]) ** 2
        lq = -lq / (2 * s * s)
        acc = np.minimum(1.0, ph[None, :] / ph[:, None] * np.exp(lq.T - lq))
    else:  # diffusion_restore: Alg. 4, no accept/reject
        rot = ct * np.stack([g[:, 1], -g[:, 0]], 1)
        return wrapped_gauss_rows(pts + h * g + rot, pts, s)
    P = q * acc
    P[np.arange(n), np.arange(n)] += 1.0 - P.sum(1)      # rejected mass stays
    return P


def tile_density(pts, rho):
    """rho / rho_lambda at the grid points for tile probabilities `rho` (R x R, row = x1 tile): R^2 w[tile]."""
    R = rho.shape[0]
    tx, ty = np.minimum((pts[:, 0] * R).astype(int), R - 1), np.minimum((pts[:, 1] * R).astype(int), R - 1)
    return R * R * rho[ty, tx]


def expected_run(method, pts, p, g, pix, s, ct, m, dt, lsp, p_lambda, rho=None):
    n = len(pts)
    ph = p + EPS
    dens = np.ones(n) if rho is None else tile_density(pts, rho)
    nu = dens / n                                  # regeneration law on the grid (f4: density rho, else uniform)
    P = local_kernel(method, pts, p, g, s, ct)
    restore = method.endswith("restore")
    fop = p / ph                                  # f = (p, p, p)
    accum = np.zeros(W * W)
    tours = 0.0
    mu = nu.copy()
    if restore:
        dt_eff = dt if method == "diffusion_restore" else 1.0
        lam = 1.0 / dt_eff                        # PAPER.md L659 / L737
        kappa = dens * (p_lambda / (m * dt_eff)) / ph    # L752, L445: (rho / rho_lambda) kappa0 / p_hat
        kill = kappa / (lam + kappa)
        hold = 1.0 / (lam + kappa)                # E[min(Exp(lam), Exp(kappa))]
        for _ in range(T + 1):
            np.add.at(accum, pix, mu * hold * fop)
            tours += (mu * kill).sum()
            mu = (mu * (1 - kill)) @ P + (mu * kill).sum() * nu
    else:
        acc_large = np.minimum(1.0, ph[None, :] / ph[:, None]) * nu[None, :]
        acc_large[np.arange(n), np.arange(n)] += 1.0 - acc_large.sum(1)
        Pf = lsp * acc_large + (1 - lsp) * P
        for _ in range(T + 1):
            np.add.at(accum, pix, mu * fop)
            mu = mu @ Pf
    return accum, tours


PARAMS = {
    "metropolis": dict(stddev=0.10, large_step_prob=0.3),
    "mala": dict(stddev=0.12, large_step_prob=0.3),
    "metropolis_restore": dict(stddev=0.10, m=5.0),
    "mala_restore": dict(stddev=0.12, m=5.0),
    "diffusion_restore": dict(stddev=0.10, c_tilde=0.006, dt=1e-2, m=5.0),
}


RB = [(m, False) for m in PARAMS] + [(m, True) for m in PARAMS if m.endswith("restore")]


@pytest.mark.parametrize("method,rb", RB, ids=[m + ("-rao_blackwell" if r else "") for m, r in RB])
def test_finite_state_brute_force(oracle, method, rb):
    """rb: Rao-Blackwellised Accumulate (f3): the weight is E[dtau | x] = 1 / (lambda + kappa), which is exactly the
    `hold` the model propagates, so the same expectations pin it."""
    sc, pts, p, g, pix = grid_model(oracle)
    kw = dict(PARAMS[method], rao_blackwell=rb)
    s, ct = kw["stddev"], kw.get("c_tilde", 0.0)
    m, dt, lsp = kw.get("m", 64.0), kw.get("dt", 1e-5), kw.get("large_step_prob", 0.0)
    p_lambda = 1.0 + EPS
    want_acc, want_tours = expected_run(method, pts, p, g, pix, s, ct, m, dt, lsp, p_lambda)
    seeds, N = 8, 30000
    accs, tours = [], []
    for seed in range(seeds):
        ch = oracle.Chains(sc, method, N, seed=100 + seed, p_lambda_override=p_lambda, **kw)
        ch.init(0)
        ch.step(T)
        accs.append(ch.accum()[:, 0] / N)
        tours.append(ch.stats()["tours"] / N)
        assert ch.stats()["mutations"] == N * (T + 1)
    accs, tours = np.array(accs), np.array(tours)
    mean, se = accs.mean(0), accs.std(0, ddof=1) / np.sqrt(seeds)
    # per pixel: within 5 standard errors (+ a 2e-3 relative allowance for the grid discretisation of min(1, .))
    z = np.abs(mean - want_acc) / (se + 2e-3 * want_acc)
    assert z.max() < 5.0, (method, z.max(), mean[z.argmax()], want_acc[z.argmax()])
    # totals: much tighter
    tot, tot_se = accs.sum(1).mean(), accs.sum(1).std(ddof=1) / np.sqrt(seeds)
    assert abs(tot - want_acc.sum()) < 5 * tot_se + 5e-4 * want_acc.sum(), (method, tot, want_acc.sum(), tot_se)
    if method.endswith("restore"):
        t_se = tours.std(ddof=1) / np.sqrt(seeds)
        assert abs(tours.mean() - want_tours) < 5 * t_se + 5e-4 * want_tours, (method, tours.mean(), want_tours)


def test_nonuniform_regeneration_density(oracle):
    """f4: regeneration from a density rho that is piecewise constant on film tiles, killing
    rate (rho / rho_lambda) kappa0 / p_hat.  (i) In the finite-state model the tour estimator stays exact for a reversible
    kernel: kappa0 nu.h = integral of f with nu = rho; (ii) the model's exact expectations after T iterations pin the oracle's
    runs with a strongly non-uniform rho; (iii) the init states follow rho."""
    sc, pts, p, g, pix = grid_model(oracle)
    rng = np.random.default_rng(8)
    rho = rng.uniform(0.2, 3.0, size=(4, 4))
    rho /= rho.sum()
    rho = rho.astype(np.float32).astype(np.float64)
    ph, n = p + EPS, len(p)
    dens = tile_density(pts, rho)
    nu = dens / n
    P = local_kernel("metropolis_restore", pts, p, g, 0.1, 0.0)
    lam, m = 1.0, 5.0
    kappa0 = ph.mean() * lam / m
    A = np.diag(lam + dens * kappa0 / ph) - lam * P
    assert np.isclose(kappa0 * (nu @ np.linalg.solve(A, p / ph)), p.mean(), rtol=1e-9)        # (i)
    p_lambda = 1.0 + EPS
    for method in ("metropolis_restore", "diffusion_restore"):
        kw = dict(PARAMS[method])
        want_acc, want_tours = expected_run(method, pts, p, g, pix, kw["stddev"], kw.get("c_tilde", 0.0), kw["m"], kw.get("dt", 1e-5),
                                            0.0, p_lambda, rho=rho)
        base_acc, _ = expected_run(method, pts, p, g, pix, kw["stddev"], kw.get("c_tilde", 0.0), kw["m"], kw.get("dt", 1e-5), 0.0, p_lambda)
        assert np.abs(want_acc - base_acc).max() > 0.05 * base_acc.max()                         # rho matters at T = 10
        seeds, N = 8, 30000
        accs, tours = [], []
        for seed in range(seeds):
            ch = oracle.Chains(sc, method, N, seed=500 + seed, p_lambda_override=p_lambda, rho=rho, **kw)
            ch.init(0)
            if seed == 0:                                                                         # (iii)
                x = ch.state()["x"]
                hist = np.histogram2d(x[:, 1], x[:, 0], bins=4, range=[[0, 1], [0, 1]])[0] / N
                assert np.abs(hist - rho).max() < 5 * np.sqrt(rho.max() / N)
            ch.step(T)
            accs.append(ch.accum()[:, 0] / N)
            tours.append(ch.stats()["tours"] / N)
        accs, tours = np.array(accs), np.array(tours)
        mean, se = accs.mean(0), accs.std(0, ddof=1) / np.sqrt(seeds)
        z = np.abs(mean - want_acc) / (se + 2e-3 * want_acc)
        assert z.max() < 5.0, (method, z.max())
        t_se = tours.std(ddof=1) / np.sqrt(seeds)
        assert abs(tours.mean() - want_tours) < 5 * t_se + 5e-4 * want_tours, (method, tours.mean(), want_tours)


def test_second_antisymmetric_pattern(oracle):
    """f4: the drift's antisymmetric part, read off the oracle by teacher forcing.  A state with a
    chosen score g is set, Diffusion Restore takes one step (always accepted), and y - x - (s^2/2) g - s xi = c~ A~ g with xi
    recomputed from the chain's Philox stream.  a_mode 0 is the paper's diag(A_block) (rotate(v) = c~ (v2, -v1), L720);
    a_mode 1 couples coordinates (4i, 4i+2) and (4i+1, 4i+3); both are antisymmetric (g . A~ g = 0, A~^T = -A~)."""
    desc = S.furnace()                                        # d = 8
    sc = oracle.Scene(desc, oracle.F64)
    d, N, s, ct = desc.dim, 64, 1e-3, 0.25
    want = {0: np.kron(np.eye(4), np.array([[0.0, 1.0], [-1.0, 0.0]])),
            1: np.kron(np.eye(2), np.array([[0, 0, 1, 0], [0, 0, 0, 1], [-1, 0, 0, 0], [0, -1, 0, 0]], dtype=float))}
    for mode in (0, 1):
        ch = oracle.Chains(sc, "diffusion_restore", N, seed=3, stddev=s, c_tilde=ct, a_mode=mode)
        ch.init(0)
        st = ch.state()
        rng = np.random.default_rng(1)
        st["x"] = rng.uniform(0.3, 0.7, size=(N, d))
        st["g"] = np.zeros((N, d))
        st["g"][:d] = np.eye(d) * 0.1                         # chains 0..d-1 probe the columns of A~
        st["g"][d:] = rng.normal(size=(N - d, d)) * 0.1
        st["killed"][:] = 0
        ch.set_state(st, 5)
        ch.step(1)
        y = ch.state()["x"]
        xi = np.zeros((N, d))
        for i in range(N):
            for j in range(d // 4):
                w = oracle.stream_block(3, i, 6, j, 1, 0)    # purpose 1 = PROP_N, iteration 6
                xi[i, 4 * j:4 * j + 2] = oracle.rng_transforms(int(w[0]), int(w[1]), oracle.F64)[2:]
                xi[i, 4 * j + 2:4 * j + 4] = oracle.rng_transforms(int(w[2]), int(w[3]), oracle.F64)[2:]
        Ag = (y - st["x"] - 0.5 * s * s * st["g"] - s * xi) / ct
        assert np.allclose(Ag, st["g"] @ want[mode].T, atol=1e-12)
        assert np.allclose(want[mode].T, -want[mode]) and np.abs(np.sum(Ag * st["g"], axis=1)).max() < 1e-12
    assert not np.allclose(want[0], want[1])


def test_rao_blackwell_weight_is_the_expected_holding_time(oracle):
    """f3: with the flag every chain accumulates 1 / (lambda + kappa0 / p_hat(x)) -- a closed form of
    its state -- the kill decisions and hence the states are those of the plain run with the same seed, and the
    per-pixel spread over seeds of the accumulation buffer shrinks."""
    sc = oracle.Scene(target(), oracle.F64)
    kw = dict(PARAMS["diffusion_restore"])
    N, p_lambda = 20000, 1.0 + EPS
    spread = {}
    for rb in (False, True):
        accs = []
        for seed in range(6):
            ch = oracle.Chains(sc, "diffusion_restore", N, seed=300 + seed, p_lambda_override=p_lambda, rao_blackwell=rb, **kw)
            ch.init(0)
            ch.step(5)
            accs.append(ch.accum()[:, 0] / N)
            if seed == 0:
                st, (_, w) = ch.state(), ch.last()
                if rb:
                    lam, kappa0 = 1.0 / kw["dt"], p_lambda / (kw["m"] * kw["dt"])
                    assert np.allclose(w, 1.0 / (lam + kappa0 / (st["p"] + EPS)), rtol=1e-13, atol=0)
                    assert np.array_equal(st["x"], x_plain) and np.array_equal(st["killed"], k_plain)
                else:
                    x_plain, k_plain = st["x"], st["killed"]
        spread[rb] = np.array(accs).std(0, ddof=1).sum()
    assert spread[True] < 0.85 * spread[False], spread


def test_path_tracing_method_is_a_plain_average(oracle):
    """f2: method 5 draws every chain anew each iteration and accumulates f with unit weight.
    Recomputed here from the definition: the Philox uniforms of (chain, iteration), the target evaluation (pinned in
    test_oracle_target.py), a numpy histogram.  And the furnace classes resolve to their closed forms."""
    desc = S.furnace()
    sc = oracle.Scene(desc, oracle.F64)
    N, T, seed = 3000, 3, 11
    ch = oracle.Chains(sc, "path_tracing", N, seed=seed)
    ch.init(2)
    ch.step(T)
    assert ch.stats()["mutations"] == N * (T + 1) and ch.stats()["tours"] == 0 and len(ch.queue()) == 0
    want = np.zeros((desc.width * desc.height, 4))
    for it in range(T + 1):
        x = np.zeros((N, desc.dim))
        for i in range(N):
            for j in range(desc.dim // 4):
                w = oracle.stream_block(seed, i, it, j, 0, 2)
                x[i, 4 * j:4 * j + 4] = (w >> 8).astype(np.float64) * 2.0 ** -24
        e = sc.eval(x, False)
        np.add.at(want[:, :3], e["pix"], e["f"])
        np.add.at(want[:, 3], e["pix"], 1.0)
        if it == T:
            assert np.array_equal(ch.state()["x"], x)
    assert np.allclose(ch.accum(), want, rtol=1e-12, atol=0)
    img, status = ch.resolve()
    assert status == 0 and np.allclose(img.reshape(-1, 3), want[:, :3] * (desc.width * desc.height / (N * (T + 1.0))), rtol=1e-12)
    # closed form (tests/golden/furnace.txt): many samples, class means 0.5 / 1.0
    ch = oracle.Chains(sc, "path_tracing", 100000, seed=1)
    ch.init(0)
    ch.step(3)
    img = ch.resolve()[0][..., 0]
    yy, xx = np.mgrid[0:64, 0:64]
    corners = [np.hypot(xx + a - 32, yy + b - 32) for a in (0, 1) for b in (0, 1)]
    assert abs(img[np.max(corners, axis=0) < 22.65].mean() - 0.5) < 0.01 and abs(img[np.min(corners, axis=0) > 22.75].mean() - 1.0) < 0.01


def test_model_identities_tour_length_and_unbiasedness(oracle):
    """Checks of the finite-state model itself against the theory it restates: for a p_hat-reversible local
    kernel, (i) expected events per tour = m + 1 exactly and (ii) kappa0 * nu.h = integral of f, where
    h solves (diag(lambda + kappa) - lambda P) h = f / p_hat  (regeneration-tour estimator)."""
    sc, pts, p, g, pix = grid_model(oracle)
    ph = p + EPS
    n = len(p)
    nu = np.full(n, 1.0 / n)
    for method, lam, m in (("metropolis_restore", 1.0, 5.0), ("mala_restore", 1.0, 64.0), ("metropolis_restore", 1e5, 3.0)):
        P = local_kernel(method, pts, p, g, 0.1, 0.0)
        kappa0 = ph.mean() * lam / m
        kappa = kappa0 / ph
        A = np.diag(lam + kappa) - lam * P
        events = nu @ np.linalg.solve(A, lam + kappa)
        # Metropolis on the grid is exactly reversible; grid MALA only up to row normalisation / nearest image
        rtol = 1e-9 if method == "metropolis_restore" else 1e-4
        assert np.isclose(events, m + 1, rtol=rtol)
        est = kappa0 * (nu @ np.linalg.solve(A, p / ph))
        assert np.isclose(est, p.mean(), rtol=rtol)
    # the unadjusted Langevin kernel is not p_hat-invariant: the identity fails (modified-kappa bias, L443-L460)
    P = local_kernel("diffusion_restore", pts, p, g, 0.1, 0.006)
    lam, m = 100.0, 5.0
    kappa0 = ph.mean() * lam / m
    A = np.diag(lam + kappa0 / ph) - lam * P
    assert abs(nu @ np.linalg.solve(A, lam + kappa0 / ph) - (m + 1)) > 1e-3


def test_brute_force_model_is_sensitive(oracle):
    """The pin has teeth: flipping the rotation sign, dropping the drift or using kappa0*p instead of
    kappa0/p moves the exact expectation by far more than the tolerance used above."""
    sc, pts, p, g, pix = grid_model(oracle)
    base, _ = expected_run("diffusion_restore", pts, p, g, pix, 0.10, 0.006, 5.0, 1e-2, 0.0, 1.0)
    flipped, _ = expected_run("diffusion_restore", pts, p, g, pix, 0.10, -0.006, 5.0, 1e-2, 0.0, 1.0)
    nodrift, _ = expected_run("diffusion_restore", pts, p, -g, pix, 0.10, 0.0, 5.0, 1e-2, 0.0, 1.0)
    assert np.abs(flipped - base).max() / base.max() > 0.01
    assert np.abs(nodrift - base).max() / base.max() > 0.05


def test_long_run_convergence_and_kill_fraction(oracle):
    """Long-run kill fraction -> 1/(m+1) for every Restore variant with a p_hat-invariant kernel, any target;
    images approach the quadrature reference as the run gets longer (transient ~ 1/iterations, Q17)."""
    sc, pts, p, g, pix = grid_model(oracle)
    ref = np.zeros(W * W)
    np.add.at(ref, pix, p / len(p))
    ref *= W * W                                  # N_pix * integral of f over the pixel
    for method in ("metropolis_restore", "mala_restore", "diffusion_restore"):
        errs = []
        for its in (300, 2400):
            ch = oracle.Chains(sc, method, 1500, seed=3, p_lambda_override=1.0, m=16.0)
            ch.init(0)
            ch.step(its)
            img, _ = ch.resolve()
            errs.append(abs(img[..., 0].mean() - 1.0))
            st = ch.stats()
        assert errs[1] < 0.4 * errs[0] + 0.004, (method, errs)
        assert abs(st["tours"] / st["mutations"] - 1 / 17) < 0.02 / 17, method
        assert np.abs(img[..., 0].ravel() - ref).max() < 0.12 * ref.max()
    for method in ("metropolis", "mala"):
        ch = oracle.Chains(sc, method, 1500, seed=3, p_lambda_override=1.0)
        ch.init(0)
        ch.step(1500)
        img, _ = ch.resolve()
        assert abs(img.mean() - 1.0) < 1e-6        # sum of f/p_hat * p_lambda / N_mut == 1 up to eps
        assert np.abs(img[..., 0].ravel() - ref).max() < 0.08 * ref.max()


def test_agreement_with_path_tracing(oracle):
    """Converged MCMC images agree with ordinary path tracing on a mesh scene (exactly
    consistent samplers; Diffusion Restore's gap is reported in DESIGN.md, not asserted)."""
    desc = S.closed_furnace(albedo=0.6, emission=1.5, width=4, height=4, max_path_len=4)
    sc = oracle.Scene(desc, oracle.F64)
    pt = sc.pt_render(600000, seed=1)
    for method in ("metropolis", "metropolis_restore"):
        # short tours (m = 4) so that the start-up transient of Alg. 3 (Q17) has died out after 600 iterations
        ch = oracle.Chains(sc, method, 3000, seed=2, m=4.0)
        ch.init(0)
        ch.step(600)
        img, _ = ch.resolve()
        assert abs(img.mean() / pt.mean() - 1.0) < 0.04, (method, img.mean(), pt.mean())
        assert oracle.rel_mse(img, pt) < 5e-3


def test_thread_count_does_not_change_results(oracle):
    desc = S.mini_machines()
    sc = oracle.Scene(desc, oracle.F32)
    outs = []
    for th in (1, 8):
        oracle.set_threads(th)
        ch = oracle.Chains(sc, "mala_restore", 600, seed=9)
        ch.init(1)
        ch.step(5)
        outs.append((ch.accum().copy(), ch.state()["x"].copy(), ch.queue().copy()))
    oracle.set_threads(oracle.max_threads())
    assert (outs[0][0] == outs[1][0]).all() and (outs[0][1] == outs[1][1]).all() and (outs[0][2] == outs[1][2]).all()


def test_queue_is_sorted_killed_ids(oracle):
    sc = oracle.Scene(S.single_mode(0.2), oracle.F64)
    ch = oracle.Chains(sc, "diffusion_restore", 5000, seed=1, m=4.0)
    ch.init(0)
    ch.step(3)
    q, k = ch.queue(), ch.state()["killed"]
    assert (q == np.nonzero(k)[0]).all() and len(q) == ch.stats()["kills_last_step"] == ch.stats()["regen_queue_len"]
