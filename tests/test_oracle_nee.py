"""Pins for the oracle's next-event estimation + MIS (Q21).

What fixes the result with no implementation to compare against:
 * direct light on a Lambert plane under a parallel rectangle = albedo * Le * form factor (closed form, the one that pins
   the Lambert map in test_oracle_lambert.py), whatever the MIS weights are as long as they sum to one per path;
 * the two weights of ONE path (found by the direction sample, found by the emitter sample) sum to one;
 * the expectation of f does not depend on the estimator: uniform-sample means with and without next-event estimation
   agree (Lambert box and the GGX / dielectric room), while the variance drops;
 * the score equals central differences of ln(p + eps) with the geometry and MIS terms live.
"""
import copy

import numpy as np

from dr_inputs import scenes as S
from test_oracle_lambert import ALBEDO, LE, RECT, form_factor_rect, grid, rect_scene


def nee_scene(desc):
    d = copy.copy(desc)
    d.nee = True
    return d


def states(G, d, u=None, v=None):
    """(film centre | vertex-1 coordinates): a G x G grid over (u1, u2) with (v1, v2) fixed, or the other way round."""
    a, b = grid(G)
    x = np.zeros((G * G, d))
    x[:, 0] = x[:, 1] = 0.5
    if u is None:
        x[:, 4], x[:, 5], x[:, 6], x[:, 7] = a, b, v[0], v[1]
    else:
        x[:, 4], x[:, 5], x[:, 6], x[:, 7] = u[0], u[1], a, b
    return x


def test_direct_light_equals_form_factor_with_nee(oracle):
    desc = nee_scene(rect_scene())
    assert desc.dim == 8
    sc = oracle.Scene(desc, oracle.F64, use_bvh=False)
    G = 1000
    u0, v0 = (0.3, 0.7), (0.4, 0.6)
    # L = 2: f(u, v) = [emitter found by the direction sample](u) + [connection to the emitter sample](v)
    fu = sc.eval(states(G, 8, v=v0), False)["f"][:, 0]
    fv = sc.eval(states(G, 8, u=u0), False)["f"][:, 0]
    f00 = sc.eval(np.array([[0.5, 0.5, 0, 0, u0[0], u0[1], v0[0], v0[1]]]), False)["f"][0, 0]
    total = fu.mean() + fv.mean() - f00
    F = form_factor_rect(**RECT)
    assert abs(total / (ALBEDO * LE) - F) <= 5e-4 * F, (total / (ALBEDO * LE), F)
    # both techniques do real work here: neither term is negligible
    assert fv.std() > 0 and (fu > f00 * 0 + fv.min() * 0).all() and (fu != fu[0]).any() and fv.mean() > 0.05 * total
    # without next-event estimation the same expectation comes from the direction sample alone (test_oracle_lambert.py)


def test_mis_weights_of_one_path_sum_to_one(oracle):
    """The same light path generated both ways: floor point P = origin, emitter point y.  w_b = f_bsdf / (albedo Le);
    w_l = f_nee p_l pi / (albedo Le cos_x), with p_l = r^2 / (cos_l A) from the geometry."""
    desc = nee_scene(rect_scene())
    sc = oracle.Scene(desc, oracle.F64, use_bvh=False)
    r = RECT
    area = (r["x2"] - r["x1"]) * (r["z2"] - r["z1"])
    rng = np.random.default_rng(3)
    for _ in range(20):
        v1, v2 = rng.uniform(0.05, 0.95, 2)
        # the oracle's emitter sample for (v1, v2): recover y from the NEE term with L = 2 and a direction sample that misses
        x = np.array([[0.5, 0.5, 0, 0, 0.999, 0.5, v1, v2]])            # u1 ~ 1: grazing direction, misses the rectangle
        f_nee = sc.eval(x, False)["f"][0, 0]
        assert f_nee > 0
        # y by the documented map: triangle by area, su = sqrt(v1'), y = v0 + e1 su (1 - v2) + e2 su v2
        quad = np.array([[r["x1"], r["h"], r["z1"]], [r["x2"], r["h"], r["z1"]], [r["x2"], r["h"], r["z2"]], [r["x1"], r["h"], r["z2"]]])
        tris = [(quad[0], quad[1], quad[2]), (quad[0], quad[2], quad[3])]       # _Mesh.quad order
        j = 0 if v1 < 0.5 else 1
        v1r = v1 * 2 - j
        a0, a1, a2 = tris[j]
        su = np.sqrt(v1r)
        y = a0 + (a1 - a0) * su * (1 - v2) + (a2 - a0) * su * v2
        P = np.array([0.0, 0.0, 0.0])
        w = (y - P) / np.linalg.norm(y - P)
        cos_x, cos_l, r2 = w[1], w[1], float(np.dot(y - P, y - P))
        p_l = r2 / (cos_l * area)
        w_l = f_nee * p_l * np.pi / (ALBEDO * LE * cos_x)
        # direction sample that reaches the same y: invert the cosine map in the Q6 frame of the floor triangle
        # (t = normalize(v1 - v0) of the first floor triangle = +z, n = +y, b = n x t = +x)
        wx, wy, wz = w[2], w[0], w[1]                                    # components along t, b, n
        u1 = 1 - wz * wz
        u2 = (np.arctan2(wy, wx) / (2 * np.pi)) % 1.0
        x = np.array([[0.5, 0.5, 0, 0, u1, u2, 0.9999, 0.9999]])
        e = sc.eval(x, False)
        f_both = e["f"][0, 0]
        # subtract the NEE term of THIS state (its own v): evaluate it with a direction that misses
        x2 = x.copy(); x2[0, 4] = 0.999; x2[0, 5] = 0.5
        f_bsdf = f_both - sc.eval(x2, False)["f"][0, 0]
        w_b = f_bsdf / (ALBEDO * LE)
        assert 0 < w_b < 1 and 0 < w_l < 1
        assert abs(w_b + w_l - 1.0) < 3e-5, (w_b, w_l)                   # eps_ray offset of the direction sample's origin: O(1e-5)


def uniform_mean(sc, n, seed):
    rng = np.random.default_rng(seed)
    x = rng.random((n, sc.dim))
    e = sc.eval(x, False)
    return e["f"][:, 0], e["nrays"]


def test_expectation_does_not_depend_on_the_estimator(oracle):
    """Uniform PSS samples: the mean of f is the image integral either way (MIS is unbiased); next-event estimation
    lowers the variance by a large factor on a small light."""
    for make in (lambda: S.cornell(width=4, height=4, max_path_len=4), lambda: S.ggx_room(width=4, height=4, max_path_len=4)):
        desc = make()
        n = 400000
        f0, _ = uniform_mean(oracle.Scene(desc, oracle.F64), n, 1)
        f1, nr = uniform_mean(oracle.Scene(nee_scene(desc), oracle.F64), n, 2)
        se = np.hypot(f0.std() / np.sqrt(n), f1.std() / np.sqrt(n))
        assert abs(f0.mean() - f1.mean()) < 4 * se, (desc.name, f0.mean(), f1.mean(), se)
        assert f1.mean() > 20 * se                                        # the comparison has resolution
        assert f1.var() < 0.8 * f0.var()
        assert (f1 > 0).mean() > 2 * (f0 > 0).mean()                      # many more uniform samples are lit (zeta)
        assert nr.mean() > 4                                              # shadow rays are counted


def test_score_matches_finite_differences_with_nee(oracle):
    for make in (S.ggx_room, S.mini_machines, lambda: S.cornell(width=8, height=8, max_path_len=4)):
        desc = nee_scene(make())
        sc = oracle.Scene(desc, oracle.F64)
        x = np.random.default_rng(5).random((3000, desc.dim))
        e = sc.eval(x, True)
        lit = np.flatnonzero(e["p"] > 1e-4)[:60]
        assert len(lit) >= 30
        checked = 0

        def fd(i, h):
            g = np.zeros(desc.dim)
            for j in range(desc.dim):
                xp, xm = x[i].copy(), x[i].copy()
                xp[j] += h; xm[j] -= h
                ep, em = sc.eval(xp[None], False), sc.eval(xm[None], False)
                if ep["sig"][0] != e["sig"][i] or em["sig"][0] != e["sig"][i]:      # a discrete decision flips inside the stencil
                    return None
                g[j] = (np.log(ep["p"][0] + 1e-8) - np.log(em["p"][0] + 1e-8)) / (2 * h)
            return g

        for i in lit:
            g, g2 = fd(i, 1e-6), fd(i, 2.5e-7)
            if g is None or g2 is None or not np.allclose(g, g2, rtol=1e-3, atol=1e-3 * (1 + np.abs(g).max())):
                continue        # the stencil straddles a kink (e.g. the choice of emitter triangle, which is not in the signature)
            checked += 1
            assert np.allclose(e["g"][i], g2, rtol=1e-3, atol=1e-3 * (1 + np.abs(g2).max())), (desc.name, i, e["g"][i], g2)
        assert checked >= 15, (desc.name, checked)
        assert (np.abs(e["g"][lit]).max(1) > 0).mean() > 0.9              # with NEE the score is live on diffuse paths too


def degenerate_emitter_appended(desc):
    """The same scene with one more emitter triangle, of zero area (three times the same vertex), LAST in triangle order."""
    d = copy.copy(desc)
    light = int(np.flatnonzero(desc.materials[:, 0] == 3)[0])
    nv = len(desc.vertices)
    d.vertices = np.concatenate([desc.vertices, np.array([[0.5, 0.5, 0.5]], dtype=np.float32)])
    d.indices = np.concatenate([desc.indices, np.array([[nv, nv, nv]], dtype=np.uint32)])
    d.tri_material = np.concatenate([desc.tri_material, np.array([light], dtype=np.uint32)])
    return d


def test_an_emitter_without_area_is_never_sampled(oracle):
    """DESIGN.md Q21 (emitters are drawn by area; PAPER.md L735, L757 leave the construction open): a zero-area emitter has
    probability zero.  Appending one to a scene changes nothing, also with v1 at the top of [0, 1); and when it is the ONLY
    emitter no vertex makes a connection: the evaluation is that of the direction sample alone, not 0/0."""
    base = nee_scene(S.cornell(width=32, height=32, max_path_len=4))
    plus = degenerate_emitter_appended(base)
    x = S.seeded_states(4000, base.dim, 21).astype(np.float64)
    x[:2000, 6::4] = 1.0 - 2.0 ** -24                      # v1 of every vertex at the top of [0, 1)
    for prec in (oracle.F32, oracle.F64):
        a = oracle.Scene(base, prec, use_bvh=False).eval(x, True)
        b = oracle.Scene(plus, prec, use_bvh=False).eval(x, True)
        assert not b["nonfinite"].any()
        for k in ("f", "p", "pix", "sig", "g"):
            assert np.array_equal(a[k], b[k]), k
        assert (a["p"][:2000] > 0).sum() > 200             # the corner case is exercised on lit paths
    # the only emitter has no area: light comes from the environment alone
    dark = copy.copy(plus)
    dark.tri_material = plus.tri_material.copy()
    dark.tri_material[:-1][plus.tri_material[:-1] == plus.tri_material[-1]] = 0     # the ceiling light becomes a white wall
    dark.env_radiance = (1.0, 0.5, 0.25)
    plain = copy.copy(dark)
    plain.nee = False
    xp = np.ascontiguousarray(x.reshape(len(x), -1, 4)[:, :, :2].reshape(len(x), -1))   # (u1, u2) of every vertex
    for prec in (oracle.F32, oracle.F64):
        a = oracle.Scene(dark, prec, use_bvh=False).eval(x, True)
        b = oracle.Scene(plain, prec, use_bvh=False).eval(xp, True)
        assert not a["nonfinite"].any() and (a["p"] > 0).mean() > 0.3
        assert np.array_equal(a["f"], b["f"]) and np.array_equal(a["pix"], b["pix"])
        g = a["g"].reshape(len(x), -1, 4)
        assert np.array_equal(np.ascontiguousarray(g[:, :, :2]).reshape(len(x), -1), b["g"]) and not g[:, :, 2:].any()
