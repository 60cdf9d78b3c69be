"""Pins for the oracle's Lambert direction map (Q6; PAPER.md L775 pbrt `diffuse`).

What the mathematics fixes: a diffuse vertex that samples the outgoing direction with density cos(theta)/pi and
carries the weight `albedo` sends, into any polygon seen from the vertex, exactly the fraction given by the
point-to-polygon form factor (Lambert's formula)
    F = 1/(2 pi) * sum_edges gamma_i * (n . Gamma_i),
gamma_i = angle subtended by edge i, Gamma_i = unit normal of the plane through the vertex and edge i.
Nothing here re-types the oracle's map to produce an expected value: expected values are closed forms.  The maps
re-typed in `DIR_MAPS` only drive the sensitivity checks (a wrong map must fail the same assertion by a wide margin).
"""
import numpy as np

from dr_inputs import scenes as S

ALBEDO = 0.5          # power of two: f / ALBEDO is exact


# ---- closed forms ---------------------------------------------------------------------------------------------------
def form_factor_polygon(p, n, verts):
    """Lambert's formula: form factor from the differential element (p, n) to the polygon `verts` (k x 3), which must
    lie in the half space n.(v - p) >= 0.  Orientation-independent (absolute value)."""
    r = verts - p
    r /= np.linalg.norm(r, axis=1, keepdims=True)
    total = 0.0
    for i in range(len(r)):
        a, b = r[i], r[(i + 1) % len(r)]
        c = np.cross(a, b)
        s = np.linalg.norm(c)
        if s == 0.0:
            continue
        gamma = np.arctan2(s, np.dot(a, b))
        total += gamma * np.dot(n, c / s)
    return abs(total) / (2.0 * np.pi)


def form_factor_corner(a, b, h):
    """Textbook configuration factor: differential element parallel to an a x b rectangle at distance h, the element's
    normal passing through one corner of the rectangle."""
    A, B = np.hypot(a, h), np.hypot(b, h)
    return (a / A * np.arctan(b / A) + b / B * np.arctan(a / B)) / (2.0 * np.pi)


def form_factor_rect(x1, x2, z1, z2, h):
    """Element at the origin (normal +y), rectangle [x1,x2] x [z1,z2] in the plane y = h: signed corner sums."""
    g = lambda x, z: np.sign(x) * np.sign(z) * form_factor_corner(abs(x), abs(z), h) if x != 0 and z != 0 else 0.0
    return g(x2, z2) - g(x1, z2) - g(x2, z1) + g(x1, z1)


def solid_angle_triangle(p, tri):
    """Van Oosterom-Strackee."""
    a, b, c = (v - p for v in tri)
    la, lb, lc = np.linalg.norm(a), np.linalg.norm(b), np.linalg.norm(c)
    num = np.dot(a, np.cross(b, c))
    den = la * lb * lc + np.dot(a, b) * lc + np.dot(a, c) * lb + np.dot(b, c) * la
    return abs(2.0 * np.arctan2(num, den))


# ---- direction maps in the local frame (x, y tangent, z normal); only "cosine" is the claimed one ---------------------
DIR_MAPS = {
    "cosine": lambda u1, u2: (np.sqrt(u1) * np.cos(2 * np.pi * u2), np.sqrt(u1) * np.sin(2 * np.pi * u2), np.sqrt(1 - u1)),
    # uniform hemisphere (z = 1 - u1): a plausible mistake, biased by 2 cos(theta) with the weight `albedo`
    "uniform": lambda u1, u2: (np.sqrt(1 - (1 - u1) ** 2) * np.cos(2 * np.pi * u2),
                               np.sqrt(1 - (1 - u1) ** 2) * np.sin(2 * np.pi * u2), 1 - u1),
    # forgotten square root on the radius
    "r_equals_u1": lambda u1, u2: (u1 * np.cos(2 * np.pi * u2), u1 * np.sin(2 * np.pi * u2), np.sqrt(1 - u1 * u1)),
}


def grid(G):
    u = (np.arange(G) + 0.5) / G
    u1, u2 = np.meshgrid(u, u, indexing="ij")
    return u1.ravel(), u2.ravel()


def probe_states(G, L):
    """x = (film centre, u1, u2, 0...) on a G x G midpoint grid of the vertex-1 coordinates."""
    u1, u2 = grid(G)
    x = np.zeros((G * G, 2 * L))
    x[:, 0] = x[:, 1] = 0.5
    x[:, 2], x[:, 3] = u1, u2
    return x


def floor_probe(extra_quads, mats, L=2):
    """Camera straight above the origin looking down at a small Lambert floor patch in the plane y = 0 (normal +y);
    `extra_quads`: list of (p0, p1, p2, p3, material)."""
    mesh = S._Mesh()
    e = 0.01
    mesh.quad((-e, 0, -e), (-e, 0, e), (e, 0, e), (e, 0, -e), 0)
    for q in extra_quads:
        mesh.quad(*q)
    v, i, m = mesh.finish()
    return S.SceneDesc(v, i, m, np.stack(mats), cam_pos=(0, 0.5, 0), cam_look=(0, 0, 0), cam_up=(0, 0, 1), vfov_deg=1.0,
                       width=1, height=1, max_path_len=L)


# ---- (a) direct light from a parallel rectangle = albedo * Le * form factor ---------------------------------------------
RECT = dict(x1=0.2, x2=1.1, z1=-0.3, z2=0.6, h=1.0)
LE = 4.0


def rect_scene():
    r = RECT
    quad = ((r["x1"], r["h"], r["z1"]), (r["x2"], r["h"], r["z1"]), (r["x2"], r["h"], r["z2"]), (r["x1"], r["h"], r["z2"]), 1)  # normal -y
    return floor_probe([quad], [S.material(S.MAT_LAMBERT, (ALBEDO,) * 3), S.material(S.MAT_EMITTER, le=(LE,) * 3)])


def hits_rect(w):
    """Does the direction w = (wx, wy_tangent, wz_normal) from the origin reach RECT?  Local z = world +y; the
    azimuth convention does not matter for a set whose measure is compared (any rotation about the normal of the
    tangent frame maps the rectangle's image to a set of equal measure only if the map is isotropic, which all
    three maps are)."""
    wx, wy, wz = w
    with np.errstate(divide="ignore", invalid="ignore"):
        t = RECT["h"] / wz
        X, Z = wx * t, wy * t
    return (wz > 0) & (X >= RECT["x1"]) & (X <= RECT["x2"]) & (Z >= RECT["z1"]) & (Z <= RECT["z2"])


def test_two_closed_forms_agree():
    r = RECT
    poly = np.array([[r["x1"], r["h"], r["z1"]], [r["x2"], r["h"], r["z1"]], [r["x2"], r["h"], r["z2"]], [r["x1"], r["h"], r["z2"]]])
    a = form_factor_polygon(np.zeros(3), np.array([0.0, 1.0, 0.0]), poly)
    b = form_factor_rect(r["x1"], r["x2"], r["z1"], r["z2"], r["h"])
    assert abs(a - b) < 1e-14 and 0.05 < a < 0.2


def test_lambert_direct_light_equals_form_factor(oracle):
    G = 2000
    sc = oracle.Scene(rect_scene(), oracle.F64, use_bvh=False)
    e = sc.eval(probe_states(G, 2), False)
    f = e["f"][:, 0]
    assert np.isin(f, [0.0, ALBEDO * LE]).all()                      # weight = albedo, emission seen once
    assert (e["nrays"] == 2).all()
    F = form_factor_rect(**RECT)
    got = f.mean() / (ALBEDO * LE)
    tol = 2e-4 * F                                                   # midpoint rule on an indicator: boundary cells / G^2
    assert abs(got - F) <= tol, (got, F)
    # sensitivity: the same quadrature with a wrong map misses by far more than 10 x the tolerance
    u1, u2 = grid(G)
    assert abs(hits_rect(DIR_MAPS["cosine"](u1, u2)).mean() - F) <= tol
    for wrong in ("uniform", "r_equals_u1"):
        miss = abs(hits_rect(DIR_MAPS[wrong](u1, u2)).mean() - F)
        assert miss > 100 * tol, (wrong, miss)


# ---- (b) the whole distribution: dome of uniquely emitting triangles -----------------------------------------------------
N_THETA, N_PHI, R_DOME = 12, 24, 8.0


def dome_scene():
    """Lat-long dome around the origin above the floor plane plus a skirt below it; triangle j emits j + 1."""
    th = np.linspace(0.0, np.pi / 2, N_THETA + 1)
    ph = np.linspace(0.0, 2 * np.pi, N_PHI + 1)
    pt = lambda t, p: R_DOME * np.array([np.sin(t) * np.cos(p), np.cos(t), np.sin(t) * np.sin(p)])
    tris = []
    for i in range(N_THETA):
        for j in range(N_PHI):
            a, b, c, d = pt(th[i], ph[j]), pt(th[i + 1], ph[j]), pt(th[i + 1], ph[j + 1]), pt(th[i], ph[j + 1])
            if i > 0:
                tris.append((a, b, d))
            tris.append((b, c, d))
    for j in range(N_PHI):                                           # skirt: horizon ring down to y = -1
        b, c = pt(np.pi / 2, ph[j]), pt(np.pi / 2, ph[j + 1])
        lo = np.array([0.0, 1.0, 0.0])
        tris += [(b, b - lo, c), (c, b - lo, c - lo)]
    mesh = S._Mesh()
    e = 0.01
    mesh.quad((-e, 0, -e), (-e, 0, e), (e, 0, e), (e, 0, -e), 0)
    mats = [S.material(S.MAT_LAMBERT, (ALBEDO,) * 3)]
    centre = np.array([0.0, 1.0, 0.0])
    for k, (a, b, c) in enumerate(tris):
        if np.dot(np.cross(b - a, c - a), centre - a) < 0:            # front (emitting) side faces inwards
            b, c = c, b
        mesh.add(np.stack([a, b, c]), [(0, 1, 2)], len(mats))
        mats.append(S.material(S.MAT_EMITTER, le=(float(k + 1),) * 3))
        tris[k] = (a, b, c)
    v, i, m = mesh.finish()
    desc = S.SceneDesc(v, i, m, np.stack(mats), cam_pos=(0, 0.5, 0), cam_look=(0, 0, 0), cam_up=(0, 0, 1), vfov_deg=1.0,
                       width=1, height=1, max_path_len=2)
    return desc, np.array([np.stack(t) for t in tris])


def test_lambert_distribution_matches_form_factors(oracle):
    desc, tris = dome_scene()
    n_up = len(tris) - 2 * N_PHI
    sc = oracle.Scene(desc, oracle.F64)
    G = 60 * N_PHI                                                    # whole grid columns per azimuth bin
    e = sc.eval(probe_states(G, 2), False)
    idx = e["f"][:, 0] / ALBEDO - 1.0
    assert (idx == np.round(idx)).all() and (idx >= 0).all()          # every path ends on exactly one emitter
    idx = idx.astype(np.int64)
    counts = np.bincount(idx, minlength=len(tris)) / float(G * G)
    # the ray starts eps_ray above the floor, so nothing lands on the skirt below the horizon
    assert counts[n_up:].sum() < 1e-4
    p0 = np.array([0.0, sc.eps_ray, 0.0])
    n = np.array([0.0, 1.0, 0.0])
    v32 = tris.astype(np.float32).astype(np.float64)                  # the scene stores float32 vertices
    F = np.array([form_factor_polygon(p0, n, t) for t in v32[:n_up]])
    assert abs(F.sum() - 1.0) < 1e-3                                  # the dome closes the hemisphere
    tol = 2.5e-5                                                      # boundary cells of a bin / G^2
    assert np.abs(counts[:n_up] - F).max() <= tol, np.abs(counts[:n_up] - F).max()
    # sensitivity: a uniform-hemisphere map would fill bin j with solid_angle_j / (2 pi)
    uni = np.array([solid_angle_triangle(p0, t) for t in v32[:n_up]]) / (2 * np.pi)
    assert abs(uni.sum() - 1.0) < 1e-3
    assert np.abs(uni - F).max() > 100 * tol
    # moments of cos(theta) and azimuthal uniformity, from the bins (centroid directions)
    c = v32[:n_up].mean(1) - p0
    c /= np.linalg.norm(c, axis=1, keepdims=True)
    cos_t = c[:, 1]
    w = counts[:n_up]
    assert abs((w * cos_t).sum() - 2.0 / 3.0) < 2e-3                  # E[w.n] = 2/3    (uniform: 1/2, r = u1: pi/4)
    assert abs((w * cos_t ** 2).sum() - 0.5) < 3e-3                   # E[(w.n)^2] = 1/2 (uniform: 1/3, r = u1: 2/3)
    phi_bin = np.floor((np.arctan2(c[:, 2], c[:, 0]) % (2 * np.pi)) / (2 * np.pi / N_PHI)).astype(int)
    per_phi = np.bincount(phi_bin, weights=w, minlength=N_PHI)
    assert np.abs(per_phi - 1.0 / N_PHI).max() < 2e-4                 # uniform azimuth


def test_lambert_two_sided_flip(oracle):
    """Seen from below, the same floor patch scatters into the lower hemisphere with the same law (Q6: the frame flips
    with the normal that faces the incoming ray)."""
    r = RECT
    quad = ((r["x1"], -r["h"], r["z1"]), (r["x1"], -r["h"], r["z2"]), (r["x2"], -r["h"], r["z2"]), (r["x2"], -r["h"], r["z1"]), 1)  # normal +y
    desc = floor_probe([quad], [S.material(S.MAT_LAMBERT, (ALBEDO,) * 3), S.material(S.MAT_EMITTER, le=(LE,) * 3)])
    desc.cam_pos = (0, -0.5, 0)
    G = 1000
    e = oracle.Scene(desc, oracle.F64, use_bvh=False).eval(probe_states(G, 2), False)
    F = form_factor_rect(**RECT)
    assert abs(e["f"][:, 0].mean() / (ALBEDO * LE) - F) <= 1e-3 * F
