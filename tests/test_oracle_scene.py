"""Pins for the oracle's closest-hit query (Q8) and camera / pixel map (Q4)."""
import numpy as np

from dr_inputs import scenes as S


def textbook_closest_hit(desc, o, d):
    """Independent definition: solve o + t d = v0 + a e1 + b e2 with numpy's linear solver per triangle."""
    v = desc.vertices.astype(np.float64)
    tri = desc.indices
    v0, e1, e2 = v[tri[:, 0]], v[tri[:, 1]] - v[tri[:, 0]], v[tri[:, 2]] - v[tri[:, 0]]
    best_t, best_i = np.inf, -1
    for i in range(len(tri)):
        A = np.stack([-d, e1[i], e2[i]], axis=1)
        if abs(np.linalg.det(A)) < 1e-14:
            continue
        t, a, b = np.linalg.solve(A, o - v0[i])
        if t > 0 and a >= 0 and b >= 0 and a + b <= 1 and t < best_t:
            best_t, best_i = t, i
    return best_t, best_i


def test_brute_force_matches_textbook_solve(oracle):
    desc = S.mini_machines(n_objects=6)
    sc = oracle.Scene(desc, oracle.F64)
    o, d = S.seeded_rays(desc, 150, 1)
    t, tri = sc.trace(o, d, brute=True)
    agree = 0
    for k in range(len(o)):
        bt, bi = textbook_closest_hit(desc, o[k].astype(np.float64), d[k].astype(np.float64))
        if bi < 0:
            assert tri[k] == -1
        else:
            # an edge-grazing ray may legitimately pick the neighbour; otherwise identical
            assert np.isclose(t[k], bt, rtol=1e-9)
            agree += int(tri[k] == bi)
    assert agree >= 0.97 * (tri >= 0).sum() and (tri >= 0).sum() > 50


def test_bvh_equals_brute_force(oracle):
    for desc in (S.mini_machines(), S.furnace(level=3), S.cornell()):
        for prec in (oracle.F64, oracle.F32):
            sc = oracle.Scene(desc, prec)
            o, d = S.seeded_rays(desc, 4000, 2)
            t1, i1 = sc.trace(o, d, brute=True)
            t2, i2 = sc.trace(o, d, brute=False)
            assert (i1 == i2).all() and (t1 == t2).all()
            assert (i1 >= 0).mean() > 0.2


def test_tie_rule_smaller_index_wins(oracle):
    # two coincident triangles: the hit must report the smaller index (Q8)
    v = np.array([[0, 0, 1], [1, 0, 1], [0, 1, 1]], dtype=np.float32)
    desc = S.SceneDesc(np.concatenate([v, v]), np.array([[3, 4, 5], [0, 1, 2]], dtype=np.uint32), np.zeros(2, dtype=np.uint32),
                       np.stack([S.material(0, (0.5,) * 3)]), width=4, height=4, max_path_len=2)
    for brute in (True, False):
        t, i = oracle.Scene(desc, oracle.F64).trace([[0.2, 0.2, 0]], [[0, 0, 1]], brute=brute)
        assert i[0] == 0 and t[0] == 1.0
    # origin on the surface: t = 0 is excluded (t_min = 0 exclusive)
    t, i = oracle.Scene(desc, oracle.F64).trace([[0.2, 0.2, 1]], [[0, 0, 1]], brute=True)
    assert i[0] == -1


def test_pixel_index_and_camera(oracle):
    """Q4: pix = min(floor(x1 H), H-1) W + min(floor(x0 W), W-1); the film centre looks along `look - pos`."""
    desc = S.furnace(width=8, height=4)
    sc = oracle.Scene(desc, oracle.F64)
    x = np.zeros((4, desc.dim))
    x[0, :2] = (0.0, 0.0)
    x[1, :2] = (0.999999, 0.0)
    x[2, :2] = (0.0, 0.999999)
    x[3, :2] = (0.5, 0.5)
    e = sc.eval(x, False)
    assert list(e["pix"]) == [0, 7, 24, 2 * 8 + 4]
    # film centre hits the sphere head-on: f = albedo * env = 0.5
    assert e["f"][3, 0] == 0.5 and e["nrays"][3] == 2
    # corner rays of a 40-degree camera 4 units away miss the unit sphere
    assert e["f"][0, 0] == 1.0 and e["nrays"][0] == 1
