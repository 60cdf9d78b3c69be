"""Pin for the oracle's Q18 branch (Q18; "non-finite f or score -> treated as p = 0, counted";
S:L35 "NaN propagation is never silent"): oracle/samplers.hpp evaluate().

What fixes the result without the branch itself: the SAME states evaluated in fp64, where nothing overflows.  The fp32
evaluation must flag exactly the states whose fp64 value does not fit fp32, return f = p = 0 and a zero score for them, and
leave every other state alone.
 * f overflows: a closed box with Lambert albedo 2 (allowed: the description only asks for finite numbers) and an emitting
   ceiling of radiance 1e38.  A path that reaches the ceiling after k bounces carries f = 2^k * 1e38 (closed form: cosine
   sampling makes the throughput of a Lambert bounce the albedo, Q6), which fits fp32 for k = 1 and not for k >= 2.
 * only the score overflows: the GGX room with its emitters scaled to 1e38.  f <= 1e38 fits, the derivative of f does not
   where |grad ln p| (p + eps) exceeds FLT_MAX.  The duals of the three colour channels can leave fp32 a little earlier than
   the gradient of their luminance, so the states with FLT_MAX / 8 < |grad p| <= FLT_MAX may go either way.
"""
import copy

import numpy as np

from dr_inputs import scenes as S

FLT_MAX = float(np.finfo(np.float32).max)


def overflow_box():
    return S.closed_furnace(albedo=2.0, emission=1e38)


def bright_ggx_room():
    d = copy.copy(S.ggx_room())
    d.materials = d.materials.copy()
    d.materials[:, 6:9] *= 1e38 / d.materials[:, 6:9].max()
    d.name = "ggx_room_1e38"
    return d


def test_overflowing_f_is_zeroed_and_counted(oracle):
    desc = overflow_box()
    x = S.seeded_states(4000, desc.dim, 31).astype(np.float64)
    for want_score in (False, True):
        a = oracle.Scene(desc, oracle.F32).eval(x, want_score)
        b = oracle.Scene(desc, oracle.F64).eval(x, want_score)
        assert (a["sig"] == b["sig"]).all() and not b["nonfinite"].any()
        k = np.round(np.log2(np.maximum(b["f"][:, 0], 1e38) / 1e38)).astype(int)         # bounces before the ceiling
        lit = b["f"][:, 0] > 0
        assert np.allclose(b["f"][lit, 0], 1e38 * 2.0 ** k[lit], rtol=1e-6) and set(np.unique(k[lit])) >= {1, 2, 3}
        overflow = lit & (k >= 2)
        assert overflow.sum() > 500 and (lit & (k == 1)).sum() > 300
        flagged = a["nonfinite"].astype(bool)
        assert np.array_equal(flagged, overflow)                                          # exactly the states whose f does not fit fp32
        assert not a["f"][flagged].any() and not a["p"][flagged].any()
        if want_score:
            assert not a["g"][flagged].any()
        keep = lit & ~overflow
        assert np.allclose(a["f"][keep], b["f"][keep], rtol=1e-6) and np.allclose(a["p"][keep], b["p"][keep], rtol=1e-6)
        assert np.isfinite(a["f"]).all() and np.isfinite(a["g"]).all()


def test_overflowing_score_is_zeroed_and_counted(oracle):
    desc = bright_ggx_room()
    x = S.seeded_states(60000, desc.dim, 32).astype(np.float64)
    a = oracle.Scene(desc, oracle.F32).eval(x, True)
    b = oracle.Scene(desc, oracle.F64).eval(x, True)
    v = oracle.Scene(desc, oracle.F32).eval(x, False)                                     # values only: nothing to overflow
    assert not b["nonfinite"].any() and not v["nonfinite"].any() and b["f"].max() <= 1e38 * (1 + 1e-6)
    same = a["sig"] == b["sig"]
    assert same.mean() > 0.999
    grad_p = np.abs(b["g"]).max(1) * (b["p"] + 1e-8)                                      # |grad p| from g = grad p / (p + eps)
    flagged = a["nonfinite"].astype(bool)
    must, must_not = same & (grad_p > FLT_MAX), same & (grad_p < FLT_MAX / 8)
    assert must.sum() >= 20 and flagged[must].all()
    assert not flagged[must_not].any() and (must_not & (b["p"] > 0)).sum() > 1000
    assert not a["f"][flagged].any() and not a["p"][flagged].any() and not a["g"][flagged].any()
    assert (v["p"][flagged] > 0).all()                     # the value alone was fine: the score is what made these states zero-contribution
    keep = same & ~flagged
    assert np.allclose(a["f"][keep], v["f"][keep], rtol=1e-5) and np.isfinite(a["g"]).all()     # the others are untouched


def test_chains_count_nonfinite_evaluations_and_never_move_onto_them(oracle):
    """Alg. 2 with Q18: a proposal whose evaluation was zeroed has p = 0, so plain Metropolis rejects it (ratio 0) and
    a Restore chain that regenerates onto it is killed again at once; the counter equals the flagged evaluations."""
    desc = overflow_box()
    sc = oracle.Scene(desc, oracle.F32)
    N = 3000
    ch = oracle.Chains(sc, "metropolis", N, seed=5, large_step_prob=1.0)                  # every proposal is a fresh uniform state
    ch.init(1)
    st0 = ch.state()
    bad0 = sc.eval(st0["x"], False)["nonfinite"].astype(bool)
    assert ch.stats()["nonfinite"] == bad0.sum() > 500 and not st0["p"][bad0].any()
    ch.step(1)
    st1, (accepted, _) = ch.state(), ch.last()
    moved = (st1["x"] != st0["x"]).any(1)
    assert (moved == accepted.astype(bool)).all() and moved.sum() > 100
    lit0 = st0["p"] > 0
    assert (lit0 & moved).sum() > 50 and (st1["p"][lit0 & moved] > 0).all()   # a lit chain never moves onto a zeroed (or dark) state: ratio eps / p_hat
    assert ch.stats()["nonfinite"] > bad0.sum()             # the step's proposals were counted too
    assert np.isfinite(ch.accum()).all()
