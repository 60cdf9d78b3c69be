"""Helpers of the GPU parity tests: GPU state vs oracle state under DESIGN.md Q15."""
import numpy as np

from oracle import oracle as O

METHODS = ["metropolis", "mala", "metropolis_restore", "mala_restore", "diffusion_restore"]


def min_image(v):
    return v - np.floor(v + 0.5)


def compare_states(gs, os_, g_last, o_last, stddev, check_score=True, fold_outliers=False):
    """Per-chain comparison after one teacher-forced step.  Returns (diverged mask, report dict).

    A chain whose discrete decisions differ (path signature, accept flag, killed flag, pixel) is counted as
    diverged; every other chain must agree: x within 1e-4 * stddev (minimal image), p and f/p_hat within 1e-4
    relative (to max(value, eps)), score within 1e-4 relative + 1e-4 * stddev / (stddev^2 / 2) absolute.
    fold_outliers (scenes with next-event estimation): a chain whose VALUES miss those tolerances is counted with the
    diverged ones instead of failing the test -- an emitter connection that grazes the emitter or is very short divides
    by a cancelled fp32 quantity (cos_l, r^2), on either side; the caller bounds the total fraction.
    """
    g_acc, g_w = g_last
    o_acc, o_w = o_last
    div = (gs["sig"] != os_["sig"]) | (g_acc != o_acc) | (gs["killed"] != os_["killed"]) | (gs["pix"] != os_["pix"])
    dx = np.abs(min_image(gs["x"].astype(np.float64) - os_["x"])).max(1)
    rel = lambda a, b: np.abs(a - b) / np.maximum(np.abs(b), 1e-8)
    dp = rel(gs["p"].astype(np.float64), os_["p"])
    dfop = rel(gs["fop"].astype(np.float64), os_["fop"]).max(1)
    dw = rel(g_w.astype(np.float64), o_w)
    out = (dx > 1e-4 * stddev) | (dp > 1e-4) | (dfop > 1e-4) | (dw > 1e-4)
    dg = None
    if check_score:
        tol = 1e-4 * np.abs(os_["g"]) + 2e-4 / stddev
        dg = (np.abs(gs["g"].astype(np.float64) - os_["g"]) - tol).max(1)
        out |= dg > 0
    n_out = int((out & ~div).sum())
    if fold_outliers:
        div = div | out
    ok = ~div
    rep = dict(diverged=int(div.sum()), frac=float(div.mean()), dx=float(dx[ok].max(initial=0)), dp=float(dp[ok].max(initial=0)),
               dfop=float(dfop[ok].max(initial=0)), dw=float(dw[ok].max(initial=0)), value_outliers=n_out)
    assert rep["dx"] <= 1e-4 * stddev, rep
    assert rep["dp"] <= 1e-4 and rep["dfop"] <= 1e-4 and rep["dw"] <= 1e-4, rep
    if check_score:
        rep["dg_excess"] = float(dg[ok].max(initial=-1))
        assert rep["dg_excess"] <= 0, rep
    return div, rep


def oracle_chains(desc, method, n, seed, prec=O.F32, **kw):
    sc = O.Scene(desc, prec)
    return sc, O.Chains(sc, method, n, seed=seed, **kw)


def splats(state, last):
    """Per-chain splat of the last Accumulate (Alg. 1 L522-L525 + the ratio channel of Q12): (pixel, [w f/p_hat, w/p_hat])."""
    _, w = last
    w = np.asarray(w, dtype=np.float64)
    p = np.asarray(state["p"], dtype=np.float64)
    on = p > 0
    v = np.concatenate([w[:, None] * np.asarray(state["fop"], dtype=np.float64), (w / (p + 1e-8))[:, None]], axis=1)
    return state["pix"], v * on[:, None]


def accum_without(accum, state, last, mask):
    """accum (npix x 4, float64) minus the splats of the chains in `mask`."""
    pix, v = splats(state, last)
    out = np.array(accum, dtype=np.float64)
    np.subtract.at(out, pix[mask], v[mask])
    return out


def largest_addend(state, last, npix):
    """Per pixel, the largest |splat| component that went into it (scale of the fp32 rounding of its atomic sum)."""
    pix, v = splats(state, last)
    out = np.zeros(npix)
    np.maximum.at(out, pix, np.abs(v).max(1))
    return out


def compare_bulk(gch, och, gs, os_, g_last, o_last, div, tours_g, tours_o):
    """Queue, tourCount delta and accumulation buffer of one teacher-forced step, with the diverged chains masked out
    (their own splats subtracted on each side) instead of skipping the comparison."""
    keep = ~div
    gq, oq = gch.queue(), och.queue()
    assert np.array_equal(gq[keep[gq]], oq[keep[oq]])                                   # regeneration queue: bit-exact, ascending
    assert np.array_equal(gq, np.flatnonzero(gs["killed"])) and np.array_equal(oq, np.flatnonzero(os_["killed"]))
    assert tours_g - int(gs["killed"][div].sum()) == tours_o - int(os_["killed"][div].sum())
    npix = gch.scene.npix
    ga = accum_without(gch.accum.cpu().numpy(), gs, g_last, div)
    oa = accum_without(och.accum(), os_, o_last, div)
    # per pixel: 1e-4 relative + rounding of an fp32 atomic sum (a few ulps of the largest addend per addend)
    big = np.maximum(largest_addend(gs, g_last, npix), largest_addend(os_, o_last, npix))
    cnt = np.bincount(os_["pix"], minlength=npix) + 2
    tol = 1e-4 * np.abs(oa) + (4e-7 * cnt * big)[:, None] + 1e-30
    bad = np.abs(ga - oa) > tol
    assert not bad.any(), (int(bad.sum()), float((np.abs(ga - oa) / tol).max()))
