"""Helpers of the GPU parity tests: GPU state vs oracle state under DESIGN.md Q15."""
import numpy as np

from oracle import oracle as O

METHODS = ["metropolis", "mala", "metropolis_restore", "mala_restore", "diffusion_restore"]


def min_image(v):
    return v - np.floor(v + 0.5)


def compare_states(gs, os_, g_last, o_last, stddev, check_score=True):
    """Per-chain comparison after one teacher-forced step.  Returns (diverged mask, report dict).

    A chain whose discrete decisions differ (path signature, accept flag, killed flag, pixel) is counted as
    diverged; every other chain must agree: x within 1e-4 * stddev (minimal image), p and f/p_hat within 1e-4
    relative (to max(value, eps)), score within 1e-4 relative + 1e-4 * stddev / (stddev^2 / 2) absolute.
    """
    g_acc, g_w = g_last
    o_acc, o_w = o_last
    div = (gs["sig"] != os_["sig"]) | (g_acc != o_acc) | (gs["killed"] != os_["killed"]) | (gs["pix"] != os_["pix"])
    ok = ~div
    dx = np.abs(min_image(gs["x"].astype(np.float64) - os_["x"])).max(1)
    rel = lambda a, b: np.abs(a - b) / np.maximum(np.abs(b), 1e-8)
    dp = rel(gs["p"].astype(np.float64), os_["p"])
    dfop = rel(gs["fop"].astype(np.float64), os_["fop"]).max(1)
    dw = rel(g_w.astype(np.float64), o_w)
    rep = dict(diverged=int(div.sum()), frac=float(div.mean()), dx=float(dx[ok].max(initial=0)), dp=float(dp[ok].max(initial=0)),
               dfop=float(dfop[ok].max(initial=0)), dw=float(dw[ok].max(initial=0)))
    assert rep["dx"] <= 1e-4 * stddev, rep
    assert rep["dp"] <= 1e-4 and rep["dfop"] <= 1e-4 and rep["dw"] <= 1e-4, rep
    if check_score:
        tol = 1e-4 * np.abs(os_["g"]) + 2e-4 / stddev
        dg = np.abs(gs["g"].astype(np.float64) - os_["g"]) - tol
        rep["dg_excess"] = float(dg[ok].max(initial=-1))
        assert rep["dg_excess"] <= 0, rep
    return div, rep


def oracle_chains(desc, method, n, seed, prec=O.F32, **kw):
    sc = O.Scene(desc, prec)
    return sc, O.Chains(sc, method, n, seed=seed, **kw)
