"""TEST INFRASTRUCTURE — ctypes front end of the CPU oracle (oracle/liboracle.so).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
may import this module.  It never touches the CUDA library.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

F32, F64 = 0, 1
METHODS = {"metropolis": 0, "mala": 1, "metropolis_restore": 2, "mala_restore": 3, "diffusion_restore": 4, "path_tracing": 5}

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        L = _lib
        vp, u32, u64, i32, f64, f32 = C.c_void_p, C.c_uint32, C.c_uint64, C.c_int, C.c_double, C.c_float
        L.orc_scene_create.restype = vp
        L.orc_scene_create.argtypes = [i32, vp, u32, vp, u32, vp, vp, u32, vp, vp, f32, u32, u32, u32, i32, i32]
        L.orc_scene_create_analytic2d.restype = vp
        L.orc_scene_create_analytic2d.argtypes = [i32, u32, vp, vp, vp, vp, u32, u32]
        L.orc_scene_destroy.argtypes = [vp]
        L.orc_scene_dim.restype = u32
        L.orc_scene_dim.argtypes = [vp]
        L.orc_scene_eps_ray.restype = f64
        L.orc_scene_eps_ray.argtypes = [vp]
        L.orc_trace.argtypes = [vp, vp, vp, u32, i32, vp, vp]
        L.orc_eval.argtypes = [vp, vp, u32, i32, vp, vp, vp, vp, vp, vp, vp]
        L.orc_pt_render.argtypes = [vp, u64, u64, vp]
        L.orc_bias_field.argtypes = [vp, f64, f64, f64, u32, u32, vp]
        L.orc_chains_create.restype = vp
        L.orc_chains_create.argtypes = [vp, i32, u32, f64, f64, f64, f64, f64, f64, u64, u32, i32]
        L.orc_chains_destroy.argtypes = [vp]
        L.orc_chains_set_f4.argtypes = [vp, i32, u32, vp]
        L.orc_chains_init.argtypes = [vp, u32]
        L.orc_chains_step.argtypes = [vp, u32]
        L.orc_chains_get_state.argtypes = [vp] * 8
        L.orc_chains_set_state.argtypes = [vp] * 7 + [u32]
        L.orc_chains_last.argtypes = [vp, vp, vp]
        L.orc_chains_accum.argtypes = [vp, vp]
        L.orc_chains_zero_accum.argtypes = [vp]
        L.orc_chains_resolve.restype = i32
        L.orc_chains_resolve.argtypes = [vp, vp]
        L.orc_chains_stats.argtypes = [vp, vp]
        L.orc_chains_queue.restype = u32
        L.orc_chains_queue.argtypes = [vp, vp]
        L.orc_philox.argtypes = [vp, vp, vp]
        L.orc_stream_block.argtypes = [u64, u32, u32, u32, u32, u32, vp]
        L.orc_rng_transforms.argtypes = [u32, u32, i32, vp]
        L.orc_wrap.restype = f64
        L.orc_wrap.argtypes = [f64, i32]
        L.orc_min_image.restype = f64
        L.orc_min_image.argtypes = [f64, i32]
        L.orc_set_threads.argtypes = [i32]
        L.orc_max_threads.restype = i32
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def set_threads(n: int):
    lib().orc_set_threads(int(n))


def max_threads() -> int:
    return int(lib().orc_max_threads())


def philox(key, ctr) -> np.ndarray:
    k = np.asarray(key, dtype=np.uint32)
    c = np.asarray(ctr, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox(_p(k), _p(c), _p(out))
    return out


def stream_block(seed, chain, iteration, slot, purpose, epoch) -> np.ndarray:
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_stream_block(int(seed), int(chain), int(iteration), int(slot), int(purpose), int(epoch), _p(out))
    return out


def rng_transforms(w, w2, prec=F32) -> np.ndarray:
    """[u in [0,1), u in (0,1], Box-Muller z0, z1] computed from words (w, w2)."""
    out = np.zeros(4, dtype=np.float64)
    lib().orc_rng_transforms(int(w), int(w2), prec, _p(out))
    return out


def wrap(v: float, prec=F64) -> float:
    return float(lib().orc_wrap(float(v), prec))


def min_image(v: float, prec=F64) -> float:
    return float(lib().orc_min_image(float(v), prec))


class Scene:
    """Oracle-side scene (mesh or analytic 2-D mixture)."""

    def __init__(self, desc, prec=F64, use_bvh=True):
        self.desc, self.prec = desc, prec
        L = lib()
        if hasattr(desc, "weights"):
            w = np.ascontiguousarray(desc.weights, dtype=np.float32).astype(np.float64)
            mx = np.ascontiguousarray(desc.means[:, 0], dtype=np.float32).astype(np.float64)
            my = np.ascontiguousarray(desc.means[:, 1], dtype=np.float32).astype(np.float64)
            s = np.ascontiguousarray(desc.stddevs, dtype=np.float32).astype(np.float64)
            self.h = L.orc_scene_create_analytic2d(prec, len(w), _p(w), _p(mx), _p(my), _p(s), desc.width, desc.height)
        else:
            v = np.ascontiguousarray(desc.vertices, dtype=np.float32)
            i = np.ascontiguousarray(desc.indices, dtype=np.uint32)
            tm = np.ascontiguousarray(desc.tri_material, dtype=np.uint32)
            m = np.ascontiguousarray(desc.materials, dtype=np.float32).astype(np.float64)
            env = np.asarray(desc.env_radiance, dtype=np.float32)
            cam = np.concatenate([np.asarray(desc.cam_pos, dtype=np.float32), np.asarray(desc.cam_look, dtype=np.float32),
                                  np.asarray(desc.cam_up, dtype=np.float32)])
            self.h = L.orc_scene_create(prec, _p(v), len(v), _p(i), len(i), _p(tm), _p(m), len(m), _p(env), _p(cam),
                                        float(desc.vfov_deg), desc.width, desc.height, desc.max_path_len, int(use_bvh),
                                        int(bool(getattr(desc, "nee", False))))
        self.dim = int(L.orc_scene_dim(self.h))
        self.npix = desc.width * desc.height

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.orc_scene_destroy(self.h)
            self.h = None

    @property
    def eps_ray(self) -> float:
        return float(lib().orc_scene_eps_ray(self.h))

    def trace(self, o, d, brute=False):
        o = np.ascontiguousarray(o, dtype=np.float64)
        d = np.ascontiguousarray(d, dtype=np.float64)
        n = len(o)
        t = np.zeros(n, dtype=np.float64)
        tri = np.zeros(n, dtype=np.int32)
        lib().orc_trace(self.h, _p(o), _p(d), n, 0 if brute else 1, _p(t), _p(tri))
        return t, tri

    def eval(self, x, want_score=True):
        x = np.ascontiguousarray(x, dtype=np.float64).reshape(-1, self.dim)
        n = len(x)
        out = dict(f=np.zeros((n, 3)), p=np.zeros(n), pix=np.zeros(n, dtype=np.uint32), nrays=np.zeros(n, dtype=np.uint32),
                   sig=np.zeros(n, dtype=np.uint32), g=np.zeros((n, self.dim)), nonfinite=np.zeros(n, dtype=np.uint8))
        lib().orc_eval(self.h, _p(x), n, int(want_score), _p(out["f"]), _p(out["p"]), _p(out["pix"]), _p(out["nrays"]),
                       _p(out["sig"]), _p(out["g"]), _p(out["nonfinite"]))
        return out

    def bias_field(self, stddev: float, c_tilde: float, dt: float, G: int = 64, M: int = 256) -> np.ndarray:
        """Appendix C: (L^* p_hat / p_hat) of the analytic target on a G x G grid (rows = x1), M x M quadrature points."""
        out = np.zeros((G, G), dtype=np.float64)
        lib().orc_bias_field(self.h, float(stddev), float(c_tilde), float(dt), int(G), int(M), _p(out))
        return out

    def pt_render(self, n_samples: int, seed: int = 0) -> np.ndarray:
        rgb = np.zeros((self.npix, 3), dtype=np.float64)
        lib().orc_pt_render(self.h, int(n_samples), int(seed), _p(rgb))
        return rgb.reshape(self.desc.height, self.desc.width, 3)


class Chains:
    """Oracle-side chain ensemble: Alg. 1-4 of the paper, one plain loop over chains."""

    def __init__(self, scene: Scene, method, n_chains, stddev=None, c_tilde=None, dt=1e-5, m=64.0, large_step_prob=None,
                 p_lambda_override=0.0, seed=0, chain_offset=0, rao_blackwell=False, a_mode=0, rho=None):
        method = METHODS[method] if isinstance(method, str) else int(method)
        if stddev is None:
            stddev = 1e-2 if method in (0, 2) else 5e-3
        if c_tilde is None:
            c_tilde = 0.5 * stddev * stddev                    # DESIGN.md Q10
        if large_step_prob is None:
            large_step_prob = 0.3 if method in (0, 1) else 0.0
        self.scene, self.method, self.N, self.d = scene, method, int(n_chains), scene.dim
        self.params = dict(stddev=stddev, c_tilde=c_tilde, dt=dt, m=m, large_step_prob=large_step_prob,
                           p_lambda_override=p_lambda_override, seed=seed)
        self.h = lib().orc_chains_create(scene.h, method, self.N, stddev, c_tilde, dt, m, large_step_prob,
                                         p_lambda_override, int(seed), int(chain_offset), int(bool(rao_blackwell)))
        if a_mode or rho is not None:      # f4: another antisymmetric pattern / a regeneration density on film tiles (float32 weights)
            w = np.zeros(0) if rho is None else np.ascontiguousarray(rho, dtype=np.float32).astype(np.float64)
            G = 0 if rho is None else int(round(np.sqrt(w.size)))
            lib().orc_chains_set_f4(self.h, int(a_mode), G, _p(w.ravel()))

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.orc_chains_destroy(self.h)
            self.h = None

    def init(self, frame=0):
        lib().orc_chains_init(self.h, int(frame))

    def step(self, iterations=1):
        lib().orc_chains_step(self.h, int(iterations))

    def state(self):
        N, d = self.N, self.d
        s = dict(x=np.zeros((N, d)), p=np.zeros(N), fop=np.zeros((N, 3)), pix=np.zeros(N, dtype=np.uint32),
                 killed=np.zeros(N, dtype=np.uint8), g=np.zeros((N, d)), sig=np.zeros(N, dtype=np.uint32))
        lib().orc_chains_get_state(self.h, _p(s["x"]), _p(s["p"]), _p(s["fop"]), _p(s["pix"]), _p(s["killed"]), _p(s["g"]),
                                   _p(s["sig"]))
        return s

    def set_state(self, s, iteration):
        a = {k: np.ascontiguousarray(s[k], dtype=np.float64) for k in ("x", "p", "fop", "g")}
        pix = np.ascontiguousarray(s["pix"], dtype=np.uint32)
        killed = np.ascontiguousarray(s["killed"], dtype=np.uint8)
        lib().orc_chains_set_state(self.h, _p(a["x"]), _p(a["p"]), _p(a["fop"]), _p(pix), _p(killed), _p(a["g"]), int(iteration))

    def last(self):
        acc = np.zeros(self.N, dtype=np.uint8)
        dtau = np.zeros(self.N, dtype=np.float64)
        lib().orc_chains_last(self.h, _p(acc), _p(dtau))
        return acc, dtau

    def accum(self) -> np.ndarray:
        a = np.zeros((self.scene.npix, 4), dtype=np.float64)
        lib().orc_chains_accum(self.h, _p(a))
        return a

    def zero_accum(self):
        lib().orc_chains_zero_accum(self.h)

    def resolve(self):
        rgb = np.zeros((self.scene.npix, 3), dtype=np.float64)
        status = lib().orc_chains_resolve(self.h, _p(rgb))
        return rgb.reshape(self.scene.desc.height, self.scene.desc.width, 3), int(status)

    def stats(self) -> dict:
        o = np.zeros(11, dtype=np.float64)
        lib().orc_chains_stats(self.h, _p(o))
        keys = ["tours", "mutations", "rays", "mh_accepts", "nonfinite", "kills_last_step", "regen_queue_len", "p_lambda",
                "kappa0", "lambda", "iteration"]
        return {k: (float(v) if k in ("p_lambda", "kappa0", "lambda") else int(v)) for k, v in zip(keys, o)}

    def queue(self) -> np.ndarray:
        n = lib().orc_chains_queue(self.h, None)
        ids = np.zeros(max(n, 1), dtype=np.uint32)
        lib().orc_chains_queue(self.h, _p(ids))
        return ids[:n]


def ratio_image(accum: np.ndarray) -> np.ndarray:
    """Per-pixel sum(w f/p_hat) / sum(w / p_hat) (Q12); NaN where a pixel got no sample."""
    with np.errstate(invalid="ignore", divide="ignore"):
        return accum[:, :3] / accum[:, 3:4]


def rel_mse(a: np.ndarray, b: np.ndarray) -> float:
    """mean (a - b)^2 / (b^2 + 1e-2) over pixels and channels."""
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return float(np.mean((a - b) ** 2 / (b * b + 1e-2)))
