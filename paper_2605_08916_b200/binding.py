"""ctypes binding of include/dr.h — same names, argument marshalling only.

`Scene` and `Chains` are small holders that keep the caller-owned torch tensors (state, accumulation buffer)
alive next to the opaque handles; every method is one C-ABI call.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("DR_LIB") or os.path.join(HERE, "libdr.so")   # DR_LIB: a build_variant() library (tests)

DR_OK, DR_WARN_NO_TOURS = 0, 1
DR_ERR_INVALID_ARG, DR_ERR_UNSUPPORTED, DR_ERR_CUDA, DR_ERR_NONFINITE, DR_ERR_OOM = -1, -2, -3, -4, -5
DR_METROPOLIS, DR_MALA, DR_METROPOLIS_RESTORE, DR_MALA_RESTORE, DR_DIFFUSION_RESTORE, DR_PATH_TRACING = range(6)
METHODS = {"metropolis": 0, "mala": 1, "metropolis_restore": 2, "mala_restore": 3, "diffusion_restore": 4, "path_tracing": 5}

EXPORTS = [
    "dr_last_error", "dr_scene_create", "dr_scene_create_analytic2d", "dr_scene_destroy", "dr_scene_get_info",
    "dr_chains_state_bytes", "dr_chains_create", "dr_chains_destroy", "dr_chains_init", "dr_step", "dr_resolve_image",
    "dr_chains_stats", "dr_chains_download", "dr_chains_upload", "dr_chains_last_step", "dr_regen_queue_download",
    "dr_trace_rays", "dr_eval_states", "dr_philox_blocks", "dr_rng_transforms", "dr_resolve_image_sharded",
    "dr_eval_work_stats", "dr_profile_enable", "dr_profile_read", "dr_chains_work_stats", "dr_eval_states_form",
    "dr_chains_set_eval_form", "dr_frame_floats", "dr_pack_frame", "dr_resolve_image_packed",
    "dr_bias_field", "dr_trace_rays_noalloc", "dr_config_default",
]
TRACE_NOALLOC_MAX_RAYS = 65536   # DR_TRACE_NOALLOC_MAX_RAYS of include/dr.h
PROF_NAMES = ["propose", "raygen", "trace", "shade", "grad", "decide", "scan", "scatter", "resolve"]


class dr_material(C.Structure):
    _fields_ = [("kind", C.c_int32), ("albedo_or_f0", C.c_float * 3), ("ior", C.c_float), ("roughness", C.c_float),
                ("emission", C.c_float * 3)]


class dr_scene_desc(C.Structure):
    _fields_ = [("host_vertices", C.c_void_p), ("nv", C.c_uint32), ("host_indices", C.c_void_p), ("nt", C.c_uint32),
                ("host_tri_material", C.c_void_p), ("host_materials", C.POINTER(dr_material)), ("nm", C.c_uint32),
                ("env_radiance", C.c_float * 3), ("cam_pos", C.c_float * 3), ("cam_look", C.c_float * 3),
                ("cam_up", C.c_float * 3), ("vfov_deg", C.c_float), ("width", C.c_uint32), ("height", C.c_uint32),
                ("max_path_len", C.c_uint32), ("nee", C.c_uint32)]


class dr_analytic2d_desc(C.Structure):
    _fields_ = [("n_components", C.c_uint32), ("host_weights", C.c_void_p), ("host_means", C.c_void_p),
                ("host_stddevs", C.c_void_p), ("width", C.c_uint32), ("height", C.c_uint32)]


class dr_config(C.Structure):
    _fields_ = [("method", C.c_int32), ("n_chains", C.c_uint32), ("stddev", C.c_float), ("c_tilde", C.c_float),
                ("dt", C.c_float), ("m", C.c_float), ("large_step_prob", C.c_float), ("p_lambda_override", C.c_float),
                ("seed", C.c_uint64), ("chain_offset", C.c_uint32), ("rao_blackwell", C.c_uint32), ("a_mode", C.c_uint32),
                ("rho_grid", C.c_uint32), ("host_rho", C.c_void_p)]


class dr_stats(C.Structure):
    _fields_ = [("tours", C.c_uint64), ("mutations", C.c_uint64), ("rays", C.c_uint64), ("mh_accepts", C.c_uint64),
                ("nonfinite", C.c_uint64), ("kills_last_step", C.c_uint32), ("regen_queue_len", C.c_uint32),
                ("iteration", C.c_uint32), ("p_lambda", C.c_float), ("kappa0", C.c_float), ("lambda_", C.c_float),
                ("no_tour_resolves", C.c_uint32), ("wave_timeouts", C.c_uint32), ("grad_states", C.c_uint64), ("lit_init", C.c_uint64)]


class dr_scene_info(C.Structure):
    _fields_ = [("n_tris", C.c_uint32), ("n_nodes", C.c_uint32), ("depth", C.c_uint32), ("smem_nodes", C.c_uint32),
                ("sah_cost", C.c_float), ("eps_ray", C.c_float), ("device_bytes", C.c_size_t)]


class DrError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"dr status {status}: {msg}")
        self.status = status


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2605_08916_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, u32, i32, u64 = C.c_void_p, C.c_uint32, C.c_int32, C.c_uint64
    L.dr_last_error.restype = C.c_char_p
    L.dr_scene_create.argtypes = [C.POINTER(dr_scene_desc), C.POINTER(vp)]
    L.dr_scene_create_analytic2d.argtypes = [C.POINTER(dr_analytic2d_desc), C.POINTER(vp)]
    L.dr_scene_destroy.argtypes = [vp]
    L.dr_scene_get_info.argtypes = [vp, C.POINTER(dr_scene_info)]
    L.dr_chains_state_bytes.restype = C.c_size_t
    L.dr_chains_state_bytes.argtypes = [vp, C.POINTER(dr_config)]
    L.dr_chains_create.argtypes = [vp, C.POINTER(dr_config), vp, C.c_size_t, vp, C.POINTER(vp)]
    L.dr_chains_destroy.argtypes = [vp]
    L.dr_chains_init.argtypes = [vp, u32, vp]
    L.dr_step.argtypes = [vp, i32, u32, vp]
    L.dr_resolve_image.argtypes = [vp, vp, vp]
    L.dr_chains_stats.argtypes = [vp, C.POINTER(dr_stats), vp]
    L.dr_chains_download.argtypes = [vp] * 9
    L.dr_chains_upload.argtypes = [vp] * 8 + [u32, vp]
    L.dr_chains_last_step.argtypes = [vp, vp, vp, vp]
    L.dr_regen_queue_download.argtypes = [vp, vp, C.POINTER(u32), vp]
    L.dr_trace_rays.argtypes = [vp, vp, vp, u32, vp, vp, vp]
    L.dr_trace_rays_noalloc.argtypes = [vp, vp, vp, u32, vp, vp, vp]
    L.dr_config_default.argtypes = [i32, C.c_double, vp]
    L.dr_eval_states.argtypes = [vp, vp, u32, vp, vp, vp, vp, vp, vp, vp]
    L.dr_eval_states_form.argtypes = [vp, vp, u32, vp, vp, vp, vp, vp, vp, i32, vp]
    L.dr_chains_set_eval_form.argtypes = [vp, i32]
    L.dr_frame_floats.restype = C.c_size_t
    L.dr_frame_floats.argtypes = [vp]
    L.dr_pack_frame.argtypes = [vp, vp, vp]
    L.dr_resolve_image_packed.argtypes = [vp, vp, vp, vp]
    L.dr_bias_field.argtypes = [vp, C.c_double, C.c_double, C.c_double, u32, u32, vp, vp]
    L.dr_resolve_image_sharded.argtypes = [vp, vp, u64, u64, vp, vp]
    L.dr_eval_work_stats.argtypes = [vp, vp, u32, vp, vp]
    L.dr_profile_enable.argtypes = [vp, i32, vp]
    L.dr_profile_read.argtypes = [vp, vp, vp, vp]
    L.dr_chains_work_stats.argtypes = [vp, vp, vp]
    L.dr_philox_blocks.argtypes = [u64, vp, u32, vp, vp]
    L.dr_rng_transforms.argtypes = [vp, u32, vp, vp]
    for name in EXPORTS:
        if name not in ("dr_last_error", "dr_chains_state_bytes", "dr_frame_floats"):
            getattr(L, name).restype = i32
    return L


lib = _load()


def _check(status, allow_warn=False):
    if status < 0 or (status > 0 and not allow_warn):
        raise DrError(status, lib.dr_last_error().decode())
    return status


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _np(a):
    return a.ctypes.data_as(C.c_void_p)


def _dp(t):
    return C.c_void_p(t.data_ptr())


class Scene:
    """dr_scene_create / dr_scene_create_analytic2d from a dr_inputs description (host arrays are copied)."""

    def __init__(self, desc):
        self.desc = desc
        h = C.c_void_p()
        if hasattr(desc, "weights"):
            w = np.ascontiguousarray(desc.weights, dtype=np.float32)
            mu = np.ascontiguousarray(desc.means, dtype=np.float32)
            s = np.ascontiguousarray(desc.stddevs, dtype=np.float32)
            d = dr_analytic2d_desc(len(w), _np(w), _np(mu), _np(s), desc.width, desc.height)
            _check(lib.dr_scene_create_analytic2d(C.byref(d), C.byref(h)))
            self.dim = 2
        else:
            v = np.ascontiguousarray(desc.vertices, dtype=np.float32)
            i = np.ascontiguousarray(desc.indices, dtype=np.uint32)
            tm = np.ascontiguousarray(desc.tri_material, dtype=np.uint32)
            mats = (dr_material * len(desc.materials))()
            for k, m in enumerate(np.asarray(desc.materials, dtype=np.float32)):
                mats[k].kind = int(m[0])
                mats[k].albedo_or_f0[:] = [float(m[1]), float(m[2]), float(m[3])]
                mats[k].ior, mats[k].roughness = float(m[4]), float(m[5])
                mats[k].emission[:] = [float(m[6]), float(m[7]), float(m[8])]
            d = dr_scene_desc()
            d.host_vertices, d.nv, d.host_indices, d.nt = _np(v), len(v), _np(i), len(i)
            d.host_tri_material, d.host_materials, d.nm = _np(tm), mats, len(mats)
            d.env_radiance[:] = [float(c) for c in desc.env_radiance]
            d.cam_pos[:] = [float(c) for c in desc.cam_pos]
            d.cam_look[:] = [float(c) for c in desc.cam_look]
            d.cam_up[:] = [float(c) for c in desc.cam_up]
            d.vfov_deg, d.width, d.height, d.max_path_len = float(desc.vfov_deg), desc.width, desc.height, desc.max_path_len
            d.nee = int(bool(getattr(desc, "nee", False)))
            _check(lib.dr_scene_create(C.byref(d), C.byref(h)))
            self.dim = desc.dim
        self.h = h
        self.width, self.height = desc.width, desc.height
        self.npix = desc.width * desc.height

    def __del__(self):
        if getattr(self, "h", None) and lib is not None:      # (module globals are gone at interpreter shutdown)
            lib.dr_scene_destroy(self.h)
            self.h = None

    def info(self) -> dict:
        o = dr_scene_info()
        _check(lib.dr_scene_get_info(self.h, C.byref(o)))
        return {k: getattr(o, k) for k, _ in o._fields_}

    def trace_rays(self, o: torch.Tensor, d: torch.Tensor):
        n = o.shape[0]
        t = torch.empty(n, dtype=torch.float32, device="cuda")
        prim = torch.empty(n, dtype=torch.int32, device="cuda")
        _check(lib.dr_trace_rays(self.h, _dp(o.contiguous()), _dp(d.contiguous()), n, _dp(t), _dp(prim), _stream()))
        return t, prim

    def trace_rays_noalloc(self, o: torch.Tensor, d: torch.Tensor, t: torch.Tensor, prim: torch.Tensor) -> None:
        """dr_trace_rays_noalloc: closest hits into the caller's own t (float32) and prim (int32) tensors, for callers that
        must not allocate GPU memory while they trace (fixed-budget frame loops and servers, hosts whose own pool owns the
        GPU, plugins inside another process).  Unlike trace_rays, nothing is created here: outputs are passed in, the
        scratch is a fixed 2.5 MiB array inside libdr.so.  At most TRACE_NOALLOC_MAX_RAYS rays per call (more is an error);
        asynchronous on the current stream; calls that overlap on the GPU race on the shared scratch (include/dr.h)."""
        n = o.shape[0]
        assert o.is_contiguous() and d.is_contiguous() and t.is_contiguous() and prim.is_contiguous()
        assert t.numel() == n and prim.numel() == n and t.dtype == torch.float32 and prim.dtype == torch.int32
        _check(lib.dr_trace_rays_noalloc(self.h, _dp(o), _dp(d), n, _dp(t), _dp(prim), _stream()))

    def bias_field(self, stddev, c_tilde, dt, G=64, M=256) -> torch.Tensor:
        out = torch.empty(G, G, dtype=torch.float64, device="cuda")
        _check(lib.dr_bias_field(self.h, float(stddev), float(c_tilde), float(dt), int(G), int(M), _dp(out), _stream()))
        return out

    def eval_work_stats(self, x: torch.Tensor) -> dict:
        out = torch.zeros(3, dtype=torch.int64, device="cuda")
        _check(lib.dr_eval_work_stats(self.h, _dp(x.contiguous()), x.shape[0], _dp(out), _stream()))
        r, n, t = (int(v) for v in out.cpu())
        return dict(rays=r, node_visits=n, tri_tests=t)

    def eval_states(self, x: torch.Tensor, want_score=True, form=0):
        x = x.contiguous()
        n = x.shape[0]
        dev = dict(device="cuda")
        out = dict(f=torch.empty(n, 3, dtype=torch.float32, **dev), p=torch.empty(n, dtype=torch.float32, **dev),
                   pix=torch.empty(n, dtype=torch.int32, **dev), nrays=torch.empty(n, dtype=torch.int32, **dev),
                   sig=torch.empty(n, dtype=torch.int32, **dev))
        g = torch.zeros(n, self.dim, dtype=torch.float32, **dev) if want_score else None
        _check(lib.dr_eval_states_form(self.h, _dp(x), n, _dp(out["f"]), _dp(out["p"]), _dp(out["pix"]),
                                       _dp(g) if want_score else None, _dp(out["nrays"]), _dp(out["sig"]), int(form), _stream()))
        out["g"] = g
        return out


class Chains:
    """dr_chains_create over caller-owned torch memory + the per-frame calls."""

    def __init__(self, scene: Scene, method, n_chains, stddev=None, c_tilde=None, dt=None, m=None, large_step_prob=None,
                 p_lambda_override=0.0, seed=0, chain_offset=0, rao_blackwell=False, a_mode=0, rho=None):
        method = METHODS[method] if isinstance(method, str) else int(method)
        dflt = dr_config()                                      # the method's parameters live in the library (dr_config_default)
        _check(lib.dr_config_default(method, 0.0 if stddev is None else float(stddev), C.byref(dflt)))
        stddev = dflt.stddev if stddev is None else stddev
        c_tilde = dflt.c_tilde if c_tilde is None else c_tilde
        dt = dflt.dt if dt is None else dt
        m = dflt.m if m is None else m
        large_step_prob = dflt.large_step_prob if large_step_prob is None else large_step_prob
        self.scene, self.method, self.N, self.d = scene, method, int(n_chains), scene.dim
        rho_arr = None if rho is None else np.ascontiguousarray(rho, dtype=np.float32).ravel()
        grid = 0 if rho is None else int(round(np.sqrt(rho_arr.size)))
        if rho is not None and grid * grid != rho_arr.size:     # dr_chains_create reads G * G floats from host_rho
            raise ValueError(f"rho must hold G x G tile probabilities, got {rho_arr.size} values")
        self.cfg = dr_config(method, self.N, stddev, c_tilde, dt, m, large_step_prob, p_lambda_override, seed, chain_offset,
                             int(bool(rao_blackwell)), int(a_mode), grid, None if rho is None else _np(rho_arr))
        nbytes = lib.dr_chains_state_bytes(scene.h, C.byref(self.cfg))
        if nbytes == 0:
            raise DrError(DR_ERR_INVALID_ARG, lib.dr_last_error().decode())
        self.state = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        self.accum = torch.zeros(scene.npix, 4, dtype=torch.float32, device="cuda")
        self.image = torch.empty(scene.height, scene.width, 3, dtype=torch.float32, device="cuda")
        h = C.c_void_p()
        _check(lib.dr_chains_create(scene.h, C.byref(self.cfg), _dp(self.state), nbytes, _dp(self.accum), C.byref(h)))
        self.h = h

    def __del__(self):
        if getattr(self, "h", None) and lib is not None:
            lib.dr_chains_destroy(self.h)
            self.h = None

    def set_eval_form(self, form: int):
        _check(lib.dr_chains_set_eval_form(self.h, int(form)))

    def init(self, frame=0):
        _check(lib.dr_chains_init(self.h, int(frame), _stream()))

    def step(self, iterations=1):
        _check(lib.dr_step(self.h, self.method, int(iterations), _stream()))

    def resolve(self):
        """Asynchronous; (image, 0).  A resolve before the first completed tour shows in stats()["status"]."""
        status = _check(lib.dr_resolve_image(self.h, _dp(self.image), _stream()), allow_warn=True)
        return self.image, status

    def resolve_sharded(self, accum_sum: torch.Tensor, tours_total: int, mutations_total: int):
        status = _check(lib.dr_resolve_image_sharded(self.h, _dp(accum_sum), int(tours_total), int(mutations_total),
                                                     _dp(self.image), _stream()), allow_warn=True)
        return self.image, status

    def pack_frame(self) -> torch.Tensor:
        """This shard's frame (accumulation buffer + counters as limbs) in one buffer, ready for one all-reduce(sum)."""
        if getattr(self, "frame", None) is None:
            self.frame = torch.empty(lib.dr_frame_floats(self.h), dtype=torch.float32, device="cuda")
        _check(lib.dr_pack_frame(self.h, _dp(self.frame), _stream()))
        return self.frame

    def resolve_packed(self, frame_sum: torch.Tensor):
        _check(lib.dr_resolve_image_packed(self.h, _dp(frame_sum), _dp(self.image), _stream()))
        return self.image

    def profile_enable(self, on=True):
        _check(lib.dr_profile_enable(self.h, int(on), _stream()))

    def profile_read(self) -> dict:
        ms = np.zeros(len(PROF_NAMES), np.float64)
        n = np.zeros(len(PROF_NAMES), np.uint64)
        _check(lib.dr_profile_read(self.h, _np(ms), _np(n), _stream()))
        return {k: dict(ms=float(a), launches=int(b)) for k, a, b in zip(PROF_NAMES, ms, n)}

    def work_stats(self) -> dict:
        o = np.zeros(3, np.uint64)
        _check(lib.dr_chains_work_stats(self.h, _np(o), _stream()))
        return dict(rays=int(o[0]), node_visits=int(o[1]), tri_tests=int(o[2]))

    def stats(self) -> dict:
        o = dr_stats()
        status = _check(lib.dr_chains_stats(self.h, C.byref(o), _stream()), allow_warn=True)
        d = {k: getattr(o, k) for k, _ in o._fields_}
        d["status"] = status
        d["lambda"] = d.pop("lambda_")
        return d

    def download(self, out: dict | None = None) -> dict:
        """Chain state as row-major host arrays.  `out`: arrays to fill (e.g. numpy views of pinned torch tensors, which
        the copies then reach by DMA); default: fresh numpy arrays."""
        N, d = self.N, self.d
        s = out if out is not None else dict(
            x=np.empty((N, d), np.float32), p=np.empty(N, np.float32), fop=np.empty((N, 3), np.float32),
            pix=np.empty(N, np.uint32), killed=np.empty(N, np.uint8), g=np.empty((N, d), np.float32),
            sig=np.empty(N, np.uint32))
        _check(lib.dr_chains_download(self.h, _np(s["x"]), _np(s["p"]), _np(s["fop"]), _np(s["pix"]), _np(s["killed"]),
                                      _np(s["g"]), _np(s["sig"]), _stream()))
        return s

    def upload(self, s: dict, iteration: int):
        a = {k: np.ascontiguousarray(s[k], dtype=np.float32) for k in ("x", "p", "fop", "g")}
        pix = np.ascontiguousarray(s["pix"], dtype=np.uint32)
        killed = np.ascontiguousarray(s["killed"], dtype=np.uint8)
        sig = np.ascontiguousarray(s["sig"], dtype=np.uint32)
        _check(lib.dr_chains_upload(self.h, _np(a["x"]), _np(a["p"]), _np(a["fop"]), _np(pix), _np(killed), _np(a["g"]),
                                    _np(sig), int(iteration), _stream()))

    def last_step(self):
        acc = np.zeros(self.N, np.uint8)
        w = np.zeros(self.N, np.float32)
        _check(lib.dr_chains_last_step(self.h, _np(acc), _np(w), _stream()))
        return acc, w

    def queue(self) -> np.ndarray:
        n = C.c_uint32()
        ids = np.zeros(self.N, np.uint32)
        _check(lib.dr_regen_queue_download(self.h, _np(ids), C.byref(n), _stream()))
        return ids[: n.value]


def philox_blocks(seed: int, ctr: torch.Tensor) -> torch.Tensor:
    out = torch.empty_like(ctr)
    _check(lib.dr_philox_blocks(int(seed), _dp(ctr.contiguous()), ctr.shape[0], _dp(out), _stream()))
    return out


def rng_transforms(words: torch.Tensor) -> torch.Tensor:
    n = words.shape[0]
    out = torch.empty(n, 4, dtype=torch.float32, device="cuda")
    _check(lib.dr_rng_transforms(_dp(words.contiguous()), n, _dp(out), _stream()))
    return out
