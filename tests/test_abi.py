"""The C-ABI library loads and exports every symbol include/dr.h declares (no compute calls: no GPU needed)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "dr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dr_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported():
    from paper_2605_08916_b200 import build
    lib = ctypes.CDLL(build.build())
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n


def test_binding_lists_the_same_names():
    from paper_2605_08916_b200 import build
    build.build()
    from paper_2605_08916_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()
    # struct sizes match the C layout
    assert ctypes.sizeof(binding.dr_material) == 36
    assert ctypes.sizeof(binding.dr_config) == 64
    assert ctypes.sizeof(binding.dr_stats) == 88
    assert ctypes.sizeof(binding.dr_scene_info) == 32


def test_config_default_holds_the_papers_parameters():
    """dr_config_default (host-only, no GPU): PAPER.md L747 (stddev 1e-2 for the random-walk samplers, 5e-3 for the Langevin-based
    ones; large steps with probability 0.3 for plain Metropolis / MALA), L754-L755 (m = 64, dt = 1e-5), Q10 (c~ = s^2 / 2)."""
    import numpy as np
    from paper_2605_08916_b200 import build
    build.build()
    from paper_2605_08916_b200 import binding
    lib = ctypes.CDLL(build.build())
    lib.dr_config_default.argtypes = [ctypes.c_int32, ctypes.c_double, ctypes.c_void_p]
    f32 = np.float32
    for method in range(6):
        c = binding.dr_config()
        c.n_chains, c.seed, c.rho_grid = 7, 9, 3                      # overwritten: the call zeroes the struct first
        assert lib.dr_config_default(method, 0.0, ctypes.byref(c)) == 0
        s = 1e-2 if method in (0, 2) else 5e-3
        assert c.method == method and f32(c.stddev) == f32(s) and f32(c.c_tilde) == f32(0.5 * s * s)
        assert f32(c.dt) == f32(1e-5) and c.m == 64.0 and f32(c.large_step_prob) == f32(0.3 if method in (0, 1) else 0.0)
        assert (c.n_chains, c.seed, c.chain_offset, c.rao_blackwell, c.a_mode, c.rho_grid, c.host_rho) == (0, 0, 0, 0, 0, 0, None)
        assert c.p_lambda_override == 0.0
        assert lib.dr_config_default(method, 0.02, ctypes.byref(c)) == 0   # the caller's step width, and the rotation that goes with it
        assert f32(c.stddev) == f32(0.02) and f32(c.c_tilde) == f32(0.5 * 0.02 * 0.02)
    c = binding.dr_config()
    assert lib.dr_config_default(6, 0.0, ctypes.byref(c)) == -1 and lib.dr_config_default(-1, 0.0, ctypes.byref(c)) == -1
    assert lib.dr_config_default(0, float("nan"), ctypes.byref(c)) == -1 and lib.dr_config_default(0, 0.0, None) == -1


def test_product_path_does_not_touch_the_oracle():
    """The oracle is test infrastructure: nothing in the package or the inputs module imports it."""
    for folder in ("paper_2605_08916_b200", "dr_inputs"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, folder)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                    text = open(os.path.join(dirpath, f)).read()
                    for needle in ("import oracle", "from oracle", "liboracle", "orc_", "oracle/", "oracle."):
                        assert needle not in text, (dirpath, f, needle)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".hpp")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2605_08916_b200" not in text and "libdr" not in text and "dr.h" not in text, f
