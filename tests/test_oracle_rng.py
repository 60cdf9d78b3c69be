"""Pins for the oracle's Philox4x32-10 and its uniform / exponential / normal transforms.

Pin: ATen's at::Philox4_32 (torch/include/ATen/core/PhiloxRNGEngine.h), an independent
implementation of the same generator (Salmon et al. 2011, cited at PAPER.md L480), is
compiled on the spot and compared word for word.  Random123's known-answer vectors are
not in this container and are not typed from memory.
"""
import os
import subprocess
import sys
import tempfile

import numpy as np
import pytest

ATEN_PROG = r"""
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdio>
#include <cstdint>
int main() {
  unsigned long long seed, sub, off;
  while (scanf("%llu %llu %llu", &seed, &sub, &off) == 3) {
    at::Philox4_32 e(seed, sub, off);
    uint32_t a = e(), b = e(), c = e(), d = e();
    printf("%u %u %u %u\n", a, b, c, d);
  }
  return 0;
}
"""


@pytest.fixture(scope="module")
def aten_philox():
    import torch
    inc = os.path.join(os.path.dirname(torch.__file__), "include")
    if not os.path.exists(os.path.join(inc, "ATen/core/PhiloxRNGEngine.h")):
        pytest.skip("ATen Philox header not present")
    tmp = tempfile.mkdtemp()
    src, exe = os.path.join(tmp, "p.cpp"), os.path.join(tmp, "p")
    open(src, "w").write(ATEN_PROG)
    subprocess.run(["g++", "-std=c++17", "-O1", "-I", inc, src, "-o", exe], check=True)

    def run(rows):
        inp = "\n".join(f"{s} {sub} {off}" for s, sub, off in rows) + "\n"
        out = subprocess.run([exe], input=inp, capture_output=True, text=True, check=True).stdout
        return np.array([[int(v) for v in line.split()] for line in out.strip().splitlines()], dtype=np.uint32)
    return run


def test_philox_matches_aten(oracle, aten_philox):
    rng = np.random.default_rng(0)
    rows = [(0, 0, 0), (2**64 - 1, 2**64 - 1, 2**64 - 1), (1, 0, 0), (0, 1, 0), (0, 0, 1)]
    rows += [tuple(int(v) for v in rng.integers(0, 2**64, size=3, dtype=np.uint64)) for _ in range(200)]
    ref = aten_philox(rows)
    for (seed, sub, off), want in zip(rows, ref):
        # ATen: key = (seed lo, hi); counter = (offset lo, hi, subsequence lo, hi)
        got = oracle.philox([seed & 0xFFFFFFFF, seed >> 32], [off & 0xFFFFFFFF, off >> 32, sub & 0xFFFFFFFF, sub >> 32])
        assert (got == want).all(), (seed, sub, off)


def test_stream_keying(oracle):
    # DESIGN.md Q14: key = (seed lo, seed hi), counter = (chain, iteration, slot, purpose | epoch << 8)
    seed, chain, it, slot, purpose, epoch = 0x123456789ABCDEF, 77, 5, 3, 2, 9
    a = oracle.stream_block(seed, chain, it, slot, purpose, epoch)
    b = oracle.philox([seed & 0xFFFFFFFF, seed >> 32], [chain, it, slot, purpose | (epoch << 8)])
    assert (a == b).all()
    # distinct coordinates -> distinct blocks
    seen = {tuple(oracle.stream_block(0, c, i, s, p, 0)) for c in range(3) for i in range(3) for s in range(3) for p in range(4)}
    assert len(seen) == 108


def test_uniform_transforms_exact(oracle):
    for w in [0, 1, 255, 256, 0x80000000, 0xFFFFFF00, 0xFFFFFFFF, 123456789]:
        for prec in (oracle.F32, oracle.F64):
            u_co, u_oc, _, _ = oracle.rng_transforms(w, 0, prec)
            assert u_co == (w >> 8) / 2.0**24          # [0,1), exact in float32
            assert u_oc == ((w >> 8) + 1) / 2.0**24    # (0,1]
            assert 0.0 <= u_co < 1.0 and 0.0 < u_oc <= 1.0


def test_box_muller_is_standard_normal(oracle):
    # moments of the N(0, I_2) draws of Alg. 4 line 3 over 2e5 Philox blocks
    n = 50000
    z = []
    for i in range(n):
        w = oracle.stream_block(3, i, 1, 0, 1, 0)
        t = oracle.rng_transforms(int(w[0]), int(w[1]), oracle.F64)
        z.append((t[2], t[3]))
    z = np.array(z)
    se = 1.0 / np.sqrt(n)
    assert abs(z[:, 0].mean()) < 4 * se and abs(z[:, 1].mean()) < 4 * se
    assert abs(z[:, 0].var() - 1) < 6 * se and abs(z[:, 1].var() - 1) < 6 * se
    assert abs(np.mean(z[:, 0] * z[:, 1])) < 4 * se
    assert abs(np.mean(z[:, 0] ** 4) - 3.0) < 0.15         # kurtosis of a Gaussian
    # Box-Muller identity: z0^2 + z1^2 = -2 ln u_a
    w = oracle.stream_block(3, 0, 1, 0, 1, 0)
    t = oracle.rng_transforms(int(w[0]), int(w[1]), oracle.F64)
    assert np.isclose(t[2] ** 2 + t[3] ** 2, -2 * np.log(t[1]), rtol=1e-12)
    # float and double agree to float rounding
    t32 = oracle.rng_transforms(int(w[0]), int(w[1]), oracle.F32)
    assert np.allclose(t32[2:], t[2:], rtol=2e-6, atol=1e-6)
