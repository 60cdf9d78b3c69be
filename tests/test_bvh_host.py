"""Host logic of the scene builder (csrc/dr_bvh.cpp) and of the traversal building blocks (csrc/dr_traverse.cuh),
without a GPU: tests/bvh_host_check.cpp is compiled with g++ against the product sources and run.

What is pinned: every triangle is referenced and stored as given; the node masks are consistent (unary triangle counts,
a slot is a leaf or an internal child, totals match); the BVH8 closest hit equals a brute-force loop over all
triangles bit for bit (same triangle test on both sides, so any wrongly culled box, wrong child index, wrong triangle
index from the trimask popcount, or wrong octant permutation shows up as a mismatch); reference pre-splitting
(long thin triangles cut into several references) changes no hit and reduces the triangle tests per ray."""
import os
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CUDA_INC = os.environ.get("CUDA_INCLUDE", "/usr/local/cuda/include")


@pytest.fixture(scope="module")
def exe(tmp_path_factory):
    if not os.path.exists(os.path.join(CUDA_INC, "vector_types.h")):
        pytest.skip("CUDA headers not found")
    out = str(tmp_path_factory.mktemp("bvh") / "bvh_host_check")
    subprocess.run(["g++", "-O2", "-std=c++17", "-I", CUDA_INC, "-o", out, os.path.join(ROOT, "tests", "bvh_host_check.cpp"),
                    os.path.join(ROOT, "paper_2605_08916_b200", "csrc", "dr_bvh.cpp")], check=True)
    return out


def run(exe, *args):
    line = subprocess.run([exe] + [str(a) for a in args], check=True, capture_output=True, text=True).stdout.strip()
    return {k: float(v) for k, v in (kv.split("=") for kv in line.split())}


@pytest.mark.parametrize("budget", [0.0, 1.0, 3.0])
def test_bvh8_closest_hit_equals_brute_force(exe, budget):
    r = run(exe, budget, 3000, 6000)
    assert r["referenced"] == r["tris"]          # every triangle has at least one reference
    assert r["bad_tri"] == 0 and r["bad_node"] == 0
    assert r["hits"] > 500                       # the rays do hit the mesh
    assert r["mismatch"] == 0                    # bit-exact closest hit (t and original id)
    if budget == 0.0:
        assert r["refs"] == r["tris"]
    else:
        assert r["tris"] < r["refs"] <= (1.0 + budget) * r["tris"] + 1


def test_presplitting_cuts_triangle_tests(exe):
    a, b = run(exe, 0.0, 3000, 4000), run(exe, 1.0, 3000, 4000)
    assert a["mismatch"] == 0 and b["mismatch"] == 0
    assert a["hits"] == b["hits"]
    assert b["tris_per_ray"] < 0.75 * a["tris_per_ray"]


def test_tiny_and_single_triangle_scenes(exe):
    for n in (1, 2, 9):
        r = run(exe, 1.0, n, 2000)
        assert r["mismatch"] == 0 and r["bad_node"] == 0 and r["referenced"] == r["tris"]


def test_optimal_collapse_beats_greedy(exe):
    """The cost-optimal BVH2 -> BVH8 cut (dr_bvh.cpp) changes no hit and needs fewer nodes, node tests and triangle
    tests per ray than opening the largest child until there are eight."""
    a, b = run(exe, 1.0, 6000, 6000, 0), run(exe, 1.0, 6000, 6000, 1)
    assert a["mismatch"] == 0 and b["mismatch"] == 0 and a["hits"] == b["hits"]
    assert b["nodes"] < 0.9 * a["nodes"]
    cost = lambda r: r["nodes_per_ray"] + 0.4 * r["tris_per_ray"]     # the collapse's own weights
    assert cost(b) < cost(a) and b["tris_per_ray"] < a["tris_per_ray"]
