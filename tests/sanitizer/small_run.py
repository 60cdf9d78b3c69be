"""Small hot-path run for compute-sanitizer: k_wave in both instantiations, the per-segment loop, and
a few iterations of two samplers on the mini machines scene, then the same with next-event estimation on the GGX room.  Usage (one tool per gpurun call, B200_PROFILING.md):
    compute-sanitizer --tool memcheck|racecheck|initcheck|synccheck python tests/sanitizer/small_run.py
"""
import os
import sys

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import paper_2605_08916_b200 as dr  # noqa: E402
from dr_inputs import scenes as S  # noqa: E402

desc = S.mini_machines()
sc = dr.Scene(desc)
x = torch.from_numpy(S.seeded_states(3001, desc.dim, 11)).cuda()
a = sc.eval_states(x, True, form=2)
b = sc.eval_states(x, True, form=1)
c = sc.eval_states(x, False, form=2)
for k in ("f", "p", "pix", "nrays", "sig", "g"):
    assert torch.equal(a[k], b[k]), k
assert torch.equal(a["f"], c["f"])
for method in ("metropolis_restore", "diffusion_restore"):
    ch = dr.Chains(sc, method, 2000, seed=3)
    ch.init(0)
    ch.step(3)
    ch.resolve()
    st = ch.stats()
    assert st["mutations"] == 4 * 2000 and st["nonfinite"] == 0
# next-event estimation (Q21): two-phase vertices and shadow rays of k_wave, up to 2L - 1 queue entries per state,
# with and without the score (the reverse sweep of dr_grad.cuh)
import copy  # noqa: E402
desc_nee = copy.copy(S.ggx_room())
desc_nee.nee = True
sc_nee = dr.Scene(desc_nee)
xn = torch.from_numpy(S.seeded_states(3001, desc_nee.dim, 12)).cuda()
an = sc_nee.eval_states(xn, True, form=2)
cn = sc_nee.eval_states(xn, False, form=2)
assert torch.equal(an["f"], cn["f"]) and torch.equal(an["nrays"], cn["nrays"])
assert int(an["nrays"].max()) > desc_nee.max_path_len          # some path made more rays than it has segments: shadow rays ran
for method in ("metropolis_restore", "diffusion_restore"):      # without / with score
    ch = dr.Chains(sc_nee, method, 2000, seed=4)
    ch.init(0)
    ch.step(3)
    ch.resolve()
    st = ch.stats()
    assert st["mutations"] == 4 * 2000 and st["nonfinite"] == 0
torch.cuda.synchronize()
print("small_run ok", int(a["nrays"].sum()))
