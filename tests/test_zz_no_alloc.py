"""dr_trace_rays_noalloc against dr_trace_rays (needs a B200).

Some users of libdr.so cannot let the library call cudaMalloc / cudaFree while it works: a frame loop or a server that
runs inside a fixed memory budget (an allocation may fail late, and cudaFree stalls the whole device), a host program
whose own pool has already taken the GPU's memory, a plugin that must not change its host process's footprint.
dr_trace_rays allocates its ray queue and hit records on every call; dr_trace_rays_noalloc runs the same kernels with
that scratch in a fixed array inside the library (include/dr.h: at most DR_TRACE_NOALLOC_MAX_RAYS rays per call).

What is checked here: on two calls in a row -- the second smaller than the first, so the array still holds the first
call's rays behind the second's -- the hits equal those of dr_trace_rays (same kernels, same rays: bit for bit, which is
inside the 1e-5 bound the closest-hit tests use against the oracle); a batch above the limit is refused with a message that
names the limit and leaves the outputs alone; the free device memory does not move across a call.

This file sorts last on purpose: pytest -x stops at the first failure, so a failure here hides no other test."""
import numpy as np
import pytest

from dr_inputs import scenes as S

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dr():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2605_08916_b200 import build
    build.build()
    import paper_2605_08916_b200 as dr_
    return dr_


def _rays(desc, n, seed):
    import torch
    o, d = S.seeded_rays(desc, n, seed)
    return torch.from_numpy(o).cuda().contiguous(), torch.from_numpy(d).cuda().contiguous()


def test_noalloc_trace_equals_the_allocating_trace_on_two_calls_in_a_row(dr):
    import torch
    desc = S.mini_machines()
    sc = dr.Scene(desc)
    first, second = _rays(desc, 20011, 5), _rays(desc, 4099, 6)     # several blocks and a ragged tail; then a shorter batch
    want = [sc.trace_rays(*first), sc.trace_rays(*second)]           # the existing path (allocates, synchronises)
    got = []
    for o, d in (first, second):                                     # two calls in a row on one stream, nothing in between
        t = torch.full((o.shape[0],), 123.0, dtype=torch.float32, device="cuda")
        prim = torch.full((o.shape[0],), 7, dtype=torch.int32, device="cuda")
        sc.trace_rays_noalloc(o, d, t, prim)
        got.append((t, prim))
    torch.cuda.synchronize()
    for (t, prim), (wt, wprim) in zip(got, want):
        assert torch.equal(prim, wprim)
        assert torch.equal(t, wt)                                    # same kernels on the same rays: identical bits
        hit = wprim >= 0
        assert int(hit.sum()) > 1000 and int((~hit).sum()) > 0       # the comparison saw hits and misses
        assert torch.all(torch.abs(t[hit] - wt[hit]) <= 1e-5 * torch.abs(wt[hit]))   # the suite's closest-hit bound, for the record
    assert not torch.equal(got[0][1][:4099], got[1][1])              # the second call traced its own rays, not the first's leftovers


def test_noalloc_trace_refuses_more_rays_than_its_scratch_holds_and_allocates_nothing(dr):
    import torch
    desc = S.cornell()
    sc = dr.Scene(desc)
    limit = dr.binding.TRACE_NOALLOC_MAX_RAYS
    o, d = _rays(desc, limit + 1, 9)
    t = torch.full((limit + 1,), 123.0, dtype=torch.float32, device="cuda")
    prim = torch.full((limit + 1,), 7, dtype=torch.int32, device="cuda")
    with pytest.raises(Exception, match=str(limit)):
        sc.trace_rays_noalloc(o, d, t, prim)
    torch.cuda.synchronize()
    assert bool((t == 123.0).all()) and bool((prim == 7).all())      # refused before anything was launched
    # exactly the limit is served, and equals the allocating path
    wt, wprim = sc.trace_rays(o[:limit].contiguous(), d[:limit].contiguous())
    sc.trace_rays_noalloc(o[:limit].contiguous(), d[:limit].contiguous(), t[:limit], prim[:limit])   # also this device's first-call set-up, if the test runs alone
    torch.cuda.synchronize()
    assert torch.equal(prim[:limit], wprim) and torch.equal(t[:limit], wt)
    # a later call neither takes nor returns device memory (driver's own figure; the torch tensors exist already)
    o2, d2 = o[:3000].contiguous(), d[:3000].contiguous()
    t2, prim2 = t[:3000], prim[:3000]
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    sc.trace_rays_noalloc(o2, d2, t2, prim2)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before
    assert torch.equal(prim2, wprim[:3000]) and torch.equal(t2, wt[:3000])
    # empty input is a no-op
    e = torch.zeros(0, 3, device="cuda")
    sc.trace_rays_noalloc(e, e, torch.zeros(0, device="cuda"), torch.zeros(0, dtype=torch.int32, device="cuda"))
