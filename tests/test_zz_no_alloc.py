"""grmhd_maxspeed_noalloc: the max-characteristic-speed reduction (row A8) for callers that cannot
allocate -- its scratch is a file-scope static device array inside libgrmhd.so.

Collected LAST on purpose (the suite runs with `pytest -x`): a failure here hides nothing.

The expected values come from the library's EXISTING path: a handle's max-speed reduction, which
accumulates into the caller-owned workspace (`grmhd_get_stats` -> maxspeed).  Both paths evaluate
the same per-state speeds and a max of non-negative doubles is exact and order independent, so they
must agree to the tolerance the parity tests use for this quantity (rtol 1e-13).  Consecutive
calls go from a large batch with fast states to a small one with slow states: anything stale left
in the shared scratch array by the earlier call would raise the later result.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2406_11669_b200 import workloads as wl

RTOL = 1e-13   # as tests/test_gpu_parity.py asserts for maxspeed right after set_prims
G = 3
I3 = (slice(G, -G),) * 3


def _states_of(solver, w, torch):
    """The interior cells of a handle as plain (8, n) / (10, n) device arrays: the primitives and
    the cell-centred B the handle holds (get_prims), and the caller's metric."""
    P = solver.get_prims()
    prim = torch.stack([p[I3].reshape(-1) for p in P]).contiguous()
    met = torch.stack([torch.from_numpy(np.ascontiguousarray(w.metric[r][I3])).reshape(-1)
                       for r in range(10)]).to(prim.device).contiguous()
    return prim, met


def test_oversize_batch_is_rejected_before_any_cuda_call():
    """n beyond the static scratch's capacity -> GRMHD_ELIMIT and a message naming the limit;
    argument checks come before any CUDA call, so this runs without a GPU."""
    from paper_2406_11669_b200 import binding
    L = binding.lib()
    o = binding.make_opts()
    a = np.ones(4)
    pp = (C.c_void_p * 8)(*[a.ctypes.data] * 8)
    mp = (C.c_void_p * 10)(*[a.ctypes.data] * 10)
    out = np.zeros(3)
    msg = C.create_string_buffer(256)
    rc = L.grmhd_maxspeed_noalloc(pp, mp, binding.NOALLOC_MAX_STATES + 1, C.byref(o),
                                  C.c_void_p(out.ctypes.data), None, msg, len(msg))
    assert rc == binding.ELIMIT == -6
    assert b"GRMHD_NOALLOC_MAX_STATES" in msg.value and b"4194304" in msg.value
    assert L.grmhd_maxspeed_noalloc(pp, mp, 0, C.byref(o), C.c_void_p(out.ctypes.data), None,
                                    msg, len(msg)) == binding.EINVAL
    assert L.grmhd_maxspeed_noalloc(pp, mp, 4, C.byref(o), None, None, None, 0) == binding.EINVAL
    assert not out.any()


@pytest.mark.gpu
def test_maxspeed_noalloc_matches_the_handle_path_on_consecutive_calls():
    import torch
    from paper_2406_11669_b200 import binding
    from tests.util import make_gpu

    out = torch.full((3,), -1.0, dtype=torch.float64, device="cuda")
    results = []
    # large + fast (W up to 10, 46 656 states = 183 blocks), then small + slow (v = 0, 1 024 states
    # = 4 blocks), then a curved metric with a shift; each right after set_prims and after a step
    for w in (wl.c2p_stress(36), wl.balsara1(64, 4, 4), wl.kerr_blob(40)):
        g = make_gpu(w)
        o = binding.make_opts(**w.opts)
        for nsteps in (0, 1):
            if nsteps:
                g.step(nsteps, w.cfl)
            want = np.array(g.stats()["maxspeed"])          # existing path (workspace scratch)
            prim, met = _states_of(g, w, torch)
            binding.maxspeed_noalloc(prim, met, o, out)     # new path (static scratch)
            got = out.cpu().numpy().copy()
            assert np.all(want > 0.0) and np.all(np.isfinite(want))
            np.testing.assert_allclose(got, want, rtol=RTOL, atol=0.0, err_msg=f"{w.name} step {nsteps}")
            results.append((w.name, nsteps, prim, met, o, got))
        g.close()
    # the calls above ran back to back on one scratch array with different sizes; now repeat each
    # of them in reverse order: identical bits, whatever the previous call left behind
    for name, nsteps, prim, met, o, got in reversed(results):
        out.fill_(-1.0)
        binding.maxspeed_noalloc(prim, met, o, out)
        assert np.array_equal(out.cpu().numpy(), got), (name, nsteps)


@pytest.mark.gpu
def test_maxspeed_noalloc_at_the_size_limit_and_without_allocating():
    """n = GRMHD_NOALLOC_MAX_STATES exactly (16 384 blocks, every partial maximum of the scratch in
    use) on the states of a handle tiled up to that size: the max is idempotent, so the result
    equals the handle's; and a call allocates no device memory (torch's allocator aside, the
    driver's free-memory figure does not move)."""
    import torch
    from paper_2406_11669_b200 import binding
    from tests.util import make_gpu

    w = wl.c2p_stress(36)
    g = make_gpu(w)
    want = np.array(g.stats()["maxspeed"])
    prim, met = _states_of(g, w, torch)
    g.close()
    o = binding.make_opts(**w.opts)
    n, nmax = prim.shape[1], binding.NOALLOC_MAX_STATES
    reps = -(-nmax // n)
    big_p = prim.repeat(1, reps)[:, :nmax].contiguous()
    big_m = met.repeat(1, reps)[:, :nmax].contiguous()
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    binding.maxspeed_noalloc(big_p, big_m, o, out)          # first use on this size: warm
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(2):                                      # two calls in a row
        out.zero_()
        binding.maxspeed_noalloc(big_p, big_m, o, out)
        np.testing.assert_allclose(out.cpu().numpy(), want, rtol=RTOL, atol=0.0)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "grmhd_maxspeed_noalloc must not allocate device memory"
    # one state more is refused, and the refusal leaves `out` alone
    one_more_p = torch.cat([big_p, big_p[:, :1]], dim=1).contiguous()
    one_more_m = torch.cat([big_m, big_m[:, :1]], dim=1).contiguous()
    before = out.cpu().numpy().copy()
    with pytest.raises(binding.GrmhdError) as ei:
        binding.maxspeed_noalloc(one_more_p, one_more_m, o, out)
    assert ei.value.code == binding.ELIMIT and "GRMHD_NOALLOC_MAX_STATES" in str(ei.value)
    assert np.array_equal(out.cpu().numpy(), before)
