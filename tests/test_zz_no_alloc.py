"""tpmc_facet_sum_static -- the one entry point of libtpmc.so that allocates no device memory -- against the path every
other test exercises (tpmc_run's own reduction F = sum_f P_f).

Why the entry point exists: some users of the library may not call cudaMalloc when they need a result -- their process
has given the GPU's memory to a pool of its own, or they sit in a loop with a deadline where an allocation's driver
locks and device-wide wait are not acceptable, or another of their threads is capturing a stream in the global mode,
under which the runtime refuses to allocate.  For them the partial sums of this reduction live in a fixed array inside
the library image instead of in memory owned by the mesh handle.  That array is shared by every call on a GPU and keeps
what the previous call left behind, which is what this file probes: calls made back to back, on inputs of different
sizes (so a later, smaller call sees partial sums of an earlier, larger one lying beyond its own), must each agree with
tpmc_run.  The tolerance is the one tests/test_gpu_parity.py uses for the same identity: 1e-12 of sum |P_f| per component
(the two reductions add in different orders, so they agree to rounding, not bit for bit).

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here should not hide the
parity tests.  It shares no state with them (its own meshes), so it passes alone in a fresh process and after them."""
import ctypes as C

import numpy as np
import pytest

import tpmc_inputs as ti


@pytest.fixture(scope="module")
def T():
    import paper_1312_3691_b200 as t
    return t


def _agree(fm, F_static, F_run):
    scale = 1e-12 * fm.abs().sum(0).cpu().numpy() + 1e-30
    a, b = F_static.cpu().numpy(), F_run.cpu().numpy()
    assert np.all(np.abs(a - b) <= scale), (a, b, scale)
    assert np.all(np.abs(a - fm.cpu().numpy().sum(0)) <= scale)       # and with a plain host sum of the same array


@pytest.mark.gpu
def test_static_scratch_sum_agrees_with_tpmc_run_on_calls_in_a_row(T):
    import torch
    # 20 480 facets (five full 4096-facet parts), ~50 k facets (ragged last part), 2 facets (one part, after the big ones)
    cases = [(ti.config("C2")[1], 200_000), (ti.config("C4")[5], 200_000), (ti.config("C1")[0], 100_000)]
    runs = []
    for cfg, count in cases:
        m = cfg.mesh()
        gm = T.Mesh(m.vertices, m.indices, m.flags)
        r = gm.run(cfg, first=0, count=count)
        assert r.stats["hits"] > 0
        runs.append((gm, r))
    out = torch.empty((2 * len(runs), 3), dtype=torch.float64, device="cuda")
    # two passes over the three bodies, six calls in a row on one stream, no synchronisation in between
    for k in range(out.shape[0]):
        _, r = runs[k % len(runs)]
        got = T.tpmc_facet_sum_static(r.facet_momentum, out=out[k])
        assert got.data_ptr() == out[k].data_ptr()                    # the wrapper wrote where it was told to
    torch.cuda.synchronize()
    for k in range(out.shape[0]):
        _, r = runs[k % len(runs)]
        _agree(r.facet_momentum, out[k], r.force)
    # the same input twice gives the same bits (fixed summation tree), whatever ran in between
    for k in range(len(runs)):
        assert torch.equal(out[k], out[k + len(runs)])
    for gm, _ in runs:
        gm.close()


@pytest.mark.gpu
def test_static_scratch_sum_on_ragged_sizes_side_stream_and_empty_input(T):
    import torch
    g = torch.Generator(device="cpu").manual_seed(7)
    side = torch.cuda.Stream()
    for nt in (1, 255, 4096, 4097, 3 * 4096 + 17, 1_035_320, 0):        # descending would hide nothing either: mixed on purpose
        fm = (torch.randn((nt, 3), generator=g, dtype=torch.float64) * 1e-7).cuda()
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            F = T.tpmc_facet_sum_static(fm)
        side.synchronize()
        ref = fm.cpu().numpy().sum(0) if nt else np.zeros(3)
        assert np.all(np.abs(F.cpu().numpy() - ref) <= 1e-12 * fm.abs().sum(0).cpu().numpy() + 1e-30), nt


def test_static_scratch_sum_refuses_what_does_not_fit(T):
    """Argument checks come before any CUDA call, so this runs without a GPU too: more facets than the fixed array
    serves is an error of its own (never a silent fallback to allocating), and the text says what the limit is."""
    L = T.lib()
    dummy = C.c_void_p(256)                                            # never dereferenced: the call must stop first
    assert L.tpmc_facet_sum_static(dummy, T.TPMC_STATIC_MAX_FACETS + 1, None, dummy) == T.TPMC_ECAPACITY
    assert str(T.TPMC_STATIC_MAX_FACETS).encode() in L.tpmc_last_cuda_error()
    assert b"capacity" in L.tpmc_strerror(T.TPMC_ECAPACITY)
    assert L.tpmc_facet_sum_static(dummy, -1, None, dummy) == T.TPMC_EINVAL
    assert L.tpmc_facet_sum_static(None, 5, None, dummy) == T.TPMC_EINVAL
    assert L.tpmc_facet_sum_static(dummy, 5, None, None) == T.TPMC_EINVAL
