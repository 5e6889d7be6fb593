"""grpic_compact_static: the order-preserving compaction for callers that cannot allocate (scratch in
a file-scope static __device__ array of the library, no workspace, no cudaMalloc) against the existing
grpic_compact, bit for bit, on two calls in a row that share the static array.  Collected last on
purpose (file name): the suite runs with `pytest -x`."""
import ctypes as C

import numpy as np
import pytest

import inputs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def G():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2503_04558_b200 import grpic
    return grpic


def _particles(p, n, seed, frac_removed):
    rng = np.random.default_rng(seed)
    ptc = inputs.make_particles(p, n, seed, "crowded", ("loguniform", 0.1, 10.0))
    ptc["flag"] = (ptc["flag"] | (2 * (rng.uniform(size=n) < frac_removed))).astype(np.uint32)
    ptc["w"] = rng.uniform(0.5, 1.5, n)
    return ptc


def test_compact_static_matches_compact_on_two_calls_in_a_row(G):
    p = inputs.grid_params(64, 64, 0.9)
    ref_ctx = G.Context(p, 1 << 20)                       # existing path: needs its workspace
    ctx = G.Context(p)
    # the context of the static path has NO workspace: the existing entry point refuses to run on it
    G._check(G.load().grpic_set_workspace(ctx.h, None, C.c_size_t(0)))
    # two calls in a row on the shared static array: the second one is smaller (fewer tiles, other
    # survivor counts), so stale words of the first call lie right behind the ones it uses
    cases = [(700001, 1, 0.15), (30011, 2, 0.6)]
    src = [G.Particles.from_numpy(_particles(p, n, seed, fr)) for n, seed, fr in cases]
    dst = [G.Particles(n) for n, _, _ in cases]
    na = [torch.full((1,), -1, dtype=torch.int64, device="cuda") for _ in cases]
    with pytest.raises(G.GrpicError):
        a, b = src[1].struct(), dst[1].struct()
        G._check(G.load().grpic_compact(ctx.h, C.byref(a), C.byref(b),
                                        C.cast(C.c_void_p(na[1].data_ptr()), C.POINTER(C.c_int64)), G._stream()))
    ctx.compact_static(src[0], dst[0], na[0])             # first call: resolves the array's address
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    ctx.compact_static(src[1], dst[1], na[1])             # second call, straight after
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before    # no device memory was taken by the call
    for k, (n, _, _) in enumerate(cases):
        ref = G.Particles(n)
        nr = torch.full((1,), -1, dtype=torch.int64, device="cuda")
        ref_ctx.compact(src[k], ref, nr)
        torch.cuda.synchronize()
        assert int(na[k].item()) == int(nr.item()) and 0 < int(nr.item()) < n
        got, want = dst[k].to_numpy(), ref.to_numpy()
        m = int(nr.item())
        for key in want:                                  # integer and byte work: bit-exact
            assert np.array_equal(got[key][:m], want[key][:m]), (k, key)
        assert np.all(got["flag"][m:] & 2) and np.array_equal(got["cell"][m:], want["cell"][m:])
    # empty input
    e_src, e_dst = G.Particles(0), G.Particles(0)
    ctx.compact_static(e_src, e_dst, na[0])
    torch.cuda.synchronize()
    assert int(na[0].item()) == 0


def test_compact_static_rejects_sizes_beyond_its_maximum(G):
    p = inputs.grid_params(16, 16, 0.5)
    ctx = G.Context(p)
    lib = G.load()
    src, dst = G.Particles(8), G.Particles(8)
    na = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    a, b = src.struct(), dst.struct()
    a.n = ctx.COMPACT_STATIC_MAX_PARTICLES + 1            # the size is checked before anything is read
    rc = lib.grpic_compact_static(ctx.h, C.byref(a), C.byref(b),
                                  C.cast(C.c_void_p(na.data_ptr()), C.POINTER(C.c_int64)), G._stream())
    torch.cuda.synchronize()
    assert rc == -5 and b"capacity" in lib.grpic_strerror(rc)
    assert int(na.item()) == -7                           # nothing was launched
