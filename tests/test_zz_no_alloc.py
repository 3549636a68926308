"""lq_energy_terms_noalloc: the energy pass for hosts that cannot allocate device memory.

Who that is: a process that has given the whole GPU to its own memory pool (a framework's caching allocator, a
service with a fixed memory budget), where a driver allocation can fail or is not allowed; and a latency-critical
loop that cannot afford the device-wide synchronisation cudaMalloc / cudaFree bring while other streams are busy.
The ordinary lq_energy_terms allocates its partial-sum buffer on first use; this variant keeps the partial sums in
a static array inside liblq.so (1.5 MiB per GPU, at most 65536 reduction blocks = a 512^3 lattice) that every call
on the GPU shares and that still holds whatever the previous call left there.

So the checks here are: the numbers equal the existing path's (tolerance of the other energy tests, and in fact
bit for bit: same kernels, same order) on calls made back to back on lattices of different size, so that stale
contents of the shared array would show; the device-output form; the size limit (exactly at it: accepted, one
block over: rejected with both numbers in the message, nothing launched); the state error.

This file is named to be collected last: `pytest -x` stops at the first failure and a failure here must not hide
the parity tests.  It does not depend on them: it passes alone in a fresh process (where its first call is the one
that looks up the array's device address) and after the rest of the suite.
"""
import numpy as np
import pytest

from paper_1911_07045_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_E = 1e-9                     # relative, as in test_parity_gpu.py / test_fullsize_gpu.py
MAX_BLOCKS = 65536               # include/lq.h: ceil(Lx/64) * ceil(Ly/4) * ceil(Lz/8)


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1911_07045_b200 import binding, build
    build.build()
    binding.load()
    return binding


def _blocks(Lx, Ly, Lz):
    return -(-Lx // 64) * -(-Ly // 4) * -(-Lz // 8)


def _same(got, ref):
    scale = np.abs(ref).sum()
    assert np.abs(got - ref).max() <= TOL_E * scale
    assert np.array_equal(got, ref)          # the header's stronger claim: identical kernels and summation order


def test_back_to_back_calls_match_the_allocating_path(lq):
    """two contexts of different size and physics share the one static array: large, small, large again"""
    big = wl.make_replica("4")               # 96 x 80 x 72, one constant, periodic: 360 blocks
    small = wl.make_replica("3")             # 64^3, L1 + L2 + L3, walls + colloid + anchoring: 128 blocks
    assert _blocks(big["Lx"], big["Ly"], big["Lz"]) > _blocks(small["Lx"], small["Ly"], small["Lz"])
    cb, cs = lq.create_from_config(big), lq.create_from_config(small)
    try:
        got = [lq.lq_energy_terms_noalloc(cb).copy(), lq.lq_energy_terms_noalloc(cs).copy(),
               lq.lq_energy_terms_noalloc(cb).copy(), lq.lq_energy_terms_noalloc(cs).copy()]
        ref_b, ref_s = lq.lq_energy_terms(cb), lq.lq_energy_terms(cs)
        assert np.all(np.isfinite(ref_b)) and ref_s[2] != 0.0      # the small case really has an anchoring term
        for g, r in zip(got, (ref_b, ref_s, ref_b, ref_s)):
            _same(g, r)
        # and once more after the allocating path has run in between, and after the state moved
        lq.lq_fire_minimize(cs, 5, 0.0, small["fire"])
        _same(lq.lq_energy_terms_noalloc(cs), lq.lq_energy_terms(cs))
        assert abs(lq.lq_energy_terms_noalloc(cs).sum() - lq.lq_energy(cs)) <= TOL_E * abs(lq.lq_energy(cs))
    finally:
        lq.lq_destroy(cb)
        lq.lq_destroy(cs)


def test_device_output_twice_in_a_row(lq):
    """where = LQ_DEVICE: the three doubles land in the caller's tensor in stream order, no host copy"""
    import torch
    c = wl.make_replica("5")                 # patterned cell: masked one-constant lattice with anchoring
    ctx = lq.create_from_config(c)
    try:
        out1 = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
        out2 = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
        assert lq.lq_energy_terms_noalloc(ctx, out1) is out1
        lq.lq_energy_terms_noalloc(ctx, out2)
        torch.cuda.synchronize()
        ref = lq.lq_energy_terms(ctx)
        _same(out1.cpu().numpy(), ref)
        _same(out2.cpu().numpy(), ref)
    finally:
        lq.lq_destroy(ctx)


def test_size_limit(lq):
    """exactly MAX_BLOCKS blocks is served (and right); one z-layer of blocks more is refused before any launch"""
    rng = np.random.default_rng(20191107)
    Lx, Ly, Lz = 4, 4096, 512
    assert _blocks(Lx, Ly, Lz) == MAX_BLOCKS
    ctx = lq.lq_create(Lx, Ly, Lz, -0.172, -2.12, 1.73, 2.32)
    try:
        lq.lq_set_Q(ctx, 0.1 * rng.standard_normal((5, Lx * Ly * Lz)))
        _same(lq.lq_energy_terms_noalloc(ctx), lq.lq_energy_terms(ctx))
    finally:
        lq.lq_destroy(ctx)
    over = lq.lq_create(Lx, Ly, Lz + 8, -0.172, -2.12, 1.73, 2.32)
    try:
        with pytest.raises(lq.LqError) as ei:         # the size test comes first: no Q is needed to be told no
            lq.lq_energy_terms_noalloc(over)
        assert ei.value.code == lq.LQ_ERR_ARG
        assert str(_blocks(Lx, Ly, Lz + 8)) in str(ei.value) and str(MAX_BLOCKS) in str(ei.value)
    finally:
        lq.lq_destroy(over)


def test_errors(lq):
    ctx = lq.lq_create(8, 8, 8, -0.172, -2.12, 1.73, 2.32)
    try:
        with pytest.raises(lq.LqError) as ei:
            lq.lq_energy_terms_noalloc(ctx)
        assert ei.value.code == lq.LQ_ERR_STATE
        with pytest.raises(lq.LqError):               # wrong length is caught by the binding
            lq.lq_energy_terms_noalloc(ctx, np.empty(2))
        assert lq.load().lq_energy_terms_noalloc(ctx.handle, None, lq.LQ_HOST) == lq.LQ_ERR_ARG
        assert lq.load().lq_energy_terms_noalloc(ctx.handle, None, 7) == lq.LQ_ERR_ARG
    finally:
        lq.lq_destroy(ctx)
