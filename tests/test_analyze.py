"""Director / order-parameter / defect-mask analysis: oracle pins and GPU parity.

The oracle is the plain definition (numpy.linalg.eigh per site).  Pins: the paper's own parametrisations, Eq. 3
(uniaxial) and Eq. 2 (biaxial), written out here and inverted by the oracle; the threshold rule; object sites.
The director is headless: parity compares n n^T through |n . n_ref| and, separately, the sign
convention; where the two largest eigenvalues are closer than 1e-6 the direction is ill-conditioned and only the
eigen-equation residual is checked.
"""
import numpy as np
import pytest

from paper_1911_07045_b200 import workloads as wl


def five(Q):
    return np.stack([Q[:, 0, 0], Q[:, 0, 1], Q[:, 0, 2], Q[:, 1, 1], Q[:, 1, 2]])


def frames(rng, N):
    """N random orthonormal frames (n, m, l = n x m)"""
    a = rng.standard_normal((N, 3))
    n = a / np.linalg.norm(a, axis=1, keepdims=True)
    b = rng.standard_normal((N, 3))
    b -= (b * n).sum(1, keepdims=True) * n
    m = b / np.linalg.norm(b, axis=1, keepdims=True)
    return n, m, np.cross(n, m)


def test_eq3_uniaxial_roundtrip(oracle_mod):
    """Q = (3/2) S (nn - I/3)  ->  largest eigenvalue S, eigenvector +-n"""
    rng = np.random.default_rng(0)
    N = 500
    n, _, _ = frames(rng, N)
    S = 0.05 + rng.random(N)
    Q = 1.5 * S[:, None, None] * (n[:, :, None] * n[:, None, :] - np.eye(3) / 3.0)
    So, no, _ = oracle_mod.analyze(five(Q))
    assert np.abs(So - S).max() < 1e-14
    assert np.abs(np.abs((no.T * n).sum(1)) - 1.0).max() < 1e-13
    k = np.argmax(np.abs(no), axis=0)
    assert np.all(no[k, np.arange(N)] > 0)           # sign convention


def test_eq2_biaxial_roundtrip_and_threshold(oracle_mod):
    """Eq. 2: eigenvalues S (n), (S_B - S)/2 (m), -(S_B + S)/2 (l); S is the largest for S_B < 3 S"""
    rng = np.random.default_rng(1)
    N = 400
    n, m, l = frames(rng, N)
    S = 0.1 + rng.random(N)
    SB = (rng.random(N) - 0.5) * S                   # |S_B| < S/2
    Q = 1.5 * S[:, None, None] * (n[:, :, None] * n[:, None, :] - np.eye(3) / 3.0) \
        + 0.5 * SB[:, None, None] * (m[:, :, None] * m[:, None, :] - l[:, :, None] * l[:, None, :])
    mask = (rng.random(N) < 0.2).astype(np.uint8)
    So, no, d = oracle_mod.analyze(five(Q), mask, threshold=0.6)
    sim = mask == 0
    assert np.abs(So[sim] - S[sim]).max() < 1e-14
    assert np.abs(np.abs((no.T * n).sum(1))[sim] - 1.0).max() < 1e-12
    assert np.array_equal(d[sim], (S[sim] < 0.6).astype(np.uint8))
    assert np.all(So[~sim] == 0) and np.all(no[:, ~sim] == 0) and np.all(d[~sim] == 0)


# ------------------------------------------------------------------ GPU parity

@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1911_07045_b200 import binding, build
    build.build()
    binding.load()
    return binding


GPU_CASES = {
    "masked_37x21x11": lambda: wl.random_masked_problem(103, 37, 21, 11, obj_frac=0.15),
    "replica3": lambda: wl.make_replica("3"),
    "replica4": lambda: wl.make_replica("4"),
    "replica5p": lambda: wl.make_replica("5p"),
    "cfg1": lambda: wl.make_config("1"),
}


def check(lq, oracle_mod, ctx, q, mask, thr):
    r = lq.lq_analyze(ctx, thr)
    S, n, d = oracle_mod.analyze(q, mask, thr)
    N = S.size
    sim = np.ones(N, bool) if mask is None else np.asarray(mask).reshape(-1) == 0
    assert np.abs(r["S"] - S).max() <= 1e-12
    q = np.asarray(q).reshape(5, -1)
    Q = np.empty((N, 3, 3))
    Q[:, 0, 0], Q[:, 0, 1], Q[:, 0, 2] = q[0], q[1], q[2]
    Q[:, 1, 0], Q[:, 1, 1], Q[:, 1, 2] = q[1], q[3], q[4]
    Q[:, 2, 0], Q[:, 2, 1], Q[:, 2, 2] = q[2], q[4], -q[0] - q[3]
    w = np.linalg.eigvalsh(Q)
    gap = w[:, 2] - w[:, 1]
    g = r["director"]
    res = np.einsum("nij,jn->in", Q, g) - r["S"] * g            # eigen-equation residual, every simulated site
    assert np.abs(res[:, sim]).max() <= 1e-10
    assert np.abs(np.linalg.norm(g[:, sim], axis=0) - 1.0).max() <= 1e-12
    well = sim & (gap > 1e-6)
    assert well.sum() > 0.9 * sim.sum()
    assert np.abs(np.abs((g * n).sum(0))[well] - 1.0).max() <= 1e-9
    k = np.argmax(np.abs(g), axis=0)
    assert np.all(g[k, np.arange(N)][sim] > 0)                     # sign convention
    clear = sim & (np.abs(S - thr) > 1e-12)
    assert np.array_equal(r["defect"][clear], d[clear])
    assert np.all(r["S"][~sim] == 0) and np.all(g[:, ~sim] == 0) and np.all(r["defect"][~sim] == 0)
    assert r["n_defect"] == int(r["defect"].sum())
    return r


@pytest.mark.gpu
@pytest.mark.parametrize("name", sorted(GPU_CASES))
def test_gpu_analysis_parity(lq, oracle_mod, name):
    """on the seeded initial state and after 30 FIRE steps (defect cores appear in the quench)"""
    c = GPU_CASES[name]()
    ctx = lq.create_from_config(c)
    thr = 0.8 * lq.lq_get_S0(ctx)
    check(lq, oracle_mod, ctx, c["q"], c["mask"], thr)
    lq.lq_fire_minimize(ctx, 30, 0.0, c["fire"])
    r = check(lq, oracle_mod, ctx, lq.lq_get_Q(ctx), c["mask"], thr)
    if name in ("replica4", "cfg1"):
        assert 0 < r["n_defect"] < r["S"].size                      # a coarsening quench has melted cores
    lq.lq_destroy(ctx)


@pytest.mark.gpu
def test_gpu_analysis_device_outputs_and_errors(lq, oracle_mod):
    import torch
    c = wl.make_replica("4")
    ctx = lq.lq_create(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], 0.0, 0.0)
    with pytest.raises(lq.LqError) as e:
        lq.lq_analyze(ctx, 0.3)
    assert e.value.code == lq.LQ_ERR_STATE
    lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
    N = c["N"]
    S = torch.empty(N, dtype=torch.float64, device="cuda")
    d = torch.empty((3, N), dtype=torch.float64, device="cuda")
    m = torch.empty(N, dtype=torch.uint8, device="cuda")
    cnt = lq.lq_analyze_device(ctx, 0.3, S, d, m)
    r = lq.lq_analyze(ctx, 0.3)
    assert np.array_equal(S.cpu().numpy(), r["S"]) and np.array_equal(d.cpu().numpy(), r["director"])
    assert np.array_equal(m.cpu().numpy(), r["defect"]) and cnt == r["n_defect"]
    only = lq.lq_analyze(ctx, 0.3, want_director=False, want_defect=False)
    assert only["director"] is None and np.array_equal(only["S"], r["S"]) and only["n_defect"] == cnt
    lq.lq_destroy(ctx)
