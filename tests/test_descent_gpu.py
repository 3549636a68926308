"""GPU parity of the gradient-descent / Nesterov minimisers against the CPU oracle, element by
element on the same seeded host arrays, through the C ABI.  Tolerances follow north_star's FIRE bar: Q after
exactly K steps max-abs 1e-8 (K = 100 on the replicas), Fmax / Frms rel 1e-9, energy rel 1e-9.
"""
import numpy as np
import pytest

from paper_1911_07045_b200 import workloads as wl

pytestmark = pytest.mark.gpu

ETA, MU = 0.004, 0.8        # stable for the three-constant stencils too (largest Hessian eigenvalue ~ 12 (3 L1 + L2 + L3))


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1911_07045_b200 import binding, build
    build.build()
    binding.load()
    return binding


def make_oracle(oracle_mod, c):
    return oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"],
                             mask=c["mask"], kind=c["kind"], W=c["W"], axis=c["axis"])


CASES = {
    "masked_5x4x6_odd": (lambda: wl.random_masked_problem(102, 5, 4, 6, obj_frac=0.25), 40),
    "masked_37x21x11": (lambda: wl.random_masked_problem(103, 37, 21, 11, obj_frac=0.15), 40),
    "masked_70x35x9_L1only": (lambda: wl.random_masked_problem(104, 70, 35, 9, obj_frac=0.1, L2=0.0, L3=0.0), 40),
    "replica3": (lambda: wl.make_replica("3"), 100),
    "replica4": (lambda: wl.make_replica("4"), 100),
    "replica5p": (lambda: wl.make_replica("5p"), 100),
    "cfg1": (lambda: wl.make_config("1"), 100),
}


@pytest.fixture(scope="module", params=sorted(CASES))
def case(request, lq, oracle_mod):
    build, K = CASES[request.param]
    c = build()
    ctx = lq.create_from_config(c)
    yield request.param, c, ctx, make_oracle(oracle_mod, c), K
    lq.lq_destroy(ctx)


@pytest.mark.parametrize("method", [0, 1])
def test_q_after_K_steps(case, lq, method):
    name, c, ctx, o, K = case
    lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
    rep = lq.lq_descent_minimize(ctx, method, K, 0.0, ETA, MU, report_energy=True)
    qref, rref = o.descent(c["q"], method, K, 0.0, ETA, MU)
    assert rep["steps"] == K and rep["converged"] == 0 and rep["launches"] >= K
    q = lq.lq_get_Q(ctx)
    assert np.abs(q - qref).max() <= 1e-8
    assert abs(rep["Fmax"] - rref["Fmax"]) <= 1e-9 * rref["Fmax"]
    assert abs(rep["Frms"] - rref["Frms"]) <= 1e-9 * rref["Frms"]
    assert abs(rep["energy"] - rref["energy"]) <= 1e-9 * abs(rref["energy"])
    if c["mask"] is not None:                      # object sites never move
        obj = np.asarray(c["mask"]).reshape(-1) != 0
        assert np.array_equal(q.reshape(5, -1)[:, obj], np.asarray(c["q"]).reshape(5, -1)[:, obj])


@pytest.mark.parametrize("method", [0, 1])
def test_general_kernel_path_matches_too(lq, oracle_mod, method):
    """fire_path = 1 runs k_descent over every site (no TMA sweep): same oracle, same tolerance; and the two GPU
    paths agree with each other far below it"""
    for name in ("masked_70x35x9_L1only", "replica5p", "replica3", "masked_37x21x11"):
        build, K = CASES[name]
        c = build()
        o = make_oracle(oracle_mod, c)
        qref, _ = o.descent(c["q"], method, K, 0.0, ETA, MU)
        got = []
        for path in (1, 0):
            ctx = lq.create_from_config(c)
            lq.lq_set_option(ctx, "fire_path", path)
            rep = lq.lq_descent_minimize(ctx, method, K, 0.0, ETA, MU)
            assert rep["steps"] == K
            got.append(lq.lq_get_Q(ctx))
            lq.lq_destroy(ctx)
            assert np.abs(got[-1] - qref).max() <= 1e-8
        assert np.abs(got[0] - got[1]).max() <= 1e-12


def test_first_step_is_q_plus_eta_F(case, lq):
    """one GD step against the force entry point of the same library and the oracle's force"""
    name, c, ctx, o, K = case
    lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
    F = lq.lq_forces(ctx)
    lq.lq_descent_minimize(ctx, 0, 1, 0.0, ETA)
    q1 = lq.lq_get_Q(ctx)
    ref = np.asarray(c["q"]).reshape(5, -1) + ETA * o.forces(c["q"], 1)
    assert np.abs(q1.reshape(5, -1) - ref).max() <= 1e-13
    assert np.abs(q1.reshape(5, -1) - (np.asarray(c["q"]).reshape(5, -1) + ETA * F.reshape(5, -1))).max() <= 1e-13


def test_stop_convention_and_chaining(lq, oracle_mod):
    """tolerance stop applies the step that measured it; a run split over several calls of GD equals one run;
    FIRE still works on the same context afterwards (buffers rotate through the velocity storage)"""
    c = wl.make_replica("4")
    o = make_oracle(oracle_mod, c)
    ctx = lq.create_from_config(c)
    rep = lq.lq_descent_minimize(ctx, 1, 50, 1e9, ETA, MU)
    assert rep["steps"] == 1 and rep["converged"] == 1
    assert not lq.lq_get_velocity(ctx).any()           # no velocity is carried (the storage served as a buffer)
    q1ref, _ = o.descent(c["q"], 1, 1, 0.0, ETA, MU)
    assert np.abs(lq.lq_get_Q(ctx) - q1ref).max() <= 1e-13
    lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
    for k in (7, 2, 11):
        lq.lq_descent_minimize(ctx, 0, k, 0.0, ETA)
    qref, _ = o.descent(c["q"], 0, 20, 0.0, ETA)
    assert np.abs(lq.lq_get_Q(ctx) - qref).max() <= 1e-10
    for k in (3, 4):                                   # odd / even Nesterov step counts leave Q in every buffer
        lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
        lq.lq_descent_minimize(ctx, 1, k, 0.0, ETA, MU)
        qn, _ = o.descent(c["q"], 1, k, 0.0, ETA, MU)
        assert np.abs(lq.lq_get_Q(ctx) - qn).max() <= 1e-11
        lq.lq_fire_minimize(ctx, 20, 0.0, c["fire"])
        qf, _ = o.fire(qn, 20, 0.0, c["fire"], variant=1)
        assert np.abs(lq.lq_get_Q(ctx) - qf).max() <= 1e-9
    lq.lq_destroy(ctx)


def test_bad_arguments(lq):
    c = wl.bulk_quench(8, 3)
    ctx = lq.lq_create(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], 0.0, 0.0)
    with pytest.raises(lq.LqError) as e:
        lq.lq_descent_minimize(ctx, 0, 5, 0.0, ETA)
    assert e.value.code == lq.LQ_ERR_STATE
    lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
    for args in ((2, 5, 0.0, ETA, MU), (0, 5, 0.0, 0.0, MU), (1, 5, 0.0, ETA, 1.0), (0, -1, 0.0, ETA, MU),
                 (0, 5, -1.0, ETA, MU)):
        with pytest.raises(lq.LqError) as e:
            lq.lq_descent_minimize(ctx, *args)
        assert e.value.code == lq.LQ_ERR_ARG
    lq.lq_destroy(ctx)
