"""Pins of the oracle's FIRE on the semi-implicit Euler step (integrator = 1; R30).

With A = B = C = 0 the force on a plane wave in the xy component is -kappa a, kappa = 2 L1 lam (7-point symbol), and
every FIRE quantity of the lattice run is a function of the single mode amplitude: the whole algorithm reduces to
a scalar recurrence, written out below from the reading (not from the oracle's loop) and run with a time step
large enough to overshoot, so that the P <= 0 branch (v = 0, dt halved, alpha reset) is exercised too.
"""
import math

import numpy as np

from paper_1911_07045_b200 import workloads as wl

A, B, Cc, L1 = wl.A_5CB, wl.B_5CB, wl.C_5CB, wl.L1_5CB


def scalar_fire_euler(a, kappa, K, fp):
    v, dt, alpha, npos, resets = 0.0, fp["dt0"], fp["alpha0"], 0, 0
    for _ in range(K):
        F = -kappa * a
        v += dt * F
        P = F * v
        if F != 0.0:
            v = (1.0 - alpha) * v + alpha * abs(v) / abs(F) * F
        dtn = dt
        if P > 0.0:
            npos += 1
            if npos > fp["Nmin"]:
                dtn = min(dt * fp["finc"], fp["dtmax"])
                alpha *= fp["falpha"]
        else:
            npos, dtn, alpha, v = 0, dt * fp["fdec"], fp["alpha0"], 0.0
            resets += 1
        a += dt * v
        dt = dtn
    return a, dt, alpha, resets


def test_single_mode_scalar_recurrence(oracle_mod):
    Lx, Ly, Lz = 8, 4, 4
    o = oracle_mod.Oracle(Lx, Ly, Lz, 0.0, 0.0, 0.0, L1)
    x = np.tile(np.arange(Lx), Ly * Lz)
    k = 2 * math.pi / Lx
    wave = np.cos(k * x)
    kappa = 2.0 * L1 * 4 * math.sin(k / 2) ** 2
    fp = dict(wl.FIRE_PARAMS, dt0=0.1, dtmax=0.6, integrator=1)
    q0 = np.zeros((5, Lx * Ly * Lz))
    q0[1] = 0.05 * wave
    for K in (1, 7, 40, 150):
        q, rep = o.fire(q0, K, 0.0, fp, variant=1)
        a, dt, alpha, resets = scalar_fire_euler(0.05, kappa, K, fp)
        assert np.abs(q[1] - a * wave).max() < 1e-13
        assert np.abs(q[[0, 2, 3, 4]]).max() < 1e-16
        assert abs(rep["dt"] - dt) < 1e-15 and abs(rep["alpha"] - alpha) < 1e-15 and rep["steps"] == K
    assert resets > 0                                # the uphill branch was taken on the way


def test_first_step_and_stop_rule(oracle_mod):
    """first step: v = dt0 F0, mixing leaves a vector parallel to F unchanged in norm ((1-a)|v| + a|v|), so
    q1 = q0 + dt0^2 F0; the stop test reads the force at the NEW q, so a huge tolerance stops with steps = 0"""
    c = wl.bulk_quench(8, 11, Ly=6, Lz=5)
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"])
    fp = dict(c["fire"], integrator=1)
    F0 = o.forces(c["q"], 1)
    q1, rep = o.fire(c["q"], 1, 0.0, fp, variant=1)
    assert np.abs(q1 - (np.asarray(c["q"]).reshape(5, -1) + fp["dt0"] ** 2 * F0)).max() < 1e-15
    q, rep = o.fire(c["q"], 10, 1e9, fp, variant=1)
    assert rep["steps"] == 0 and rep["converged"] == 1 and np.array_equal(q, np.asarray(c["q"]).reshape(5, -1))


def test_converges_to_uniform_ground_state_and_lowers_energy(oracle_mod):
    L = 6
    N = L ** 3
    q0v = oracle_mod.q0_of(A, B, Cc)
    rng = np.random.default_rng(4)
    q = np.zeros((5, N))
    q[0] = q[3] = -q0v / 3.0
    q += 0.02 * rng.standard_normal((5, N))
    o = oracle_mod.Oracle(L, L, L, A, B, Cc, L1)
    fp = dict(wl.FIRE_PARAMS, integrator=1)
    qf, rep = o.fire(q, 5000, 1e-10, fp, variant=1)
    f0 = A / 3.0 * q0v ** 2 + 2.0 * B / 27.0 * q0v ** 3 + Cc / 9.0 * q0v ** 4
    assert rep["converged"] == 1
    assert abs(rep["energy"] - N * f0) < 1e-10 * abs(N * f0)
    assert rep["energy"] < o.energy(q, 1)


# ------------------------------------------------------------------ GPU parity
import pytest


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
    "masked_70x35x9_L1only": lambda: wl.random_masked_problem(104, 70, 35, 9, obj_frac=0.1, L2=0.0, L3=0.0),
    "replica3": lambda: wl.make_replica("3"),
    "replica4": lambda: wl.make_replica("4"),
    "replica5p": lambda: wl.make_replica("5p"),
}


@pytest.mark.gpu
@pytest.mark.parametrize("path", [0, 1, 2])
@pytest.mark.parametrize("name", sorted(GPU_CASES))
def test_gpu_euler_fire_matches_oracle(lq, oracle_mod, name, path):
    """Q after exactly 100 steps max-abs 1e-8; dt, alpha, steps exact; Fmax / Frms / P / energy rel 1e-9;
    on the fused sweeps (path 0: default, 2: stored force) and on the four-launch general path (1)"""
    c = GPU_CASES[name]()
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"], mask=c["mask"],
                          kind=c["kind"], W=c["W"], axis=c["axis"])
    fp = dict(c["fire"], integrator=1)
    ctx = lq.create_from_config(c)
    lq.lq_set_option(ctx, "fire_path", path)
    for K in (1, 2, 100):
        lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
        rep = lq.lq_fire_minimize(ctx, K, 0.0, fp, report_energy=True)
        qref, rref = o.fire(c["q"], K, 0.0, fp, variant=1)
        assert rep["steps"] == K and rep["converged"] == 0
        assert np.abs(lq.lq_get_Q(ctx) - qref).max() <= 1e-8
        assert rep["dt"] == rref["dt"] and abs(rep["alpha"] - rref["alpha"]) <= 1e-15
        for key in ("Fmax", "Frms", "P", "energy"):
            assert abs(rep[key] - rref[key]) <= 1e-9 * abs(rref[key]), key
    lq.lq_destroy(ctx)


@pytest.mark.gpu
def test_gpu_euler_fire_stop_rule_and_convergence(lq, oracle_mod):
    c = wl.bulk_quench(12, 5)
    fp = dict(c["fire"], integrator=1)
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"])
    ctx = lq.create_from_config(c)
    rep = lq.lq_fire_minimize(ctx, 50, 1e9, fp)
    assert rep["steps"] == 0 and rep["converged"] == 1
    assert np.array_equal(lq.lq_get_Q(ctx), np.asarray(c["q"]).reshape(lq.lq_get_Q(ctx).shape))
    rep = lq.lq_fire_minimize(ctx, 20000, 1e-9, fp, report_energy=True)
    qref, rref = o.fire(c["q"], 20000, 1e-9, fp, variant=1)
    assert rep["converged"] == 1 and rref["converged"] == 1
    assert abs(rep["steps"] - rref["steps"]) <= 2
    assert abs(rep["energy"] - rref["energy"]) <= 1e-6 * abs(rref["energy"])
    lq.lq_destroy(ctx)
