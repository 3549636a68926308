"""Cubic distortion term L6/2 Q_lk dQ_ij/dx_l dQ_ij/dx_k of Eq. 10: oracle pins, GPU parity.

Pins: the paper's PRINTED map between (L1, L2, L3, L6) and the Frank constants inverted by hand,
    K2 = (9 S^2/2) L1 - (9 S^3/4) L6,   K1 = K2 + (9 S^2/4)(L2 + L3),   K3 = K1 + (27 S^3/4) L6,
checked on long-wavelength twist, splay-dominated and bend-dominated director fields against the Frank-Oseen
density of Eq. 9, 1/2 [K1 (div n)^2 + K2 (n.curl n)^2 + K3 |n x curl n|^2]; literal == factorised; force == minus
central differences of the energy on a masked lattice with every constant on; a uniform field feels nothing.
"""
import numpy as np
import pytest

from paper_1911_07045_b200 import workloads as wl

A, B, Cc, L1 = wl.A_5CB, wl.B_5CB, wl.C_5CB, wl.L1_5CB


@pytest.mark.parametrize("L2,L3,L6", [(0.0, 0.0, 0.8), (1.0, 0.5, -0.6), (0.3, -0.2, 1.1)])
def test_frank_oseen_limit_with_printed_map(oracle_mod, L2, L3, L6):
    S = oracle_mod.S0_of(A, B, Cc)
    K2 = 4.5 * S ** 2 * L1 - 2.25 * S ** 3 * L6
    K1 = K2 + 2.25 * S ** 2 * (L2 + L3)
    K3 = K1 + 6.75 * S ** 3 * L6
    L = 64
    u = np.arange(L)
    th1 = 0.4 * np.sin(2 * np.pi * u / L)
    dth = 0.4 * 2 * np.pi / L * np.cos(2 * np.pi * u / L)
    c2, s2 = np.cos(th1) ** 2, np.sin(th1) ** 2
    # n = (cos t, sin t, 0): varying along z = pure twist; along x: bend cos^2 + splay sin^2; along y: the reverse
    dens = {"z": 0.5 * K2 * dth ** 2, "x": 0.5 * (K3 * c2 + K1 * s2) * dth ** 2, "y": 0.5 * (K1 * c2 + K3 * s2) * dth ** 2}
    for ax, dims in (("z", (4, 4, L)), ("x", (L, 4, 4)), ("y", (4, L, 4))):
        Lx, Ly, Lz = dims
        zz, yy, xx = np.meshgrid(np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
        coord = {"z": zz, "x": xx, "y": yy}[ax].reshape(-1)
        th = 0.4 * np.sin(2 * np.pi * coord / L)
        q = wl.uniaxial_q(np.stack([np.cos(th), np.sin(th), 0 * th]), 1.5 * S)
        o = oracle_mod.Oracle(Lx, Ly, Lz, A, B, Cc, L1, L2, L3, L6=L6)
        for v in (0, 1):
            e_el = o.energy(q, v, terms=True)[1][1]
            assert abs(e_el / (16 * np.sum(dens[ax])) - 1) < 4e-3
    assert abs(K3 - K1) > 0.05                       # the test separates bend from splay


def test_literal_equals_factorised_and_fd_gradient(oracle_mod):
    c = wl.random_masked_problem(13, 5, 4, 6)
    o = oracle_mod.Oracle(5, 4, 6, c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"], mask=c["mask"], kind=c["kind"],
                          W=c["W"], axis=c["axis"], L4=0.6, L6=-0.8)
    q = np.asarray(c["q"]).reshape(5, -1).copy()
    e0, e1 = o.energy(q, 0), o.energy(q, 1)
    assert abs(e0 - e1) < 1e-12 * abs(e0)
    F0, F1 = o.forces(q, 0), o.forces(q, 1)
    assert np.abs(F0 - F1).max() < 1e-12 * np.abs(F0).max()
    rng = np.random.default_rng(0)
    sim = np.flatnonzero(np.asarray(c["mask"]).reshape(-1) == 0)
    h = 1e-5
    for _ in range(30):
        a, s = rng.integers(5), rng.choice(sim)
        qp, qm = q.copy(), q.copy()
        qp[a, s] += h
        qm[a, s] -= h
        fd = -(o.energy(qp, 0) - o.energy(qm, 0)) / (2 * h)
        assert abs(fd - F0[a, s]) < 2e-7 * max(1.0, np.abs(F0).max())


def test_uniform_field_feels_nothing(oracle_mod):
    c = wl.random_masked_problem(12, 6, 5, 4)
    q = np.repeat(np.array([0.3, -0.1, 0.2, -0.25, 0.05])[:, None], c["N"], axis=1)
    oa = oracle_mod.Oracle(6, 5, 4, A, B, Cc, L1, mask=c["mask"])
    ob = oracle_mod.Oracle(6, 5, 4, A, B, Cc, L1, mask=c["mask"], L6=0.9)
    assert abs(oa.energy(q, 0) - ob.energy(q, 0)) < 1e-13
    assert np.abs(oa.forces(q, 1) - ob.forces(q, 1)).max() < 1e-14


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
    "masked_70x35x9_L1only": lambda: wl.random_masked_problem(104, 70, 35, 9, obj_frac=0.1, L2=0.0, L3=0.0),
    "replica3": lambda: wl.make_replica("3"),
    "replica4": lambda: wl.make_replica("4"),
    "replica5p": lambda: wl.make_replica("5p"),
}


@pytest.mark.gpu
@pytest.mark.parametrize("name", sorted(GPU_CASES))
@pytest.mark.parametrize("L4,L6", [(0.0, 0.7), (-0.45, -0.5)])
def test_gpu_parity_with_cubic_term(lq, oracle_mod, name, L4, L6):
    """all of Eq. 10 on: forces rel 1e-10, energy and its three terms rel 1e-9, Q after 40 FIRE / GD / Nesterov
    steps max-abs 1e-8; L6 = L4 = 0 restores the force bit for bit"""
    c = GPU_CASES[name]()
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"], mask=c["mask"],
                          kind=c["kind"], W=c["W"], axis=c["axis"], L4=L4, L6=L6)
    ctx = lq.create_from_config(c)
    F0 = lq.lq_forces(ctx)
    lq.lq_set_chiral(ctx, L4)
    lq.lq_set_cubic(ctx, L6)
    Fref = o.forces(c["q"], 1)
    assert np.abs(lq.lq_forces(ctx) - Fref).max() <= 1e-10 * np.abs(Fref).max()
    eref, tref = o.energy(c["q"], 1, terms=True)
    assert abs(lq.lq_energy(ctx) - eref) <= 1e-9 * abs(eref)
    assert np.abs(lq.lq_energy_terms(ctx) - tref).max() <= 1e-9 * np.abs(tref).max()
    rep = lq.lq_fire_minimize(ctx, 40, 0.0, c["fire"], report_energy=True)
    qref, rref = o.fire(c["q"], 40, 0.0, c["fire"], variant=1)
    assert np.abs(lq.lq_get_Q(ctx) - qref).max() <= 1e-8
    assert abs(rep["energy"] - rref["energy"]) <= 1e-9 * abs(rref["energy"])
    for method in (0, 1):
        lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
        lq.lq_descent_minimize(ctx, method, 40, 0.0, 0.003, 0.8)
        qd, _ = o.descent(c["q"], method, 40, 0.0, 0.003, 0.8)
        assert np.abs(lq.lq_get_Q(ctx) - qd).max() <= 1e-8
    lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
    lq.lq_set_chiral(ctx, 0.0)
    lq.lq_set_cubic(ctx, 0.0)
    assert np.array_equal(lq.lq_forces(ctx), F0)
    lq.lq_destroy(ctx)


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["masked_37x21x11", "replica3", "replica5p"])
def test_gpu_everything_on(lq, oracle_mod, name):
    """L1..L6, both external fields, anchoring and objects together; FIRE (both integrators), GD and Nesterov"""
    c = GPU_CASES[name]()
    Hf, chi, Ef, eps, L4, L6 = (0.3, -0.5, 0.8), 0.7, (0.6, 0.2, -0.4), -0.9, 0.35, -0.4
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"], mask=c["mask"],
                          kind=c["kind"], W=c["W"], axis=c["axis"], H=Hf, chi=chi, E=Ef, eps=eps, L4=L4, L6=L6)
    ctx = lq.create_from_config(c)
    lq.lq_set_field(ctx, Hf, chi, Ef, eps)
    lq.lq_set_chiral(ctx, L4)
    lq.lq_set_cubic(ctx, L6)
    Fref = o.forces(c["q"], 1)
    assert np.abs(lq.lq_forces(ctx) - Fref).max() <= 1e-10 * np.abs(Fref).max()
    eref = o.energy(c["q"], 1)
    assert abs(lq.lq_energy(ctx) - eref) <= 1e-9 * abs(eref)
    for integ in (0, 1):
        fp = dict(c["fire"], integrator=integ)
        lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
        lq.lq_fire_minimize(ctx, 30, 0.0, fp)
        qref, _ = o.fire(c["q"], 30, 0.0, fp, variant=1)
        assert np.abs(lq.lq_get_Q(ctx) - qref).max() <= 1e-8
    for method in (0, 1):
        lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
        lq.lq_descent_minimize(ctx, method, 30, 0.0, 0.003, 0.8)
        qd, _ = o.descent(c["q"], method, 30, 0.0, 0.003, 0.8)
        assert np.abs(lq.lq_get_Q(ctx) - qd).max() <= 1e-8
    a = lq.lq_analyze(ctx, 0.3)
    Sref, _, _ = oracle_mod.analyze(lq.lq_get_Q(ctx), c["mask"], 0.3)
    assert np.abs(a["S"] - Sref).max() <= 1e-10
    lq.lq_destroy(ctx)
