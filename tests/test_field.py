"""External-field term, Eq. 13: oracle pins (CPU) and GPU parity.

Pins: the uniaxial limit the paper PRINTS under Eq. 13, "-1/2 S mu0 dchi (H.n)^2 - 1/2 S eps0 deps (E.n)^2" with
Q = (3/2) S (nn - I/3) (Eq. 3); the force as minus central finite differences of the total energy; the constant
force written out by hand; "positive dchi ... will favor alignment of n with H" as the end state of a minimisation.
"""
import numpy as np
import pytest

from paper_1911_07045_b200 import workloads as wl

A, B, Cc, L1 = wl.A_5CB, wl.B_5CB, wl.C_5CB, wl.L1_5CB
H, CHI, E, EPS = (0.3, -0.5, 0.8), 0.7, (0.6, 0.2, -0.4), -0.9


def uniaxial(n, q0, N):
    n = np.asarray(n, float) / np.linalg.norm(n)
    Q = q0 * (np.outer(n, n) - np.eye(3) / 3.0)
    return np.repeat(np.array([Q[0, 0], Q[0, 1], Q[0, 2], Q[1, 1], Q[1, 2]])[:, None], N, axis=1)


def test_printed_uniaxial_limit(oracle_mod):
    """E(n) - E(n') = -1/2 S chi [(H.n)^2 - (H.n')^2] - 1/2 S eps [(E.n)^2 - (E.n')^2] per site, S = q0 / 1.5"""
    N = 4 * 4 * 4
    q0 = oracle_mod.q0_of(A, B, Cc)
    S = q0 / 1.5
    o = oracle_mod.Oracle(4, 4, 4, A, B, Cc, L1, H=H, chi=CHI, E=E, eps=EPS)
    rng = np.random.default_rng(1)
    n1, n2 = rng.standard_normal(3), rng.standard_normal(3)
    n1 /= np.linalg.norm(n1)
    n2 /= np.linalg.norm(n2)
    for variant in (0, 1):
        d = o.energy(uniaxial(n1, q0, N), variant) - o.energy(uniaxial(n2, q0, N), variant)
        ref = -0.5 * S * CHI * (np.dot(H, n1) ** 2 - np.dot(H, n2) ** 2) - 0.5 * S * EPS * (np.dot(E, n1) ** 2 - np.dot(E, n2) ** 2)
        assert abs(d - N * ref) < 1e-12


def test_constant_force_by_hand(oracle_mod):
    """f = -T_ab Q_ab, T = (chi HH + eps EE)/3, Qzz = -Qxx - Qyy  =>  F = (Txx - Tzz, 2Txy, 2Txz, Tyy - Tzz, 2Tyz)"""
    c = wl.bulk_quench(5, 2, Ly=4, Lz=6)
    o0 = oracle_mod.Oracle(5, 4, 6, A, B, Cc, L1)
    o1 = oracle_mod.Oracle(5, 4, 6, A, B, Cc, L1, H=H, chi=CHI, E=E, eps=EPS)
    T = (CHI * np.outer(H, H) + EPS * np.outer(E, E)) / 3.0
    ref = np.array([T[0, 0] - T[2, 2], 2 * T[0, 1], 2 * T[0, 2], T[1, 1] - T[2, 2], 2 * T[1, 2]])
    for variant in (0, 1):
        dF = o1.forces(c["q"], variant) - o0.forces(c["q"], variant)
        assert np.abs(dF - ref[:, None]).max() < 1e-13


def test_force_is_minus_fd_gradient_with_field(oracle_mod):
    c = wl.random_masked_problem(7, 5, 4, 6)
    o = oracle_mod.Oracle(5, 4, 6, c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"], mask=c["mask"], kind=c["kind"],
                          W=c["W"], axis=c["axis"], H=H, chi=CHI, E=E, eps=EPS)
    q = np.asarray(c["q"]).reshape(5, -1).copy()
    F = o.forces(q, 1)
    rng = np.random.default_rng(0)
    sim = np.flatnonzero(np.asarray(c["mask"]).reshape(-1) == 0)
    h = 1e-5
    for _ in range(25):
        a, s = rng.integers(5), rng.choice(sim)
        qp, qm = q.copy(), q.copy()
        qp[a, s] += h
        qm[a, s] -= h
        fd = -(o.energy(qp, 0) - o.energy(qm, 0)) / (2 * h)
        assert abs(fd - F[a, s]) < 2e-7 * max(1.0, np.abs(F).max())


def test_positive_chi_aligns_director_with_H(oracle_mod):
    """'Positive dchi ... will favor alignment of n with H'; negative favours the perpendicular plane"""
    L = 4
    N = L ** 3
    q0 = oracle_mod.q0_of(A, B, Cc)
    q = uniaxial((1.0, 0.2, 0.1), q0, N)
    Hdir = np.array([0.0, 0.0, 1.0])
    for chi, want in ((+0.5, 1.0), (-0.5, 0.0)):
        o = oracle_mod.Oracle(L, L, L, A, B, Cc, L1, H=Hdir, chi=chi)
        qf, rep = o.fire(q, 20000, 1e-10, wl.FIRE_PARAMS, variant=1)
        assert rep["converged"] == 1
        Q = np.array([[qf[0, 0], qf[1, 0], qf[2, 0]], [qf[1, 0], qf[3, 0], qf[4, 0]], [qf[2, 0], qf[4, 0], -qf[0, 0] - qf[3, 0]]])
        w, v = np.linalg.eigh(Q)
        assert abs(abs(v[2, -1]) - want) < 1e-6        # z component of the director


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
def test_gpu_parity_with_field(lq, oracle_mod, name):
    """forces rel 1e-10, energy rel 1e-9, Q after 50 FIRE steps and after 50 GD / Nesterov steps max-abs 1e-8, with
    both fields on; and switching the field off restores the field-free force bit for bit"""
    c = GPU_CASES[name]()
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"], mask=c["mask"],
                          kind=c["kind"], W=c["W"], axis=c["axis"], H=H, chi=CHI, E=E, eps=EPS)
    ctx = lq.create_from_config(c)
    F0 = lq.lq_forces(ctx)
    lq.lq_set_field(ctx, H, CHI, E, EPS)
    Fref = o.forces(c["q"], 1)
    assert np.abs(lq.lq_forces(ctx) - Fref).max() <= 1e-10 * np.abs(Fref).max()
    eref, tref = o.energy(c["q"], 1, terms=True)
    assert abs(lq.lq_energy(ctx) - eref) <= 1e-9 * abs(eref)
    rep = lq.lq_fire_minimize(ctx, 50, 0.0, c["fire"], report_energy=True)
    qref, rref = o.fire(c["q"], 50, 0.0, c["fire"], variant=1)
    assert np.abs(lq.lq_get_Q(ctx) - qref).max() <= 1e-8
    assert abs(rep["energy"] - rref["energy"]) <= 1e-9 * abs(rref["energy"])
    for method in (0, 1):
        lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
        lq.lq_descent_minimize(ctx, method, 50, 0.0, 0.004, 0.8)
        qd, _ = o.descent(c["q"], method, 50, 0.0, 0.004, 0.8)
        assert np.abs(lq.lq_get_Q(ctx) - qd).max() <= 1e-8
    lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
    lq.lq_set_field(ctx, None, 0.0, None, 0.0)
    assert np.array_equal(lq.lq_forces(ctx), F0)
    with pytest.raises(lq.LqError):
        lq.lq_set_field(ctx, (float("nan"), 0, 0), 1.0)
    lq.lq_destroy(ctx)
