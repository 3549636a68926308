"""Chiral distortion term L4/2 eps_lik Q_lj dQ_ij/dx_k of Eq. 10: oracle pins and GPU parity.

Pins (none retypes the oracle's loops):
  * a uniform helix n = (cos qz, sin qz, 0): worked out by hand from Eq. 10 with centred differences the chiral energy
    per site is L4 q0^2 sin(2q)/4; in the continuum limit that is -q0_ch K2 theta' with the paper's PRINTED map
    L4 = -(8 / 9 S^2) q0_ch K2, the cross term of the Frank-Oseen twist energy K2/2 (n.curl n + q0_ch)^2
    (Eq. 9), n.curl n = -theta';
  * with L1 and L4 the helix of lowest energy on the lattice has tan(q) L1-term balance: dE/dq = 0 <=> the closed
    form below; a minimisation started near it converges to it;
  * literal (enumerated sign combinations) == factorised; force == -central finite differences on masked lattices;
    a uniform field feels no chiral force; the term is odd under mirror reflection.
"""
import numpy as np
import pytest

from paper_1911_07045_b200 import workloads as wl

A, B, Cc, L1 = wl.A_5CB, wl.B_5CB, wl.C_5CB, wl.L1_5CB


def helix(q0, L, m, nxy=4, handed=+1):
    """Q = q0 (nn - I/3), n = (cos(qz), handed sin(qz), 0), q = 2 pi m / L, lattice nxy x nxy x L"""
    z = np.repeat(np.arange(L), nxy * nxy)
    th = 2 * np.pi * m / L * z
    return wl.uniaxial_q(np.stack([np.cos(th), handed * np.sin(th), 0 * th]), q0)


def test_uniform_helix_closed_form_and_printed_map(oracle_mod):
    S0 = oracle_mod.S0_of(A, B, Cc)
    q0 = 1.5 * S0
    L, L4 = 48, 0.37
    for m in (1, 2, 5):
        q = 2 * np.pi * m / L
        o0 = oracle_mod.Oracle(4, 4, L, A, B, Cc, L1)
        o4 = oracle_mod.Oracle(4, 4, L, A, B, Cc, L1, L4=L4)
        for v in (0, 1):
            d = o4.energy(helix(q0, L, m), v) - o0.energy(helix(q0, L, m), v)
            assert abs(d - 16 * L * L4 * q0 ** 2 * np.sin(2 * q) / 4) < 1e-11
            dm = o4.energy(helix(q0, L, m, handed=-1), v) - o0.energy(helix(q0, L, m, handed=-1), v)
            assert abs(dm + d) < 1e-11                      # mirror image: opposite sign
    # continuum limit with the printed map: L4 = -(8/(9 S^2)) qch K2  =>  f4 -> -qch K2 theta'
    K2, qch, m = 4.5 * S0 ** 2 * L1, 0.2, 1
    L4p = -8.0 / (9.0 * S0 ** 2) * qch * K2
    q = 2 * np.pi * m / 256
    per_site = L4p * q0 ** 2 * np.sin(2 * q) / 4
    assert abs(per_site / (-qch * K2 * q) - 1) < 1e-3


def test_literal_equals_factorised_and_fd_gradient(oracle_mod):
    c = wl.random_masked_problem(11, 5, 4, 6)
    o = oracle_mod.Oracle(5, 4, 6, c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"], mask=c["mask"], kind=c["kind"],
                          W=c["W"], axis=c["axis"], L4=0.6)
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
    obj = np.asarray(c["mask"]).reshape(-1) != 0
    assert np.all(F0[:, obj] == 0)


def test_uniform_field_has_no_chiral_energy_and_no_bulk_force(oracle_mod):
    """every difference vanishes, so the chiral ENERGY is 0 on any mask; the term is linear in the gradient, so
    its force on a uniform field cancels between the two neighbours of a bond pair only where none is missing:
    0 on an object-free periodic lattice, a surface torque next to objects"""
    c = wl.random_masked_problem(12, 6, 5, 4)
    N = c["N"]
    q = np.repeat(np.array([0.3, -0.1, 0.2, -0.25, 0.05])[:, None], N, axis=1)
    oa = oracle_mod.Oracle(6, 5, 4, A, B, Cc, L1, mask=c["mask"])
    ob = oracle_mod.Oracle(6, 5, 4, A, B, Cc, L1, mask=c["mask"], L4=0.9)
    assert abs(oa.energy(q, 0) - ob.energy(q, 0)) < 1e-13
    dF = ob.forces(q, 1) - oa.forces(q, 1)
    assert np.abs(dF).max() > 1e-3                   # the surface torque exists
    oc, od = oracle_mod.Oracle(6, 5, 4, A, B, Cc, L1), oracle_mod.Oracle(6, 5, 4, A, B, Cc, L1, L4=0.9)
    assert np.abs(oc.forces(q, 1) - od.forces(q, 1)).max() < 1e-14


def test_preferred_pitch(oracle_mod):
    """helices theta = q z, q = 2 pi m / L: E(q)/site = L1 q0^2 (1 - cos 2q)... each z bond carries L1 q0^2 sin^2(q)
    (test_frank_oseen pin) and the chiral term L4 q0^2 sin(2q)/4, so E'(q) = 0 <=> tan(2q) = -L4 / (2 L1); the
    commensurate helix nearest to that pitch has the lowest energy and FIRE leaves it in place (it is a stationary
    point of the lattice energy by symmetry) while a neighbouring winding number has a higher energy"""
    S0 = oracle_mod.S0_of(A, B, Cc)
    q0 = 1.5 * S0
    L, m_star = 40, 3
    qs = 2 * np.pi * m_star / L
    L4 = -2.0 * L1 * np.tan(2 * qs)
    o = oracle_mod.Oracle(4, 4, L, A, B, Cc, L1, L4=L4)
    E = {m: o.energy(helix(q0, L, m), 1) for m in range(0, 7)}
    assert min(E, key=E.get) == m_star
    for m in E:                                      # closed form of the whole curve (bulk part is m-independent)
        qm = 2 * np.pi * m / L
        ref = 16 * L * (L1 * q0 ** 2 * np.sin(qm) ** 2 + L4 * q0 ** 2 * np.sin(2 * qm) / 4)
        assert abs((E[m] - E[0]) - ref) < 1e-10
    # at the optimal commensurate pitch the force only relaxes the degree of order; the director field stays
    qf, rep = o.fire(helix(q0, L, m_star), 3000, 1e-9, wl.FIRE_PARAMS, variant=1)
    assert rep["converged"] == 1
    Sf, nf, _ = oracle_mod.analyze(qf)
    th = 2 * np.pi * m_star / L * np.repeat(np.arange(L), 16)
    nref = np.stack([np.cos(th), np.sin(th), 0 * th])
    assert np.abs(np.abs((nf * nref).sum(0)) - 1).max() < 1e-8          # the helix stayed where it was
    assert rep["energy"] <= o.energy(helix(q0, L, m_star), 1) + 1e-12


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
def test_gpu_parity_with_chiral_term(lq, oracle_mod, name):
    """forces rel 1e-10, energy rel 1e-9, Q after 40 FIRE / GD / Nesterov steps max-abs 1e-8 with L4 on; L4 = 0
    restores the achiral force bit for bit"""
    c = GPU_CASES[name]()
    L4 = -0.45
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"], mask=c["mask"],
                          kind=c["kind"], W=c["W"], axis=c["axis"], L4=L4)
    ctx = lq.create_from_config(c)
    F0 = lq.lq_forces(ctx)
    lq.lq_set_chiral(ctx, L4)
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
        lq.lq_descent_minimize(ctx, method, 40, 0.0, 0.004, 0.8)
        qd, _ = o.descent(c["q"], method, 40, 0.0, 0.004, 0.8)
        assert np.abs(lq.lq_get_Q(ctx) - qd).max() <= 1e-8
    lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
    lq.lq_set_chiral(ctx, 0.0)
    assert np.array_equal(lq.lq_forces(ctx), F0)
    with pytest.raises(lq.LqError):
        lq.lq_set_chiral(ctx, float("inf"))
    lq.lq_destroy(ctx)


@pytest.mark.gpu
def test_gpu_helix_energy_closed_form(lq):
    """the hand-derived helix value straight against the CUDA energy (no oracle in between)"""
    L, m, L4 = 48, 2, 0.37
    ctx = lq.lq_create(4, 4, L, A, B, Cc, L1, 0.0, 0.0)
    q0 = 1.5 * lq.lq_get_S0(ctx)
    q = np.ascontiguousarray(helix(q0, L, m))
    lq.lq_set_Q(ctx, q)
    e0 = lq.lq_energy(ctx)
    lq.lq_set_chiral(ctx, L4)
    assert abs((lq.lq_energy(ctx) - e0) - 16 * L * L4 * q0 ** 2 * np.sin(2 * 2 * np.pi * m / L) / 4) < 1e-10
    lq.lq_destroy(ctx)
