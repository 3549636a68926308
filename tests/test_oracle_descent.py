"""Pins of the oracle's gradient-descent / Nesterov minimisers (R23, R24).

The paper names both minimisers but prints neither formula nor numbers, so
the pins are closed forms the mathematics fixes, none of them a retyping of the oracle's own loop:
  * a spatially uniform uniaxial field reduces both methods to a scalar recurrence on the order parameter S
    through the paper's Eq. 6 -- derived here from Eq. 6, not from the tensor code;
  * with A = B = C = 0 the energy is the quadratic form (L1/2) sum_bonds |dQ|^2, a plane
    wave is an eigenmode, and both methods become linear recurrences with the eigenvalue 2 L1 lambda(k);
  * invariants: object sites never move, small-step GD never raises the energy, the stopping convention.
"""
import math

import numpy as np

from paper_1911_07045_b200 import workloads as wl

A, B, Cc, L1 = wl.A_5CB, wl.B_5CB, wl.C_5CB, wl.L1_5CB


def uniaxial_z(S, N):
    """Q = S (zz - I/3) on N sites, stored (xx, xy, xz, yy, yz)"""
    q = np.zeros((5, N))
    q[0] = -S / 3.0
    q[3] = -S / 3.0
    return q


def fprime(S):
    """d/dS of Eq. 6 in the normalisation Q = S (nn - I/3): f = A/3 S^2 + 2B/27 S^3 + C/9 S^4
    (tr Q^2 = 2 S^2/3, tr Q^3 = 2 S^3/9 put into Eq. 5)"""
    return 2.0 * A / 3.0 * S + 2.0 * B / 9.0 * S * S + 4.0 * Cc / 9.0 * S ** 3


def test_uniform_field_reduces_to_scalar_recurrence(oracle_mod):
    """xx = yy = -S/3 stays symmetric; dS = -3 dxx and df/dxx = -(3/2) f'(S) give S <- S - (9/2) eta f'(S)"""
    o = oracle_mod.Oracle(6, 5, 4, A, B, Cc, L1)
    N, eta, mu, S_init = 120, 0.05, 0.6, 0.3
    for method in (0, 1):
        q, rep = o.descent(uniaxial_z(S_init, N), method, 25, 0.0, eta, mu)
        S, Sp = S_init, S_init
        for _ in range(25):
            y = S + (mu * (S - Sp) if method == 1 else 0.0)
            S, Sp = y - 4.5 * eta * fprime(y), S
        assert rep["steps"] == 25 and rep["converged"] == 0
        assert np.allclose(q[0], -S / 3.0, rtol=0, atol=1e-14) and np.allclose(q[3], -S / 3.0, rtol=0, atol=1e-14)
        assert np.abs(q[[1, 2, 4]]).max() == 0.0
        assert abs(S - S_init) > 0.05          # the recurrence actually moved


def test_plane_wave_linear_recurrence(oracle_mod):
    """A = B = C = 0: F = L1 M lap(q); for the xy component M = 2, so a plane wave of wave vector k decays as
    a <- (1 - 2 eta L1 lam) a (GD) and a_{k+1} = (1 - 2 eta L1 lam)((1 + mu) a_k - mu a_{k-1}) (Nesterov),
    lam = sum_k 4 sin^2(k_k / 2) (7-point Laplacian symbol)."""
    Lx, Ly, Lz = 8, 6, 4
    o = oracle_mod.Oracle(Lx, Ly, Lz, 0.0, 0.0, 0.0, L1)
    z, y, x = np.meshgrid(np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    kx, ky, kz = 2 * math.pi / Lx, 2 * 2 * math.pi / Ly, 2 * math.pi / Lz
    wave = np.cos(kx * x + ky * y + kz * z).reshape(-1)
    lam = 4 * (math.sin(kx / 2) ** 2 + math.sin(ky / 2) ** 2 + math.sin(kz / 2) ** 2)
    q0 = np.zeros((5, Lx * Ly * Lz))
    q0[1] = 0.01 * wave
    eta, mu, K = 0.02, 0.5, 12
    g = 1.0 - 2.0 * eta * L1 * lam
    for method in (0, 1):
        q, _ = o.descent(q0, method, K, 0.0, eta, mu)
        a, ap = 0.01, 0.01
        for _ in range(K):
            yk = a + (mu * (a - ap) if method == 1 else 0.0)
            a, ap = g * yk, a
        assert np.allclose(q[1], a * wave, rtol=0, atol=1e-15)
        assert np.abs(q[[0, 2, 3, 4]]).max() < 1e-18


def test_xx_yy_block_eigenmodes(oracle_mod):
    """the (xx, yy) block of M is [[2, 1], [1, 2]]: xx = yy decays with 3 L1 lam, xx = -yy with 1 L1 lam"""
    Lx, Ly, Lz = 8, 4, 4
    o = oracle_mod.Oracle(Lx, Ly, Lz, 0.0, 0.0, 0.0, L1)
    x = np.tile(np.arange(Lx), Ly * Lz)
    k = 2 * math.pi / Lx
    wave = np.sin(k * x)
    lam = 4 * math.sin(k / 2) ** 2
    eta = 0.03
    for sign, ev in ((+1.0, 3.0), (-1.0, 1.0)):
        q0 = np.zeros((5, Lx * Ly * Lz))
        q0[0], q0[3] = 0.02 * wave, sign * 0.02 * wave
        q, _ = o.descent(q0, 0, 5, 0.0, eta)
        a = 0.02 * (1.0 - eta * ev * L1 * lam) ** 5
        assert np.allclose(q[0], a * wave, rtol=0, atol=1e-15) and np.allclose(q[3], sign * a * wave, rtol=0, atol=1e-15)


def test_masked_invariants_and_energy_descent(oracle_mod):
    """object sites never move; with a small step plain GD lowers the energy every step (descent lemma);
    Nesterov ends below its start"""
    c = wl.random_masked_problem(5, 7, 6, 5)
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"],
                          mask=c["mask"], kind=c["kind"], W=c["W"], axis=c["axis"])
    obj = c["mask"].reshape(-1) != 0
    assert obj.any()
    q, rep, tr = o.descent(c["q"], 0, 40, 0.0, 0.01, trace=True, trace_energy=True)
    assert np.array_equal(q[:, obj], c["q"].reshape(5, -1)[:, obj])
    e0 = o.energy(c["q"], 1)
    e = np.concatenate([[e0], tr[:, 2]])
    assert np.all(np.diff(e) < 0.0)
    assert abs(rep["energy"] - tr[-1, 2]) <= 1e-12 * abs(rep["energy"])
    qn, repn = o.descent(c["q"], 1, 40, 0.0, 0.01, 0.8)
    assert np.array_equal(qn[:, obj], c["q"].reshape(5, -1)[:, obj])
    assert repn["energy"] < e0
    assert repn["energy"] < rep["energy"]      # momentum gets further in the same number of steps


def test_stopping_convention_and_first_step(oracle_mod):
    """the test uses F(y_k) of the step and the step's update is still applied: a huge tolerance stops after one
    step with q_1 = q_0 + eta F(q_0) (F from lqo_forces, itself pinned by finite differences); Nesterov's first
    step equals GD's (q_{-1} = q_0)"""
    c = wl.bulk_quench(8, 11, Ly=6, Lz=5)
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"])
    F0 = o.forces(c["q"], 1)
    for method in (0, 1):
        q, rep = o.descent(c["q"], method, 10, 1e9, 0.004, 0.9)
        assert rep["steps"] == 1 and rep["converged"] == 1
        assert rep["Fmax"] == np.abs(F0).max()
        assert np.array_equal(q, c["q"].reshape(5, -1) + 0.004 * F0)
    q, rep = o.descent(c["q"], 0, 0, 0.0, 0.004)
    assert rep["steps"] == 0 and np.array_equal(q, c["q"].reshape(5, -1))


def test_gd_converges_to_uniform_ground_state(oracle_mod):
    """smooth start near a uniform director: GD relaxes to N f0 (Fig. 2 'uniform texture')"""
    L = 6
    N = L ** 3
    q0v = oracle_mod.q0_of(A, B, Cc)
    rng = np.random.default_rng(3)
    q = uniaxial_z(q0v, N) + 0.02 * rng.standard_normal((5, N))
    o = oracle_mod.Oracle(L, L, L, A, B, Cc, L1)
    qf, rep = o.descent(q, 1, 4000, 1e-10, 0.008, 0.7)
    f0 = A / 3.0 * q0v ** 2 + 2.0 * B / 27.0 * q0v ** 3 + Cc / 9.0 * q0v ** 4
    assert rep["converged"] == 1
    assert abs(rep["energy"] - N * f0) < 1e-10 * abs(N * f0)
