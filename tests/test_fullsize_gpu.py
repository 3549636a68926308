"""GPU parity at BASELINE.json's FULL sizes (configs 2, 3, 4, 5, 5'), in the launch configuration bench.py times.

What the oracle can do at these sizes in a few minutes it does in full: classification, energy, force field and
exactly 100 FIRE steps (north_star's gate) on configs 2, 3, 5, 5' at full size, every site (oracle: OpenMP variant,
measured on the GPU box's 16 host cores: about 1-4 minutes per config).  Config 4 (512^3, 134M sites) uses sampled
sites for forces and the first FIRE step, plus properties that hold at any size (lattice-translation equivariance of
the fused trajectory, agreement of the fused sweep with the unfused generic path), and its 256^3 periodic crop runs
the full 100 steps against the oracle in the SAME launch configuration as the 512^3 run (64-plane z-chunks, many
waves of CTAs).  north_star's converged-energy gate (rel 1e-6): config 2 at full size against the oracle and the
closed form 980000 f0; configs 3, 5, 5' on their declared replicas (the full-size runs need 5000 /
30000 steps of a 16M-site oracle).  The oracle leg of the config-2 convergence run (7.3 min) is opt-in:
LQ_FULL_PARITY=1; its passing logs are kept in profiles/r02_parity_fullsize.txt and r03_parity_fullsize.txt.  Also at full size: gradient descent and
Nesterov on configs 5 and 3, the analysis kernel at 512^3 on sampled sites, and config 3's lattice with every energy
term switched on (chiral, cubic, both fields).
"""
import os

import numpy as np
import pytest

from paper_1911_07045_b200 import workloads as wl

pytestmark = pytest.mark.gpu
TOL_F, TOL_E, TOL_Q = 1e-10, 1e-9, 1e-8
FULL = os.environ.get("LQ_FULL_PARITY", "0") == "1"


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available()
    from paper_1911_07045_b200 import binding, build
    build.build()
    binding.load()
    return binding


def make_oracle(oracle_mod, c):
    return oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"],
                             mask=c["mask"], kind=c["kind"], W=c["W"], axis=c["axis"])


@pytest.mark.parametrize("name,steps", [("2", 100), ("3", 100), ("5", 100), ("5p", 100)])
def test_full_size_masked_configs(lq, oracle_mod, name, steps):
    c = wl.make_config(name)
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    # classification: bit-exact
    ref = o.classify()
    assert np.array_equal(lq.lq_get_flags(ctx), ref)
    assert lq.lq_get_info(ctx, "n_object") == int(np.sum((ref & 3) == 2))
    # force field and energy on the seeded initial state, every site
    Fref = o.forces(c["q"], 1)
    F = lq.lq_forces(ctx)
    assert np.abs(F - Fref).max() <= TOL_F * np.abs(Fref).max()
    del F
    eref, tref = o.energy(c["q"], 1, terms=True)
    assert abs(lq.lq_energy(ctx) - eref) <= TOL_E * abs(eref)
    # FIRE: exactly `steps` fused steps vs the oracle, every site
    rep = lq.lq_fire_minimize(ctx, steps, 0.0, c["fire"], report_energy=True)
    qref, rref = o.fire(c["q"], steps, 0.0, c["fire"], variant=1)
    q = lq.lq_get_Q(ctx)
    assert rep["steps"] == steps
    assert np.abs(q - qref).max() <= TOL_Q
    assert abs(rep["energy"] - rref["energy"]) <= TOL_E * abs(rref["energy"])
    assert abs(rep["dt"] - rref["dt"]) <= 1e-15 and abs(rep["alpha"] - rref["alpha"]) <= 1e-15
    assert rep["energy"] < eref                                   # DESIGN.md R18
    obj = c["mask"] == 1
    assert np.array_equal(q[:, obj], c["q"][:, obj])
    lq.lq_destroy(ctx)


def test_config3_classification_counts(lq):
    """integer geometry rules of DESIGN.md section 4, counted on the GPU (lattice-point counts)"""
    c = wl.make_config("3")
    ctx = lq.create_from_config(c)
    L = 256
    idx = np.arange(-128, 128)
    n_sph = int(np.sum(idx[:, None, None] ** 2 + idx[None, :, None] ** 2 + idx[None, None, :] ** 2 <= 625))
    n_wall = L ** 3 - (L - 2) ** 3
    assert lq.lq_get_info(ctx, "n_object") == n_wall + n_sph
    f = lq.lq_get_flags(ctx)
    assert int(np.sum(((f & 3) == 1) & (c["W"] == 0.5))) == (L - 2) ** 3 - (L - 4) ** 3
    assert lq.lq_get_info(ctx, "n_simulated") == L ** 3 - n_wall - n_sph
    lq.lq_destroy(ctx)


def test_config4_full_size(lq, oracle_mod):
    """512^3 periodic quench: sampled forces, full energy, first FIRE step on sampled sites (closed form of the
    kick-drift from the oracle's force), translation equivariance and fused-vs-unfused agreement."""
    c = wl.make_config("4")
    L = 512
    N = c["N"]
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    rng = np.random.default_rng(4)
    sites = rng.integers(0, L, size=(3000, 3))
    sites[:64] = np.array([[x, y, z] for x in (0, 1, 510, 511) for y in (0, 17, 495, 511) for z in (0, 63, 64, 511)])
    F = lq.lq_forces(ctx)
    Fs = np.array([o.force_at(c["q"], x, y, z, 1) for x, y, z in sites])
    sidx = sites[:, 0] + L * (sites[:, 1] + L * sites[:, 2])
    scale = np.abs(F).max()
    assert np.abs(F[:, sidx].T - Fs).max() <= TOL_F * scale
    eref = o.energy(c["q"], 1)
    assert abs(lq.lq_energy(ctx) - eref) <= TOL_E * abs(eref)
    # one fused step: q1 = q0 + dt0 * (dt0/2) F0 at every sampled site (v0 = 0; Alg. 1)
    dt0 = c["fire"]["dt0"]
    rep = lq.lq_fire_minimize(ctx, 1, 0.0, c["fire"])
    q1 = lq.lq_get_Q(ctx)
    assert rep["steps"] == 1 and rep["sweep_launches"] == 1
    assert np.abs(q1[:, sidx].T - (c["q"][:, sidx].T + dt0 * 0.5 * dt0 * Fs)).max() <= 1e-13
    assert abs(rep["Fmax"] - np.abs(lq.lq_forces(ctx)).max()) <= 1e-9 * scale
    del F
    # K fused steps vs K unfused steps (independent generic kernels), every site
    K = 6
    lq.lq_set_Q(ctx, c["q"])
    lq.lq_fire_minimize(ctx, K, 0.0, c["fire"])
    qa = lq.lq_get_Q(ctx)
    lq.lq_set_option(ctx, "fire_path", 1)
    lq.lq_set_Q(ctx, c["q"])
    lq.lq_fire_minimize(ctx, K, 0.0, c["fire"])
    qb = lq.lq_get_Q(ctx)
    lq.lq_set_option(ctx, "fire_path", 0)
    assert np.abs(qa - qb).max() <= 1e-11
    del qb
    # translation equivariance of the fused trajectory (periodic lattice): roll by (37, 5, 130) sites
    sh = (130, 5, 37)                                              # (z, y, x)
    qr = np.ascontiguousarray(np.roll(c["q"].reshape(5, L, L, L), sh, axis=(1, 2, 3)).reshape(5, N))
    lq.lq_set_Q(ctx, qr)
    del qr
    lq.lq_fire_minimize(ctx, K, 0.0, c["fire"])
    qc = lq.lq_get_Q(ctx)
    assert np.abs(qc.reshape(5, L, L, L) - np.roll(qa.reshape(5, L, L, L), sh, axis=(1, 2, 3))).max() <= 1e-11
    lq.lq_destroy(ctx)


def test_config4_crop_256_100_steps(lq, oracle_mod):
    """north_star: Q after exactly 100 FIRE steps, max-abs 1e-8, on the 256^3 periodic crop of config 4 (SURVEY 8(d)
    allows the crop: the 512^3 oracle needs 16 GB and hours).  256^3 takes the same launch configuration of
    k_sweep_rc as 512^3: 64-plane z-chunks, 1024 CTAs = 7 waves on 148 SMs, x/y/z ghost shells written by face
    CTAs -- the configuration bench.py times, oracle-checked over many steps."""
    c = wl.bulk_quench(256, wl.SEED_BASE + 4)
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    rep = lq.lq_fire_minimize(ctx, 100, 0.0, c["fire"], report_energy=True)
    assert rep["steps"] == 100 and rep["sweep_launches"] == 100 and rep["launches"] == 100
    qref, rref = o.fire(c["q"], 100, 0.0, c["fire"], variant=1)
    assert np.abs(lq.lq_get_Q(ctx) - qref).max() <= TOL_Q
    assert abs(rep["energy"] - rref["energy"]) <= TOL_E * abs(rref["energy"])
    assert abs(rep["dt"] - rref["dt"]) <= 1e-15 and abs(rep["alpha"] - rref["alpha"]) <= 1e-15
    assert abs(rep["P"] - rref["P"]) <= 1e-6 * abs(rref["P"])
    lq.lq_destroy(ctx)


TOL_ECONV = 1e-6


def test_config2_converged_energy_full_size(lq, oracle_mod):
    """north_star: converged minimised energy rel 1e-6.  Config 2 at full size (100^3 slab, homeotropic walls) to
    max|F| < 1e-9: against the closed form 980000 f0 (uniform z texture: zero bulk force, zero elastic energy, both
    wall terms zero, Eq. 6-8) and against the oracle run the same way (about 6700 steps
    of a 1M-site lattice: a few minutes on the box's host cores)."""
    c = wl.make_config("2")
    ctx = lq.create_from_config(c)
    rep = lq.lq_fire_minimize(ctx, c["max_steps"], c["tol"], c["fire"], report_energy=True)
    S0 = lq.lq_get_S0(ctx)
    f0 = 0.75 * c["A"] * S0 ** 2 + 0.25 * c["B"] * S0 ** 3 + 9.0 / 16.0 * c["C"] * S0 ** 4
    assert rep["converged"] == 1 and rep["Fmax"] < c["tol"]
    assert abs(rep["energy"] - 980000 * f0) <= TOL_ECONV * abs(980000 * f0)
    if not FULL:
        # the oracle leg takes 7.3 min on the GPU box's 16 cores (measured; passing logs: profiles/r02_parity_fullsize.txt, r03_parity_fullsize.txt):
        # opt in with LQ_FULL_PARITY=1 so that the default -m gpu suite stays near ten minutes
        lq.lq_destroy(ctx)
        return
    o = make_oracle(oracle_mod, c)
    qref, rref = o.fire(c["q"], c["max_steps"], c["tol"], c["fire"], variant=1)
    assert rref["converged"] == 1
    assert abs(rep["energy"] - rref["energy"]) <= TOL_ECONV * abs(rref["energy"])
    assert abs(rep["steps"] - rref["steps"]) <= max(5, rref["steps"] // 100)      # chaotic late-stage schedule
    lq.lq_destroy(ctx)


@pytest.mark.parametrize("name", ["3", "5", "5p"])
def test_replica_converged_energy(lq, oracle_mod, name):
    """north_star: converged minimised energy rel 1e-6 on the declared replicas of configs 3, 5, 5' (full size:
    5000 / 30000 steps of a 16M-site oracle).  Both sides run to max|F| < 1e-8 or 2000 steps, whichever comes first;
    the energies at the end agree to 1e-6 relative and the energy has dropped."""
    c = wl.make_replica(name)
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    e0 = lq.lq_energy(ctx)
    rep = lq.lq_fire_minimize(ctx, 2000, 1e-8, c["fire"], report_energy=True)
    qref, rref = o.fire(c["q"], 2000, 1e-8, c["fire"], variant=1)
    assert rep["converged"] == rref["converged"]
    assert abs(rep["steps"] - rref["steps"]) <= 3
    assert abs(rep["energy"] - rref["energy"]) <= TOL_ECONV * abs(rref["energy"])
    assert rep["energy"] < e0
    lq.lq_destroy(ctx)


@pytest.mark.parametrize("name", ["5", "3"])
def test_full_size_descent(lq, oracle_mod, name):
    """Gradient descent and Nesterov at full size, in the launch configuration bench.py --method times:
    10 steps of each (20 with LQ_FULL_PARITY=1) against the oracle's lqo_descent, every site.  Config 5 runs the
    one-constant sweep with bond codes (every simulated site in the one kernel), config 3 the 19-point sweep + the list
    kernel (opt-in, LQ_FULL_PARITY=1: 72 s of oracle; test_full_size_every_term_on runs the same kernels on the same
    lattice by default)."""
    if name == "3" and not FULL:
        pytest.skip("config 3 leg is opt-in (LQ_FULL_PARITY=1); passing logs: profiles/r02_parity_fullsize.txt, profiles/r03_parity_fullsize.txt")
    c = wl.make_config(name)
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    K, eta, mu = (20 if FULL else 10), 0.004, 0.8
    for method in (0, 1):
        lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
        rep = lq.lq_descent_minimize(ctx, method, K, 0.0, eta, mu)
        qref, rref = o.descent(c["q"], method, K, 0.0, eta, mu)
        q = lq.lq_get_Q(ctx)
        assert rep["steps"] == K
        assert np.abs(q - qref).max() <= TOL_Q
        assert abs(rep["Fmax"] - rref["Fmax"]) <= 1e-9 * rref["Fmax"]
        obj = c["mask"] == 1
        assert np.array_equal(q[:, obj], c["q"][:, obj])
        del q, qref
    lq.lq_destroy(ctx)


def test_full_size_analysis_sampled(lq, oracle_mod):
    """lq_analyze at 512^3 in the configuration bench.py --method analyze times, after 60 FIRE steps of
    the quench (melted cores exist): S, director and defect flag on 400 000 sampled sites against numpy.linalg.eigh
    (the oracle computes them one by one), and the device-side defect count against the returned mask."""
    c = wl.make_config("4")
    ctx = lq.create_from_config(c)
    lq.lq_fire_minimize(ctx, 60, 0.0, c["fire"])
    q = lq.lq_get_Q(ctx)
    rng = np.random.default_rng(20)
    idx = np.sort(rng.choice(c["N"], size=400_000, replace=False))
    # the caller's threshold: the median order of the sample, so that both outcomes of the defect rule occur
    thr = float(np.median(oracle_mod.analyze(np.ascontiguousarray(q[:, idx]), None, 0.0)[0]))
    r = lq.lq_analyze(ctx, thr)
    lq.lq_destroy(ctx)
    S, n, d = oracle_mod.analyze(np.ascontiguousarray(q[:, idx]), None, thr)
    assert np.abs(r["S"][idx] - S).max() <= 1e-12
    g = r["director"][:, idx]
    assert np.abs(np.linalg.norm(g, axis=0) - 1.0).max() <= 1e-12
    Q = np.empty((idx.size, 3, 3))
    qs = q[:, idx]
    Q[:, 0, 0], Q[:, 0, 1], Q[:, 0, 2] = qs[0], qs[1], qs[2]
    Q[:, 1, 0], Q[:, 1, 1], Q[:, 1, 2] = qs[1], qs[3], qs[4]
    Q[:, 2, 0], Q[:, 2, 1], Q[:, 2, 2] = qs[2], qs[4], -qs[0] - qs[3]
    assert np.abs(np.einsum("nij,jn->in", Q, g) - S * g).max() <= 1e-10          # eigen-equation residual
    w = np.linalg.eigvalsh(Q)
    well = (w[:, 2] - w[:, 1]) > 1e-6
    assert well.sum() > 0.9 * idx.size
    assert np.abs(np.abs((g * n).sum(0))[well] - 1.0).max() <= 1e-9
    clear = np.abs(S - thr) > 1e-12
    assert np.array_equal(r["defect"][idx][clear], d[clear])
    assert r["n_defect"] == int(r["defect"].sum())
    assert 0.4 * c["N"] < r["n_defect"] < 0.6 * c["N"]


def test_full_size_every_term_on(lq, oracle_mod):
    """Config 3's lattice (256^3, walls + colloid, L1 L2 L3) with the chiral (L4) and cubic (L6) distortion terms of
    Eq. 10 and both external fields of Eq. 13 switched on: 10 FIRE steps and 5 steps each of GD and Nesterov against the
    oracle, every site.  This is the size at which the cubic-term sweeps (32 x 8 tiles of 256 threads) run many CTAs
    over several z-chunks."""
    c = wl.make_config("3")
    Hf, chi, Ef, eps, L4, L6 = (0.3, -0.5, 0.8), 0.7, (0.6, 0.2, -0.4), -0.9, 0.35, -0.4
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"], mask=c["mask"],
                          kind=c["kind"], W=c["W"], axis=c["axis"], H=Hf, chi=chi, E=Ef, eps=eps, L4=L4, L6=L6)
    ctx = lq.create_from_config(c)
    lq.lq_set_field(ctx, Hf, chi, Ef, eps)
    lq.lq_set_chiral(ctx, L4)
    lq.lq_set_cubic(ctx, L6)
    lq.lq_fire_minimize(ctx, 10, 0.0, c["fire"])
    qref, _ = o.fire(c["q"], 10, 0.0, c["fire"], variant=1)
    assert np.abs(lq.lq_get_Q(ctx) - qref).max() <= TOL_Q
    del qref
    for method in (0, 1):
        lq.lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
        lq.lq_descent_minimize(ctx, method, 5, 0.0, 0.003, 0.8)
        qd, _ = o.descent(c["q"], method, 5, 0.0, 0.003, 0.8)
        assert np.abs(lq.lq_get_Q(ctx) - qd).max() <= TOL_Q
        del qd
    lq.lq_destroy(ctx)
