"""z-slab domain decomposition on the B200: N sub-domains of one process on one GPU
must reproduce the undivided lattice -- flags bit-exact, forces and energy within north_star's tolerances, and Q after
exactly 100 FIRE steps within 1e-8 of the ORACLE (which knows nothing of sub-domains).  Both drivers are checked: the C
group driver lq_slabs_fire_minimize and the per-rank pieces (halo export / import, step_local, step_commit) strung
together by parallel.fire_minimize_emulated, the protocol a one-rank-per-GPU run follows."""
import numpy as np
import pytest

from paper_1911_07045_b200 import parallel, workloads as wl

pytestmark = pytest.mark.gpu
TOL_F, TOL_E, TOL_Q100 = 1e-10, 1e-9, 1e-8


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


CASES = {
    "replica4": lambda: wl.make_replica("4"),               # periodic, one constant: recompute sweep, unmasked
    "replica5p": lambda: wl.make_replica("5p"),             # walls (object planes at the slab faces of rank 0 / n-1), Eq. 14 + 15
    "replica3": lambda: wl.make_replica("3"),               # three constants, walls + colloid: stored-force sweep + fix-up
    "masked_37x21x23": lambda: wl.random_masked_problem(203, 37, 21, 23, obj_frac=0.15, L2=0.0, L3=0.0),
}


@pytest.fixture(scope="module", params=sorted(CASES))
def case(request, oracle_mod):
    c = CASES[request.param]()
    o = make_oracle(oracle_mod, c)
    qref, rref = o.fire(c["q"], 100, 0.0, c["fire"], variant=1)
    return request.param, c, o, qref, rref


@pytest.mark.parametrize("nslabs", [2, 4, 3])
def test_slabs_static_quantities(case, lq, nslabs):
    name, c, o, _, _ = case
    if c["Lz"] < 4 * nslabs:
        pytest.skip("too few planes")
    ctxs = parallel.make_slabs(lq, c, nslabs)
    lq.lq_slabs_exchange(ctxs, lq.LQ_HALO_Q)
    flags = np.concatenate([lq.lq_get_flags(x) for x in ctxs])
    assert np.array_equal(flags, o.classify())
    F = parallel.gather(lq.lq_forces, ctxs)
    Fref = o.forces(c["q"], 1)
    assert np.abs(F - Fref).max() <= TOL_F * np.abs(Fref).max()
    e = sum(lq.lq_energy(x) for x in ctxs)
    eref = o.energy(c["q"], 1)
    assert abs(e - eref) <= TOL_E * abs(eref)
    for x in ctxs:
        lq.lq_destroy(x)


@pytest.mark.parametrize("nslabs", [2, 4])
def test_slabs_100_fire_steps_vs_oracle(case, lq, nslabs):
    name, c, o, qref, rref = case
    if c["Lz"] < 4 * nslabs:
        pytest.skip("too few planes")
    ctxs = parallel.make_slabs(lq, c, nslabs)
    rep = lq.lq_slabs_fire_minimize(ctxs, 100, 0.0, c["fire"], report_energy=True)
    q = parallel.gather(lq.lq_get_Q, ctxs)
    assert rep["steps"] == 100 and rep["converged"] == 0
    assert np.abs(q - qref).max() <= TOL_Q100, "%s x%d: Q err %.3e" % (name, nslabs, np.abs(q - qref).max())
    assert abs(rep["energy"] - rref["energy"]) <= TOL_E * abs(rref["energy"])
    assert abs(rep["dt"] - rref["dt"]) <= 1e-15 and abs(rep["alpha"] - rref["alpha"]) <= 1e-15
    assert abs(rep["Fmax"] - rref["Fmax"]) <= 1e-7 * max(rref["Fmax"], 1e-3)
    assert abs(rep["Frms"] - rref["Frms"]) <= 1e-7 * max(rref["Frms"], 1e-3)
    if c["mask"] is not None:
        obj = c["mask"] == 1
        assert np.array_equal(q[:, obj], c["q"][:, obj])
    for x in ctxs:
        lq.lq_destroy(x)


@pytest.mark.parametrize("name", ["replica4", "replica3"])
def test_rank_protocol_pieces_vs_oracle(lq, oracle_mod, name):
    """halo export / import + step_local / step_commit, rank by rank in one process (parallel.fire_minimize_emulated):
    the pieces a one-rank-per-GPU run uses, against the oracle and bit-identical to the C group driver"""
    c = CASES[name]()
    o = make_oracle(oracle_mod, c)
    qref, _ = o.fire(c["q"], 60, 0.0, c["fire"], variant=1)
    ctxs = parallel.make_slabs(lq, c, 3)
    assert lq.lq_get_info(ctxs[0], "stored_force") == (1.0 if (c["L2"] != 0 or c["L3"] != 0) else 0.0)
    rep = parallel.fire_minimize_emulated(lq, ctxs, 60, 0.0, c["fire"])
    q = parallel.gather(lq.lq_get_Q, ctxs)
    assert rep["steps"] == 60
    assert np.abs(q - qref).max() <= TOL_Q100
    ctxs2 = parallel.make_slabs(lq, c, 3)
    lq.lq_slabs_fire_minimize(ctxs2, 60, 0.0, c["fire"])
    assert np.array_equal(parallel.gather(lq.lq_get_Q, ctxs2), q)
    for x in ctxs + ctxs2:
        lq.lq_destroy(x)


@pytest.mark.parametrize("name", ["replica4", "replica3"])
def test_slabs_semi_implicit_euler_and_velocity(lq, oracle_mod, name):
    """integrator = 1 through the group driver (extra sweep, dt_prev, no FIRST instantiation) against the oracle, and
    lq_get_velocity on sub-domain contexts (pending lazy rescale + a force pass that needs the final ghost planes)
    against the oracle and the undivided context, for both integrators"""
    c = CASES[name]()
    o = make_oracle(oracle_mod, c)
    for integrator in (1, 0):
        fire = dict(c["fire"], integrator=integrator)
        qref, rref, vref = o.fire(c["q"], 60, 0.0, fire, variant=1, return_v=True)
        ctxs = parallel.make_slabs(lq, c, 2)
        rep = lq.lq_slabs_fire_minimize(ctxs, 60, 0.0, fire)
        q, v = parallel.gather(lq.lq_get_Q, ctxs), parallel.gather(lq.lq_get_velocity, ctxs)
        assert rep["steps"] == 60 == rref["steps"]
        assert np.abs(q - qref).max() <= TOL_Q100, "%s integrator %d: Q err %.3e" % (name, integrator, np.abs(q - qref).max())
        assert abs(rep["dt"] - rref["dt"]) <= 1e-15 and abs(rep["alpha"] - rref["alpha"]) <= 1e-15
        vscale = max(np.abs(vref).max(), 1e-3)
        assert np.abs(v - vref).max() <= 1e-7 * vscale
        whole = lq.create_from_config(c)
        lq.lq_fire_minimize(whole, 60, 0.0, fire)
        assert np.abs(v - lq.lq_get_velocity(whole)).max() <= 1e-7 * vscale
        for x in ctxs + [whole]:
            lq.lq_destroy(x)


def test_slabs_converge_and_stop(lq, oracle_mod):
    """stop test across sub-domains: an 8x8x16 quench converges at the same step as the oracle; a uniform field stops
    at step 0 with Q untouched"""
    c = wl.bulk_quench(8, 12345, Lz=16)
    o = make_oracle(oracle_mod, c)
    qref, rref = o.fire(c["q"], 4000, 1e-9, c["fire"], variant=1)
    ctxs = parallel.make_slabs(lq, c, 2)
    rep = lq.lq_slabs_fire_minimize(ctxs, 4000, 1e-9, c["fire"], report_energy=True)
    assert rep["converged"] == 1 and rref["converged"] == 1 and abs(rep["steps"] - rref["steps"]) <= 1
    assert np.abs(parallel.gather(lq.lq_get_Q, ctxs) - qref).max() < 1e-8
    assert abs(rep["energy"] - rref["energy"]) <= 1e-6 * abs(rref["energy"])
    qu = wl.uniaxial_q(np.repeat(np.array([[0.0], [0.6], [0.8]]), c["N"], axis=1), wl.Q0_5CB)
    for x, (z0, nz) in zip(ctxs, parallel.split_z(16, 2)):
        lq.lq_set_Q(x, parallel.slice_planes(qu, (8, 8, 16), z0, nz, 0, (5,)))
    rep = lq.lq_slabs_fire_minimize(ctxs, 10, 1e-9, c["fire"])
    assert rep["converged"] == 1 and rep["steps"] == 0
    assert np.array_equal(parallel.gather(lq.lq_get_Q, ctxs), qu)
    # the sweep count of the step-wise protocol is only defined while a run is open
    with pytest.raises(lq.LqError) as ei:
        lq.lq_get_info(ctxs[0], "fire_sweeps_total")
    assert ei.value.code == lq.LQ_ERR_STATE
    lq.lq_fire_begin(ctxs[0], 7, 0.0, c["fire"])
    assert lq.lq_get_info(ctxs[0], "fire_sweeps_total") == 7 and lq.lq_get_info(ctxs[0], "stored_force") == 0
    lq.lq_fire_end(ctxs[0])
    lq.lq_fire_begin(ctxs[0], 7, 0.0, dict(c["fire"], integrator=1))
    assert lq.lq_get_info(ctxs[0], "fire_sweeps_total") == 8
    lq.lq_fire_end(ctxs[0])
    # misuse: a sub-domain context refuses the single-domain minimisers
    with pytest.raises(lq.LqError) as ei:
        lq.lq_fire_minimize(ctxs[0], 1, 0.0, c["fire"])
    assert ei.value.code == lq.LQ_ERR_STATE
    for x in ctxs:
        lq.lq_destroy(x)
