"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded host arrays.  Tolerances are BASELINE.json's north_star:
  flags bit-exact; forces  max|dF| <= 1e-10 * max|F_ref|; energy rel 1e-9;
  Q after exactly 100 FIRE steps max-abs 1e-8; converged energy rel 1e-6.
"""
import os

import numpy as np
import pytest

from paper_1911_07045_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_F, TOL_E, TOL_Q100, TOL_ECONV = 1e-10, 1e-9, 1e-8, 1e-6


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


SMALL_CASES = {
    # name -> builder; sizes span several 32x16 tiles with ragged tails in x, y and z
    "masked_4x4x4": lambda: wl.random_masked_problem(101, 4, 4, 4, obj_frac=0.2),
    "masked_5x4x6_odd": lambda: wl.random_masked_problem(102, 5, 4, 6, obj_frac=0.25),
    "masked_37x21x11": lambda: wl.random_masked_problem(103, 37, 21, 11, obj_frac=0.15),
    "masked_70x35x9_L1only": lambda: wl.random_masked_problem(104, 70, 35, 9, obj_frac=0.1, L2=0.0, L3=0.0),
    "dense_objects_12^3": lambda: wl.random_masked_problem(105, 12, 12, 12, obj_frac=0.6),
    "replica3": lambda: wl.make_replica("3"),
    "replica4": lambda: wl.make_replica("4"),
    "replica5": lambda: wl.make_replica("5"),
    "replica5p": lambda: wl.make_replica("5p"),
    "cfg1": lambda: wl.make_config("1"),
}


@pytest.fixture(scope="module", params=sorted(SMALL_CASES))
def case(request, lq, oracle_mod):
    c = SMALL_CASES[request.param]()
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    yield request.param, c, ctx, o
    lq.lq_destroy(ctx)


def test_flags_bit_exact(case, lq):
    name, c, ctx, o = case
    ref = o.classify()
    got = lq.lq_get_flags(ctx)
    assert np.array_equal(got, ref), "%s: %d flag bytes differ" % (name, int(np.sum(got != ref)))
    sim = int(np.sum((ref & 3) != 2))
    assert lq.lq_get_info(ctx, "n_simulated") == sim
    assert lq.lq_get_info(ctx, "n_boundary") == int(np.sum((ref & 3) == 1)) or c["mask"] is None


def test_forces_match_oracle(case, lq):
    name, c, ctx, o = case
    lq.lq_set_Q(ctx, c["q"])
    F = lq.lq_forces(ctx)
    Fref = o.forces(c["q"], 1)
    scale = np.abs(Fref).max()
    err = np.abs(F - Fref).max()
    assert err <= TOL_F * scale, "%s: force err %.3e (scale %.3e)" % (name, err, scale)
    if c["mask"] is not None:
        assert np.abs(F[:, c["mask"] == 1]).max(initial=0.0) == 0.0


def test_energy_matches_oracle(case, lq):
    name, c, ctx, o = case
    lq.lq_set_Q(ctx, c["q"])
    e = lq.lq_energy(ctx)
    t = lq.lq_energy_terms(ctx)
    eref, tref = o.energy(c["q"], 1, terms=True)
    assert abs(e - eref) <= TOL_E * abs(eref), "%s: E %.15g vs %.15g" % (name, e, eref)
    assert np.all(np.abs(t - tref) <= TOL_E * np.maximum(np.abs(tref), abs(eref) * 1e-3))


@pytest.mark.parametrize("path", [0, 1, 2])
def test_q_after_100_fire_steps(case, lq, path):
    name, c, ctx, o = case
    lq.lq_set_option(ctx, "fire_path", path)
    lq.lq_set_Q(ctx, c["q"])
    rep = lq.lq_fire_minimize(ctx, 100, 0.0, c["fire"], report_energy=True)
    q = lq.lq_get_Q(ctx)
    v = lq.lq_get_velocity(ctx)
    qref, rref, vref = o.fire(c["q"], 100, 0.0, c["fire"], variant=1, return_v=True)
    assert rep["steps"] == 100 and rep["converged"] == 0
    assert np.abs(q - qref).max() <= TOL_Q100, "%s: Q err %.3e" % (name, np.abs(q - qref).max())
    assert abs(rep["energy"] - rref["energy"]) <= TOL_E * abs(rref["energy"])
    assert abs(rep["dt"] - rref["dt"]) <= 1e-15 and abs(rep["alpha"] - rref["alpha"]) <= 1e-15
    assert abs(rep["Fmax"] - rref["Fmax"]) <= 1e-7 * max(rref["Fmax"], 1e-3)
    assert abs(rep["P"] - rref["P"]) <= 1e-6 * max(abs(rref["P"]), 1e-6)
    # velocities: Algorithm 1's v at the end of the step, i.e. after the rescale (lq.h, lq_get_velocity)
    assert np.abs(v - vref).max() <= 1e-7 * max(np.abs(vref).max(), 1e-3), "%s: v err %.3e" % (name, np.abs(v - vref).max())
    if c["mask"] is not None:
        obj = c["mask"] == 1
        assert np.array_equal(q[:, obj], c["q"][:, obj])       # object sites never move (R17)
        assert np.abs(v[:, obj]).max(initial=0.0) == 0.0
    lq.lq_set_option(ctx, "fire_path", 0)


@pytest.mark.parametrize("name", ["masked_70x35x9_L1only", "masked_37x21x11", "replica5p"])
def test_anchoring_records_off_boundary_are_ignored(lq, oracle_mod, name):
    """SURVEY 8(c) O5 / DESIGN.md R9: an anchoring term exists iff class == boundary and kind != 0.  Here EVERY site
    (bulk, boundary, object) carries a record with kind in {1, 2}; forces, energy and 100 FIRE steps (fused sweeps,
    both the recompute and the stored-force path) must equal the oracle's, which is pinned to ignore the records
    off the boundary class (tests/test_oracle_pins.py::test_anchoring_only_on_boundary_class_sites)."""
    c = dict(SMALL_CASES[name]())
    rng = np.random.default_rng(4242)
    N = c["N"]
    c["kind"] = rng.integers(1, 3, size=N).astype(np.uint8)
    c["W"] = 0.2 + 3.0 * rng.random(N)
    ax = rng.standard_normal((3, N))
    c["axis"] = ax / np.linalg.norm(ax, axis=0, keepdims=True)
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    Fref = o.forces(c["q"], 1)
    assert np.abs(lq.lq_forces(ctx) - Fref).max() <= TOL_F * np.abs(Fref).max()
    eref = o.energy(c["q"], 1)
    assert abs(lq.lq_energy(ctx) - eref) <= TOL_E * abs(eref)
    qref, _ = o.fire(c["q"], 100, 0.0, c["fire"], variant=1)
    for path in (0, 2):
        lq.lq_set_option(ctx, "fire_path", path)
        lq.lq_set_Q(ctx, c["q"])
        lq.lq_fire_minimize(ctx, 100, 0.0, c["fire"])
        assert np.abs(lq.lq_get_Q(ctx) - qref).max() <= TOL_Q100
    lq.lq_destroy(ctx)


@pytest.mark.parametrize("name", ["replica4", "masked_70x35x9_L1only"])
def test_stored_path_then_recompute_path_without_set_Q(lq, oracle_mod, name):
    """The stored-force sweep (fire_path = 2) must leave the full 2-wide ghost shell of q current, because the
    recompute sweep that may run next on the same context reads q with a 2-site halo.  40 steps on path 2, then 60
    on path 0 with no lq_set_Q in between == the oracle run the same way (two calls, each restarting v, dt, alpha;
    DESIGN.md R13)."""
    c = SMALL_CASES[name]()
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    lq.lq_set_option(ctx, "fire_path", 2)
    lq.lq_fire_minimize(ctx, 40, 0.0, c["fire"])
    lq.lq_set_option(ctx, "fire_path", 0)
    lq.lq_fire_minimize(ctx, 60, 0.0, c["fire"])
    q1, _ = o.fire(c["q"], 40, 0.0, c["fire"], variant=1)
    q2, _ = o.fire(q1, 60, 0.0, c["fire"], variant=1)
    assert np.abs(lq.lq_get_Q(ctx) - q2).max() <= TOL_Q100
    lq.lq_destroy(ctx)


@pytest.mark.parametrize("name", ["replica4", "replica5p", "replica3"])
def test_fused_steps_are_bit_reproducible(lq, name):
    """per-CTA partials are reduced in index order by the last CTA to finish, no floating-point atomics anywhere:
    two runs of 100 fused steps from the same state give bit-identical Q, v and schedule"""
    c = SMALL_CASES[name]()
    ctx = lq.create_from_config(c)
    out = []
    for _ in range(2):
        lq.lq_set_Q(ctx, c["q"])
        rep = lq.lq_fire_minimize(ctx, 100, 0.0, c["fire"])
        out.append((lq.lq_get_Q(ctx), lq.lq_get_velocity(ctx), rep["dt"], rep["alpha"], rep["P"], rep["Fmax"]))
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert out[0][2:] == out[1][2:]
    lq.lq_destroy(ctx)


def test_fused_and_unfused_paths_agree(case, lq):
    name, c, ctx, o = case
    out = []
    for path in (0, 1, 2):
        lq.lq_set_option(ctx, "fire_path", path)
        lq.lq_set_Q(ctx, c["q"])
        lq.lq_fire_minimize(ctx, 37, 0.0, c["fire"])
        out.append(lq.lq_get_Q(ctx))
    lq.lq_set_option(ctx, "fire_path", 0)
    assert np.abs(out[0] - out[1]).max() <= 1e-11
    assert np.abs(out[2] - out[1]).max() <= 1e-11


# ------------------------------------------------------------------ convergence

def test_config1_converged_energy(lq, oracle_mod):
    """config 1 to max|F| < 1e-9 or 2000 steps; energy vs the oracle (rel 1e-6) and vs the closed form
    N f0 of the uniform texture (Fig. 2; Eq. 6 at S0)."""
    c = wl.make_config("1")
    ctx = lq.create_from_config(c)
    rep = lq.lq_fire_minimize(ctx, c["max_steps"], c["tol"], c["fire"], report_energy=True)
    o = make_oracle(oracle_mod, c)
    qref, rref = o.fire(c["q"], c["max_steps"], c["tol"], c["fire"], variant=1)
    assert abs(rep["energy"] - rref["energy"]) <= TOL_ECONV * abs(rref["energy"])
    S0 = lq.lq_get_S0(ctx)
    f0 = 0.75 * c["A"] * S0 ** 2 + 0.25 * c["B"] * S0 ** 3 + 9.0 / 16.0 * c["C"] * S0 ** 4
    assert abs(rep["energy"] - c["N"] * f0) <= TOL_ECONV * abs(c["N"] * f0)
    assert rep["converged"] == rref["converged"]
    assert abs(rep["steps"] - rref["steps"]) <= 2
    lq.lq_destroy(ctx)


def test_converges_and_stops_early(lq, oracle_mod):
    """8^3 quench converges well inside the step budget: same step count as the oracle, Q is the state the
    last force was computed on."""
    c = wl.bulk_quench(8, 12345)
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    for path in (0, 1, 2):
        lq.lq_set_option(ctx, "fire_path", path)
        lq.lq_set_Q(ctx, c["q"])
        rep = lq.lq_fire_minimize(ctx, 4000, 1e-9, c["fire"], report_energy=True)
        qref, rref = o.fire(c["q"], 4000, 1e-9, c["fire"], variant=1)
        assert rep["converged"] == 1 and rref["converged"] == 1
        assert abs(rep["steps"] - rref["steps"]) <= 1
        assert rep["Fmax"] < 1e-9
        assert np.abs(lq.lq_get_Q(ctx) - qref).max() < 1e-8
        assert np.abs(lq.lq_forces(ctx)).max() < 1e-9
    lq.lq_destroy(ctx)


# ------------------------------------------------------------------ edge cases

def test_edge_cases(lq, oracle_mod):
    A, B, Cc, L1 = wl.A_5CB, wl.B_5CB, wl.C_5CB, wl.L1_5CB
    fire = wl.FIRE_PARAMS
    # before set_Q
    ctx = lq.lq_create(6, 6, 6, A, B, Cc, L1)
    for fn in (lambda: lq.lq_get_Q(ctx), lambda: lq.lq_energy(ctx), lambda: lq.lq_forces(ctx),
               lambda: lq.lq_fire_minimize(ctx, 1, 0.0, fire)):
        with pytest.raises(lq.LqError) as ei:
            fn()
        assert ei.value.code == lq.LQ_ERR_STATE
    q = wl.random_director_q(5, 216)
    lq.lq_set_Q(ctx, q)
    # max_steps = 0: nothing moves, report has the initial force
    rep = lq.lq_fire_minimize(ctx, 0, 0.0, fire)
    assert rep["steps"] == 0 and np.array_equal(lq.lq_get_Q(ctx), q)
    o = oracle_mod.Oracle(6, 6, 6, A, B, Cc, L1)
    assert abs(rep["Fmax"] - np.abs(o.forces(q, 1)).max()) < 1e-12
    # already converged: a uniform field at S0
    qu = wl.uniaxial_q(np.repeat(np.array([[0.0], [0.6], [0.8]]), 216, axis=1), wl.Q0_5CB)
    lq.lq_set_Q(ctx, qu)
    rep = lq.lq_fire_minimize(ctx, 10, 1e-9, fire)
    assert rep["converged"] == 1 and rep["steps"] == 0 and np.array_equal(lq.lq_get_Q(ctx), qu)
    # bad parameters
    for bad in (dict(fire, dt0=0.0), dict(fire, dtmax=0.001), dict(fire, falpha=1.5), dict(fire, integrator=2)):
        with pytest.raises(lq.LqError) as ei:
            lq.lq_fire_minimize(ctx, 1, 0.0, bad)
        assert ei.value.code == lq.LQ_ERR_ARG
    with pytest.raises(lq.LqError):
        lq.lq_set_sites(ctx, np.full(216, 2, np.uint8))
    with pytest.raises(lq.LqError):
        lq.lq_set_Q(ctx, q[:, :100].copy())
    # every site an object: nothing simulated, everything is zero, FIRE "converges" at step 0 iff tol > 0
    lq.lq_set_sites(ctx, np.ones(216, np.uint8))
    lq.lq_set_Q(ctx, q)
    assert lq.lq_energy(ctx) == 0.0 and np.abs(lq.lq_forces(ctx)).max() == 0.0
    rep = lq.lq_fire_minimize(ctx, 5, 0.0, fire)
    assert rep["steps"] == 5 and np.array_equal(lq.lq_get_Q(ctx), q)
    # reset to all-bulk
    lq.lq_set_sites(ctx, None)
    assert np.all(lq.lq_get_flags(ctx) == 0xFC)
    lq.lq_destroy(ctx)

    # a site sandwiched between objects along x (R6) and an isolated site
    mask = np.zeros((6, 6, 6), np.uint8)
    mask[2, 2, 1] = mask[2, 2, 3] = 1
    mask[4, 3:6, 3:6] = 1
    mask[4, 4, 4] = 0
    mask[3, 4, 4] = mask[5, 4, 4] = 1
    c = wl.random_masked_problem(7, 6, 6, 6)
    c["mask"] = mask.reshape(-1)
    c["kind"] = np.where(wl.neighbour_is_object(mask) & (mask == 0), np.maximum(c["kind"].reshape(6, 6, 6), 1), 0).astype(np.uint8).reshape(-1)
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    assert np.array_equal(lq.lq_get_flags(ctx), o.classify())
    Fref = o.forces(c["q"], 0)
    assert np.abs(lq.lq_forces(ctx) - Fref).max() <= TOL_F * np.abs(Fref).max()
    eref = o.energy(c["q"], 0)
    assert abs(lq.lq_energy(ctx) - eref) <= TOL_E * abs(eref)
    lq.lq_fire_minimize(ctx, 100, 0.0, c["fire"])
    qref, _ = o.fire(c["q"], 100, 0.0, c["fire"], variant=0)
    assert np.abs(lq.lq_get_Q(ctx) - qref).max() <= TOL_Q100
    lq.lq_destroy(ctx)


def test_device_buffers_and_stream(lq):
    """LQ_DEVICE buffers (torch tensors) and a non-default torch stream give the same results as host buffers"""
    import torch
    c = wl.make_replica("5p")
    ctx = lq.create_from_config(c)
    Fh = lq.lq_forces(ctx)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        ctx2 = lq.lq_create(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"])
        lq.lq_set_stream(ctx2, s.cuda_stream)
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        lq.lq_set_sites(ctx2, dev(c["mask"]), dev(c["kind"]), dev(c["W"]), dev(c["axis"]))
        lq.lq_set_Q(ctx2, dev(c["q"]))
        Fd = torch.empty(5, c["N"], dtype=torch.float64, device="cuda")
        lq.lq_forces(ctx2, Fd)
        fl = torch.empty(c["N"], dtype=torch.uint8, device="cuda")
        lq.lq_get_flags(ctx2, fl)
    s.synchronize()
    assert np.array_equal(Fd.cpu().numpy(), Fh)
    assert np.array_equal(fl.cpu().numpy(), lq.lq_get_flags(ctx))
    lq.lq_destroy(ctx)
    lq.lq_destroy(ctx2)


@pytest.mark.parametrize("name", ["cfg1", "masked_70x35x9_L1only", "masked_5x4x6_L1"])
def test_resident_kernel_matches_streaming_sweeps_and_oracle(lq, oracle_mod, name):
    """Small one-constant lattices run lq_fire_minimize as ONE cooperative launch with the state on chip
    (lq_resident.cu); "resident" = 0 forces the streaming sweep on the same context.  Both against the oracle
    (100 steps, 1e-8) and against each other; the resident run reports a single launch of the fused kernel."""
    if name == "masked_5x4x6_L1":
        c = wl.random_masked_problem(106, 5, 4, 6, obj_frac=0.25, L2=0.0, L3=0.0)
    else:
        c = SMALL_CASES[name]()
    ctx = lq.create_from_config(c)
    o = make_oracle(oracle_mod, c)
    qref, rref, vref = o.fire(c["q"], 100, 0.0, c["fire"], variant=1, return_v=True)
    out = {}
    for resident in (1, 0):
        lq.lq_set_option(ctx, "resident", resident)
        lq.lq_set_Q(ctx, c["q"])
        rep = lq.lq_fire_minimize(ctx, 100, 0.0, c["fire"], report_energy=True)
        q, v = lq.lq_get_Q(ctx), lq.lq_get_velocity(ctx)
        assert rep["steps"] == 100 and rep["converged"] == 0
        assert rep["sweep_launches"] == (1 if resident else 100)
        assert np.abs(q - qref).max() <= TOL_Q100
        assert np.abs(v - vref).max() <= 1e-7 * max(np.abs(vref).max(), 1e-3)
        assert abs(rep["energy"] - rref["energy"]) <= TOL_E * abs(rref["energy"])
        assert abs(rep["dt"] - rref["dt"]) <= 1e-15 and abs(rep["alpha"] - rref["alpha"]) <= 1e-15
        # ghost shell left current: the generic force kernel (reads neighbours through the ghosts) agrees with the oracle
        Fref = o.forces(qref, 1)
        assert np.abs(lq.lq_forces(ctx) - Fref).max() <= 1e-7 * np.abs(Fref).max()
        out[resident] = q
    assert np.abs(out[0] - out[1]).max() <= 1e-11
    lq.lq_destroy(ctx)


def test_fp64_fma_microbenchmark_reports_a_plausible_roof(lq):
    """lq_get_info("fp64_fma_tflops") runs the register-only FMA microbenchmark (SURVEY 8(d)'s secondary roof):
    a B200 has 148 SMs x 64 fp64 FMA per clock, 37 TFLOP/s at 1.965 GHz; anything between a third of that and
    a little above it is a believable measurement, anything else a broken timer or kernel."""
    c = wl.make_replica("4")
    ctx = lq.create_from_config(c)
    t = lq.lq_get_info(ctx, "fp64_fma_tflops")
    assert 12.0 < t < 42.0, t
    lq.lq_destroy(ctx)
