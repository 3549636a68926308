"""Seeded synthetic inputs shaped like the paper's workloads (numpy only).

This module serves BOTH the CUDA path and the test oracle and therefore holds
none of the method's arithmetic: no energies, forces, differences or FIRE.  It
produces host arrays only -- lattice sizes, constants, the object mask, the
per-site anchoring records and the initial Q field -- from integer geometry
rules and ``numpy.random.default_rng(seed)`` (PCG64).  The same arrays are
handed to both sides, so no RNG or libm parity between them is needed.

The five configs are BASELINE.json's; they stand in for the paper's workloads
(Fig. 2 bulk quench, Fig. 3/5 colloid in a box, Fig. 6 patterned cell,
PAPER.md:205-211, 237-275), whose own geometry files are not available.
Recipe details: DESIGN.md section 4.

Layout of every field: SoA ``[5][N]`` in component order (xx, xy, xz, yy, yz)
(PAPER.md:173), site index ``s = x + Lx*(y + Ly*z)``.
"""
from __future__ import annotations

import numpy as np

# 5CB constants in lattice units and BASELINE.json's FIRE parameters
A_5CB, B_5CB, C_5CB, L1_5CB = -0.172, -2.12, 1.73, 2.32
# amplitude of the uniaxial tensor Q = q0 (nn - I/3), q0 = (3/2) S0 with S0 of
# Eq. 7.  Stored as data (input recipe); tests pin it against the
# oracle's and the library's own evaluation of Eq. 7.
Q0_5CB = 0.7992969232035255
FIRE_PARAMS = dict(dt0=0.002, dtmax=0.02, alpha0=0.1, Nmin=5, finc=1.1, fdec=0.5, falpha=0.99)
SEED_BASE = 1911070450

SITE_LC, SITE_OBJECT = 0, 1
ANCH_NONE, ANCH_ORIENTED, ANCH_DEGENERATE_PLANAR = 0, 1, 2


def uniaxial_q(n, q0):
    """5 stored components of q0*(n n - I/3) for directors n [3][N]."""
    nx, ny, nz = n
    q = np.empty((5, nx.size), dtype=np.float64)
    q[0] = q0 * (nx * nx - 1.0 / 3.0)
    q[1] = q0 * (nx * ny)
    q[2] = q0 * (nx * nz)
    q[3] = q0 * (ny * ny - 1.0 / 3.0)
    q[4] = q0 * (ny * nz)
    return q


def random_directors(rng, N):
    """n uniform on S^2: z = 2u1-1, phi = 2 pi u2."""
    z = 2.0 * rng.random(N) - 1.0
    phi = 2.0 * np.pi * rng.random(N)
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([r * np.cos(phi), r * np.sin(phi), z])


def random_director_q(seed, N, q0=Q0_5CB):
    return uniaxial_q(random_directors(np.random.default_rng(seed), N), q0)


def noisy_uniform_q(seed, N, n=(0.0, 0.0, 1.0), sigma=0.01, q0=Q0_5CB, sim=None):
    """uniform director n at q0 plus N(0, sigma^2) on each stored component of simulated sites."""
    nn = np.asarray(n, dtype=np.float64)
    nn = nn / np.linalg.norm(nn)
    q = uniaxial_q(np.repeat(nn[:, None], N, axis=1), q0)
    noise = sigma * np.random.default_rng(seed).standard_normal((5, N))
    if sim is not None:
        noise *= sim[None, :]
    return q + noise


def neighbour_is_object(mask3):
    """[Lz][Ly][Lx] bool: some face neighbour (periodic wrap) is an object site."""
    m = mask3.astype(bool)
    out = np.zeros_like(m)
    for ax in range(3):
        out |= np.roll(m, 1, axis=ax) | np.roll(m, -1, axis=ax)
    return out


def _base(Lx, Ly, Lz, L1=L1_5CB, L2=0.0, L3=0.0):
    return dict(Lx=Lx, Ly=Ly, Lz=Lz, N=Lx * Ly * Lz, A=A_5CB, B=B_5CB, C=C_5CB,
                L1=L1, L2=L2, L3=L3, q0=Q0_5CB, fire=dict(FIRE_PARAMS),
                mask=None, kind=None, W=None, axis=None)


def bulk_quench(L, seed, Ly=None, Lz=None):
    """configs 1 and 4: periodic, object-free, random-director quench (Fig. 2's shape)."""
    Ly = L if Ly is None else Ly
    Lz = L if Lz is None else Lz
    c = _base(L, Ly, Lz)
    c["q"] = random_director_q(seed, c["N"])
    return c


def homeotropic_slab(Lx, Ly, Lz, seed, W=1.0):
    """config 2: object layers z=0 and z=Lz-1; boundary layers z=1, Lz-2 oriented along z."""
    c = _base(Lx, Ly, Lz)
    N = c["N"]
    mask3 = np.zeros((Lz, Ly, Lx), dtype=np.uint8)
    mask3[0] = SITE_OBJECT
    mask3[Lz - 1] = SITE_OBJECT
    bnd = neighbour_is_object(mask3) & (mask3 == 0)
    kind = np.where(bnd, ANCH_ORIENTED, ANCH_NONE).astype(np.uint8)
    Wf = np.where(bnd, W, 0.0)
    axis = np.zeros((3, Lz, Ly, Lx))
    axis[2][bnd] = 1.0
    c.update(mask=mask3.reshape(N), kind=kind.reshape(N), W=Wf.reshape(N), axis=axis.reshape(3, N))
    c["q"] = random_director_q(seed, N)
    return c


def colloid_in_box(L, R, seed, W_wall=0.5, W_colloid=5.0, L2=1.0, L3=0.5, sigma=0.01):
    """config 3: object shell (any index in {0, L-1}) with planar anchoring along x on the
    wall-adjacent sites; central sphere dx^2+dy^2+dz^2 <= R^2 about (L/2, L/2, L/2), masked inside,
    homeotropic (radial) anchoring on its adjacent sites.  Sites adjacent to both take the colloid's."""
    c = _base(L, L, L, L2=L2, L3=L3)
    N = c["N"]
    i = np.arange(L)
    Z, Y, X = np.meshgrid(i, i, i, indexing="ij")
    wall = (X == 0) | (X == L - 1) | (Y == 0) | (Y == L - 1) | (Z == 0) | (Z == L - 1)
    cx = L // 2
    dx, dy, dz = X - cx, Y - cx, Z - cx
    sphere = (dx * dx + dy * dy + dz * dz) <= R * R
    mask3 = (wall | sphere).astype(np.uint8)
    sim = mask3 == 0
    near_wall = neighbour_is_object(wall) & sim
    near_sph = neighbour_is_object(sphere) & sim
    kind = np.where(near_wall | near_sph, ANCH_ORIENTED, ANCH_NONE).astype(np.uint8)
    Wf = np.zeros((L, L, L))
    Wf[near_wall] = W_wall
    Wf[near_sph] = W_colloid
    axis = np.zeros((3, L, L, L))
    axis[0][near_wall] = 1.0
    rr = np.sqrt((dx * dx + dy * dy + dz * dz).astype(np.float64))
    rr[rr == 0] = 1.0
    for a, d in enumerate((dx, dy, dz)):
        axis[a][near_sph] = (d / rr)[near_sph]
    c.update(mask=mask3.reshape(N), kind=kind.reshape(N), W=Wf.reshape(N), axis=axis.reshape(3, N))
    c["q"] = noisy_uniform_q(seed, N, sigma=sigma, sim=sim.reshape(N).astype(np.float64))
    return c


def patterned_cell(Lx, Ly, Lz, seed, ndef=8, spacing=50, W_bottom=2.0, W_top=1.0,
                   top_kind=ANCH_ORIENTED, sigma=0.01):
    """config 5 (top_kind=1) and 5' (top_kind=2, the paper's degenerate-planar opposite wall,
    PAPER.md:269).  Bottom boundary layer z=1: oriented anchoring along (cos t, sin t, 0),
    t(x,y) = sum_ij s_ij atan2(y - y_j, x - x_i), ndef x ndef defects at (spacing/2 - 0.5 + spacing*i),
    charges (-1)^(i+j), no periodic images.  Top boundary layer z=Lz-2: axis z."""
    c = _base(Lx, Ly, Lz)
    N = c["N"]
    mask3 = np.zeros((Lz, Ly, Lx), dtype=np.uint8)
    mask3[0] = SITE_OBJECT
    mask3[Lz - 1] = SITE_OBJECT
    kind = np.zeros((Lz, Ly, Lx), dtype=np.uint8)
    Wf = np.zeros((Lz, Ly, Lx))
    axis = np.zeros((3, Lz, Ly, Lx))
    yy, xx = np.meshgrid(np.arange(Ly, dtype=np.float64), np.arange(Lx, dtype=np.float64), indexing="ij")
    theta = np.zeros((Ly, Lx))
    off = 0.5 * spacing - 0.5
    for i in range(ndef):
        for j in range(ndef):
            sgn = 1.0 if (i + j) % 2 == 0 else -1.0
            theta += sgn * np.arctan2(yy - (off + spacing * j), xx - (off + spacing * i))
    kind[1] = ANCH_ORIENTED
    Wf[1] = W_bottom
    axis[0, 1] = np.cos(theta)
    axis[1, 1] = np.sin(theta)
    kind[Lz - 2] = top_kind
    Wf[Lz - 2] = W_top
    axis[2, Lz - 2] = 1.0
    c.update(mask=mask3.reshape(N), kind=kind.reshape(N), W=Wf.reshape(N), axis=axis.reshape(3, N))
    sim = (mask3 == 0).reshape(N).astype(np.float64)
    c["q"] = noisy_uniform_q(seed, N, sigma=sigma, sim=sim)
    return c


# name -> (builder, run spec).  tol/max_steps are BASELINE.json's stopping rules.
def make_config(name: str):
    """The five BASELINE.json configs at full size ('1'..'5', '5p' = config 5')."""
    if name == "1":
        c = bulk_quench(32, SEED_BASE + 1)
        c.update(name="cfg1_32^3_periodic_L1", tol=1e-9, max_steps=2000)
    elif name == "2":
        c = homeotropic_slab(100, 100, 100, SEED_BASE + 2)
        c.update(name="cfg2_100^3_homeotropic_walls_L1", tol=1e-9, max_steps=20000)
    elif name == "3":
        c = colloid_in_box(256, 25, SEED_BASE + 3)
        c.update(name="cfg3_256^3_walls_colloid_L1L2L3", tol=0.0, max_steps=5000)
    elif name == "4":
        c = bulk_quench(512, SEED_BASE + 4)
        c.update(name="cfg4_512^3_periodic_L1", tol=0.0, max_steps=1000)
    elif name == "5":
        c = patterned_cell(400, 400, 100, SEED_BASE + 5)
        c.update(name="cfg5_400x400x100_patterned_L1", tol=1e-8, max_steps=30000)
    elif name == "5p":
        c = patterned_cell(400, 400, 100, SEED_BASE + 5, top_kind=ANCH_DEGENERATE_PLANAR)
        c.update(name="cfg5p_400x400x100_patterned_FGtop_L1", tol=1e-8, max_steps=30000)
    else:
        raise KeyError(name)
    return c


def make_replica(name: str):
    """Declared scaled-down replicas of configs 3, 4, 5, 5' that the oracle finishes in seconds;
    same structure (walls, colloid, defect array), several tiles and ragged tails."""
    if name == "3":
        c = colloid_in_box(64, 6, SEED_BASE + 30)
        c.update(name="replica3_64^3_R6", tol=0.0, max_steps=100)
    elif name == "4":
        c = bulk_quench(96, SEED_BASE + 40, Ly=80, Lz=72)
        c.update(name="replica4_96x80x72", tol=0.0, max_steps=100)
    elif name == "5":
        c = patterned_cell(100, 100, 50, SEED_BASE + 50, ndef=2)
        c.update(name="replica5_100x100x50_2x2", tol=0.0, max_steps=100)
    elif name == "5p":
        c = patterned_cell(100, 100, 50, SEED_BASE + 50, ndef=2, top_kind=ANCH_DEGENERATE_PLANAR)
        c.update(name="replica5p_100x100x50_2x2", tol=0.0, max_steps=100)
    else:
        raise KeyError(name)
    return c


def random_masked_problem(seed, Lx, Ly, Lz, obj_frac=0.2, L2=0.7, L3=0.4, amp=0.3):
    """Tiny stress case: random object sites, random anchoring kinds / W / axes on every
    boundary site, random (non-uniaxial) Q.  Used by the pin and parity tests."""
    rng = np.random.default_rng(seed)
    c = _base(Lx, Ly, Lz, L2=L2, L3=L3)
    N = c["N"]
    mask3 = (rng.random((Lz, Ly, Lx)) < obj_frac).astype(np.uint8)
    bnd = neighbour_is_object(mask3) & (mask3 == 0)
    kind = np.where(bnd, rng.integers(0, 3, size=(Lz, Ly, Lx)), 0).astype(np.uint8)
    Wf = np.where(bnd, 0.2 + rng.random((Lz, Ly, Lx)) * 3.0, 0.0)
    ax = rng.standard_normal((3, Lz, Ly, Lx))
    ax /= np.linalg.norm(ax, axis=0, keepdims=True)
    c.update(mask=mask3.reshape(N), kind=kind.reshape(N), W=Wf.reshape(N), axis=ax.reshape(3, N))
    c["q"] = amp * rng.standard_normal((5, N))
    c.update(name="random_masked_%dx%dx%d" % (Lx, Ly, Lz), tol=0.0, max_steps=50)
    return c
