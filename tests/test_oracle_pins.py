"""Pins for the CPU oracle.

None of these re-type the oracle's loops: they use closed forms, conservation
laws, special cases, the survey's independent reference numbers, and a brute
force written in a deliberately different formulation (pull form, velocity set
generated from c.c <= 2, tensor-form equilibrium).
"""
import itertools
import json
import os

import numpy as np
import pytest

from paper_2112_08264_b200 import workloads as w

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "p12_config0_trajectory.json")))


# ----------------------------------------------------------------------------
# an independent D3Q19 description: generated, not typed in
# ----------------------------------------------------------------------------
def generated_lattice():
    vel = [c for c in itertools.product((-1, 0, 1), repeat=3) if sum(a * a for a in c) <= 2]
    wt = {0: 1 / 3, 1: 1 / 18, 2: 1 / 36}
    return vel, [wt[sum(a * a for a in c)] for c in vel]


def test_lattice_table_is_d3q19(oracle_mod):
    c, wgt = oracle_mod.lattice()
    vel, _ = generated_lattice()
    assert len(vel) == 19
    assert sorted(map(tuple, c.tolist())) == sorted(vel)
    assert tuple(c[0]) == (0, 0, 0)
    for i in range(1, 19, 2):                                      # reading S1: opp(i) = i+1 for odd i
        assert np.array_equal(c[i], -c[i + 1])
    c2 = (c * c).sum(1)
    assert np.array_equal(wgt, np.where(c2 == 0, 1 / 3, np.where(c2 == 1, 1 / 18, 1 / 36)))
    # isotropy the method relies on: sum w = 1, sum w c = 0, sum w c c = (1/3) I
    assert abs(wgt.sum() - 1) < 1e-15
    assert np.abs((wgt[:, None] * c).sum(0)).max() < 1e-17
    assert np.allclose(np.einsum("i,ia,ib->ab", wgt, c, c), np.eye(3) / 3, atol=1e-16)
    # S1 explicit order
    want = [(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1),
            (1, 1, 0), (-1, -1, 0), (1, -1, 0), (-1, 1, 0), (1, 0, 1), (-1, 0, -1), (1, 0, -1),
            (-1, 0, 1), (0, 1, 1), (0, -1, -1), (0, 1, -1), (0, -1, 1)]
    assert list(map(tuple, c.tolist())) == want


# P1 ------------------------------------------------------------------------
def test_p1_equilibrium_moments(oracle_mod):
    c, _ = oracle_mod.lattice()
    rng = np.random.default_rng(1)
    for _ in range(200):
        rho = rng.uniform(0.1, 3.0)
        u = rng.normal(size=3)
        u *= rng.uniform(0, 0.1) / np.linalg.norm(u)
        fe = oracle_mod.feq(rho, *u)
        ulp = np.spacing(rho)
        assert abs(fe.sum() - rho) <= 4 * ulp
        assert np.abs(fe @ c - rho * u).max() <= 4 * ulp
        # second moment of Eq. 10: rho (c_s^2 delta + u u)
        pi = np.einsum("i,ia,ib->ab", fe, c, c)
        assert np.abs(pi - rho * (np.eye(3) / 3 + np.outer(u, u))).max() <= 8 * ulp
    # Eq. 10 at rest is w_i rho exactly
    _, wgt = oracle_mod.lattice()
    assert np.array_equal(oracle_mod.feq(1.0, 0, 0, 0), wgt)


def _config0(oracle_mod, n=32, **kw):
    cfg = w.CONFIGS[0]
    rr, rb = w.mixture_fields(n, n, n, cfg.seed)
    o = oracle_mod.Oracle(n, n, n, **kw)
    o.set_fields(rr, rb)
    return o, rr, rb


# P2, P3 --------------------------------------------------------------------
def test_p2_p3_mass_and_momentum_periodic(oracle_mod):
    o, rr, rb = _config0(oracle_mod, 16, tau_r=0.8, tau_b=1.3, G=0.9)
    m0, p0 = o.get_diagnostics()
    assert abs(m0[0] - rr.sum()) < 1e-10 and abs(m0[1] - rb.sum()) < 1e-10
    assert np.abs(p0).max() < 1e-13
    o.step(50)
    m1, p1 = o.get_diagnostics()
    assert np.abs(m1 / m0 - 1).max() < 2e-14          # per-component mass (Eq. 11 analogue)
    assert np.abs(p1).max() < 2e-13                    # pair forces cancel link by link


def test_p2_mass_with_solids(oracle_mod):
    n = 16
    rr, rb = w.mixture_fields(n, n, n, 5)
    mask = w.solid_mask_from_spheres(n, n, n, np.array([[8.0, 8.0, 8.0], [1.5, 14.2, 3.3]]), radius=3.5)
    o = oracle_mod.Oracle(n, n, n, 0.9, 1.1, 1.0)
    o.set_solid_mask(mask)
    o.set_fields(rr, rb)
    m0, _ = o.get_diagnostics()
    fl = mask == 0
    assert abs(m0[0] - rr[fl].sum()) < 1e-10
    o.step(40)
    m1, _ = o.get_diagnostics()
    assert np.abs(m1 / m0 - 1).max() < 2e-14
    f = o.get_populations().reshape(38, -1)
    assert np.all(f[:, mask == 1] == 0.0)             # S8: solid nodes hold exactly 0
    # mask-then-fields and fields-then-mask agree
    o2 = oracle_mod.Oracle(n, n, n, 0.9, 1.1, 1.0)
    o2.set_fields(rr, rb)
    o2.set_solid_mask(mask)
    o2.step(40)
    assert np.array_equal(o2.get_populations().reshape(38, -1), f)


# P4 ------------------------------------------------------------------------
@pytest.mark.parametrize("tau,G", [((1.0, 1.0), 1.2), ((0.8, 1.3), 0.9), ((0.6, 0.6), -2.0)])
def test_p4_uniform_rest_state(oracle_mod, tau, G):
    n = 6
    o = oracle_mod.Oracle(n, n, n, tau[0], tau[1], G)
    o.set_fields(np.full(n ** 3, 0.7), np.full(n ** 3, 1.3))
    f0 = o.get_populations().copy()
    o.step(5)
    f1 = o.get_populations()
    # F = 0 because sum_i w_i c_i = 0, and u' = 0 exactly (opposite pairs cancel in order);
    # what is left is the rounding of the 19-term sum rho = sum_i f_i, <= 18 eps rho per step.
    # (SURVEY P4 says "bit-exact at tau = 1"; in fp64 even sum_i w_i is not exactly 1, so the
    # pin is this bound.  A spurious force of order G*rho would show as ~1e-1.)
    assert np.abs(f1 - f0).max() <= 5 * 18 * 2.0 ** -53 * 1.3


# P5 ------------------------------------------------------------------------
@pytest.mark.parametrize("tau,tol", [(1.0, 1e-4), (0.8, 2e-2), (0.6, 2e-2)])
def test_p5_shear_wave_decay(oracle_mod, tau, tol):
    nx, ny, nz, U, steps = 4, 32, 4, 1e-3, 200
    y = np.arange(ny)
    ux = np.broadcast_to((U * np.sin(2 * np.pi * y / ny))[None, :, None], (nz, ny, nx)).reshape(-1).copy()
    o = oracle_mod.Oracle(nx, ny, nz, tau, tau, 0.0)           # G = 0, identical components
    o.set_fields(np.full(nx * ny * nz, 0.5), np.full(nx * ny * nz, 0.5), ux, None, None)
    amp = []
    for _ in range(steps + 1):
        u = o.get_moments()[2].reshape(nz, ny, nx)
        amp.append(2.0 / ny * (u[0, :, 0] * np.sin(2 * np.pi * y / ny)).sum())
        o.step(1)
    amp = np.array(amp)
    k2 = (2 * np.pi / ny) ** 2
    nu = (tau - 0.5) / 3.0                                       # Eq. 2
    rate = -np.polyfit(np.arange(100, steps + 1), np.log(amp[100:]), 1)[0]
    assert abs(rate / (nu * k2) - 1) < tol


def test_p5_single_fluid_reduction(oracle_mod):
    """rho_b = 0 turns the two-component update into the plain single-fluid BGK of Eq. 1 (reading S6: no division by
    rho^k; the empty component exerts no force and stays exactly empty), for any G.  Pinned by the same shear wave:
    nu = c_s^2 (tau - 1/2), Eq. 2 PAPER.md:84.  This is the oracle of the single-fluid calibration path (lbs_*)."""
    nx, ny, nz, U, steps, tau = 4, 32, 4, 1e-3, 200, 0.8
    y = np.arange(ny)
    ux = np.broadcast_to((U * np.sin(2 * np.pi * y / ny))[None, :, None], (nz, ny, nx)).reshape(-1).copy()
    o = oracle_mod.Oracle(nx, ny, nz, tau, 1.7, 1.2)            # the blue relaxation time and G must not matter
    o.set_fields(np.ones(nx * ny * nz), np.zeros(nx * ny * nz), ux, None, None)
    amp = []
    for _ in range(steps + 1):
        u = o.get_moments()[2].reshape(nz, ny, nx)
        amp.append(2.0 / ny * (u[0, :, 0] * np.sin(2 * np.pi * y / ny)).sum())
        o.step(1)
    f = o.get_populations()
    assert np.all(f[1] == 0.0)                                   # the empty component stays exactly empty
    assert np.all(np.isfinite(f[0]))
    k2 = (2 * np.pi / ny) ** 2
    rate = -np.polyfit(np.arange(100, steps + 1), np.log(np.array(amp)[100:]), 1)[0]
    assert abs(rate / ((tau - 0.5) / 3.0 * k2) - 1) < 0.02


# P6 ------------------------------------------------------------------------
def test_p6_force_on_sine_profile(oracle_mod):
    nx, ny, nz, G, a, b = 32, 3, 5, 1.2, 1.0, 0.2
    x = np.arange(nx)
    kx = 2 * np.pi * 3 / nx
    rb = np.broadcast_to(a + b * np.sin(kx * x), (nz, ny, nx)).reshape(-1).copy()
    rr = np.broadcast_to(0.8 + 0.1 * np.cos(kx * x), (nz, ny, nx)).reshape(-1).copy()
    o = oracle_mod.Oracle(nx, ny, nz, 1.0, 1.0, G)
    o.set_fields(rr, rb)
    Fr, Fb = o.get_force()
    want = -G * rr * (b / 3.0) * np.sin(kx) * np.cos(kx * np.tile(x, ny * nz))
    assert np.abs(Fr[0] - want).max() < 1e-15
    assert np.abs(Fr[1]).max() < 1e-17 and np.abs(Fr[2]).max() < 1e-17
    # the force on blue from red's cosine profile: d/dx cos = -sin
    want_b = -G * rb * (0.1 / 3.0) * np.sin(kx) * (-np.sin(kx * np.tile(x, ny * nz)))
    assert np.abs(Fb[0] - want_b).max() < 1e-15


# P7 ------------------------------------------------------------------------
def test_p7_point_perturbation(oracle_mod):
    n, G, eps = 8, 1.2, 1e-3
    c, wgt = oracle_mod.lattice()
    rb = np.ones(n ** 3)
    p = (3, 4, 5)
    rb[p[0] + n * (p[1] + n * p[2])] += eps
    o = oracle_mod.Oracle(n, n, n, 1.0, 1.0, G)
    o.set_fields(np.ones(n ** 3), rb)
    Fr, Fb = o.get_force()
    Fr = Fr.reshape(3, n, n, n)
    want = np.zeros_like(Fr)
    for i in range(1, 19):
        q = [(p[a] - c[i][a]) % n for a in range(3)]            # node p - c_i sees p along +c_i
        want[:, q[2], q[1], q[0]] = -G * wgt[i] * eps * c[i]
    assert np.abs(Fr - want).max() < 5e-16          # signal is G*w*eps ~ 3e-5..7e-5
    # red is uniform, so blue feels nothing except through its own density factor: F_b = 0
    assert np.abs(Fb).max() < 5e-16


# P8 ------------------------------------------------------------------------
def test_p8_forcing_variants_agree_at_tau1_only(oracle_mod):
    oa, _, _ = _config0(oracle_mod, 12)
    ob, _, _ = _config0(oracle_mod, 12)
    ob.set_forcing(1)
    oa.step(1), ob.step(1)
    fa, fb = oa.get_populations(), ob.get_populations()
    assert np.abs(fa - fb).max() / np.abs(fa).max() < 5e-16
    oc, _, _ = _config0(oracle_mod, 12, tau_r=0.8, tau_b=0.8, G=1.2)
    od, _, _ = _config0(oracle_mod, 12, tau_r=0.8, tau_b=0.8, G=1.2)
    od.set_forcing(1)
    oc.step(10), od.step(10)
    d = np.abs(oc.get_populations() - od.get_populations()).max() / np.abs(oc.get_populations()).max()
    assert 1e-8 < d < 1e-3                                      # they are different schemes off tau = 1


# P9 ------------------------------------------------------------------------
def brute_force_step(f, solid, n, tau, G):
    """One update in PULL form with a generated velocity set (no shared tables).

    f: dict {(k, c): array[z][y][x]} keyed by the velocity vector itself."""
    vel, wt = generated_lattice()
    W = dict(zip(vel, wt))
    cs2 = 1.0 / 3.0
    nx, ny, nz = n

    def feq(c, rho, u):
        cu = sum(ci * ui for ci, ui in zip(c, u))
        return W[c] * rho * (1 + cu / cs2 + cu * cu / (2 * cs2 * cs2) - sum(ui * ui for ui in u) / (2 * cs2))

    post = {}
    rho = {k: sum(f[(k, c)] for c in vel) * (1 - solid) for k in (0, 1)}
    for z, y, x in itertools.product(range(nz), range(ny), range(nx)):
        if solid[z, y, x]:
            continue
        om = [1 / tau[0], 1 / tau[1]]
        mom = [[sum(f[(k, c)][z, y, x] * c[a] for c in vel) for a in range(3)] for k in (0, 1)]
        den = om[0] * rho[0][z, y, x] + om[1] * rho[1][z, y, x]
        u = [(om[0] * mom[0][a] + om[1] * mom[1][a]) / den if den else 0.0 for a in range(3)]
        for k in (0, 1):
            F = [0.0, 0.0, 0.0]                               # F^k = -G psi^k sum_c w_c psi^kbar(x+c) c
            for c in vel:
                nbv = rho[1 - k][(z + c[2]) % nz, (y + c[1]) % ny, (x + c[0]) % nx]
                for a in range(3):
                    F[a] -= G * rho[k][z, y, x] * W[c] * nbv * c[a]
            rk = rho[k][z, y, x]
            ush = [u[a] + (F[a] / rk if rk else 0.0) for a in range(3)]
            for c in vel:
                fe = feq(c, rk, u)
                post[(k, c, z, y, x)] = f[(k, c)][z, y, x] + om[k] * (fe - f[(k, c)][z, y, x]) + (feq(c, rk, ush) - fe)
    g = {key: np.zeros((nz, ny, nx)) for key in f}
    for z, y, x in itertools.product(range(nz), range(ny), range(nx)):
        if solid[z, y, x]:
            continue
        for k in (0, 1):
            for c in vel:                                       # what arrives at (x,y,z) moving along c
                sx, sy, sz = (x - c[0]) % nx, (y - c[1]) % ny, (z - c[2]) % nz
                if solid[sz, sy, sx]:                           # came off a wall: my own reversed population
                    g[(k, c)][z, y, x] = post[(k, tuple(-a for a in c), z, y, x)]
                else:
                    g[(k, c)][z, y, x] = post[(k, c, sz, sy, sx)]
    return g


@pytest.mark.parametrize("n,tau,G,with_solid", [((4, 4, 4), (1.0, 1.0), 1.2, False),
                                                ((4, 4, 4), (0.8, 1.3), 0.9, False),
                                                ((4, 3, 5), (0.7, 1.1), 1.5, True)])
def test_p9_brute_force_small_lattice(oracle_mod, n, tau, G, with_solid):
    nx, ny, nz = n
    c, _ = oracle_mod.lattice()
    rng = np.random.default_rng(42)
    fin = rng.uniform(0.01, 0.1, size=(2, 19, nz, ny, nx))     # random NON-equilibrium populations
    solid = np.zeros((nz, ny, nx), dtype=np.uint8)
    if with_solid:
        solid[1, 1, 2] = 1
        solid[3, 0, 0] = 1
        solid[3, 0, 1] = 1
    o = oracle_mod.Oracle(nx, ny, nz, tau[0], tau[1], G)
    o.set_solid_mask(solid)
    o.set_populations(fin)
    f = {(k, tuple(c[i])): fin[k, i] * (1 - solid) for k in (0, 1) for i in range(19)}
    for _ in range(3):
        o.step(1)
        f = brute_force_step(f, solid, n, tau, G)
        got = o.get_populations()
        for k in (0, 1):
            for i in range(19):
                assert np.abs(got[k, i] - f[(k, tuple(c[i]))]).max() <= 1e-14


# P10 -----------------------------------------------------------------------
def test_p10_demixing_threshold(oracle_mod):
    def contrast_ratio(G):
        o, _, _ = _config0(oracle_mod, 16, G=G)
        o.step(100)
        a = np.std(o.get_moments()[0] - o.get_moments()[1])
        o.step(100)
        b = np.std(o.get_moments()[0] - o.get_moments()[1])
        return b / a
    assert contrast_ratio(0.4) < 0.9        # mixes: long-wave estimate G_c*rho ~ (tau-1/2)/tau = 0.5
    assert contrast_ratio(0.6) > 1.1        # demixes


# P11 -----------------------------------------------------------------------
def _popcount(a):
    return int(np.unpackbits(a.view(np.uint8)).sum())


def test_p11_bounce_back_geometry(oracle_mod):
    g = GOLD["geometry"]
    n = 32
    for key, ctr in (("sphere_R5.5_on_node", 16.0), ("sphere_R5.5_on_cell_centre", 16.5)):
        mask = w.solid_mask_from_spheres(n, n, n, np.array([[ctr] * 3]))
        o = oracle_mod.Oracle(n, n, n)
        o.set_solid_mask(mask)
        links = o.get_link_mask()
        assert _popcount(links) == g[key]["links"]
        assert np.all(links[mask == 1] == 0)
    # one solid node: 18 links, one per direction, each on the node it points from
    c, _ = oracle_mod.lattice()
    mask = np.zeros((5, 5, 5), np.uint8)
    mask[2, 2, 2] = 1
    o = oracle_mod.Oracle(5, 5, 5)
    o.set_solid_mask(mask)
    links = o.get_link_mask().reshape(5, 5, 5)
    assert _popcount(links) == 18
    for i in range(1, 19):
        assert links[2 - c[i][2], 2 - c[i][1], 2 - c[i][0]] == 1 << i
    # flat wall z = 0 in a 4x4x6 box: plane z=1 sees the 5 directions with c_z=-1, plane z=5 (periodic) c_z=+1
    mask = np.zeros((6, 4, 4), np.uint8)
    mask[0] = 1
    o = oracle_mod.Oracle(4, 4, 6)
    o.set_solid_mask(mask)
    links = o.get_link_mask().reshape(6, 4, 4)
    down = sum(1 << i for i in range(19) if c[i][2] == -1)
    up = sum(1 << i for i in range(19) if c[i][2] == 1)
    assert np.all(links[1] == down) and np.all(links[5] == up) and np.all(links[2:5] == 0) and np.all(links[0] == 0)


def test_bounce_back_wall_reflects(oracle_mod):
    """A population aimed at a wall comes back reversed on the same node one step later (Eq. 23-24, u_b=0)."""
    c, _ = oracle_mod.lattice()
    mask = np.zeros((6, 4, 4), np.uint8)
    mask[0] = 1
    o = oracle_mod.Oracle(4, 4, 6, 1e9, 1e9, 0.0)              # omega ~ 0: collision is the identity
    o.set_solid_mask(mask)
    f = np.zeros((2, 19, 6, 4, 4))
    f[0, 6, 1, 2, 3] = 1.0                                       # direction 6 = -z, sitting next to the wall
    f[1, 12, 1, 2, 3] = 2.0                                      # direction 12 = (-1,0,-1)
    o.set_populations(f)
    o.step(1)
    g = o.get_populations()
    assert abs(g[0, 5, 1, 2, 3] - 1.0) < 1e-8 and abs(g[1, 11, 1, 2, 3] - 2.0) < 1e-8
    assert abs(g.sum() - 3.0) < 1e-8


# P12 -----------------------------------------------------------------------
def test_p12_reference_trajectory_config0(oracle_mod):
    o, _, _ = _config0(oracle_mod)
    seen = {}
    t = 0
    for target in (0, 1, 2, 10, 100):
        o.step(target - t)
        t = target
        f = o.get_populations()
        rr, rb = o.get_moments()[:2]
        phi = (rr - rb) / (rr + rb)
        seen[str(t)] = (f[0, 1, 0, 0, 0], f[1, 7, 3, 2, 1], (f * f).sum(), phi.std(), np.abs(phi).max())
    for t, (a, b, s2, ps, pm) in seen.items():
        tol = 2e-12 if int(t) <= 10 else 5e-9
        assert abs(a / GOLD["f_r1_000"][t] - 1) < tol
        if t in GOLD["f_b7_x1y2z3"]:
            assert abs(b / GOLD["f_b7_x1y2z3"][t] - 1) < tol
        if t in GOLD["sum_f2"]:
            assert abs(s2 / GOLD["sum_f2"][t] - 1) < max(tol, 2e-12)
        if t in GOLD["phi_std"]:
            assert abs(ps / GOLD["phi_std"][t] - 1) < max(tol, 2e-9)
    assert abs(seen["100"][4] - GOLD["phi_absmax_100"]) < 1e-5
    m, p = o.get_diagnostics()
    assert np.abs(m / np.array(GOLD["mass"]) - 1).max() < 1e-13
    assert np.abs(p).max() < 1e-12


def test_p12_general_tau(oracle_mod):
    gt = GOLD["general_tau"]
    o, _, _ = _config0(oracle_mod, tau_r=gt["tau_r"], tau_b=gt["tau_b"], G=gt["G"])
    o.step(gt["t"])
    f = o.get_populations()
    assert abs(f[0, 1, 0, 0, 0] / gt["f_r1_000"] - 1) < 2e-12
    assert abs((f * f).sum() / gt["sum_f2"] - 1) < 2e-12


# moments / API behaviour -----------------------------------------------------
def test_moments_return_the_fields_that_were_set(oracle_mod):
    n = 6
    rng = np.random.default_rng(3)
    rr, rb = rng.uniform(0.5, 1.5, n ** 3), rng.uniform(0.5, 1.5, n ** 3)
    u = rng.uniform(-0.05, 0.05, (3, n ** 3))
    o = oracle_mod.Oracle(n, n, n)
    o.set_fields(rr, rb, *u)
    got = o.get_moments()
    assert np.abs(got[0] - rr).max() < 1e-15 and np.abs(got[1] - rb).max() < 1e-15
    for a in range(3):
        assert np.abs(got[2 + a] - u[a]).max() < 1e-16


def test_oracle_argument_checks(oracle_mod):
    with pytest.raises(ValueError):
        oracle_mod.Oracle(0, 4, 4)
    with pytest.raises(ValueError):
        oracle_mod.Oracle(4, 4, 4, 0.5, 1.0, 1.0)              # Eq. 2 needs 0 < omega < 2
    with pytest.raises(ValueError):
        oracle_mod.Oracle(4, 4, 4, 1.0, 1.0, float("nan"))
    o = oracle_mod.Oracle(4, 4, 4)
    with pytest.raises(RuntimeError):
        o.step(1)                                               # no fields yet


def test_rounding_noise_floor_fma_vs_no_fma(oracle_mod):
    """S12: the same source with FMA contraction differs after 100 unstable steps by ~1e-12 (normalised)."""
    if not oracle_mod.host_has_fma():
        pytest.skip("host CPU has no FMA")
    oa, rr, rb = _config0(oracle_mod)
    ob = oracle_mod.Oracle(32, 32, 32, variant="fma")
    ob.set_fields(rr, rb)
    oa.step(100), ob.step(100)
    fa, fb = oa.get_populations(), ob.get_populations()
    floor = np.abs(fa - fb).max() / np.abs(fa).max()
    print(f"fp64 rounding-noise floor, config 0, t=100 (normalised max): {floor:.3e}")
    assert floor < 1e-11
