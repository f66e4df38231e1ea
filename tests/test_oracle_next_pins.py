"""Pins of the oracle's two later operators: what the paper and the mathematics fix, never the
oracle's own formula retyped.

N1 colour gradient: conservation constraints Eq. 11-12; the isotropy the B_i table must have (Eq. 18,
through the second moment of Eq. 17, a closed form); colour-blindness of the total populations (recolouring Eq. 20-21 only
redistributes sum_k f_i^k); the viscosity of a pure component (Eq. 2); Laplace's law with the surface tension of Eq. 19.
N2 moving walls: reduction to plain bounce-back at rest; exact invariance of a uniform flow
that moves with the wall (Eq. 24 with Eq. 10); momentum balance between fluid and spheres; cubic symmetry of the drag.
"""
import numpy as np
import pytest

from paper_2112_08264_b200 import workloads as w


def _two_phase(nx, ny, nz, seed):
    rng = np.random.default_rng(seed)
    phi = rng.uniform(-0.9, 0.9, nx * ny * nz)
    rho = 1.0 + 0.05 * rng.uniform(-1, 1, nx * ny * nz)
    return rho * (1 + phi) / 2, rho * (1 - phi) / 2, rng.uniform(-0.02, 0.02, (3, nx * ny * nz))


# ------------------------------------------------------------------------------------------ N1
def test_cg_mass_and_momentum_conserved(oracle_mod):
    """Eq. 11-12: per-component mass and total momentum, periodic box, unequal viscosities."""
    nx, ny, nz = 12, 10, 8
    rr, rb, u = _two_phase(nx, ny, nz, 1)
    o = oracle_mod.Oracle(nx, ny, nz, 0.8, 1.4, 0.0)
    o.set_colour_gradient(0.02, 0.7)
    o.set_fields(rr, rb, *u)
    m0, p0 = o.get_diagnostics()
    o.step(30)
    m1, p1 = o.get_diagnostics()
    assert np.abs(m1 / m0 - 1).max() < 1e-13
    assert np.abs(p1 - p0).max() < 1e-12
    assert np.all(np.isfinite(o.get_populations()))


def test_cg_perturbation_moments_closed_form(oracle_mod):
    """Eq. 17 with the weights and B_i of PAPER.md:393-398: zeroth and first moments vanish (Eq. 11-12) and, by the lattice
    isotropy sum_i w_i c_a c_b c_c c_d = c_s^4 (3 delta-pairings) together with Eq. 18, the second moment is
    (A / 9) |g| (g g / |g|^2 - I): no stress along the interface normal, -A |g| / 9 in the interface plane."""
    c, _ = oracle_mod.lattice()
    rng = np.random.default_rng(3)
    for _ in range(20):
        g = rng.normal(size=3) * 10 ** rng.uniform(-3, 0)
        A = rng.uniform(0.001, 0.1)
        om2 = oracle_mod.cg_perturbation(A, *g)
        gn = np.linalg.norm(g)
        assert abs(om2.sum()) < 1e-16 * (1 + A * gn) + 1e-18
        assert np.abs(om2 @ c).max() < 1e-17 + 1e-15 * A * gn
        second = np.einsum("i,ia,ib->ab", om2, c, c)
        want = A / 9.0 * gn * (np.outer(g, g) / gn ** 2 - np.eye(3))
        assert np.abs(second - want).max() < 1e-14 * A * gn + 1e-18
    assert np.all(oracle_mod.cg_perturbation(0.05, 0.0, 0.0, 0.0) == 0.0)        # no gradient, no perturbation


def test_cg_total_populations_are_colour_blind(oracle_mod):
    """With sigma = 0 and equal viscosities the total populations sum_k f_i^k follow a single BGK fluid whatever the colours do
    (recolouring only redistributes f*_i, Eq. 20-21): the same totals as the Shan-Chen operator with G = 0, for any beta."""
    nx, ny, nz = 10, 8, 6
    rr, rb, u = _two_phase(nx, ny, nz, 5)
    ref = oracle_mod.Oracle(nx, ny, nz, 0.9, 0.9, 0.0)
    ref.set_fields(rr, rb, *u)
    ref.step(20)
    tot = ref.get_populations().sum(axis=0)
    for beta in (0.0, 0.5, 0.99):
        o = oracle_mod.Oracle(nx, ny, nz, 0.9, 0.9, 0.0)
        o.set_colour_gradient(0.0, beta)
        o.set_fields(rr, rb, *u)
        o.step(20)
        f = o.get_populations()
        assert np.abs(f.sum(axis=0) - tot).max() < 1e-14
    # and beta does act on the colours: it segregates (the phase field's spread grows with beta)
    spreads = []
    for beta in (0.0, 0.99):
        o = oracle_mod.Oracle(nx, ny, nz, 0.9, 0.9, 0.0)
        o.set_colour_gradient(0.0, beta)
        o.set_fields(rr, rb, *u)
        o.step(20)
        spreads.append(o.get_phase_field()[0].std())
    assert spreads[1] > 1.5 * spreads[0]


def test_cg_pure_component_is_bgk_with_its_own_viscosity(oracle_mod):
    """rho^2 = 0: Theta = 1 everywhere, no gradient; the shear wave decays with nu_1 = c_s^2 (tau_1 - 1/2) (Eq. 2 PAPER.md:84;
    reading C2: omega = 2 / (6 nu + 1))."""
    nx, ny, nz, U, steps, tau = 4, 32, 4, 1e-3, 200, 0.8
    y = np.arange(ny)
    ux = np.broadcast_to((U * np.sin(2 * np.pi * y / ny))[None, :, None], (nz, ny, nx)).reshape(-1).copy()
    o = oracle_mod.Oracle(nx, ny, nz, tau, 1.9, 0.0)
    o.set_colour_gradient(0.03, 0.7)
    o.set_fields(np.ones(nx * ny * nz), np.zeros(nx * ny * nz), ux, None, None)
    amp = []
    for _ in range(steps + 1):
        uu = o.get_moments()[2].reshape(nz, ny, nx)
        amp.append(2.0 / ny * (uu[0, :, 0] * np.sin(2 * np.pi * y / ny)).sum())
        o.step(1)
    rate = -np.polyfit(np.arange(100, steps + 1), np.log(np.array(amp)[100:]), 1)[0]
    assert abs(rate / ((tau - 0.5) / 3.0 * (2 * np.pi / ny) ** 2) - 1) < 0.02
    assert np.all(o.get_populations()[1] == 0.0)


def test_cg_flat_interface_stays_flat_and_laplace_law(oracle_mod):
    """(a) A planar interface keeps its symmetry exactly (fields independent of y, z).  (b) A cylindrical droplet (nz = 1)
    relaxes to a pressure jump sigma / R with p = c_s^2 rho and the sigma of Eq. 19."""
    nx, ny, nz = 24, 4, 3
    x = np.arange(nx)
    prof = 0.5 * (1 + np.tanh((np.minimum(x, nx - 1 - x) - nx / 4) / 1.5))
    rr = np.broadcast_to(prof[None, None, :], (nz, ny, nx)).reshape(-1).copy()
    o = oracle_mod.Oracle(nx, ny, nz, 1.0, 1.0, 0.0)
    o.set_colour_gradient(0.02, 0.7)
    o.set_fields(rr, 1.0 - rr)
    o.step(50)
    f = o.get_populations()
    assert np.abs(f - f[:, :, :1, :1, :]).max() < 1e-15                           # still a function of x only
    # droplet
    n, R, sigma = 48, 12.0, 0.02
    yy, xx = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    d = np.sqrt((xx - n / 2 + 0.5) ** 2 + (yy - n / 2 + 0.5) ** 2)
    rr = (0.5 * (1 - np.tanh((d - R) / 1.5))).reshape(-1)
    o = oracle_mod.Oracle(n, n, 1, 1.0, 1.0, 0.0)
    o.set_colour_gradient(sigma, 0.7)
    o.set_fields(rr, 1.0 - rr)
    o.step(3000)
    r1, r2 = o.get_moments()[:2]
    rho = (r1 + r2).reshape(n, n)
    inside = rho[d < R / 2].mean()
    outside = rho[d > 1.6 * R].mean()
    # the radius of the relaxed droplet from the red mass (sharp-interface area)
    Reff = np.sqrt(r1.sum() / (np.pi * inside))
    dp = (inside - outside) / 3.0
    assert abs(dp / (sigma / Reff) - 1) < 0.15, (dp, sigma / Reff)


# ------------------------------------------------------------------------------------------ N2
def _one_sphere(n=20, c=(10.0, 10.0, 10.0)):
    return np.array([c]), 5.5


def test_moving_wall_reduces_to_bounce_back_at_rest(oracle_mod):
    """v_p = omega_p = 0 gives the usual bounce-back: bit-identical to the plain-mask path; the mask is reading S9's
    (739 nodes for a sphere centred on a node, pin P11)."""
    n = 20
    centres, R = _one_sphere(n)
    rr, rb = w.mixture_fields(n, n, n, 21)
    a = oracle_mod.Oracle(n, n, n, 0.9, 1.2, 0.8)
    a.set_spheres(centres, R)
    mask = a.get_solid_mask()
    assert int(mask.sum()) == 739
    assert np.array_equal(mask, w.solid_mask_from_spheres(n, n, n, centres, R))
    b = oracle_mod.Oracle(n, n, n, 0.9, 1.2, 0.8)
    b.set_solid_mask(mask)
    a.set_fields(rr, rb), b.set_fields(rr, rb)
    a.step(5), b.step(5)
    assert np.array_equal(a.get_populations(), b.get_populations())


def test_moving_wall_comoving_uniform_flow_is_invariant(oracle_mod):
    """A uniform equilibrium flow u around a sphere translating with v_p = u: Eq. 24 with Eq. 10 returns exactly the
    equilibrium population of the opposite direction (f_i^eq - 2 rho w_i 3 c_i.u = f_opp(i)^eq), so nothing changes and the
    force is the hydrostatic one, which sums to zero over the closed surface of a centred sphere."""
    n = 16
    centres, R = np.array([[8.0, 8.0, 8.0]]), 4.5
    u = np.array([0.03, -0.02, 0.01])
    N = n ** 3
    for model in ("sc", "cg"):
        o = oracle_mod.Oracle(n, n, n, 0.8, 0.8, 0.0)
        if model == "cg":
            o.set_colour_gradient(0.0, 0.0)
        o.set_spheres(centres, R, vel=u)
        o.set_fields(np.full(N, 0.6), np.full(N, 0.4), np.full(N, u[0]), np.full(N, u[1]), np.full(N, u[2]))
        f0 = o.get_populations().copy()
        o.step(3)
        assert np.abs(o.get_populations() - f0).max() < 2e-16
        F, T = o.get_sphere_forces()
        assert np.abs(F).max() < 1e-13 and np.abs(T).max() < 1e-12


@pytest.mark.parametrize("model", ["sc", "cg"])
def test_moving_wall_momentum_balance(oracle_mod, model):
    """What the fluid loses in a step is what the spheres receive (reading M3; Eq. 25-26), exactly, with translating and
    rotating spheres; the Shan-Chen coupling is switched off (a solid neighbour's psi = 0 makes that force unbalanced)."""
    n = 24
    centres = np.array([[7.3, 8.1, 6.6], [17.2, 15.9, 16.4]])
    vel = np.array([[0.02, 0.0, -0.01], [0.0, 0.015, 0.0]])
    omg = np.array([[0.0, 0.0, 0.004], [0.003, -0.002, 0.0]])
    rr, rb = w.mixture_fields(n, n, n, 22)
    o = oracle_mod.Oracle(n, n, n, 0.9, 1.1, 0.0)
    if model == "cg":
        o.set_colour_gradient(0.01, 0.5)
    o.set_spheres(centres, 4.5, vel, omg)
    o.set_fields(rr, rb)
    for _ in range(4):
        _, p0 = o.get_diagnostics()
        o.step(1)
        _, p1 = o.get_diagnostics()
        F, _ = o.get_sphere_forces()
        assert np.abs((p1 - p0) + F.sum(axis=0)).max() < 1e-12


def test_moving_wall_drag_has_cubic_symmetry(oracle_mod):
    """A node-centred sphere in fluid at rest: translation along x, y or z gives the same drag magnitude, antiparallel to the
    velocity, with no torque; rotation about an axis gives a torque along that axis (sign by the paper's Eq. 22 / Eq. 27 convention:
    it opposes the rotation's power, T . omega < 0) and no force."""
    n = 20
    centres, R = _one_sphere(n)
    N = n ** 3
    drags = []
    for axis in range(3):
        v = np.zeros((1, 3))
        v[0, axis] = 0.01
        o = oracle_mod.Oracle(n, n, n, 1.0, 1.0, 0.0)
        o.set_spheres(centres, R, vel=v)
        o.set_fields(np.full(N, 0.5), np.full(N, 0.5))
        o.step(1)
        F, T = o.get_sphere_forces()
        assert F[0, axis] < 0 and np.abs(np.delete(F[0], axis)).max() < 1e-12
        assert np.abs(T).max() < 1e-12
        drags.append(F[0, axis])
        om = np.zeros((1, 3))
        om[0, axis] = 0.002
        o = oracle_mod.Oracle(n, n, n, 1.0, 1.0, 0.0)
        o.set_spheres(centres, R, omega=om)
        o.set_fields(np.full(N, 0.5), np.full(N, 0.5))
        o.step(1)
        F, T = o.get_sphere_forces()
        assert np.abs(F).max() < 1e-12
        assert T[0, axis] * om[0, axis] < 0 and np.abs(np.delete(T[0], axis)).max() < 1e-12
    assert np.ptp(drags) < 1e-12
