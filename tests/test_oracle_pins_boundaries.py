"""Pins for the parts of the CPU oracle that round 1 left without one ("parity unpinned"):
step 2f (periodic wrap sequence, non-periodic deactivation), the diagnostics (energies, charge, Gauss
residual) and the zero-read rule of the field solver on a non-periodic axis (reading Q6). Every expected
value below is worked out here in Python from the definition, never by
calling the oracle twice. No GPU."""
import math

import numpy as np
import pytest

from oracle import Oracle
from workloads import C_LIGHT as c, EPS0, M_E, M_P, Q_E


def _free_particle_sim(n, dx, dt, periodic=(1, 1, 1), order=1):
    """zero fields: Boris leaves u unchanged exactly (u + kq*0, rotation by t = 0)"""
    return Oracle(n, dx, dt, order, periodic=periodic, tile=(1, 1, 1), sort_interval=0)


def _moved(x, u3, dt):
    """step 2d in the oracle's operation order, IEEE double: x + (dt*u)/gamma"""
    inv_c2 = 1.0 / (c * c)
    g = math.sqrt(1.0 + (u3[0] * u3[0] + u3[1] * u3[1] + u3[2] * u3[2]) * inv_c2)
    return [x[d] + dt * u3[d] / g for d in range(3)]


# --------------------------------------------------------------------------- step 2f, periodic
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("direction", [-1, +1])
def test_2f_periodic_wrap_lands_at_exactly_x_plus_minus_L(axis, direction):
    """A free particle pushed across a periodic face lands at x~ + L (low face) or x~ - L (high face),
    bit for bit; the other two coordinates just advance."""
    n, dx = (6, 5, 7), (1.0e-6, 0.8e-6, 0.5e-6)
    dt = 0.9 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    L = [n[d] * dx[d] for d in range(3)]
    o = _free_particle_sim(n, dx, dt)
    x = [2.3e-6, 1.7e-6, 1.9e-6]
    x[axis] = 0.05 * dx[axis] if direction < 0 else L[axis] - 0.05 * dx[axis]
    u = [0.02 * c, -0.03 * c, 0.01 * c]
    u[axis] = direction * 2.0 * c                      # v = 0.894 c: moves 0.3-0.5 cell, enough to cross
    o.add_species([x[0]], [x[1]], [x[2]], [u[0]], [u[1]], [u[2]], [0.0], -Q_E, M_E)
    o.step(1)
    p = o.get_particles()
    xt = _moved(x, u, dt)
    assert (xt[axis] < 0.0) if direction < 0 else (xt[axis] >= L[axis])      # it did cross
    want = list(xt)
    want[axis] = xt[axis] + L[axis] if direction < 0 else xt[axis] - L[axis]
    got = [p["x"][0], p["y"][0], p["z"][0]]
    assert got == want
    assert 0.0 <= got[axis] < L[axis]
    assert [p["ux"][0], p["uy"][0], p["uz"][0]] == u   # zero fields: momentum untouched
    assert o.diagnostics()["deactivated"] == 0


def test_2f_minus_tiny_goes_to_L_and_then_to_zero():
    """The second test comes after the first: -tiny + L rounds to L, which is >= L, so the particle lands
    on 0 exactly (and never on L, which is outside [0, L))."""
    n, dx = (8, 8, 8), (1e-6,) * 3
    dt = 0.9 * 1e-6 / (c * math.sqrt(3))
    L = 8e-6
    o = _free_particle_sim(n, dx, dt)
    u = -1e-20                                         # x~ = 0 + dt*u = -3e-36: -tiny
    o.add_species([0.0], [3e-6], [4e-6], [u], [0.0], [0.0], [0.0], -Q_E, M_E)
    o.step(1)
    p = o.get_particles()
    xt = _moved([0.0, 3e-6, 4e-6], [u, 0.0, 0.0], dt)[0]
    assert xt < 0.0 and xt + L == L                    # the case is the one meant
    assert p["x"][0] == 0.0
    assert p["y"][0] == 3e-6 and p["z"][0] == 4e-6


def test_2f_particles_inside_are_left_alone_and_wrap_is_per_axis():
    n, dx = (8, 8, 8), (1e-6,) * 3
    dt = 0.9 * 1e-6 / (c * math.sqrt(3))
    o = _free_particle_sim(n, dx, dt)
    x = np.array([[4.1e-6, 0.02e-6, 7.99e-6], [0.5e-6, 6.5e-6, 3.5e-6]])
    u = np.array([[0.3 * c, -2.0 * c, 2.0 * c], [0.1 * c, 0.2 * c, -0.3 * c]])
    o.add_species(x[:, 0], x[:, 1], x[:, 2], u[:, 0], u[:, 1], u[:, 2], [0.0, 0.0], -Q_E, M_E)
    o.step(1)
    p = o.get_particles()
    for i in range(2):
        xt = _moved(list(x[i]), list(u[i]), dt)
        want = [v + 8e-6 if v < 0 else (v - 8e-6 if v >= 8e-6 else v) for v in xt]
        assert [p["x"][i], p["y"][i], p["z"][i]] == want
    # particle 0 crossed the low y face and the high z face at once; particle 1 crossed nothing
    assert p["y"][0] > 7e-6 and p["z"][0] < 1e-6 and p["x"][0] == _moved(list(x[0]), list(u[0]), dt)[0]


# --------------------------------------------------------------------------- step 2f, non-periodic (Q6)
def test_2f_nonperiodic_exit_deactivates_clamps_and_counts_once():
    n, dx = (8, 8, 8), (1e-6,) * 3
    dt = 0.9 * 1e-6 / (c * math.sqrt(3))
    L = 8e-6
    o = _free_particle_sim(n, dx, dt, periodic=(1, 1, 0))
    #            leaves at the top      leaves at the bottom   stays                 crosses periodic x only
    z = [L - 0.05e-6, 0.05e-6, 4.0e-6, 4.0e-6]
    uz = [2.0 * c, -2.0 * c, 0.5 * c, 0.0]
    xx = [1e-6, 2e-6, 3e-6, 0.05e-6]
    ux = [0.0, 0.0, 0.0, -2.0 * c]
    w = [1e3, 2e3, 3e3, 4e3]
    o.add_species(xx, [4e-6] * 4, z, ux, [0.0] * 4, uz, w, -Q_E, M_E)
    o.step(1)
    p = o.get_particles()
    assert p["w"].tolist() == [0.0, 0.0, 3e3, 4e3]
    assert p["z"][0] == math.nextafter(L, 0.0)          # clamped to the last value inside [0, L)
    assert p["z"][1] == 0.0
    assert p["z"][2] == _moved([3e-6, 4e-6, 4.0e-6], [0.0, 0.0, 0.5 * c], dt)[2]
    assert p["x"][3] == _moved([0.05e-6, 4e-6, 4e-6], [-2.0 * c, 0.0, 0.0], dt)[0] + L   # x is still periodic
    assert o.diagnostics()["deactivated"] == 2
    # a particle that is already switched off is not counted again (it sits on the face and leaves again)
    o.step(1)
    assert o.diagnostics()["deactivated"] == 2
    assert o.get_particles()["w"].tolist() == [0.0, 0.0, 3e3, 4e3]
    # charge diagnostic follows the weights that are left
    assert o.diagnostics()["charge"] == pytest.approx(-Q_E * 7e3, rel=1e-15)


# --------------------------------------------------------------------------- diagnostics (Q15)
def test_diagnostics_kinetic_energy_of_known_gamma_and_charge():
    """KE = sum w m c^2 (gamma - 1) at the stored u; gamma = 5/4 for |u| = 3c/4, 13/12 for 5c/12."""
    n, dx = (8, 8, 8), (1e-6,) * 3
    dt = 0.5 * 1e-6 / (c * math.sqrt(3))
    o = Oracle(n, dx, dt, 2, tile=(1, 1, 1), sort_interval=0)
    o.add_species([1e-6, 5e-6], [2e-6, 5e-6], [3e-6, 1e-6], [0.75 * c, 0.0], [0.0, 0.0], [0.0, -5.0 * c / 12.0],
                  [2e4, 3e4], -Q_E, M_E)
    o.add_species([4e-6], [4e-6], [4e-6], [0.0], [0.45 * c], [0.6 * c], [7e3], Q_E, M_P)
    d = o.diagnostics()
    ke = 2e4 * M_E * c * c * 0.25 + 3e4 * M_E * c * c * (13.0 / 12.0 - 1.0) + 7e3 * M_P * c * c * 0.25
    assert d["kinetic"] == pytest.approx(ke, rel=2e-15)
    assert d["charge"] == pytest.approx(-Q_E * 5e4 + Q_E * 7e3, rel=1e-15)
    assert d["field_E"] == 0.0 and d["field_B"] == 0.0
    # non-relativistic limit: (gamma - 1) m c^2 -> u^2 / 2m without cancellation
    o2 = Oracle(n, dx, dt, 1, tile=(1, 1, 1), sort_interval=0)
    o2.add_species([1e-6], [1e-6], [1e-6], [1e-3], [0.0], [0.0], [1.0], -Q_E, M_E)
    assert o2.diagnostics()["kinetic"] == pytest.approx(0.5 * M_E * 1e-6, rel=1e-14)


def test_diagnostics_field_energy_of_uniform_fields():
    """1/2 eps0 E^2 V and 1/2 eps0 c^2 B^2 V over the whole box, anisotropic cells."""
    n, dx = (6, 4, 5), (1.0e-6, 0.5e-6, 0.25e-6)
    dt = 0.5 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    o = Oracle(n, dx, dt, 1, tile=(1, 1, 1), sort_interval=0)
    shp = (n[2], n[1], n[0])
    Ev, Bv = (3e9, -4e9, 12e9), (0.3, 0.4, -1.2)
    o.set_fields([np.full(shp, v) for v in Ev], [np.full(shp, v) for v in Bv])
    d = o.diagnostics()
    V = np.prod(n) * np.prod(dx)
    assert d["field_E"] == pytest.approx(0.5 * EPS0 * (13e9) ** 2 * V, rel=1e-14)
    assert d["field_B"] == pytest.approx(0.5 * EPS0 * c * c * 1.3 ** 2 * V, rel=1e-14)
    assert d["kinetic"] == 0.0 and d["charge"] == 0.0
    assert d["gauss_max"] == 0.0                        # uniform field on a periodic box: no divergence


def test_diagnostics_gauss_residual_and_rho_of_known_configurations():
    n, dx = (8, 4, 4), (1.0e-6, 0.5e-6, 0.25e-6)
    dt = 0.5 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    shp = (n[2], n[1], n[0])
    zero = np.zeros(shp)
    # Ex = E0 * i on a NON-periodic x axis: (Ex[i] - Ex[i-1]) / dx = E0 / dx at every node, Ex[-1] reads 0
    o = Oracle(n, dx, dt, 1, periodic=(0, 1, 1), tile=(1, 1, 1), sort_interval=0)
    E0 = 2.5e8
    Ex = np.broadcast_to(E0 * np.arange(n[0]), shp).copy()
    o.set_fields([Ex, zero, zero], [zero, zero, zero])
    d = o.diagnostics()
    assert d["gauss_max"] == pytest.approx(E0 / dx[0], rel=1e-14)
    assert d["rho_max"] == 0.0
    # one particle exactly on a node, order 1: all its charge on that node, rho = q w / dV
    o = Oracle(n, dx, dt, 1, tile=(1, 1, 1), sort_interval=0)
    o.add_species([3 * dx[0]], [2 * dx[1]], [1 * dx[2]], [0.0], [0.0], [0.0], [4e4], -Q_E, M_E)
    d = o.diagnostics()
    rho = Q_E * 4e4 / np.prod(dx)
    assert d["rho_max"] == pytest.approx(rho / EPS0, rel=1e-14)
    assert d["gauss_max"] == pytest.approx(rho / EPS0, rel=1e-14)      # E = 0: the residual is rho itself
    r = o.rho()
    assert r[1, 2, 3] == pytest.approx(-rho, rel=1e-14) and np.count_nonzero(r) == 1


# --------------------------------------------------------------------------- Yee on a truncated axis (Q6)
def test_yee_truncated_axis_equals_periodic_until_the_field_reaches_a_face():
    """A pulse that stays away from the z faces cannot tell a zero-guard axis from a periodic one."""
    n, dx = (4, 4, 40), (1e-6, 1e-6, 0.5e-6)
    dt = 0.95 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    rng = np.random.default_rng(5)
    shp = (n[2], n[1], n[0])
    E = [np.zeros(shp) for _ in range(3)]
    B = [np.zeros(shp) for _ in range(3)]
    for a in E:
        a[18:22] = rng.standard_normal((4, n[1], n[0])) * 1e9
    for a in B:
        a[18:22] = rng.standard_normal((4, n[1], n[0]))
    res = []
    for per in ((1, 1, 1), (1, 1, 0)):
        o = Oracle(n, dx, dt, 1, periodic=per, tile=(1, 1, 1), sort_interval=0)
        o.set_fields(E, B)
        o.field_step(6)                                # support grows by <= 2 planes per step: 18-12 .. 21+12
        res.append(o.get_fields())
    for grp in range(2):
        for d in range(3):
            assert np.array_equal(res[0][grp][d], res[1][grp][d])
            assert np.any(res[0][grp][d][10:30] != 0)
    assert all(np.all(res[1][0][d][:4] == 0) and np.all(res[1][0][d][-4:] == 0) for d in range(3))


def test_yee_pulse_on_the_face_loses_exactly_the_terms_that_read_outside():
    """Ey = A on the plane k = 0 only, uniform in x and y: a 1-D problem in (Ey, Bx) whose first step can be
    done by hand. With a = dt/(2 dz), e = c^2 dt/dz:
      zero-guard z:  B half  Bx[0] = -aA                       (Bx[N-1] reads Ey[N] = 0 and Ey[N-1] = 0)
                     E       Ey[0] = A(1 - ea), Ey[1] = eaA    (Ey[0] reads Bx[-1] = 0)
                     B half  Bx[0] = aA(2ea - 2), Bx[1] = -e a^2 A
      periodic z:    B half  Bx[0] = -aA, Bx[N-1] = +aA        (reads Ey[N] = Ey[0] = A)
                     E       Ey[0] = A(1 - 2ea), Ey[1] = Ey[N-1] = eaA
                     B half  Bx[0] = aA(3ea - 2), Bx[1] = -e a^2 A, Bx[N-1] = aA(2 - 3ea), Bx[N-2] = e a^2 A"""
    n, dx = (4, 4, 12), (1e-6, 1e-6, 0.4e-6)
    dt = 0.9 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    a, e, A = dt / (2 * dx[2]), c * c * dt / dx[2], 3e8
    shp = (n[2], n[1], n[0])
    zero = np.zeros(shp)
    Ey = np.zeros(shp)
    Ey[0] = A
    out = {}
    for per in ((1, 1, 1), (1, 1, 0)):
        o = Oracle(n, dx, dt, 1, periodic=per, tile=(1, 1, 1), sort_interval=0)
        o.set_fields([zero, Ey, zero], [zero, zero, zero])
        o.field_step(1)
        Ef, Bf, _ = o.get_fields()
        assert np.all(Ef[0] == 0) and np.all(Ef[2] == 0) and np.all(Bf[1] == 0) and np.all(Bf[2] == 0)
        assert all(np.all(Ef[1][k] == Ef[1][k][0, 0]) and np.all(Bf[0][k] == Bf[0][k][0, 0]) for k in range(n[2]))
        out[per] = (Ef[1][:, 0, 0], Bf[0][:, 0, 0])
    ap = lambda v: pytest.approx(v, rel=1e-14)
    ey, bx = out[(1, 1, 0)]
    assert ey[0] == ap(A * (1 - e * a)) and ey[1] == ap(e * a * A)
    assert bx[0] == ap(a * A * (2 * e * a - 2)) and bx[1] == ap(-e * a * a * A)
    assert np.all(ey[2:] == 0) and np.all(bx[2:] == 0)                 # nothing came round the top
    ey, bx = out[(1, 1, 1)]
    assert ey[0] == ap(A * (1 - 2 * e * a)) and ey[1] == ap(e * a * A) and ey[-1] == ap(e * a * A)
    assert bx[0] == ap(a * A * (3 * e * a - 2)) and bx[1] == ap(-e * a * a * A)
    assert bx[-1] == ap(a * A * (2 - 3 * e * a)) and bx[-2] == ap(e * a * a * A)
    assert np.all(ey[2:-1] == 0) and np.all(bx[2:-2] == 0)
