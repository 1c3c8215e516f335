"""Pins for the CPU oracle (T1..T11 of SURVEY.md §8(c)): each test fixes a part of oracle/ with
something the method or the mathematics fixes — closed forms, invariants, brute force — so that
a dropped term, wrong sign/index or swapped operand anywhere in it fails here. No GPU."""
import math

import numpy as np
import pytest

import oracle
from oracle import Oracle
from workloads import C_LIGHT as c, EPS0, M_E, Q_E


# --------------------------------------------------------------------------- T1 shapes
@pytest.mark.parametrize("order", [1, 2, 3])
def test_T1_shape_partition_of_unity_and_first_moment(order):
    rng = np.random.default_rng(11)
    xis = np.concatenate([rng.uniform(-5, 5, 400), [0.0, 1.0, -1.0, 0.5, -0.5, 2.999999999, -3.0]])
    for xi in xis:
        l, w = oracle.shape(order, xi)
        assert len(w) == order + 1
        assert np.all(w >= -1e-16)
        assert abs(w.sum() - 1.0) < 4e-16
        # B-splines of order >= 1 reproduce linear functions: sum (l+a) w_a = xi
        assert abs(np.dot(l + np.arange(order + 1), w) - xi) < 1e-14
        if order >= 2:   # ... and the second central moment is order+1 over 12
            assert abs(np.dot((l + np.arange(order + 1) - xi) ** 2, w) - (order + 1) / 12.0) < 1e-14


@pytest.mark.parametrize("order", [1, 2, 3])
def test_T1_shape_is_the_cardinal_bspline(order):
    """Weights equal the cardinal B-spline (n-fold convolution of the box) at node distance."""
    def bspline(n, d):
        d = abs(d)
        if n == 1:
            return max(0.0, 1 - d)
        if n == 2:
            return 0.75 - d * d if d <= 0.5 else (0.5 * (1.5 - d) ** 2 if d <= 1.5 else 0.0)
        return (4 - 6 * d * d + 3 * d ** 3) / 6 if d <= 1 else ((2 - d) ** 3 / 6 if d <= 2 else 0.0)
    rng = np.random.default_rng(12)
    for xi in rng.uniform(-4, 4, 300):
        l, w = oracle.shape(order, xi)
        for a in range(order + 1):
            assert abs(w[a] - bspline(order, xi - (l + a))) < 1e-15
        # support is complete: the neighbours outside carry no weight
        assert bspline(order, xi - (l - 1)) < 1e-15 and bspline(order, xi - (l + order + 1)) < 1e-15


def test_T1_shape_fp32():
    rng = np.random.default_rng(13)
    for order in (1, 2, 3):
        for xi in rng.uniform(-5, 100, 200):
            l, w = oracle.shape(order, np.float32(xi), dtype=np.float32)
            l64, w64 = oracle.shape(order, float(np.float32(xi)))
            assert l == l64
            assert np.max(np.abs(w - w64)) < 2e-6


# --------------------------------------------------------------------------- T2 Boris in B
def test_T2_boris_gyration_angle_norm_and_sense():
    B = 5.0
    dt = 2e-13
    q, m = -Q_E, M_E
    u0 = np.array([0.3 * c, 0.0, 0.1 * c])
    gamma = math.sqrt(1 + u0.dot(u0) / c ** 2)
    wc = abs(q) * B / (gamma * m)
    theta = 2 * math.atan(wc * dt / 2)
    kq = q * dt / (2 * m)
    u = u0.copy()
    for _ in range(200):
        un = oracle.boris(kq, [0, 0, 0], [0, 0, B], u)
        assert abs(np.linalg.norm(un) - np.linalg.norm(u0)) < 1e-15 * np.linalg.norm(u0) * 50
        ang = math.atan2(un[1], un[0]) - math.atan2(u[1], u[0])
        ang = (ang + math.pi) % (2 * math.pi) - math.pi
        # q<0, B along +z: counter-clockwise in (x,y), by exactly 2*atan(wc*dt/2)
        assert abs(ang - theta) < 1e-14
        assert un[2] == pytest.approx(u0[2], rel=1e-15)
        u = un


def _single_particle_sim(n_cells, dx, dt, E=None, B=None, order=1):
    o = Oracle(n_cells, dx, dt, order, tile=(1, 1, 1), sort_interval=0)
    shp = (n_cells[2], n_cells[1], n_cells[0])
    Ef = [np.full(shp, (E or (0, 0, 0))[d]) for d in range(3)]
    Bf = [np.full(shp, (B or (0, 0, 0))[d]) for d in range(3)]
    o.set_fields(Ef, Bf)
    return o


@pytest.mark.parametrize("order", [1, 2, 3])
def test_T2_larmor_circle_radius(order):
    """Positions of the pushed particle lie on a circle of radius (v/wc)*sqrt(1+(wc dt/2)^2)."""
    n, dx = (16, 16, 4), (1e-6,) * 3
    dt = 0.9 * dx[0] / (c * math.sqrt(3))
    Bz = 8.0e2
    o = _single_particle_sim(n, dx, dt, B=(0, 0, Bz), order=order)
    u_perp = 0.5 * c
    gamma = math.sqrt(1 + (u_perp / c) ** 2)
    v = u_perp / gamma
    wc = Q_E * Bz / (gamma * M_E)
    R = v / wc * math.sqrt(1 + (wc * dt / 2) ** 2)
    assert 1e-6 < R < 5e-6
    o.add_species([8e-6], [8e-6], [2e-6], [u_perp], [0.0], [0.0], [0.0], -Q_E, M_E)   # weight 0: no J
    pts = []
    for _ in range(120):
        o.step(1)
        p = o.get_particles()
        pts.append((p["x"][0], p["y"][0]))
        assert abs(math.hypot(p["ux"][0], p["uy"][0]) - u_perp) < 1e-14 * u_perp * 100
    pts = (np.array(pts) - 8e-6) / 1e-6      # centred, in micrometres: well-conditioned fit
    R = R / 1e-6
    # circle through the points: algebraic fit
    A = np.c_[2 * pts, np.ones(len(pts))]
    sol = np.linalg.lstsq(A, (pts ** 2).sum(1), rcond=None)[0]
    Rfit = math.sqrt(sol[2] + sol[0] ** 2 + sol[1] ** 2)
    assert abs(Rfit - R) < 1e-9 * R
    assert np.max(np.abs(np.hypot(pts[:, 0] - sol[0], pts[:, 1] - sol[1]) - R)) < 1e-9 * R


# --------------------------------------------------------------------------- T3 Boris in E
def test_T3_hyperbolic_motion_second_order():
    n, dx = (64, 4, 4), (1e-6,) * 3
    dt0 = 0.5 * dx[0] / (c * math.sqrt(3))
    T = 100 * dt0
    a = c / T                       # a*T/c = 1: relativistic by the end
    Ex = a * M_E / (-Q_E)           # electron: qE/m = a
    errs = []
    for k in (1, 2, 4):
        dt = dt0 / k
        o = _single_particle_sim(n, dx, dt, E=(Ex, 0, 0))
        o.add_species([1e-6], [2e-6], [2e-6], [-a * dt / 2], [0.0], [0.0], [0.0], -Q_E, M_E)
        o.step(100 * k)
        p = o.get_particles()
        # u advances by exactly (qE/m) dt each step
        assert abs(p["ux"][0] - a * (100 * k - 0.5) * dt) < 1e-13 * a * T
        exact = 1e-6 + c * c / a * (math.sqrt(1 + (a * T / c) ** 2) - 1)
        errs.append(abs(p["x"][0] - exact))
    assert errs[0] > 1e-12
    assert 3.8 < errs[0] / errs[1] < 4.2 and 3.8 < errs[1] / errs[2] < 4.2


# --------------------------------------------------------------------------- gather
@pytest.mark.parametrize("order", [1, 2, 3])
def test_gather_reproduces_linear_fields_at_staggered_locations(order):
    """B-spline interpolation reproduces linear functions: with each component set to a linear
    function of ITS OWN Yee location, the gathered value is that function at x_p."""
    n, dx = (12, 10, 8), (1.0e-6, 0.8e-6, 0.5e-6)
    dt = 0.5 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    o = Oracle(n, dx, dt, order, tile=(1, 1, 1), sort_interval=0)
    stag = [(.5, 0, 0), (0, .5, 0), (0, 0, .5), (0, .5, .5), (.5, 0, .5), (.5, .5, 0)]
    rng = np.random.default_rng(5)
    coef = rng.standard_normal((6, 4))
    comps = []
    for cmp in range(6):
        xs = (np.arange(n[0]) + stag[cmp][0]) * dx[0]
        ys = (np.arange(n[1]) + stag[cmp][1]) * dx[1]
        zs = (np.arange(n[2]) + stag[cmp][2]) * dx[2]
        comps.append(coef[cmp, 0] + coef[cmp, 1] * xs[None, None, :] / dx[0]
                     + coef[cmp, 2] * ys[None, :, None] / dx[1] + coef[cmp, 3] * zs[:, None, None] / dx[2])
    o.set_fields(comps[:3], comps[3:])
    m = 200   # keep the support away from the periodic seam
    x = rng.uniform(3, n[0] - 3.5, m) * dx[0]
    y = rng.uniform(3, n[1] - 3.5, m) * dx[1]
    z = rng.uniform(3, n[2] - 3.5, m) * dx[2]
    g = o.gather(x, y, z)
    for cmp in range(6):
        want = coef[cmp, 0] + coef[cmp, 1] * x / dx[0] + coef[cmp, 2] * y / dx[1] + coef[cmp, 3] * z / dx[2]
        assert np.max(np.abs(g[:, cmp] - want)) < 1e-12


def test_gather_periodic_seam_and_delta_field():
    """A field that is 1 at one node and 0 elsewhere returns exactly that node's weight, also
    through the periodic seam."""
    n, dx = (6, 6, 6), (1e-6,) * 3
    dt = 0.5 * dx[0] / (c * math.sqrt(3))
    for order in (1, 2, 3):
        o = Oracle(n, dx, dt, order, tile=(1, 1, 1), sort_interval=0)
        Ez = np.zeros((6, 6, 6))
        Ez[5, 0, 0] = 1.0           # Ez[i=0,j=0,k=5] lives at z=(5+1/2)dz
        zero = np.zeros((6, 6, 6))
        o.set_fields([zero, zero, Ez], [zero, zero, zero])
        xp, yp, zp = 0.2e-6, 5.9e-6, 0.1e-6    # neighbours wrap in y and z
        g = o.gather([xp], [yp], [zp])[0]
        lx, wx = oracle.shape(order, xp / 1e-6)
        ly, wy = oracle.shape(order, yp / 1e-6)
        lz, wz = oracle.shape(order, zp / 1e-6 - 0.5)
        want = 0.0
        for a in range(order + 1):
            for b in range(order + 1):
                for cc in range(order + 1):
                    if (lx + a) % 6 == 0 and (ly + b) % 6 == 0 and (lz + cc) % 6 == 5:
                        want += wx[a] * wy[b] * wz[cc]
        assert want > 0
        assert abs(g[2] - want) < 1e-15
        assert np.all(g[[0, 1, 3, 4, 5]] == 0)


# --------------------------------------------------------------------------- T4 Yee
def test_T4_yee_plane_wave_numerical_dispersion():
    n, dx = (8, 12, 16), (1.0e-6, 0.8e-6, 0.5e-6)
    dt = 0.99 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    mode = (1, 2, 1)
    k = np.array([2 * math.pi * mode[d] / (n[d] * dx[d]) for d in range(3)])
    K = np.array([2 / dx[d] * math.sin(k[d] * dx[d] / 2) for d in range(3)])
    s2 = (c * dt) ** 2 * sum(math.sin(k[d] * dx[d] / 2) ** 2 / dx[d] ** 2 for d in range(3))
    om = 2 / dt * math.asin(math.sqrt(s2))
    Om = 2 / dt * math.sin(om * dt / 2)
    E0 = np.cross(K, [0.3, -0.2, 1.0])
    E0 *= 1e9 / np.linalg.norm(E0)          # polarisation perpendicular to K
    B0 = np.cross(K, E0) / Om
    stag = [(.5, 0, 0), (0, .5, 0), (0, 0, .5), (0, .5, .5), (.5, 0, .5), (.5, .5, 0)]

    def phase(cmp):
        xs = (np.arange(n[0]) + stag[cmp][0]) * dx[0]
        ys = (np.arange(n[1]) + stag[cmp][1]) * dx[1]
        zs = (np.arange(n[2]) + stag[cmp][2]) * dx[2]
        return k[0] * xs[None, None, :] + k[1] * ys[None, :, None] + k[2] * zs[:, None, None]

    def exact(t):
        E = [E0[d] * np.cos(phase(d) - om * t) for d in range(3)]
        B = [B0[d] * math.cos(om * dt / 2) * np.cos(phase(3 + d) - om * t) for d in range(3)]
        return E, B

    o = Oracle(n, dx, dt, 1, tile=(1, 1, 1), sort_interval=0)
    o.set_fields(*exact(0.0))
    nsteps = 200
    o.field_step(nsteps)
    E, B, _ = o.get_fields()
    Ee, Be = exact(nsteps * dt)
    for d in range(3):
        assert np.max(np.abs(E[d] - Ee[d])) < 1e-12 * 1e9
        assert np.max(np.abs(B[d] - Be[d])) < 1e-12 * np.linalg.norm(B0)
    # the wave really moved (phase advanced by many radians) and a wrong dispersion fails:
    assert om * nsteps * dt > 20
    assert np.max(np.abs(E[0] - exact(nsteps * dt * 1.001)[0][0])) > 1e-4 * 1e9


# --------------------------------------------------------------------------- T5/T6/T7 Esirkepov
def _moves(rng, n, dx, npart, maxmove=0.999):
    x0 = rng.uniform(0, 1, (npart, 3)) * (np.array(n) * np.array(dx))
    x1 = x0 + rng.uniform(-maxmove, maxmove, (npart, 3)) * np.array(dx)
    # the deposit requires |l1-l0| <= 1, guaranteed by |move| < 1 cell
    return x0, x1


def _div_back(J, dx):
    Jx, Jy, Jz = J
    return ((Jx - np.roll(Jx, 1, axis=2)) / dx[0] + (Jy - np.roll(Jy, 1, axis=1)) / dx[1]
            + (Jz - np.roll(Jz, 1, axis=0)) / dx[2])


@pytest.mark.parametrize("order", [1, 2, 3])
def test_T5_esirkepov_continuity(order):
    n, dx = (7, 6, 8), (1.0e-6, 0.8e-6, 0.5e-6)
    dt = 0.5 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    rng = np.random.default_rng(20 + order)
    x0, x1 = _moves(rng, n, dx, 300)
    w = rng.uniform(0.5, 2.0, 300) * 1e5
    L = np.array(n) * np.array(dx)
    mk = lambda: Oracle(n, dx, dt, order, tile=(1, 1, 1), sort_interval=0)
    z = np.zeros(300)
    a = mk(); a.add_species(x0[:, 0], x0[:, 1], x0[:, 2], z, z, z, w, -Q_E, M_E)
    x1w = np.mod(x1, L)
    b = mk(); b.add_species(x1w[:, 0], x1w[:, 1], x1w[:, 2], z, z, z, w, -Q_E, M_E)
    rho0, rho1 = a.rho(), b.rho()
    J = a.deposit_moves(0, x0, x1, w)
    res = (rho1 - rho0) / dt + _div_back(J, dx)
    scale = np.max(np.abs(rho1 - rho0)) / dt
    assert scale > 0
    assert np.max(np.abs(res)) < 5e-14 * scale


@pytest.mark.parametrize("order", [1, 2, 3])
def test_T6_esirkepov_first_moment_and_sign(order):
    n, dx = (8, 8, 8), (1.0e-6, 0.8e-6, 0.5e-6)
    dt = 0.5 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    rng = np.random.default_rng(30 + order)
    o = Oracle(n, dx, dt, order, tile=(1, 1, 1), sort_interval=0)
    o.add_species([0.], [0.], [0.], [0.], [0.], [0.], [1.], -Q_E, M_E)
    dv = dx[0] * dx[1] * dx[2]
    for _ in range(20):
        x0, x1 = _moves(rng, n, dx, 1)
        w = np.array([3.7e5])
        J = o.deposit_moves(0, x0, x1, w)
        for d in range(3):
            want = -Q_E * w[0] * (x1[0, d] - x0[0, d]) / dt
            assert abs(J[d].sum() * dv - want) < 1e-12 * abs(Q_E * w[0] * dx[d] / dt)


def _dense_shape(order, xi, N):
    """Dense periodic length-N vector of nodal weights (indices wrapped)."""
    l, w = oracle.shape(order, xi)
    S = np.zeros(N)
    for a in range(order + 1):
        S[(l + a) % N] += w[a]
    return S


@pytest.mark.parametrize("order", [1, 2, 3])
def test_T7_deposit_vs_brute_force_dense(order):
    """Brute force: dense S0,S1 on all N nodes, W on all N^3 nodes, integrate the defining
    difference J(i+1/2)-J(i-1/2) = -q w W[i]/(dt dy dz) along each line from a node outside the
    particle's support; must equal the windowed prefix-sum deposit."""
    n, dx = (8, 7, 6), (1.0e-6, 0.8e-6, 0.5e-6)
    dt = 0.5 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    rng = np.random.default_rng(40 + order)
    o = Oracle(n, dx, dt, order, tile=(1, 1, 1), sort_interval=0)
    q = -Q_E
    o.add_species([0.], [0.], [0.], [0.], [0.], [0.], [1.], q, M_E)
    cases = [_moves(rng, n, dx, 1) for _ in range(12)]
    # moves that cross the periodic seam on every axis, both directions
    Lx = np.array(n) * np.array(dx)
    cases.append((np.array([[0.1e-6, 0.05e-6, 0.02e-6]]), np.array([[-0.5e-6, -0.3e-6, -0.2e-6]])))
    cases.append((Lx[None, :] - 1e-8, Lx[None, :] + 0.4 * np.array(dx)[None, :]))
    for x0, x1 in cases:
        w = 2.5e5
        J = o.deposit_moves(0, x0, x1, np.array([w]))
        S0 = [_dense_shape(order, x0[0, d] / dx[d], n[d]) for d in range(3)]
        S1 = [_dense_shape(order, x1[0, d] / dx[d], n[d]) for d in range(3)]
        DS = [S1[d] - S0[d] for d in range(3)]

        def Wd(d):
            a, b = [(1, 2), (0, 2), (0, 1)][d]
            br = (np.multiply.outer(S0[a], S0[b]) + 0.5 * np.multiply.outer(DS[a], S0[b])
                  + 0.5 * np.multiply.outer(S0[a], DS[b]) + np.multiply.outer(DS[a], DS[b]) / 3.0)
            return DS[d], br      # W[d-index, a-index, b-index] = DS[d] * br[a,b]

        area = [dx[1] * dx[2], dx[0] * dx[2], dx[0] * dx[1]]
        for d in range(3):
            ds, br = Wd(d)
            # start just after a node where both S0 and S1 vanish along d; J there is 0
            outside = [i for i in range(n[d]) if S0[d][i] == 0 and S1[d][i] == 0]
            assert outside
            start = outside[0]
            line = np.zeros(n[d])           # line[i] = J at (i+1/2)
            acc = 0.0
            for s in range(1, n[d] + 1):
                i = (start + s) % n[d]
                acc += ds[i]
                line[i] = acc
            assert abs(acc) < 1e-15          # closes: sum DS = 0
            Jd = -q * w / (dt * area[d]) * np.multiply.outer(line, br)   # [d, a, b]
            # to numpy layout (z, y, x)
            if d == 0:
                want = Jd.transpose(2, 1, 0)        # [x,y,z] -> [z,y,x]
            elif d == 1:
                want = Jd.transpose(2, 0, 1)        # [y,x,z] -> [z,y,x]
            else:
                want = Jd.transpose(0, 2, 1)        # [z,x,y] -> [z,y,x]
            scale = np.max(np.abs(want))
            assert scale > 0
            assert np.max(np.abs(J[d] - want)) < 1e-13 * scale


# --------------------------------------------------------------------------- T8 whole loop
def _c1_like(order, n=(8, 8, 8), ppc=2, seed=3, sigma=0.05, density=1e24, sort_interval=4, shuffle=None):
    dx = (1e-6,) * 3
    dt = 0.99 * dx[0] / (c * math.sqrt(3))
    rng = np.random.default_rng(seed)
    npart = ppc * n[0] * n[1] * n[2]
    pos = rng.uniform(0, 1, (3, npart)) * (np.array(n)[:, None] * 1e-6)
    u = rng.standard_normal((3, npart)) * sigma * c
    w = np.full(npart, density * 1e-18 / ppc)
    if shuffle is not None:
        p = np.random.default_rng(shuffle).permutation(npart)
        pos, u, w = pos[:, p], u[:, p], w[p]
    o = Oracle(n, dx, dt, order, tile=(4, 4, 4), sort_interval=sort_interval)
    o.add_species(pos[0], pos[1], pos[2], u[0], u[1], u[2], w, -Q_E, M_E)
    return o, dx, dt


@pytest.mark.parametrize("order", [1, 2, 3])
def test_T8_gauss_law_residual_is_constant(order):
    o, dx, dt = _c1_like(order)
    def residual():
        E, _, _ = o.get_fields()
        return _div_back(E, dx) - o.rho() / EPS0
    r0 = residual()
    scale = np.max(np.abs(o.rho() / EPS0))
    for _ in range(6):
        o.step(25)
        assert np.max(np.abs(residual() - r0)) < 2e-13 * scale
    E, B, _ = o.get_fields()
    assert np.max(np.abs(E[0])) > 0 and np.max(np.abs(B[0])) > 0      # the loop did something


# --------------------------------------------------------------------------- T9 plasma oscillation
@pytest.mark.parametrize("order,expect", [(1, 0.991), (2, 0.984), (3, 0.978)])
def test_T9_cold_plasma_oscillation_frequency(order, expect):
    n, dx = (16, 4, 4), (1e-6,) * 3
    dt = 0.99 * dx[0] / (c * math.sqrt(3))
    dens = 1e24
    wp = math.sqrt(dens * Q_E ** 2 / (EPS0 * M_E))
    # quiet start: 2x2x2 lattice per cell
    g = (np.arange(2) + 0.5) / 2
    cx, cy, cz = np.meshgrid(np.arange(n[0]), np.arange(n[1]), np.arange(n[2]), indexing="ij")
    xs, ys, zs = [], [], []
    for a in g:
        for b in g:
            for cc in g:
                xs.append((cx + a).ravel()); ys.append((cy + b).ravel()); zs.append((cz + cc).ravel())
    x = np.concatenate(xs) * dx[0]; y = np.concatenate(ys) * dx[1]; z = np.concatenate(zs) * dx[2]
    Lx = n[0] * dx[0]
    ux = 1e-4 * c * np.sin(2 * math.pi * x / Lx)
    w = np.full(len(x), dens * 1e-18 / 8)
    o = Oracle(n, dx, dt, order, tile=(4, 4, 4), sort_interval=4)
    o.add_species(x, y, z, ux, 0 * x, 0 * x, w, -Q_E, M_E)
    trace = []
    for _ in range(400):
        o.step(1)
        trace.append(o.get_fields()[0][0][0, 0, 4])
    trace = np.array(trace)
    t = (np.arange(400) + 1) * dt
    sgn = np.sign(trace)
    idx = np.where(sgn[:-1] * sgn[1:] < 0)[0]
    assert len(idx) >= 6
    tz = t[idx] - trace[idx] * (t[idx + 1] - t[idx]) / (trace[idx + 1] - trace[idx])
    omega = math.pi * (len(tz) - 1) / (tz[-1] - tz[0])
    ratio = omega / wp
    assert 0.96 < ratio < 1.0005          # finite-grid smoothing lowers it slightly; never above leapfrog limit
    assert abs(ratio - expect) < 4e-3     # SURVEY.md §8(c) T9 soft pin


# --------------------------------------------------------------------------- T10 sort
@pytest.mark.parametrize("key_mode", [0, 1])
def test_T10_stable_counting_sort_matches_numpy(key_mode):
    n, dx = (16, 8, 8), (1.0e-6, 0.8e-6, 0.5e-6)
    dt = 0.5 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    T = (8, 4, 2)
    rng = np.random.default_rng(50)
    npart = 5000
    pos = rng.uniform(0, 1, (3, npart)) * (np.array(n) * np.array(dx))[:, None]
    pos[0, :5] = np.nextafter(n[0] * dx[0], 0)         # just below L: may round to N -> clamp
    pos[1, 5:9] = 0.0
    u = rng.standard_normal((3, npart))
    w = rng.uniform(1, 2, npart)
    o = Oracle(n, dx, dt, 1, tile=T, sort_interval=4, sort_key_mode=key_mode)
    o.add_species(pos[0], pos[1], pos[2], u[0], u[1], u[2], w, -Q_E, M_E)
    o.sort_now()
    cell, perm = o.get_sort_state()
    ci = [np.clip(np.floor(pos[d] * (1.0 / dx[d])).astype(np.int64), 0, n[d] - 1) for d in range(3)]
    nt = [n[d] // T[d] for d in range(3)]
    tile = ci[0] // T[0] + nt[0] * (ci[1] // T[1] + nt[1] * (ci[2] // T[2]))
    rem = ci[0] % T[0] + T[0] * (ci[1] % T[1] + T[1] * (ci[2] % T[2]))
    key = tile * (T[0] * T[1] * T[2]) + rem if key_mode == 0 else tile
    want = np.argsort(key, kind="stable")
    assert np.array_equal(perm, want.astype(np.int32))
    lin = (ci[0] + n[0] * (ci[1] + n[1] * ci[2])).astype(np.int32)
    assert np.array_equal(cell, lin[want])
    p = o.get_particles()
    assert np.array_equal(p["id"], want)
    for name, src in zip(("x", "y", "z", "ux", "uy", "uz", "w"), (pos[0], pos[1], pos[2], u[0], u[1], u[2], w)):
        assert np.array_equal(p[name], src[want])
    # idempotent: sorting sorted data is the identity permutation
    o.sort_now()
    _, perm2 = o.get_sort_state()
    assert np.array_equal(perm2, np.arange(npart, dtype=np.int32))
    assert np.array_equal(o.get_particles()["id"], want)


# --------------------------------------------------------------------------- T11 order independence
def test_T11_particle_order_does_not_change_the_physics():
    a, dx, dt = _c1_like(3, sort_interval=0)
    b, _, _ = _c1_like(3, sort_interval=1, shuffle=99)
    a.step(8); b.step(8)
    Ea, Ba, Ja = a.get_fields()
    Eb, Bb, Jb = b.get_fields()
    for fa, fb in ((Ea, Eb), (Ba, Bb), (Ja, Jb)):
        scale = max(np.max(np.abs(v)) for v in fa)
        for d in range(3):
            assert np.max(np.abs(fa[d] - fb[d])) < 1e-12 * scale
    pa, pb = a.get_particles(), b.get_particles()
    # b was shuffled by rng(99) and then sorted: match by original identity
    p = np.random.default_rng(99).permutation(len(pa["x"]))
    orig = p[pb["id"]]
    for k in ("x", "ux", "uy", "uz"):
        va = pa[k][orig]
        assert np.max(np.abs(va - pb[k])) < 1e-12 * np.max(np.abs(pa[k]))


# --------------------------------------------------------------------------- misc
def test_energy_is_nearly_conserved_and_charge_exactly():
    o, dx, dt = _c1_like(2, sigma=0.01)
    d0 = o.diagnostics()
    o.step(60)
    d1 = o.diagnostics()
    assert d1["charge"] == d0["charge"]
    e0 = d0["field_E"] + d0["field_B"] + d0["kinetic"]
    e1 = d1["field_E"] + d1["field_B"] + d1["kinetic"]
    assert d1["field_E"] > 0
    assert abs(e1 - e0) < 0.05 * e0


def test_create_rejects_bad_arguments():
    dx = (1e-6,) * 3
    dt_ok = 0.99 * 1e-6 / (c * math.sqrt(3))
    with pytest.raises(ValueError):
        Oracle((8, 8, 8), dx, dt_ok * 1.02, 1)          # CFL
    with pytest.raises(ValueError):
        Oracle((8, 8, 8), dx, dt_ok, 4)                 # order
    with pytest.raises(ValueError):
        Oracle((12, 8, 8), dx, dt_ok, 1, tile=(8, 8, 8))  # tile must divide


def test_nonperiodic_axis_reads_zero_and_drops_writes():
    """Reading Q6: on a non-periodic axis J written outside is dropped and fields outside read 0."""
    n, dx = (6, 6, 8), (1e-6,) * 3
    dt = 0.5 * 1e-6 / (c * math.sqrt(3))
    per = Oracle(n, dx, dt, 3, periodic=(1, 1, 1), tile=(1, 1, 1), sort_interval=0)
    npz = Oracle(n, dx, dt, 3, periodic=(1, 1, 0), tile=(1, 1, 1), sort_interval=0)
    for o in (per, npz):
        o.add_species([0.], [0.], [0.], [0.], [0.], [0.], [1.], -Q_E, M_E)
    x0 = np.array([[3.2e-6, 3.1e-6, 0.3e-6]])
    x1 = np.array([[3.3e-6, 3.3e-6, 0.6e-6]])
    Jp = per.deposit_moves(0, x0, x1, np.array([1e5]))
    Jn = npz.deposit_moves(0, x0, x1, np.array([1e5]))
    for d in range(3):
        # identical where the window is inside; what wrapped to the top planes is absent
        assert np.array_equal(Jn[d][:5], Jp[d][:5])
        assert np.all(Jn[d][5:] == 0)
    assert any(np.any(Jp[d][5:] != 0) for d in range(3))


# --------------------------------------------------------------------------- T13 Vay pusher (NEXT-4)
def test_T13_vay_keeps_the_ExB_drift_exactly_and_boris_does_not():
    """Defining property of the Vay pusher (ref [21]): a particle that moves with the
    drift velocity v = E x B / B^2 (E perpendicular to B, E < cB) feels no net force, at any gamma and any
    time step; the Boris rotation leaves a spurious force of order (omega_c dt)^2."""
    rng = np.random.default_rng(130)
    for _ in range(50):
        B = rng.normal(size=3)
        Bn = np.linalg.norm(B)
        e = np.cross(B, rng.normal(size=3))
        e /= np.linalg.norm(e)
        beta = rng.uniform(0.05, 0.98)
        E = beta * c * Bn * e                      # |E| = beta c |B|, perpendicular to B
        vd = np.cross(E, B) / Bn ** 2
        assert abs(np.linalg.norm(vd) / c - beta) < 1e-12
        u0 = vd / math.sqrt(1 - beta * beta)
        kq = rng.uniform(0.05, 1.5) / Bn * rng.choice([-1.0, 1.0])     # |omega_c dt / 2| up to 1.5
        uv = oracle.vay(kq, E, B, u0)
        assert np.linalg.norm(uv - u0) < 1e-13 * np.linalg.norm(u0)
        ub = oracle.boris(kq, E, B, u0)
        if beta > 0.5 and abs(kq) * Bn > 0.3:
            assert np.linalg.norm(ub - u0) > 1e-4 * np.linalg.norm(u0)


def test_T13_vay_limits_pure_E_pure_B_and_agreement_with_boris():
    rng = np.random.default_rng(131)
    for _ in range(30):
        u0 = rng.normal(size=3) * c * rng.uniform(0.01, 3.0)
        E = rng.normal(size=3) * 1e9
        B = rng.normal(size=3)
        kq = rng.uniform(-1.0, 1.0) * 1e-1
        # B = 0: u += 2 kq E exactly, as for Boris
        assert np.allclose(oracle.vay(kq, E, 0 * B, u0), u0 + 2 * kq * E, rtol=1e-15, atol=0)
        # E = 0: |u| is conserved (gamma_new = gamma, shown in closed form in DESIGN.md)
        assert abs(np.linalg.norm(oracle.vay(kq, 0 * E, B, u0)) / np.linalg.norm(u0) - 1) < 1e-14
    # both pushers are second order: their difference shrinks as dt^3 per step
    u0 = np.array([0.3, -0.2, 0.5]) * c
    E = np.array([1.0, 2.0, -1.5]) * 1e10
    B = np.array([0.5, -1.0, 2.0])
    d = [np.linalg.norm(oracle.vay(kq, E, B, u0) - oracle.boris(kq, E, B, u0)) for kq in (-5e-4, -2.5e-4, -1.25e-4)]
    assert 7.0 < d[0] / d[1] < 10.0 and 7.0 < d[1] / d[2] < 10.0 and d[1] / d[2] < d[0] / d[1]


def test_T13_vay_gyration_conserves_energy_and_closes_the_orbit():
    """Uniform B through the whole oracle loop with pusher = Vay: |u| stays constant to roundoff and
    the rotation per step is the same 2 atan(omega_c dt / 2) as Boris (for E = 0 the two coincide:
    u' = u + u x t, then the same normalisation)."""
    n, dx = (8, 8, 8), (1e-6, 1e-6, 1e-6)
    dt = 0.5 * dx[0] / (c * math.sqrt(3))
    B0 = 2.0e3
    o = Oracle(n, dx, dt, 1, sort_interval=0, pusher=oracle.PUSHER_VAY)
    Bz = np.full((8, 8, 8), B0)
    zf = np.zeros((8, 8, 8))
    o.set_fields([zf, zf, zf], [zf, zf, Bz])
    u0 = 0.5 * c
    o.add_species([4e-6], [4e-6], [4e-6], [u0], [0.0], [0.0], [0.0], -Q_E, M_E)      # weight 0: no J
    gam = math.sqrt(1 + (u0 / c) ** 2)
    wc = Q_E * B0 / (gam * M_E)
    theta = 2 * math.atan(wc * dt / 2)
    ang = []
    for _ in range(40):
        o.step(1)
        p = o.get_particles(0)
        assert abs(math.hypot(p["ux"][0], p["uy"][0]) / u0 - 1) < 1e-13
        ang.append(math.atan2(p["uy"][0], p["ux"][0]))
    dth = np.diff(np.unwrap(ang))
    assert np.all(dth > 0)                         # electron, B along +z: counter-clockwise
    assert np.max(np.abs(dth - theta)) < 1e-12


# --------------------------------------------------------------------------- T14 Galerkin gather (NEXT-2)
_STAG = [(1, 0, 0), (0, 1, 0), (0, 0, 1), (0, 1, 1), (1, 0, 1), (1, 1, 0)]   # Ex Ey Ez Bx By Bz


def _cardinal_bspline(m, d):
    """Centred cardinal B-spline of degree m at distance d, from scipy's B-spline basis (an
    implementation that shares nothing with oracle.shape)."""
    from scipy.interpolate import BSpline
    knots = np.arange(m + 2) - (m + 1) / 2.0
    b = BSpline.basis_element(knots, extrapolate=False)
    v = b(d)
    return 0.0 if np.isnan(v) else float(v)


@pytest.mark.parametrize("order", [1, 2, 3])
@pytest.mark.parametrize("mode", [0, 1])
def test_T14_gather_equals_the_tensor_product_of_library_bsplines(order, mode):
    """Both gather variants against a dense sum over ALL nodes of a small periodic grid with 1-D
    weights from scipy.interpolate.BSpline: degree n on every axis (uniform), or n-1 along the axes on
    which the component is staggered (Galerkin). Fixes offsets, orders and indices."""
    n, dx = (6, 5, 7), (1.0e-6, 0.8e-6, 0.5e-6)
    dt = 0.5 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    rng = np.random.default_rng(140 + order)
    o = Oracle(n, dx, dt, order, sort_interval=0, gather_mode=mode)
    F = [rng.normal(size=(n[2], n[1], n[0])) for _ in range(6)]
    o.set_fields(F[:3], F[3:])
    npart = 12
    pos = rng.uniform(0, 1, size=(npart, 3)) * np.array(n) * np.array(dx)
    got = o.gather(pos[:, 0], pos[:, 1], pos[:, 2])
    for p in range(npart):
        for comp in range(6):
            W = []
            for d in range(3):
                deg = order - 1 if (mode == 1 and _STAG[comp][d]) else order
                xi = pos[p, d] / dx[d] - 0.5 * _STAG[comp][d]
                w = np.zeros(n[d])
                for i in range(-4, n[d] + 4):          # periodic images
                    if deg == 0:
                        w[i % n[d]] += 1.0 if -0.5 <= xi - i < 0.5 else 0.0
                    else:
                        w[i % n[d]] += _cardinal_bspline(deg, xi - i)
                W.append(w)
            want = np.einsum("kji,k,j,i->", F[comp], W[2], W[1], W[0])
            assert abs(got[p, comp] - want) < 1e-13 * (1 + abs(want)), (p, comp)


@pytest.mark.parametrize("order", [1, 2, 3])
def test_T14_galerkin_gather_is_the_small_move_limit_of_the_esirkepov_deposit(order):
    """Energy exchange identity that gives the variant its name: for a move delta along one axis, the
    work of the field on the deposited current, sum_nodes J_d E_d dV dt, equals q w delta E_d gathered at
    the midpoint with the Galerkin weights, up to O(delta^2) (d/dx of a degree-n B-spline is the
    difference of two degree n-1 ones at the staggered points). The deposit is pinned by T5-T7."""
    n, dx = (7, 6, 8), (1.0e-6, 0.8e-6, 0.5e-6)
    dt = 0.5 / (c * math.sqrt(sum(1 / d ** 2 for d in dx)))
    rng = np.random.default_rng(150 + order)
    E = [rng.normal(size=(n[2], n[1], n[0])) for _ in range(3)]
    zf = np.zeros((n[2], n[1], n[0]))
    og = Oracle(n, dx, dt, order, sort_interval=0, gather_mode=1)
    ou = Oracle(n, dx, dt, order, sort_interval=0, gather_mode=0)
    for o in (og, ou):
        o.set_fields(E, [zf, zf, zf])
        o.add_species([0.], [0.], [0.], [0.], [0.], [0.], [1.], -Q_E, M_E)
    dv = dx[0] * dx[1] * dx[2]
    w = np.array([2.5e5])
    worst_uniform = 0.0
    for trial in range(12):
        d = trial % 3
        xm = rng.uniform(0.2, 0.8, 3) * np.array(n) * np.array(dx)
        delta = 1e-4 * dx[d]
        x0, x1 = xm.copy(), xm.copy()
        x0[d] -= delta / 2
        x1[d] += delta / 2
        J = og.deposit_moves(0, x0[None, :], x1[None, :], w)
        work = float(np.sum(J[d] * E[d])) * dv * dt
        eg = og.gather([xm[0]], [xm[1]], [xm[2]])[0, d]
        eu = ou.gather([xm[0]], [xm[1]], [xm[2]])[0, d]
        scale = Q_E * w[0] * delta * np.max(np.abs(E[d]))
        assert abs(work - (-Q_E) * w[0] * delta * eg) < 1e-6 * scale
        worst_uniform = max(worst_uniform, abs(work - (-Q_E) * w[0] * delta * eu) / scale)
    assert worst_uniform > 1e-3          # the uniform-order gather does NOT satisfy it: the pin discriminates


# --------------------------------------------------------------------------- T15 CKC solver (NEXT-4)
def _ckc_symbol(k, dx, alpha, beta, gamma):
    """S_a(k) = alpha_a + 2 beta_ab cos(k_b dx_b) + 2 beta_ac cos(k_c dx_c) + 4 gamma_a cos cos: the Fourier
    symbol of the transverse smoothing of the difference along a."""
    S = []
    for a in range(3):
        b, cc = (a + 1) % 3, (a + 2) % 3
        cb, cz = math.cos(k[b] * dx[b]), math.cos(k[cc] * dx[cc])
        S.append(alpha[a] + 2 * beta[a][b] * cb + 2 * beta[a][cc] * cz + 4 * gamma[a] * cb * cz)
    return np.array(S)


def test_T15_ckc_coefficients_cubic_values_consistency_and_von_neumann_stability():
    """Cubic cells: the published 7/12, 1/12, 1/48 (ref [12]). Any cells: the weights of every smoothed
    difference sum to 1 (second-order consistency), and with c dt = min(dx) — beyond Yee's limit — the
    amplification stays on the unit circle for every wave vector: 0 <= (c dt)^2 sum_a S_a sin^2(k_a dx_a/2)
    / dx_a^2 <= 1 (the property the coefficients are built for)."""
    o = Oracle((8, 8, 8), (1e-6,) * 3, 1e-6 / c, 1, sort_interval=0, solver=oracle.SOLVER_CKC)
    al, be, ga = o.ckc_coefficients()
    assert np.allclose(al, 7 / 12, rtol=1e-15) and np.allclose(ga, 1 / 48, rtol=1e-14)
    assert np.allclose(be[~np.eye(3, dtype=bool)], 1 / 12, rtol=1e-14)
    for dx in [(1e-6, 1e-6, 1e-6), (1e-6, 0.8e-6, 0.5e-6), (0.1e-6, 0.1e-6, 0.025e-6), (2e-6, 1e-6, 1e-6)]:
        dmin = min(dx)
        dt = dmin / c
        o = Oracle((8, 8, 8), dx, dt, 1, sort_interval=0, solver=oracle.SOLVER_CKC)
        al, be, ga = o.ckc_coefficients()
        for a in range(3):
            b, cc = (a + 1) % 3, (a + 2) % 3
            assert abs(al[a] + 2 * be[a][b] + 2 * be[a][cc] + 4 * ga[a] - 1) < 1e-15
        worst = 0.0
        for kx in np.linspace(0, math.pi, 25):
            for ky in np.linspace(0, math.pi, 25):
                for kz in np.linspace(0, math.pi, 25):
                    k = np.array([kx / dx[0], ky / dx[1], kz / dx[2]])
                    S = _ckc_symbol(k, dx, al, be, ga)
                    s2 = (c * dt) ** 2 * sum(S[a] * math.sin(k[a] * dx[a] / 2) ** 2 / dx[a] ** 2 for a in range(3))
                    assert s2 > -1e-14
                    worst = max(worst, s2)
        assert worst <= 1 + 1e-12
        assert worst > 0.999                    # the limit is reached: c dt = min(dx) is the edge
        with pytest.raises(ValueError):         # Yee cannot run this time step
            Oracle((8, 8, 8), dx, dt, 1, sort_interval=0)


@pytest.mark.parametrize("frac", [0.7, 1.0])
def test_T15_ckc_plane_wave_dispersion(frac):
    """A discrete plane wave with omega from the CKC relation sin^2(omega dt/2) = (c dt)^2 sum_a S_a(k)
    sin^2(k_a dx_a/2)/dx_a^2, E perpendicular to K, B = K' x E / Omega with K'_a = S_a K_a, is reproduced to
    roundoff over hundreds of steps on an anisotropic grid, also at c dt = min(dx)."""
    n, dx = (8, 12, 16), (1.0e-6, 0.8e-6, 0.5e-6)
    dt = frac * min(dx) / c
    o = Oracle(n, dx, dt, 1, tile=(1, 1, 1), sort_interval=0, solver=oracle.SOLVER_CKC)
    al, be, ga = o.ckc_coefficients()
    mode = (1, 2, 1)
    k = np.array([2 * math.pi * mode[d] / (n[d] * dx[d]) for d in range(3)])
    S = _ckc_symbol(k, dx, al, be, ga)
    K = np.array([2 / dx[d] * math.sin(k[d] * dx[d] / 2) for d in range(3)])
    Kp = S * K
    s2 = (c * dt) ** 2 * sum(S[d] * math.sin(k[d] * dx[d] / 2) ** 2 / dx[d] ** 2 for d in range(3))
    om = 2 / dt * math.asin(math.sqrt(s2))
    Om = 2 / dt * math.sin(om * dt / 2)
    E0 = np.cross(K, [0.3, -0.2, 1.0])
    E0 *= 1e9 / np.linalg.norm(E0)
    B0 = np.cross(Kp, E0) / Om
    stag = [(.5, 0, 0), (0, .5, 0), (0, 0, .5), (0, .5, .5), (.5, 0, .5), (.5, .5, 0)]

    def phase(cmp):
        xs = (np.arange(n[0]) + stag[cmp][0]) * dx[0]
        ys = (np.arange(n[1]) + stag[cmp][1]) * dx[1]
        zs = (np.arange(n[2]) + stag[cmp][2]) * dx[2]
        return k[0] * xs[None, None, :] + k[1] * ys[None, :, None] + k[2] * zs[:, None, None]

    def exact(t):
        E = [E0[d] * np.cos(phase(d) - om * t) for d in range(3)]
        B = [B0[d] * math.cos(om * dt / 2) * np.cos(phase(3 + d) - om * t) for d in range(3)]
        return E, B

    o.set_fields(*exact(0.0))
    nsteps = 300
    o.field_step(nsteps)
    E, B, _ = o.get_fields()
    Ee, Be = exact(nsteps * dt)
    for d in range(3):
        assert np.max(np.abs(E[d] - Ee[d])) < 1e-11 * 1e9
        assert np.max(np.abs(B[d] - Be[d])) < 1e-11 * np.linalg.norm(B0)
    assert om * nsteps * dt > 20
    # the Yee relation (S = 1) is a different wave: the pin discriminates
    s2y = (c * dt) ** 2 * sum(math.sin(k[d] * dx[d] / 2) ** 2 / dx[d] ** 2 for d in range(3))
    assert abs(s2y - s2) > 1e-3 * s2


def test_T15_ckc_no_dispersion_along_the_axis_at_the_magic_time_step():
    """Cubic cells, c dt = dx: a wave along an axis has omega = c k exactly (S = 1 for transverse k = 0,
    sin(omega dt/2) = sin(k dx/2)), for every resolvable k — the reason the scheme exists."""
    n, dx = (16, 4, 4), (1e-6, 1e-6, 1e-6)
    dt = dx[0] / c
    o = Oracle(n, dx, dt, 1, tile=(1, 1, 1), sort_interval=0, solver=oracle.SOLVER_CKC)
    rng = np.random.default_rng(151)
    f = rng.normal(size=n[0]) * 1e9                       # any profile: every Fourier mode moves at c
    Ey = np.broadcast_to(f[None, None, :], (n[2], n[1], n[0])).copy()
    zf = np.zeros_like(Ey)
    # forward wave: Bz(i+1/2) at the integer time = average of the two half-step values f(i), f(i+1) / c
    Bz = np.broadcast_to(((f + np.roll(f, -1)) / (2 * c))[None, None, :], Ey.shape).copy()
    o.set_fields([zf, Ey, zf], [zf, zf, Bz])
    o.field_step(5)
    E, B, _ = o.get_fields()
    assert np.max(np.abs(E[1][0, 0, :] - np.roll(f, 5))) < 1e-12 * np.max(np.abs(f))
    assert np.max(np.abs(E[0])) == 0 and np.max(np.abs(E[2])) == 0


# --------------------------------------------------------------------------- T12 OpenMP variant
@pytest.mark.parametrize("case", ["C1", "o3_truncated_two_species"])
def test_T12_openmp_variant_equals_the_serial_oracle(case):
    """The OpenMP variant (tiles to threads, thread-private J buffers flushed with one atomic per cell — the
    paper's CPU scheme) runs the same per-particle arithmetic as the canonical serial
    oracle and differs only in the order J is summed: after many steps every array agrees to 1e-13 of its
    family's max, the sort permutations are identical, and so is the deactivation count."""
    import workloads as W
    if case == "C1":
        cfg = W.CONFIGS["C1"]
        steps = cfg.steps
    else:
        cfg = W.scaled(W.CONFIGS["C5"], (16, 8, 24), periodic=(1, 1, 0), tile=(8, 4, 8), dx=(1e-6, 0.8e-6, 0.6e-6))
        steps = 9
    species, _, _ = W.generate(cfg)
    sims = []
    for _ in range(2):
        o = Oracle(cfg.n_cells, cfg.dx, cfg.dt, cfg.order, periodic=cfg.periodic, tile=cfg.tile,
                   sort_interval=cfg.sort_interval)
        for spec, a in species:
            o.add_species(*[a[k] for k in ("x", "y", "z", "ux", "uy", "uz", "w")], spec.charge, spec.mass)
        sims.append(o)
    sims[0].step(steps)
    assert sims[1].step_omp(steps, threads=4) == 4
    fa, fb = sims[0].get_fields(), sims[1].get_fields()
    for grp in range(3):
        scale = max(np.max(np.abs(a)) for a in fa[grp])
        assert scale > 0
        for a, b in zip(fa[grp], fb[grp]):
            assert np.max(np.abs(a - b)) <= 1e-13 * scale
    for s in range(len(species)):
        assert all(np.array_equal(a, b) for a, b in zip(sims[0].get_sort_state(s), sims[1].get_sort_state(s)))
        pa, pb = sims[0].get_particles(s), sims[1].get_particles(s)
        assert np.array_equal(pa["id"], pb["id"])
        for fam in (("x", "y", "z"), ("ux", "uy", "uz"), ("w",)):
            scale = max(np.max(np.abs(pa[k])) for k in fam)
            assert all(np.max(np.abs(pa[k] - pb[k])) <= 1e-13 * scale for k in fam)
    da, db = sims[0].diagnostics(), sims[1].diagnostics()
    assert da["deactivated"] == db["deactivated"]
    if case != "C1":
        assert da["deactivated"] > 0          # hot particles did leave through the truncated faces
