"""Pins of the tracer-particle oracle (oracle/tracers_oracle.hpp; Sec. VI, Eq. 20-22) against
what the paper and the mathematics fix: exactness of cloud-in-cell weights on (tri)linear data, the periodic wrap,
a library routine (scipy.ndimage.map_coordinates, order 1, grid-wrap), and the closed-form rotation of the Boris
scheme in a uniform field.  CPU only."""
import math

import numpy as np
import pytest
from scipy import ndimage

import oracle

L = 2 * math.pi


def idx_grid(N):
    iz, iy, ix = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    return ix.astype(float), iy.astype(float), iz.astype(float)


def rand_pos(n, rng, lo=0.0, hi=L):
    return [rng.uniform(lo, hi, n) for _ in range(3)]


def test_tp1_weights_sum_to_one():
    """Reading T1: a uniform field is reproduced wherever the particle sits.  The weights are formed from coordinate
    differences |x_p - x_grid| / dx, each good to |x| eps / dx <= N eps, so their sum is 1 to a few N eps."""
    N = 16
    rng = np.random.default_rng(1)
    pos = rand_pos(1000, rng)
    out = oracle.cic([np.full((N, N, N), 3.25)], pos)[0]
    assert np.max(np.abs(out - 3.25)) <= 4 * N * np.finfo(float).eps * 3.25


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_tp2_linear_field_exact_per_axis(axis):
    """Eq. 20 weights, axis by axis: g = index along one axis is interpolated to x/dx exactly (interior cells).  A
    weight attached to the wrong corner, or x and z swapped, fails."""
    N = 16
    dx = L / N
    ix, iy, iz = idx_grid(N)
    g = [ix, iy, iz][axis]
    rng = np.random.default_rng(2 + axis)
    pos = rand_pos(2000, rng, 0.0, (N - 1) * dx * 0.999)
    out = oracle.cic([g], pos)[0]
    assert np.max(np.abs(out - pos[axis] / dx)) <= 1e-13 * N


def test_tp3_trilinear_monomial_exact():
    """Trilinear interpolation reproduces ix*iy*iz (all 8 corner weights are needed for this)."""
    N = 8
    dx = L / N
    ix, iy, iz = idx_grid(N)
    rng = np.random.default_rng(5)
    pos = rand_pos(2000, rng, 0.0, (N - 1) * dx * 0.999)
    out = oracle.cic([ix * iy * iz], pos)[0]
    ref = (pos[0] / dx) * (pos[1] / dx) * (pos[2] / dx)
    assert np.max(np.abs(out - ref)) <= 1e-12 * N ** 3


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_tp4_periodic_wrap(axis):
    """L255: a particle in the last cell feels the grid at index 0 of the opposite boundary."""
    N = 8
    dx = L / N
    g = np.zeros((N, N, N))
    sl = [slice(None)] * 3
    sl[2 - axis] = 0                      # array order is [z][y][x]
    g[tuple(sl)] = 1.0
    f = np.array([0.0, 0.25, 0.5, 0.875])
    pos = [np.full(4, 2.5 * dx) for _ in range(3)]
    pos[axis] = (N - 1 + f) * dx
    out = oracle.cic([g], pos)[0]
    assert np.max(np.abs(out - f)) <= 1e-14


def test_tp5_library_special_case():
    """CIC with periodic wrap = scipy's order-1 spline interpolation in grid-wrap mode."""
    N = 12
    dx = L / N
    rng = np.random.default_rng(7)
    g = rng.standard_normal((N, N, N))
    pos = rand_pos(5000, rng)
    out = oracle.cic([g], pos)[0]
    coords = np.stack([pos[2] / dx, pos[1] / dx, pos[0] / dx])       # array axes are z, y, x
    ref = ndimage.map_coordinates(g, coords, order=1, mode="grid-wrap")
    assert np.max(np.abs(out - ref)) <= 1e-13


def rodrigues(v, axis_unit, angle):
    k = axis_unit
    return v * math.cos(angle) + np.cross(k, v) * math.sin(angle) + k * np.dot(k, v) * (1 - math.cos(angle))


def test_tp6_boris_is_exact_rotation_about_B():
    """Eq. 21 as printed: one push in a uniform field rotates v about B by -2 atan(|B| dt/2) (dv/dt = v x B, q = M = 1):
    fixes every sign and index of the two cross products and the factor 2/(1+t^2)."""
    N = 8
    rng = np.random.default_rng(11)
    for trial in range(5):
        B0 = rng.standard_normal(3) * 3.0
        dt = 0.05 * (trial + 1)
        B = [np.full((N, N, N), B0[c]) for c in range(3)]
        v0 = rng.standard_normal(3)
        pos = [np.array([1.0]), np.array([2.0]), np.array([3.0])]
        p1, v1 = oracle.tracers_push(B, pos, [np.array([v0[c]]) for c in range(3)], dt, 1)
        bn = np.linalg.norm(B0)
        ref = rodrigues(v0, B0 / bn, -2.0 * math.atan(bn * dt / 2))
        got = np.array([v1[c][0] for c in range(3)])
        assert np.max(np.abs(got - ref)) <= 1e-14 * np.linalg.norm(v0)
        assert abs(np.linalg.norm(got) - np.linalg.norm(v0)) <= 1e-15 * np.linalg.norm(v0) * 4
        # Eq. 22: x(t+dt) = x(t) + v(t+dt) dt, wrapped into [0, L)
        xref = (np.array([1.0, 2.0, 3.0]) + got * dt) % L
        assert np.max(np.abs(np.array([p1[c][0] for c in range(3)]) - xref)) <= 1e-15 * L


def test_tp7_gyration_closed_form():
    """n pushes in B = B0 z^: v_n = (v0 cos n th, -v0 sin n th, vz), th = 2 atan(B0 dt/2); x_n = x_0 + dt sum_j v_j;
    the orbit is a circle of radius v0 dt / (2 sin(th/2)) in the (x, y) plane."""
    N = 8
    B0, dt, n = 2.0, 0.01, 400
    B = [np.zeros((N, N, N)), np.zeros((N, N, N)), np.full((N, N, N), B0)]
    v0, vz = 0.7, 0.3
    x0 = np.array([3.0, 3.0, 1.0])
    th = 2 * math.atan(B0 * dt / 2)
    j = np.arange(1, n + 1)
    xs = x0[0] + dt * np.cumsum(v0 * np.cos(j * th))
    ys = x0[1] + dt * np.cumsum(-v0 * np.sin(j * th))
    p = [np.array([x0[c]]) for c in range(3)]
    v = [np.array([v0]), np.array([0.0]), np.array([vz])]
    traj = []
    for s in range(n):
        p, v = oracle.tracers_push(B, p, v, dt, 1)
        traj.append((p[0][0], p[1][0], p[2][0]))
    traj = np.array(traj)
    assert np.max(np.abs(traj[:, 0] - xs)) <= 1e-13 and np.max(np.abs(traj[:, 1] - ys)) <= 1e-13
    assert np.max(np.abs(traj[:, 2] - (x0[2] + vz * dt * j))) <= 1e-13
    assert abs(v[0][0] - v0 * math.cos(n * th)) <= 1e-13 and abs(v[1][0] + v0 * math.sin(n * th)) <= 1e-13
    # circle: centre from the first three points' closed form, radius r' = v0 dt / (2 sin(th/2)) ~ v0/B0
    r = v0 * dt / (2 * math.sin(th / 2))
    assert abs(r - v0 / B0) <= 1e-4 * v0 / B0
    # centre of the discrete orbit from three of its points, then every point must lie at distance r' from it
    (x1, y1), (x2, y2), (x3, y3) = traj[0, :2], traj[100, :2], traj[250, :2]
    a = np.array([[x2 - x1, y2 - y1], [x3 - x1, y3 - y1]])
    b = 0.5 * np.array([x2 ** 2 - x1 ** 2 + y2 ** 2 - y1 ** 2, x3 ** 2 - x1 ** 2 + y3 ** 2 - y1 ** 2])
    cx, cy = np.linalg.solve(a, b)
    rad = np.hypot(traj[:, 0] - cx, traj[:, 1] - cy)
    assert np.max(np.abs(rad - r)) <= 1e-11


def test_tp8_many_steps_equals_repeated_single_steps_and_wrap():
    N = 8
    rng = np.random.default_rng(3)
    B = [rng.standard_normal((N, N, N)) for _ in range(3)]
    pos = rand_pos(50, rng)
    vel = [rng.standard_normal(50) * 5 for _ in range(3)]      # fast: crosses the box several times
    pa, va = oracle.tracers_push(B, pos, vel, 0.1, 30)
    pb, vb = pos, vel
    for _ in range(30):
        pb, vb = oracle.tracers_push(B, pb, vb, 0.1, 1)
    for c in range(3):
        assert np.array_equal(pa[c], pb[c]) and np.array_equal(va[c], vb[c])
        assert np.all(pa[c] >= 0) and np.all(pa[c] < L)
    # |v| is conserved by every push even in a non-uniform field
    s0 = np.sqrt(sum(v ** 2 for v in vel))
    s1 = np.sqrt(sum(v ** 2 for v in va))
    assert np.max(np.abs(s1 - s0) / s0) <= 1e-13


def test_tp9_attached_to_solver():
    """Tracers attached to the MHD solver: initial velocity = CIC(u) (reading T3); on a uniform state (a stationary
    solution, pin P3) stepping the solver equals pushing in the frozen field; B is taken at the start of each step."""
    N = 16
    rng = np.random.default_rng(9)
    u0 = np.array([0.3, -0.2, 0.1])
    B0 = np.array([0.5, 1.0, -0.7])
    prim = [np.full((N, N, N), 1.3)] + [np.full((N, N, N), u0[c]) for c in range(3)] + [np.full((N, N, N), 2.0)] \
        + [np.full((N, N, N), B0[c]) for c in range(3)]
    o = oracle.Oracle(N, L, 5.0 / 3.0, 0.01, 0.01, 0.02)
    o.set_fields(prim, "primitive")
    pos = rand_pos(20, rng)
    o.tracers_set(pos)
    p0, v0 = o.tracers_get()
    for c in range(3):
        assert np.max(np.abs(v0[c] - u0[c])) <= 1e-14
    o.step(7)
    p1, v1 = o.tracers_get()
    pr, vr = oracle.tracers_push(prim[5:8], pos, [np.full(20, u0[c]) for c in range(3)], 0.02, 7)
    for c in range(3):
        assert np.max(np.abs(p1[c] - pr[c])) <= 1e-12 and np.max(np.abs(v1[c] - vr[c])) <= 1e-12


def test_tp10_time_varying_field_uses_start_of_step_B():
    """Damped standing B wave (pin P7/P12 regime): B_y = b(t) sin x with u = 0 decays as the field steps; the attached
    tracers must see b(t_n) at step n: equals pushing by hand with the oracle's own field history."""
    N = 16
    b = 1e-3
    x = np.arange(N) * L / N
    X = np.broadcast_to(x[None, None, :], (N, N, N))
    prim = [np.ones((N, N, N)), np.zeros((N, N, N)), np.zeros((N, N, N)), np.zeros((N, N, N)), np.ones((N, N, N)),
            np.zeros((N, N, N)), b * np.sin(X), np.zeros((N, N, N))]
    dt = 0.05
    o = oracle.Oracle(N, L, 5.0 / 3.0, 0.0, 0.5, dt)
    o.set_fields(prim, "primitive")
    rng = np.random.default_rng(4)
    pos = rand_pos(10, rng)
    vel = [rng.standard_normal(10) for _ in range(3)]
    o.tracers_set(pos, vel)
    o2 = oracle.Oracle(N, L, 5.0 / 3.0, 0.0, 0.5, dt)
    o2.set_fields(prim, "primitive")
    p, v = pos, vel
    for s in range(5):
        Bn = o2.get_fields("conservative")[5:8]
        p, v = oracle.tracers_push(Bn, p, v, dt, 1)
        o2.step(1)
    o.step(5)
    p1, v1 = o.tracers_get()
    for c in range(3):
        assert np.array_equal(p1[c], p[c]) and np.array_equal(v1[c], v[c])
    # and the field did change (so that the order matters)
    assert abs(o.get_fields()[6].max() / b - 1.0) > 0.05


def test_tp11_particle_on_a_cell_face_and_at_the_box_edge():
    """Edge cases of Eq. 20 that a wrong cell index or weight-to-corner assignment gets wrong: a particle exactly on a grid
    plane takes the value of that plane (weight 1, whichever of the two adjacent cells floor() picks); at x = L - 1 ulp it
    feels plane 0 through the periodic wrap (L255) with weight 1 - O(ulp); at x = 0 it feels plane 0 only."""
    N = 8
    dx = L / N
    ix, iy, iz = idx_grid(N)
    g = 100.0 * iz + 10.0 * iy + ix                     # every grid point has its own value
    # on the faces x = 3 dx, y = 5 dx, z = 2 dx simultaneously: exactly g[2, 5, 3]
    out = oracle.cic([g], [np.array([3 * dx]), np.array([5 * dx]), np.array([2 * dx])])[0]
    assert abs(out[0] - 253.0) <= 1e-12
    # on one face only, half-way inside the cell on the other two axes: mean of the 4 corners of that face
    out = oracle.cic([g], [np.array([3 * dx]), np.array([5.5 * dx]), np.array([2.5 * dx])])[0]
    assert abs(out[0] - (3 + 10 * 5.5 + 100 * 2.5)) <= 1e-12
    # x = L - 1 ulp: in the last cell, next to plane 0 of the opposite boundary
    edge = np.nextafter(L, 0.0)
    for axis in range(3):
        pos = [np.array([0.0]) for _ in range(3)]
        pos[axis] = np.array([edge])
        out = oracle.cic([g], pos)[0]
        assert abs(out[0] - 0.0) <= 1e-12 * 1000, axis          # g[0,0,0] = 0; plane N-1 (value 7, 70 or 700) has weight ~1e-16
    out = oracle.cic([g], [np.array([0.0])] * 3)[0]
    assert out[0] == 0.0


def test_tp12_crossing_zero_with_negative_velocity():
    """Eq. 22 + periodic wrap: a particle that leaves through x = 0 re-enters at x = L - |overshoot|; one that lands on
    x = -tiny (which rounds to L after the shift) is stored as 0, never as L."""
    N = 8
    Z = [np.zeros((N, N, N)) for _ in range(3)]          # B = 0: straight-line motion
    dt = 0.1
    p, v = oracle.tracers_push(Z, [np.array([0.02]), np.array([1.0]), np.array([L - 0.01])],
                               [np.array([-0.5]), np.array([0.0]), np.array([0.3])], dt, 1)
    assert abs(p[0][0] - (L - 0.03)) <= 2e-15 * L and p[1][0] == 1.0 and abs(p[2][0] - 0.02) <= 2e-15 * L
    tiny = 1e-20
    p, v = oracle.tracers_push(Z, [np.array([0.0]), np.array([0.0]), np.array([0.0])],
                               [np.array([-tiny / dt]), np.array([0.0]), np.array([0.0])], dt, 1)
    assert p[0][0] == 0.0
    # many box lengths in one push, both directions
    p, v = oracle.tracers_push(Z, [np.array([1.0]), np.array([1.0]), np.array([1.0])],
                               [np.array([-(5 * L + 0.25) / dt]), np.array([(7 * L + 0.5) / dt]), np.array([0.0])], dt, 1)
    assert abs(p[0][0] - 0.75) <= 1e-13 and abs(p[1][0] - 1.5) <= 1e-13
    for c in range(3):
        assert 0.0 <= p[c][0] < L


def test_tp13_initial_velocity_is_cic_of_the_grid_point_velocity_with_nonuniform_density():
    """Reading T3 (the tracers start with the fluid velocity) on a NON-uniform density: the oracle's own
    attach path (orc_tracers_set with no velocities) interpolates u = m/rho formed AT THE GRID POINTS.  With
    rho = 1.5 + 0.5 cos x, u = (a sin x, b cos 2y, c) every conservative field is band-limited (the projection of
    set_fields leaves it alone), the fields do not depend on z, and Eq. 20 reduces to linear interpolation between the
    neighbouring grid values: v0_x = (1-w_x) a sin x_i + w_x a sin x_{i+1}, v0_y likewise in y, v0_z = c.
    The tempting alternatives differ at the 1e-2 level and fail: CIC(m)/CIC(rho), m without the division, and a rho taken
    from a neighbouring corner (TP9's uniform rho cannot tell these apart)."""
    N = 16
    h = L / N
    a, b, c = 0.7, -0.4, 0.25
    x = np.arange(N) * h
    X = np.broadcast_to(x[None, None, :], (N, N, N))
    Y = np.broadcast_to(x[None, :, None], (N, N, N))
    rho = 1.5 + 0.5 * np.cos(X)
    prim = [rho, a * np.sin(X), b * np.cos(2 * Y), np.full((N, N, N), c), np.full((N, N, N), 2.0),
            np.full((N, N, N), 0.1), np.full((N, N, N), 0.2), np.full((N, N, N), 0.3)]
    o = oracle.Oracle(N, L, 5.0 / 3.0, 0.0, 0.0, 1e-3)
    o.set_fields([np.ascontiguousarray(p) for p in prim], "primitive")
    rng = np.random.default_rng(13)
    pos = rand_pos(200, rng)
    o.tracers_set(pos)
    _, v0 = o.tracers_get()

    def lin(f, s):                       # linear interpolation of the periodic grid function f(x_i) at positions s
        i = np.floor(s / h).astype(int)
        w = s / h - i
        return (1 - w) * f(x[i % N]) + w * f(x[(i + 1) % N])

    want = [lin(lambda t: a * np.sin(t), pos[0]), lin(lambda t: b * np.cos(2 * t), pos[1]), np.full(200, c)]
    for k in range(3):
        assert np.max(np.abs(v0[k] - want[k])) <= 1e-13, k
    # what the wrong readings would give (x component): all are far from `want`
    rho_f = lambda t: 1.5 + 0.5 * np.cos(t)
    m_f = lambda t: rho_f(t) * a * np.sin(t)
    ratio_of_means = lin(m_f, pos[0]) / lin(rho_f, pos[0])
    momentum = lin(m_f, pos[0])
    shifted = lin(lambda t: m_f(t) / rho_f(t + h), pos[0])
    for wrong in (ratio_of_means, momentum, shifted):
        assert np.max(np.abs(wrong - want[0])) >= 5e-3
        assert np.max(np.abs(v0[0] - wrong)) >= 5e-3
