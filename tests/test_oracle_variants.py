"""Pins of the oracle's equation-set variants: the barotropic closure P = C_s^2 rho of
PAPER.md Eq. 5 / Eq. 18 (L63, L192), the ABC forcing rho f of Eq. 18 / L215, and the switched-off equation subsets
of L199 / L205 — against closed forms.  CPU only."""
import math

import numpy as np
import pytest

import oracle
from paper_1810_12707_b200 import inputs

L = 2 * math.pi
G = 5.0 / 3.0


def full(N, v):
    return np.full((N, N, N), float(v))


def test_v1_forcing_on_a_fluid_at_rest():
    """rho = rho0, u = 0, B = 0: R_m = rho0 f_ABC exactly (each component, amplitude, k_f), everything else 0."""
    N, rho0, f0, kf = 16, 1.7, 0.3, 2
    X, Y, Z = inputs.grid(N)
    o = oracle.Oracle(N, L, G, 0.01, 0.01, 1e-3)
    o.set_variant(f0=f0, kf=kf)
    o.set_fields([full(N, rho0), full(N, 0), full(N, 0), full(N, 0), full(N, 1.0), full(N, 0), full(N, 0), full(N, 0)])
    R = o.rhs()
    sh = (N, N, N)
    fx = f0 * np.broadcast_to(np.sin(kf * Z) + np.cos(kf * Y), sh)
    fy = f0 * np.broadcast_to(np.sin(kf * X) + np.cos(kf * Z), sh)
    fz = f0 * np.broadcast_to(np.sin(kf * Y) + np.cos(kf * X), sh)
    for c, f in enumerate((fx, fy, fz)):
        assert np.max(np.abs(R[1 + c] - rho0 * f)) <= 1e-14
    for c in (0, 4, 5, 6, 7):
        assert np.max(np.abs(R[c])) <= 1e-14


def test_v1_forcing_work_term_and_balance_with_viscosity():
    """ABC flow (pin P4) + forcing with f0 = mu k_f^2 U0 and k_f = 1: the viscous term -mu u is cancelled exactly,
    R_m = -grad q, and the energy equation gains the work m.f = f0/U0 |u|^2 (reading V1)."""
    N, U0, mu = 16, 0.5, 0.02
    ux, uy, uz = inputs.abc_flow(N, U0, 1)
    o = oracle.Oracle(N, L, G, mu, 0.0, 1e-3)
    prim = [full(N, 1.0), ux, uy, uz, full(N, 3.0), full(N, 0), full(N, 0), full(N, 0)]
    o.set_fields(prim)
    R0 = o.rhs()
    o.set_variant(f0=mu * U0, kf=1)
    R1 = o.rhs()
    u = [ux, uy, uz]
    for c in range(3):
        assert np.max(np.abs((R1[1 + c] - R0[1 + c]) - mu * u[c])) <= 1e-14      # + rho f = + mu u
    work = mu * (ux * ux + uy * uy + uz * uz)
    assert np.max(np.abs((R1[4] - R0[4]) - work)) <= 1e-14
    for c in (0, 5, 6, 7):
        assert np.array_equal(R1[c], R0[c])


def test_v2_barotropic_pressure_gradient_and_no_energy_equation():
    """P = C_s^2 rho: rho = rho0 + a sin(k x), u = 0, B = 0 -> R_mx = -C_s^2 a k cos(k x), R_E = 0 (whatever E holds)."""
    N, rho0, a, k, cs2 = 32, 2.0, 0.1, 3, 1.44
    X, _, _ = inputs.grid(N)
    rho = rho0 + a * np.broadcast_to(np.sin(k * X), (N, N, N))
    o = oracle.Oracle(N, L, G, 0.0, 0.0, 1e-3)
    o.set_variant(cs2=cs2)
    o.set_fields([rho, full(N, 0), full(N, 0), full(N, 0), full(N, 7.0), full(N, 0), full(N, 0), full(N, 0)])
    R = o.rhs()
    ref = -cs2 * a * k * np.broadcast_to(np.cos(k * X), (N, N, N))
    assert np.max(np.abs(R[1] - ref)) <= 1e-13
    for c in (0, 2, 3, 4, 5, 6, 7):
        assert np.max(np.abs(R[c])) <= 1e-13


def test_v2_barotropic_sound_speed():
    """Linear sound wave under the barotropic closure travels at C_s (not sqrt(gamma P/rho)): phase of rho^(k)."""
    N, k, cs2, amp = 32, 2, 0.81, 1e-6
    cs = math.sqrt(cs2)
    X, _, _ = inputs.grid(N)
    s = np.broadcast_to(np.sin(k * X), (N, N, N))
    dt, n = 2e-3, 200
    o = oracle.Oracle(N, L, G, 0.0, 0.0, dt)
    o.set_variant(cs2=cs2)
    # right-going eigenmode: rho' = amp sin(kx), u_x = cs rho'/rho0
    o.set_fields([1.0 + amp * s, cs * amp * s, full(N, 0), full(N, 0), full(N, 1.0), full(N, 0), full(N, 0), full(N, 0)])
    o.step(n)
    rho = o.get_fields()[0]
    ph = np.angle(np.fft.fft(rho[0, 0, :])[k])            # sin(kx - w t) -> phase -pi/2 - w t
    w = (-(ph + math.pi / 2)) % (2 * math.pi) / (n * dt)
    assert abs(w - k * cs) <= 2e-4 * k * cs


def test_v3_switched_off_equations():
    """Kinematic dynamo (L205 'turn off Eq. 17 and 18'): only B moves and R_B is the full-system R_B; hydrodynamic
    (L199 'turn off Eq. 19'): B frozen."""
    N = 16
    st = inputs.random_smooth_state(N, 5)
    o = oracle.Oracle(N, L, G, 0.01, 0.02, 1e-3)
    o.set_fields(st, "primitive")
    R = o.rhs()
    o.set_variant(evolve=2)
    Rk = o.rhs()
    for c in range(5):
        assert not np.any(Rk[c])
    for c in range(5, 8):
        assert np.array_equal(Rk[c], R[c])
    o.set_variant(evolve=1)
    Rh = o.rhs()
    for c in range(5):
        assert np.array_equal(Rh[c], R[c])
    for c in range(5, 8):
        assert not np.any(Rh[c])
    # kinematic: the velocity field stays what it was
    o.set_variant(evolve=2)
    U0 = o.get_fields()
    o.step(5)
    U1 = o.get_fields()
    for c in range(5):
        assert np.array_equal(U0[c], U1[c])
    assert not np.array_equal(U0[5], U1[5])


# ---- V4: the viscous terms of Eq. 11-12 (2 nu rho S with the traceless rate of strain of Eq. 3-4) -----------------------
def _visc_part(N, prim, nu):
    """R(stress form, nu) - R(nu = 0): the viscous terms alone."""
    o = oracle.Oracle(N, L, G, nu, 0.0, 1e-3)
    o.set_stress(True)
    o.set_fields(prim)
    R1 = o.rhs()
    o0 = oracle.Oracle(N, L, G, 0.0, 0.0, 1e-3)
    o0.set_fields(prim)
    R0 = o0.rhs()
    return [a - b for a, b in zip(R1, R0)]


def test_v4_shear_and_compression_closed_forms():
    N, k, a, rho0, nu = 16, 2, 0.3, 1.7, 0.05
    X, _, _ = inputs.grid(N)
    s, c = (np.broadcast_to(f(k * X), (N, N, N)) for f in (np.sin, np.cos))
    s2, c2 = (np.broadcast_to(f(2 * k * X), (N, N, N)) for f in (np.sin, np.cos))
    z = full(N, 0)
    # shear u = (0, a sin kx, 0): S_xy = a k cos(kx)/2, theta = 0
    D = _visc_part(N, [full(N, rho0), z, a * s, z, full(N, 2.0), z, z, z], nu)
    assert np.max(np.abs(D[2] + nu * rho0 * a * k * k * s)) <= 1e-14
    assert np.max(np.abs(D[4] - nu * rho0 * a * a * k * k * c2)) <= 1e-14
    for f in (0, 1, 3, 5, 6, 7):
        assert np.max(np.abs(D[f])) <= 1e-14
    # compression u = (a sin kx, 0, 0): S_xx = theta - theta/3 = (2/3) a k cos kx  -> the factor 4/3 of the bulk part
    D = _visc_part(N, [full(N, rho0), a * s, z, z, full(N, 2.0), z, z, z], nu)
    assert np.max(np.abs(D[1] + (4.0 / 3.0) * nu * rho0 * a * k * k * s)) <= 1e-14
    assert np.max(np.abs(D[4] - (4.0 / 3.0) * nu * rho0 * a * a * k * k * c2)) <= 1e-14
    # S_yy = S_zz = -theta/3 do not act on a flow that depends on x only
    for f in (0, 2, 3, 5, 6, 7):
        assert np.max(np.abs(D[f])) <= 1e-14


def test_v4_density_sits_inside_the_divergence():
    """rho = rho0 + r cos kx, u = (0, a sin kx, 0): d_x(nu rho a k cos kx) = -nu a k^2 (rho0 sin kx + r sin 2kx)."""
    N, k, a, rho0, r, nu = 16, 2, 0.3, 1.7, 0.4, 0.05
    X, _, _ = inputs.grid(N)
    s, c = (np.broadcast_to(f(k * X), (N, N, N)) for f in (np.sin, np.cos))
    s2 = np.broadcast_to(np.sin(2 * k * X), (N, N, N))
    z = full(N, 0)
    D = _visc_part(N, [rho0 + r * c, z, a * s, z, full(N, 2.0), z, z, z], nu)
    assert np.max(np.abs(D[2] + nu * a * k * k * (rho0 * s + r * s2))) <= 1e-14


def test_v4_abc_flow_against_the_laplacian_form():
    """Solenoidal Beltrami flow, rho = 1: div(2 nu S) = nu lap u = -nu u (as R3's form), while the work term is
    d_j(2 nu u_i S_ij) = nu (lap q + div(u.grad u)) = 2 nu lap q, twice R3's mu lap q."""
    N, U0, nu = 16, 0.5, 0.02
    ux, uy, uz = inputs.abc_flow(N, U0, 1)
    z = full(N, 0)
    D = _visc_part(N, [full(N, 1.0), ux, uy, uz, full(N, 3.0), z, z, z], nu)
    for cidx, u in enumerate((ux, uy, uz)):
        assert np.max(np.abs(D[1 + cidx] + nu * u)) <= 1e-14
    q = 0.5 * (ux * ux + uy * uy + uz * uz)
    lap_q = -2.0 * (q - 1.5 * U0 * U0)                 # pin P4
    assert np.max(np.abs(D[4] - 2 * nu * lap_q)) <= 1e-14
