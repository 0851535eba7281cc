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
