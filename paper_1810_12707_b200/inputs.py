"""Seeded synthetic initial conditions — shared by the oracle and the CUDA path.

This module holds NONE of the method's arithmetic (no RHS, no derivative operator, no time step): it
only manufactures the primitive fields (rho, ux, uy, uz, P, Bx, By, Bz) at t = 0 that are handed, bit
for bit, to both `oracle/` and `libmhd` through their `set_fields(kind=primitive)` entry points.

The paper measures on its own runs, not on a public data set (Sec. VIII), and prints the
ABC-flow setup of its dynamo runs (Sec. V-B: A=B=C=1, k_f=1, U0=1, rho0=1); the configs
here are the ones BASELINE.json lists, built from those closed forms plus a random-phase solenoidal
field generator.  numpy's FFT is used here only to synthesise inputs (allowed for the harness; it is
never on the product path).

Array convention everywhere in this repo: `f[z][y][x]`, x fastest, x_i = i*L/N.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

GAMMA = 5.0 / 3.0
TWO_PI = 2.0 * math.pi
_MASK64 = (1 << 64) - 1


# ----------------------------------------------------------------------------------------------------
# counter-based phases: independent of N and of loop order
# ----------------------------------------------------------------------------------------------------
def splitmix64(x: int) -> int:
    """One splitmix64 output step (Steele/Lea/Flood mixer) on a 64-bit integer."""
    x = (x + 0x9E3779B97F4A7C15) & _MASK64
    z = x
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK64
    return z ^ (z >> 31)


def phase(seed: int, stream: int, comp: int, nx: int, ny: int, nz: int) -> float:
    """phi = 2*pi*(h >> 11)/2^53 with h chained over (seed, stream, comp, nx, ny, nz)."""
    h = 0
    for v in (seed, stream, comp, nx, ny, nz):
        h = splitmix64(h ^ (v & 0xFFFFFFFF))
    return TWO_PI * float(h >> 11) / float(1 << 53)


def half_space_modes(kmin: float, kmax: float):
    """One of each +-n pair with kmin <= |n| <= kmax: nx>0, or nx=0 and ny>0, or nx=ny=0 and nz>0."""
    m = int(math.floor(kmax))
    out = []
    for nx in range(0, m + 1):
        for ny in range(-m, m + 1):
            for nz in range(-m, m + 1):
                if nx == 0 and (ny < 0 or (ny == 0 and nz <= 0)):
                    continue
                r2 = nx * nx + ny * ny + nz * nz
                if kmin * kmin <= r2 <= kmax * kmax:
                    out.append((nx, ny, nz))
    return out


def random_solenoidal(N: int, kmin: float, kmax: float, p: float, seed: int, stream: int, rms: float):
    """G(kmin,kmax,p,seed,stream,rms): V = curl A, A_c(x) = sum_n |n|^p cos(n.x + phi_{n,c}), scaled to rms.

    Returns (Vx, Vy, Vz), each float64 [N][N][N] (z,y,x).  L = 2*pi so wavenumber == integer mode.
    Built spectrally (V^ = i n x A^): exactly solenoidal and band-limited to |n| <= kmax.
    """
    if kmax >= N // 2:
        raise ValueError("kmax must stay below the Nyquist mode")
    modes = half_space_modes(kmin, kmax)
    nh = N // 2 + 1
    scale = 0.5 * float(N) ** 3  # cos(n.x+phi) = (e^{i(n.x+phi)} + c.c.)/2 ; the inverse FFT divides by N^3
    entries = [[], [], []]       # per component: ((iz, iy, ix), value) of the half spectrum
    for (nx, ny, nz) in modes:
        amp = (nx * nx + ny * ny + nz * nz) ** (0.5 * p)
        a = [amp * complex(math.cos(ph), math.sin(ph)) * scale
             for ph in (phase(seed, stream, c, nx, ny, nz) for c in range(3))]
        # V^ = i n x A^
        v = (1j * (ny * a[2] - nz * a[1]), 1j * (nz * a[0] - nx * a[2]), 1j * (nx * a[1] - ny * a[0]))
        for c in range(3):
            entries[c].append(((nz % N, ny % N, nx), v[c]))
            if nx == 0:  # the kx = 0 plane holds both members of the pair
                entries[c].append((((-nz) % N, (-ny) % N, 0), v[c].conjugate()))
    V = [_synthesise(N, nh, entries[c]) for c in range(3)]
    ms = float(np.mean(V[0] ** 2) + np.mean(V[1] ** 2) + np.mean(V[2] ** 2))
    f = rms / math.sqrt(ms)
    for v in V:
        v *= f
    return tuple(V)


def _synthesise(N: int, nh: int, entries):
    """Real field [N][N][N] from a sparse list of half-spectrum entries (inverse real FFT, input synthesis only).
    Large grids use torch's FFT on the GPU when one is present (minutes -> seconds at 1024^3); the harness may use
    a library FFT, the product path never does."""
    if N >= 512:
        try:
            import torch
            if torch.cuda.is_available():
                Vh = torch.zeros((N, N, nh), dtype=torch.complex128, device="cuda")
                for (iz, iy, ix), val in entries:
                    Vh[iz, iy, ix] += val
                out = torch.fft.irfftn(Vh, s=(N, N, N), dim=(0, 1, 2))
                del Vh
                res = out.cpu().numpy()
                del out
                torch.cuda.empty_cache()
                return res
        except ImportError:
            pass
    Vh = np.zeros((N, N, nh), dtype=np.complex128)
    for (iz, iy, ix), val in entries:
        Vh[iz, iy, ix] += val
    return np.ascontiguousarray(np.fft.irfftn(Vh, s=(N, N, N), axes=(0, 1, 2)))


# ----------------------------------------------------------------------------------------------------
# closed-form flows
# ----------------------------------------------------------------------------------------------------
def grid(N: int, L: float = TWO_PI):
    """(X, Y, Z) broadcastable coordinate arrays for the [z][y][x] layout."""
    c = np.arange(N, dtype=np.float64) * (L / N)
    return c[None, None, :], c[None, :, None], c[:, None, None]


def abc_flow(N: int, U0: float = 1.0, k: int = 1):
    """ABC flow with A=B=C=1: u = U0 (sin kz + cos ky, sin kx + cos kz, sin ky + cos kx)."""
    X, Y, Z = grid(N)
    shape = (N, N, N)
    ux = U0 * np.broadcast_to(np.sin(k * Z) + np.cos(k * Y), shape)
    uy = U0 * np.broadcast_to(np.sin(k * X) + np.cos(k * Z), shape)
    uz = U0 * np.broadcast_to(np.sin(k * Y) + np.cos(k * X), shape)
    return tuple(np.ascontiguousarray(a) for a in (ux, uy, uz))


# ----------------------------------------------------------------------------------------------------
# the configs of BASELINE.json / SURVEY.md §8(d)
# ----------------------------------------------------------------------------------------------------
@dataclass
class Config:
    name: str
    N: int
    L: float
    gamma: float
    mu: float
    eta: float
    dt: float
    nsteps: int
    prim: list = field(repr=False)  # [rho, ux, uy, uz, P, Bx, By, Bz], each float64 [N][N][N]


def _full(N, v):
    return np.full((N, N, N), v, dtype=np.float64)


def config1(N: int = 32) -> Config:
    """32^3: rho=1, P=1, ABC velocity x0.1, seed B = G(1,4,p=0,seed 1,stream 0,rms 1e-3)."""
    ux, uy, uz = abc_flow(N, 0.1)
    bx, by, bz = random_solenoidal(N, 1, 4, 0.0, 1, 0, 1e-3)
    return Config("config1_abc_seedB", N, TWO_PI, GAMMA, 0.01, 0.01, 1e-4, 10,
                  [_full(N, 1.0), ux, uy, uz, _full(N, 1.0), bx, by, bz])


def config2(N: int = 64) -> Config:
    """64^3 3-D Orszag-Tang type: rho=gamma^2, P=gamma, u=(-sin y, sin x, 0)(1+0.1 sin z), B=(-sin y, sin 2x, 0)."""
    X, Y, Z = grid(N)
    shape = (N, N, N)
    mod = 1.0 + 0.1 * np.sin(Z)
    ux = np.ascontiguousarray(np.broadcast_to(-np.sin(Y) * mod, shape))
    uy = np.ascontiguousarray(np.broadcast_to(np.sin(X) * mod, shape))
    bx = np.ascontiguousarray(np.broadcast_to(-np.sin(Y), shape))
    by = np.ascontiguousarray(np.broadcast_to(np.sin(2 * X), shape))
    return Config("config2_orszag_tang3d", N, TWO_PI, GAMMA, 5e-3, 5e-3, 5e-4, 200,
                  [_full(N, GAMMA ** 2), ux, uy, _full(N, 0.0), _full(N, GAMMA), bx, by, _full(N, 0.0)])


def config3(N: int = 128, kmax: int = 8, seed: int = 3, mu: float = 2e-3, dt: float = 2e-4,
            nsteps: int = 500) -> Config:
    """Decaying turbulence: solenoidal random-phase u and B, E(k) ~ k^-5/3 (p = -17/6), rms 0.5, Mach 0.3."""
    p = -17.0 / 6.0
    ux, uy, uz = random_solenoidal(N, 1, kmax, p, seed, 0, 0.5)
    bx, by, bz = random_solenoidal(N, 1, kmax, p, seed, 1, 0.5)
    P0 = 0.25 / (GAMMA * 0.09)
    return Config("config3_decaying_turbulence", N, TWO_PI, GAMMA, mu, mu, dt, nsteps,
                  [_full(N, 1.0), ux, uy, uz, _full(N, P0), bx, by, bz])


def config45(N: int = 256) -> Config:
    """256^3 / 512^3 ABC kinematic-to-nonlinear dynamo: ABC amplitude 1, seed B rms 1e-4 (seed 5), Mach 0.1."""
    ux, uy, uz = abc_flow(N, 1.0)
    bx, by, bz = random_solenoidal(N, 1, 4, 0.0, 5, 0, 1e-4)
    P0 = 1.0 / (GAMMA * 0.01)
    return Config("config45_abc_dynamo", N, TWO_PI, GAMMA, 1e-3, 1e-3, 1e-4, 100,
                  [_full(N, 1.0), ux, uy, uz, _full(N, P0), bx, by, bz])


def config6(N: int = 1024) -> Config:
    """1024^3 out-of-core: config-3 style turbulence with modes 1 <= |n| <= 16 (seed 6)."""
    c = config3(N, kmax=16, seed=6, mu=5e-4, dt=5e-5, nsteps=10)
    c.name = "config6_out_of_core"
    return c


def by_name(name: str, N: int | None = None) -> Config:
    table = {"1": (config1, 32), "2": (config2, 64), "3": (config3, 128), "4": (config45, 256),
             "5": (config45, 512), "6": (config6, 1024)}
    fn, n0 = table[str(name)]
    return fn(N if N is not None else n0)


def random_smooth_state(N: int, seed: int, kmax: int = 3, amp: float = 0.2):
    """A generic smooth, strictly positive primitive state for parity tests (not a paper config):
    every field is 'mean + amp * band-limited random-phase sum', B is solenoidal."""
    s = [random_solenoidal(N, 1, kmax, -1.0, seed, k, 1.0) for k in range(4)]
    rho = 1.0 + amp * s[0][0] / np.max(np.abs(s[0][0]))
    P = 1.0 + amp * s[0][1] / np.max(np.abs(s[0][1]))
    ux, uy, uz = (amp * a for a in s[1])
    bx, by, bz = random_solenoidal(N, 1, kmax, -1.0, seed, 7, amp)
    # a non-solenoidal velocity part so that div u != 0 is exercised too
    ux = ux + 0.5 * amp * s[2][0]
    return [np.ascontiguousarray(a, dtype=np.float64) for a in (rho, ux, uy, uz, P, bx, by, bz)]
