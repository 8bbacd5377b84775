"""Seeded synthetic initial fields for the spin-2 QLGA workloads.

This module only *generates inputs*: closed-form fields of the paper's runs
(§III-§VI) sampled on a lattice, plus seeded noise.  It contains none
of the method's arithmetic (no collide / stream / interaction / observables),
imports only numpy, and is the one module both the CPU oracle's tests and the
CUDA path's tests/bench draw their arrays from.

Conventions:
  * channel index j = 0..4  <->  m_f = +2, +1, 0, -1, -2
  * psi has shape (5, Ny, Nx) complex128, x fastest; 1D lattices have Ny = 1
  * amplitudes/densities of BASELINE.json are in the paper's unscaled solution
    units; the lattice field is psi_lat(r) = a * psi_sol(a r), a = 1/width
    (the paper's own scaling psi_m -> sqrt(gamma) psi_m, gamma = a^2,
    PAPER.md:1005-1022, eq. 105-106).

Every generator takes the lattice size as an argument so that parity tests can
run the same recipe on lattices the oracle finishes in seconds.
"""
from __future__ import annotations

import dataclasses
import numpy as np

M_VALUES = (2, 1, 0, -1, -2)


def j_of_m(m: int) -> int:
    """Channel index of Zeeman level m (m=+2 -> 0 ... m=-2 -> 4)."""
    return 2 - m


@dataclasses.dataclass
class Workload:
    name: str
    ndim: int
    dims: tuple          # (Nx, Ny); Ny = 1 in 1D
    couplings: tuple     # (c0, c1, c2) = the paper's (g0, g1, g2), eq. (32)-(34)
    steps: int           # BASELINE.json step count for the full-size config
    psi: np.ndarray      # (5, Ny, Nx) complex128
    note: str = ""


def seed_for(config_number: int) -> int:
    return 1000 + int(config_number)


# --------------------------------------------------------------------------
# closed-form profiles
# --------------------------------------------------------------------------
def sech(x):
    with np.errstate(over="ignore"):          # cosh overflows to inf far from the soliton: sech -> 0
        return 1.0 / np.cosh(x)


def pade_profile(s, a1=11.0 / 32.0, b1=1.0 / 3.0, a2=11.0 / 384.0):
    """Radial Pade vortex amplitude of eq. (86), PAPER.md:737:
    sqrt((a2 s^4 + a1 s^2) / (a2 s^4 + b1 s^2 + 1)).  The default coefficients
    are the scalar Pade vortex that Tables III/IV reduce to at E = g."""
    s2 = s * s
    s4 = s2 * s2
    return np.sqrt((a2 * s4 + a1 * s2) / (a2 * s4 + b1 * s2 + 1.0))


def vortex_factor(X, Y, cx, cy, a, winding):
    """P(a |r - c|) * exp(i * winding * theta) for one vortex at (cx, cy)."""
    dx = X - cx
    dy = Y - cy
    r = np.sqrt(dx * dx + dy * dy)
    theta = np.arctan2(dy, dx)
    return pade_profile(a * r) * np.exp(1j * winding * theta)


def _grid(nx, ny):
    x = np.arange(nx, dtype=np.float64)
    y = np.arange(ny, dtype=np.float64)
    return np.meshgrid(x, y, indexing="xy")  # shapes (ny, nx)


# --------------------------------------------------------------------------
# the five BASELINE.json configurations (sizes overridable)
# --------------------------------------------------------------------------
def config1(L=1024, width=32.0, amplitude=1.0):
    """1D stationary bright soliton in m_f=+2 (Table I row 1 at E=-2,
    PAPER.md:380, 533-542): psi_{+2} = A c a sech(a (x - L/2))."""
    c0, c1, c2 = -1.0, -0.5, 0.2
    a = 1.0 / width
    c = np.sqrt(2.0 / abs(c0 + 4.0 * c1))
    x = np.arange(L, dtype=np.float64)
    psi = np.zeros((5, 1, L), dtype=np.complex128)
    psi[j_of_m(2), 0] = amplitude * c * a * sech(a * (x - L / 2))
    return Workload("cfg1_bright_1d", 1, (L, 1), (c0, c1, c2), 1000, psi)


def config2(L=65536, width=64.0, kick=0.05, centres=None):
    """1D, two kicked bright solitons in m_f=+1 and m_f=-1 (Table I rows 3-4).
    `centres=(xa, xb)` overrides L/4, 3L/4 (used for the real-collision variant)."""
    c0, c1, c2 = -1.0, -0.5, 0.2
    a = 1.0 / width
    c = np.sqrt(2.0 / abs(c0 + c1))
    xa, xb = (L / 4, 3 * L / 4) if centres is None else centres
    x = np.arange(L, dtype=np.float64)
    psi = np.zeros((5, 1, L), dtype=np.complex128)
    psi[j_of_m(1), 0] = 1.0 * c * a * sech(a * (x - xa)) * np.exp(+1j * kick * x)
    psi[j_of_m(-1), 0] = 0.8 * c * a * sech(a * (x - xb)) * np.exp(-1j * kick * x)
    return Workload("cfg2_bright_pair_1d", 1, (L, 1), (c0, c1, c2), 50000, psi)


def config3(L=1 << 22, healing=16.0, sigma=1e-3, seed=None):
    """1D dark-soliton pair (eq. 84) in m_f=0 on a background in
    m_f=+-2, plus seeded complex Gaussian noise on all five channels."""
    c0, c1, c2 = 1.0, 0.3, -0.1
    a = 1.0 / healing
    rng = np.random.default_rng(seed_for(3) if seed is None else seed)
    x = np.arange(L, dtype=np.float64)
    T = np.tanh(a * (x - L / 4)) * np.tanh(a * (3 * L / 4 - x))
    psi = np.zeros((5, 1, L), dtype=np.complex128)
    psi[j_of_m(0), 0] = a * T
    psi[j_of_m(2), 0] = a * np.sqrt(0.5)
    psi[j_of_m(-2), 0] = a * np.sqrt(0.5)
    for j in range(5):
        n_re = rng.standard_normal(L)
        n_im = rng.standard_normal(L)
        psi[j, 0] += a * sigma * (n_re + 1j * n_im) / np.sqrt(2.0)
    return Workload("cfg3_dark_pair_noise_1d", 1, (L, 1), (c0, c1, c2), 20000, psi)


def config4(L=2048, core=8.0):
    """2D Pade-vortex quadrupole: winding +-1 in m_f=+-2 on
    a uniform background in all five channels."""
    c0, c1, c2 = 1.0, 0.3, -0.1
    a = 1.0 / core
    X, Y = _grid(L, L)
    V = np.ones((L, L), dtype=np.complex128)
    for cx, cy, w in ((L / 4, L / 4, +1), (3 * L / 4, L / 4, -1),
                      (L / 4, 3 * L / 4, -1), (3 * L / 4, 3 * L / 4, +1)):
        V *= vortex_factor(X, Y, cx, cy, a, w)
    psi = np.empty((5, L, L), dtype=np.complex128)
    psi[j_of_m(2)] = a * V
    psi[j_of_m(-2)] = a * np.conj(V)
    psi[j_of_m(1)] = a
    psi[j_of_m(0)] = a
    psi[j_of_m(-1)] = a
    return Workload("cfg4_quadrupole_2d", 2, (L, L), (c0, c1, c2), 10000, psi)


def config5(L=8192, core=12.0, kick=0.03, sigma=1e-3, spacing=96.0, offset=256.0,
            seed=None):
    """2D, two Pade vortex-antivortex dipoles in m_f=+1 and m_f=-2 kicked toward
    each other along y, uniform background elsewhere, seeded phase noise.
    For reduced lattices pass smaller `spacing`/`offset`."""
    c0, c1, c2 = 1.0, 0.3, -0.1
    a = 1.0 / core
    rng = np.random.default_rng(seed_for(5) if seed is None else seed)
    X, Y = _grid(L, L)

    def dipole(cx, cy):
        h = spacing / 2.0
        return (vortex_factor(X, Y, cx + h, cy, a, +1) *
                vortex_factor(X, Y, cx - h, cy, a, -1))

    psi = np.empty((5, L, L), dtype=np.complex128)
    psi[j_of_m(1)] = a * dipole(L / 2, L / 2 - offset) * np.exp(+1j * kick * Y)
    psi[j_of_m(-2)] = a * dipole(L / 2, L / 2 + offset) * np.exp(-1j * kick * Y)
    psi[j_of_m(2)] = a
    psi[j_of_m(0)] = a
    psi[j_of_m(-1)] = a
    for j in range(5):
        psi[j] *= np.exp(1j * sigma * rng.standard_normal((L, L)))
    return Workload("cfg5_dipoles_2d", 2, (L, L), (c0, c1, c2), 5000, psi)


def config3d(L=256, core=12.0, kick=0.03, sigma=1e-3, spacing=48.0, seed=None):
    """3D workload for SURVEY.md section 8(f) row 3 (the paper quotes "a three dimensional cube of
    512 sites" as capacity, and no 3D run): config 5's recipe extruded along z --
    a straight Pade vortex-antivortex line pair in m_f=+1 kicked along y, uniform background in
    the other channels, seeded phase noise.  psi: (5, L, L, L)."""
    c0, c1, c2 = 1.0, 0.3, -0.1
    a = 1.0 / core
    rng = np.random.default_rng(seed_for(6) if seed is None else seed)
    X, Y = _grid(L, L)
    h = spacing / 2.0
    D = (vortex_factor(X, Y, L / 2 + h, L / 2, a, +1) * vortex_factor(X, Y, L / 2 - h, L / 2, a, -1))
    plane = a * D * np.exp(1j * kick * Y)
    psi = np.empty((5, L, L, L), dtype=np.complex128)
    psi[:] = a
    psi[j_of_m(1)] = plane[None, :, :]
    for j in range(5):
        psi[j] *= np.exp(1j * sigma * rng.standard_normal((L, L, L)))
    return Workload("cfg3d_vortex_lines", 3, (L, L, L), (c0, c1, c2), 1000, psi)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


# --------------------------------------------------------------------------
# generic seeded fields for unit / parity tests
# --------------------------------------------------------------------------
def random_field(dims, seed, amplitude=0.1):
    """Smooth-free seeded complex Gaussian field on all five channels."""
    nx, ny = dims
    rng = np.random.default_rng(seed)
    re = rng.standard_normal((5, ny, nx))
    im = rng.standard_normal((5, ny, nx))
    return amplitude * (re + 1j * im) / np.sqrt(2.0)


def random_spinor_state(dims, seed, amplitude=0.1):
    """Seeded random full spinor state q of shape (5, 2, Ny, Nx) (dims = (Nx, Ny)) or
    (5, 2, Nz, Ny, Nx) (dims = (Nx, Ny, Nz)) complex128, both spinor components
    independent, i.e. with an antisymmetric part."""
    shape = (5, 2) + tuple(reversed(tuple(dims)))
    rng = np.random.default_rng(seed)
    re = rng.standard_normal(shape)
    im = rng.standard_normal(shape)
    return amplitude * (re + 1j * im) / np.sqrt(2.0)


def smooth_random_field(dims, seed, amplitude=0.1, kmax=3):
    """Seeded band-limited field: a few low Fourier modes per channel."""
    nx, ny = dims
    rng = np.random.default_rng(seed)
    X, Y = _grid(nx, ny)
    psi = np.zeros((5, ny, nx), dtype=np.complex128)
    for j in range(5):
        for kx in range(-kmax, kmax + 1):
            for ky in (range(-kmax, kmax + 1) if ny > 1 else (0,)):
                coef = (rng.standard_normal() + 1j * rng.standard_normal())
                psi[j] += coef * np.exp(2j * np.pi * (kx * X / nx + ky * Y / max(ny, 1)))
    psi *= amplitude / np.sqrt(np.mean(np.abs(psi) ** 2) * 5.0)
    return psi


def table1_state(row, E, couplings, free=(0.3, 0.2)):
    """Thomas-Fermi coefficient vector (c_2, c_1, c_0, c_-1, c_-2) of Table I
     for the rows with printed numeric coefficients.  `free`
    supplies the free parameters (c_2, c_1) of rows 11, 12, 16.  The formulas are
    read from tests/golden/table1.json by the tests; this helper is the plain
    transcription used to build workloads (e.g. bright-soliton amplitudes)."""
    g0, g1, g2 = couplings
    s = np.sqrt
    c2f, c1f = free
    if row == 1:
        c = (s(E / (g0 + 4 * g1)), 0, 0, 0, 0)
    elif row == 2:
        c = (0, 0, 0, 0, s(E / (g0 + 4 * g1)))
    elif row == 3:
        c = (0, s(E / (g0 + g1)), 0, 0, 0)
    elif row == 4:
        c = (0, 0, 0, s(E / (g0 + g1)), 0)
    elif row == 5:
        c = (0, 0, s(5 * E / (5 * g0 + g2)), 0, 0)
    elif row == 6:
        v = s(5 * E / (10 * g0 + 2 * g2))
        c = (v, 0, 0, 0, v)
    elif row == 7:
        v = s(5 * E / (10 * g0 + 2 * g2))
        c = (0, v, 0, v, 0)
    elif row == 8:
        c = (s(E / (3 * g0)), 0, 0, s(2 * E / (3 * g0)), 0)
    elif row == 9:
        c = (0, s(2 * E / (3 * g0)), 0, 0, s(E / (3 * g0)))
    elif row == 10:
        c = (s(E / (4 * g0)), 0, s(E / (2 * g0)), 0, -s(E / (4 * g0)))
    elif row == 11:
        c = (c2f, 0, s((5 * E - 10 * c2f**2 * g0 - 2 * c2f**2 * g2) / (5 * g0 + g2)), 0, c2f)
    elif row == 12:
        c = (0, c1f, s((5 * E - 10 * c1f**2 * g0 - 2 * c1f**2 * g2) / (5 * g0 + g2)), -c1f, 0)
    elif row == 13:
        v = s(E / (4 * g0 + 4 * g1))
        c = (v, v, 0, -v, -v)
    elif row == 14:
        c = (s(3 * E / (16 * g0)), s(E / (4 * g0)), -s(E / (8 * g0)),
             s(E / (4 * g0)), s(3 * E / (16 * g0)))
    elif row == 15:
        u = s(E / (g0 + 4 * g1))
        c = (u / 4, u / 2, 0.5 * s(3 * E / (2 * g0 + 8 * g1)), u / 2, u / 4)
    elif row == 16:
        c = (c2f, c1f,
             s((5 * E - (c2f**2 + c1f**2) * (10 * g0 + 2 * g2)) / (5 * g0 + g2)),
             -c1f, c2f)
    else:
        raise ValueError("Table I row must be 1..16")
    return np.array(c, dtype=np.float64)


# --------------------------------------------------------------------------
# kicked solitons of the dispersion experiment (Fig. 5) and the paper's prediction
# --------------------------------------------------------------------------
def kicked_soliton(kind, row, couplings, L, k, n_kick):
    """psi[5][1][L]: Table I coefficients of `row` (E = -2 bright / +2 dark) times the
    soliton profile of inverse width k times exp(i 2 pi n x / L)."""
    x = np.arange(L, dtype=np.float64)
    if kind == "bright":
        prof = k * sech(k * (x - L / 2))
        cm = table1_state(row, -2.0, couplings)
    elif kind == "dark":
        prof = k * np.tanh(k * (x - L / 4)) * np.tanh(k * (3 * L / 4 - x))
        cm = table1_state(row, 2.0, couplings)
    else:
        raise ValueError(kind)
    psi = np.zeros((5, 1, L), dtype=np.complex128)
    psi[:, 0, :] = cm[:, None] * prof * np.exp(2j * np.pi * n_kick * x / L)
    return psi


def predicted_energy(kind, k, p):
    """The paper's dispersion relations: E = p^2 - k^2 (bright, eq. 74), E = p^2 + 2 k^2
    (dark)."""
    return p * p - k * k if kind == "bright" else p * p + 2.0 * k * k


def kicked_quadrupole(L, core=8.0, n_kick=0, axis="x", couplings=(1.0, 0.3, -0.1), m=2, offset=0.5):
    """Single-channel Pade-vortex quadrupole in channel m with the paper's kick
    exp(i 2 pi n x / L) (or y; Figs. 15-16): psi_m = a V(r) e^{i 2 pi n x/L} / sqrt(g),
    g = c0 + 4 c1 (m = +-2), c0 + c1 (m = +-1) or c0 + c2/5 (m = 0) (Table I rows 1-5 at E = 1), a = 1/core.
    A stationary state of the paper for n = 0; kicked, the whole pattern drifts at 2 p = 4 pi n / L sites per
    step (eq. 71; units pinned by the printed drift times).  The vortex centres sit at
    (L/4, 3L/4) + offset so that no zero of the field falls on a lattice site."""
    c0, c1, c2 = couplings
    g = {2: c0 + 4 * c1, 1: c0 + c1, 0: c0 + c2 / 5.0}[abs(m)]
    a = 1.0 / core
    X, Y = _grid(L, L)
    lo, hi = L / 4 + offset, 3 * L / 4 + offset
    V = np.ones((L, L), dtype=np.complex128)
    for cx, cy, w in ((lo, lo, +1), (hi, lo, -1), (lo, hi, -1), (hi, hi, +1)):
        V *= vortex_factor(X, Y, cx, cy, a, w)
    psi = np.zeros((5, L, L), dtype=np.complex128)
    psi[j_of_m(m)] = a / np.sqrt(g) * V * np.exp(2j * np.pi * n_kick * (X if axis == "x" else Y) / L)
    return Workload("kicked_quadrupole_2d", 2, (L, L), tuple(couplings), 0, psi)
