"""Pins of the oracle's full time step: unitarity, closed-form soliton
eigenstates (§III.C, eq. 67-83), Galilean drift (eq. 71), the printed
drift times, exact covariances of the discrete map, and the
double vs long-double builds.  CPU only; sized to run in about a minute."""
import numpy as np
import pytest
from scipy.linalg import expm

from paper_1907_12834_b200 import inputs
from conftest import rel_l2, norm2, table1_coeffs, load_golden


def _centre(dens):
    """Circular centre of mass of a 1D density on a periodic lattice."""
    L = dens.size
    ang = 2 * np.pi * np.arange(L) / L
    return (np.angle(np.sum(dens * np.exp(1j * ang))) % (2 * np.pi)) * L / (2 * np.pi)


@pytest.mark.parametrize("order", [0, 1])
def test_unitarity_norm_q_1e13_per_1000_steps(oracle, order):
    # north_star pin: total norm conserved to 1e-13 relative per 1000 steps (fp64).
    # Multi-channel state with an antisymmetric part so every operator is exercised.
    c = (1.0, 0.3, -0.1)
    psi = inputs.smooth_random_field((96, 1), seed=4, amplitude=0.08)
    q0 = oracle.split_psi(psi) + inputs.random_spinor_state((96, 1), seed=6, amplitude=1e-3)
    qn = oracle.step(q0, 1, c, order, 1000)
    assert abs(norm2(qn) / norm2(q0) - 1) < 1e-13
    # norm of psi alone is only approximately conserved (leakage into q1 - q2)
    n_psi0 = norm2(oracle.psi_of_q(q0)); n_psi = norm2(oracle.psi_of_q(qn))
    assert abs(n_psi / n_psi0 - 1) < 1e-2


def test_unitarity_2d(oracle):
    c = (1.0, 0.3, -0.1)
    psi = inputs.smooth_random_field((12, 10), seed=5, amplitude=0.1)
    q0 = oracle.split_psi(psi) + inputs.random_spinor_state((12, 10), seed=7, amplitude=1e-3)
    for order in (0, 1):
        qn = oracle.step(q0, 2, c, order, 200)
        assert abs(norm2(qn) / norm2(q0) - 1) < 2e-14


@pytest.mark.parametrize("row", [1, 5, 8, 13])        # the four states of Fig. 2
def test_bright_soliton_is_stationary_with_phase_k2(oracle, row):
    # eq. (67), (71) with p = 0: psi_m = c_m k sech(kx) with the
    # Table I coefficients at E = -2 keeps |psi|^2 and rotates as exp(+i k^2 t).
    c = (-1.0, -0.5, 0.2)
    L, k = 512, 1.0 / 16
    cm = table1_coeffs(row, -2.0, c)
    x = np.arange(L)
    prof = k * inputs.sech(k * (x - L / 2))
    psi = np.zeros((5, 1, L), complex); psi[:, 0, :] = cm[:, None] * prof
    q0 = oracle.split_psi(psi)
    n = 400
    qn = oracle.step(q0, 1, c, 1, n)
    pn = oracle.psi_of_q(qn)
    d0 = np.sum(np.abs(psi) ** 2, axis=0)[0]; dn = np.sum(np.abs(pn) ** 2, axis=0)[0]
    assert np.sqrt(np.sum((dn - d0) ** 2) / np.sum(d0 ** 2)) < 5e-3
    j = int(np.argmax(np.abs(cm)))
    phase = np.angle(pn[j, 0, L // 2] / psi[j, 0, L // 2])
    assert abs(phase - k * k * n) < 0.02 * k * k * n
    # a wrong sign of U or of the kinetic phase disperses the soliton: the same test
    # with the couplings negated loses the profile
    qbad = oracle.step(q0, 1, tuple(-v for v in c), 1, n)
    db = np.sum(np.abs(oracle.psi_of_q(qbad)) ** 2, axis=0)[0]
    assert np.sqrt(np.sum((db - d0) ** 2) / np.sum(d0 ** 2)) > 0.1


def test_dark_soliton_pair_stationary_interleaved_beats_plain(oracle):
    # eq. (76)-(84) and §VII.B.2: dark pair of
    # state 5 (A00 soliton) at E = 2 stays put; interleaving is what keeps it.
    c = (1.0, 0.3, -0.1)
    L, k = 512, 1.0 / 8
    cm = table1_coeffs(5, 2.0, c)
    x = np.arange(L)
    T = np.tanh(k * (x - L / 4)) * np.tanh(k * (3 * L / 4 - x))
    psi = np.zeros((5, 1, L), complex); psi[:, 0, :] = cm[:, None] * k * T
    q0 = oracle.split_psi(psi)
    d0 = np.sum(np.abs(psi) ** 2, axis=0)[0]
    err = {}
    for order in (0, 1):
        pn = oracle.psi_of_q(oracle.step(q0, 1, c, order, 1000))
        dn = np.sum(np.abs(pn) ** 2, axis=0)[0]
        err[order] = np.sqrt(np.sum((dn - d0) ** 2) / np.sum(d0 ** 2))
    assert err[1] < 1e-2
    assert err[0] > 10 * err[1]
    # phase rotation exp(-i 2 k^2 t) of the background (eq. 81 with p = 0)
    pn = oracle.psi_of_q(oracle.step(q0, 1, c, 1, 100))
    ph = np.angle(pn[2, 0, L // 2] / psi[2, 0, L // 2])
    assert abs(ph + 2 * k * k * 100) < 0.02 * 2 * k * k * 100


def test_galilean_drift_of_kicked_bright_soliton(oracle):
    # eq. (71): centre moves as x0 + 2 p t, p = 2 pi n / L.
    c = (-1.0, -0.5, 0.2)
    L, k, n_kick = 1024, 1.0 / 16, 6
    p = 2 * np.pi * n_kick / L
    cm = table1_coeffs(1, -2.0, c)
    x = np.arange(L)
    psi = np.zeros((5, 1, L), complex)
    psi[:, 0, :] = cm[:, None] * k * inputs.sech(k * (x - L / 4)) * np.exp(1j * p * x)
    q0 = oracle.split_psi(psi)
    steps = 1500
    pn = oracle.psi_of_q(oracle.step(q0, 1, c, 1, steps))
    moved = _centre(np.sum(np.abs(pn) ** 2, axis=0)[0]) - L / 4
    assert abs(moved - 2 * p * steps) < 0.01 * 2 * p * steps
    # opposite kick moves the other way
    psi2 = np.conj(psi)
    pn2 = oracle.psi_of_q(oracle.step(oracle.split_psi(psi2), 1, c, 1, 300))
    assert _centre(np.sum(np.abs(pn2) ** 2, axis=0)[0]) < L / 4


def test_printed_drift_times_fix_the_units(oracle):
    # [R3] PAPER.md:906, 922: half of a 512 lattice in ~5000 steps at n=2 and ~3500
    # at n=3, i.e. speed 2p = 4 pi n / L sites per step (one step = unit time, one
    # site = unit length).  Measure the oracle's drift speed on L = 512 directly.
    g = load_golden("printed_numbers.json")["drift_times"]
    L = g["L"]
    c = (-1.0, -0.5, 0.2)
    k = 1.0 / 12
    cm = table1_coeffs(1, -2.0, c)
    x = np.arange(L)
    for case in g["cases"]:
        p = 2 * np.pi * case["n"] / L
        psi = np.zeros((5, 1, L), complex)
        psi[:, 0, :] = cm[:, None] * k * inputs.sech(k * (x - L / 4)) * np.exp(1j * p * x)
        steps = 600
        pn = oracle.psi_of_q(oracle.step(oracle.split_psi(psi), 1, c, 1, steps))
        speed = (_centre(np.sum(np.abs(pn) ** 2, axis=0)[0]) - L / 4) / steps
        t_half = (L / 2) / speed
        assert abs(t_half / case["steps"] - 1) < 0.06          # "approximately"
        assert abs(t_half - L * L / (8 * np.pi * case["n"])) < 0.02 * t_half


def test_translation_covariance_is_bit_exact(oracle):
    c = (1.0, 0.3, -0.1)
    psi = inputs.random_field((10, 7), seed=12, amplitude=0.3)
    q0 = oracle.split_psi(psi)
    a = oracle.step(q0, 2, c, 1, 2)
    b = oracle.step(np.roll(q0, (2, 3), axis=(2, 3)), 2, c, 1, 2)
    assert np.array_equal(np.roll(a, (2, 3), axis=(2, 3)), b)


def test_global_phase_and_spin_rotation_covariance(oracle):
    c = (1.0, 0.3, -0.1)
    q0 = inputs.random_spinor_state((8, 6), seed=13, amplitude=0.3)
    a = oracle.step(q0, 2, c, 1, 2)
    ph = np.exp(0.7j)
    assert rel_l2(oracle.step(ph * q0, 2, c, 1, 2), ph * a) < 1e-14
    # psi -> D(R) psi with a spin-2 Wigner matrix D = exp(-i phi n.f) commutes with a step
    fx, fy, fz = oracle.spin_matrices()
    nvec = np.array([0.3, -0.5, 0.8]); nvec /= np.linalg.norm(nvec)
    D = expm(-1j * 1.1 * (nvec[0] * fx + nvec[1] * fy + nvec[2] * fz))
    rot = lambda q: np.einsum("ab,bsyx->asyx", D, q)
    for order in (0, 1):
        a = oracle.step(q0, 2, c, order, 2)
        assert rel_l2(oracle.step(rot(q0), 2, c, order, 2), rot(a)) < 1e-13


def test_scalar_limit_is_channel_independent(oracle):
    # c1 = c2 = 0: a field living in one channel evolves the same in any channel.
    c = (0.9, 0.0, 0.0)
    base = inputs.smooth_random_field((64, 1), seed=3, amplitude=0.2)[0]
    outs = []
    for j in range(5):
        psi = np.zeros((5, 1, 64), complex); psi[j] = base
        outs.append(oracle.step(oracle.split_psi(psi), 1, c, 1, 20)[j])
    for j in range(1, 5):
        assert np.allclose(outs[j], outs[0], atol=1e-16)


def test_plain_and_interleaved_differ_but_agree_to_splitting_order(oracle):
    c = (1.0, 0.3, -0.1)
    psi = inputs.smooth_random_field((64, 1), seed=9, amplitude=0.05)
    q0 = oracle.split_psi(psi)
    a = oracle.step(q0, 1, c, 0, 10); b = oracle.step(q0, 1, c, 1, 10)
    d = rel_l2(a, b)
    assert 1e-9 < d < 1e-3


def test_double_and_long_double_builds_agree(oracle, oracle_ld):
    c = (1.0, 0.3, -0.1)
    w = inputs.config3(L=256)
    q0 = oracle.split_psi(w.psi)
    a = oracle.step(q0, 1, c, 1, 200)
    b = oracle_ld.step(q0.astype(np.clongdouble), 1, c, 1, 200)
    assert rel_l2(a, b.astype(np.complex128)) < 1e-13
    # the long-double build conserves the norm three orders better
    assert abs(norm2(b) / norm2(q0) - 1) < 1e-16
