"""Pins of the oracle's observables (eq. 3-5, 59-60, 85, 32) and lattice
vorticity (eq. 99-104) against the paper's Table II, dispersion relations
(eq. 74), and topological invariants.  CPU only."""
import numpy as np
import pytest

from paper_1907_12834_b200 import inputs
from conftest import table1_coeffs, load_golden, eval_expr


@pytest.mark.parametrize("row", [1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 13])
def test_table2_characteristics(oracle, row):
    # Table II: |F_par|, |F_perp|, |A00| per site of the Table I states.
    c = (1.0, 0.3, -0.1)
    E = 0.3
    g0, g1, g2 = c
    cm = table1_coeffs(row, E, c)
    exp = [eval_expr(e, E=E, g0=g0, g1=g1, g2=g2) for e in load_golden("table2.json")["rows"][str(row)]]
    N = 6
    psi = np.zeros((5, 1, N), complex); psi[:, 0, :] = cm[:, None]
    ob = oracle.observables(oracle.split_psi(psi), 1, c)
    assert abs(abs(ob["F_z"]) / N - exp[0]) < 1e-14
    assert abs(np.hypot(ob["F_x"], ob["F_y"]) / N - exp[1]) < 1e-14
    assert abs(np.hypot(ob["A00_re"], ob["A00_im"]) / N - exp[2]) < 1e-14
    assert abs(ob["A00_abs2"] / N - exp[2] ** 2) < 1e-14
    assert abs(ob["norm_psi"] / N - np.sum(cm ** 2)) < 1e-14
    assert abs(ob["norm_q"] / N - np.sum(cm ** 2) / 2) < 1e-14      # q1 = q2 = psi/2


def test_spin_density_signs_and_Fy(oracle):
    # F_z = 2(|psi_2|^2 - |psi_-2|^2) + |psi_1|^2 - |psi_-1|^2 (eq. 59a);
    # F_+ = <psi|f_+|psi>: a state (psi_2, psi_1) = (1, i)/sqrt2 has F_+ = 2 conj(psi_2) psi_1 = i
    c = (1.0, 0.3, -0.1)
    psi = np.zeros((5, 1, 1), complex); psi[0] = 1 / np.sqrt(2); psi[1] = 1j / np.sqrt(2)
    ob = oracle.observables(oracle.split_psi(psi), 1, c)
    assert abs(ob["F_z"] - 1.5) < 1e-15 and abs(ob["F_x"]) < 1e-15 and abs(ob["F_y"] - 1.0) < 1e-15
    psi = np.zeros((5, 1, 1), complex); psi[4] = 1.0
    assert abs(oracle.observables(oracle.split_psi(psi), 1, c)["F_z"] + 2.0) < 1e-15


def test_energy_functional_of_plane_wave_and_uniform_state(oracle):
    # e_kin of exp(ipx) is sum |e^{ip} - 1|^2 = N (2 - 2 cos p) -> p^2 N; interaction
    # energies of a uniform Table-I state: E_int/N = (1/2) E rho (homogeneous cubic GP).
    c = (1.0, 0.3, -0.1)
    N = 64
    p = 2 * np.pi * 3 / N
    psi = np.zeros((5, 1, N), complex); psi[2, 0] = 0.5 * np.exp(1j * p * np.arange(N))
    ob = oracle.observables(oracle.split_psi(psi), 1, c)
    assert abs(ob["e_kin"] - 0.25 * N * (2 - 2 * np.cos(p))) < 1e-12
    for row in (1, 5, 13, 14, 16):
        E = 0.2
        cm = table1_coeffs(row, E, c)
        psi = np.zeros((5, 3, 4), complex); psi[:] = cm[:, None, None]
        ob = oracle.observables(oracle.split_psi(psi), 2, c)
        rho = np.sum(cm ** 2)
        assert abs(ob["e_kin"]) < 1e-28
        assert abs((ob["e_c0"] + ob["e_c1"] + ob["e_c2"]) / 12 - 0.5 * E * rho) < 1e-15
        assert abs(ob["e_total"] - (ob["e_kin"] + ob["e_c0"] + ob["e_c1"] + ob["e_c2"])) < 1e-15


def test_eq85_energy_of_uniform_state(oracle):
    # eq. (85): for psi(t) = e^{-iE} psi(t - tau), E_dt = i (1 - e^{+iE}) ~ E.
    c = (1.0, 0.3, -0.1)
    E = 0.05
    cm = table1_coeffs(13, E, c)
    psi = np.zeros((5, 1, 8), complex); psi[:, 0, :] = cm[:, None]
    q0 = oracle.split_psi(psi); q1 = oracle.step(q0, 1, c, 1, 1)
    ob = oracle.observables(q1, 1, c, qprev=q0)
    e = ob["e_dt_re"] + 1j * ob["e_dt_im"]
    assert abs(e - 1j * (1 - np.exp(1j * E))) < 1e-15
    assert np.isnan(oracle.observables(q1, 1, c)["e_dt_re"])


@pytest.mark.parametrize("n_kick", [0, 4, 8])
def test_bright_soliton_dispersion_eq74(oracle, n_kick):
    # Fig. 5 / eq. (72)-(74): E = (p^2 - k^2) per unit norm, measured with eq. (85).
    c = (-1.0, -0.5, 0.2)
    L, k = 1024, 1.0 / 16
    p = 2 * np.pi * n_kick / L
    cm = table1_coeffs(3, -2.0, c)
    x = np.arange(L)
    psi = np.zeros((5, 1, L), complex)
    psi[:, 0, :] = cm[:, None] * k * inputs.sech(k * (x - L / 2)) * np.exp(1j * p * x)
    q0 = oracle.split_psi(psi)
    qa = oracle.step(q0, 1, c, 1, 20); qb = oracle.step(qa, 1, c, 1, 1)
    ob = oracle.observables(qb, 1, c, qprev=qa)
    assert abs(ob["e_dt_re"] - (p * p - k * k)) < 0.02 * (p * p + k * k)


def _quadrupole(L, core, shift=0.5):
    """Pade quadrupole like config 4 but with vortex centres between lattice sites
    (no site has psi == 0 exactly, so every plaquette phase is defined)."""
    a = 1.0 / core
    X, Y = np.meshgrid(np.arange(L, dtype=float), np.arange(L, dtype=float), indexing="xy")
    V = np.ones((L, L), complex)
    for cx, cy, wd in ((L / 4, L / 4, +1), (3 * L / 4, L / 4, -1),
                       (L / 4, 3 * L / 4, -1), (3 * L / 4, 3 * L / 4, +1)):
        V *= inputs.vortex_factor(X, Y, cx + shift, cy + shift, a, wd)
    psi = np.empty((5, L, L), complex)
    psi[0] = a * V; psi[4] = a * np.conj(V); psi[1:4] = a
    return psi


def test_vorticity_invariants_on_quadrupole(oracle):
    # [R8] pins: sum omega = 0; every value a multiple of pi/2 (omega is a quarter of
    # the wrapped phase circulation around the diagonal plaquette); box sum around an
    # isolated Pade vortex = 2 pi x winding; a uniform channel has omega = 0.
    L = 64
    psi = _quadrupole(L, 4.0)
    om = oracle.vorticity(oracle.split_psi(psi))
    assert om.shape == (5, L, L)
    assert abs(om.sum()) < 1e-12
    assert np.allclose(om / (np.pi / 2), np.round(om / (np.pi / 2)), atol=1e-12)
    assert set(np.unique(np.round(om / (np.pi / 2)))) <= {-1.0, 0.0, 1.0}
    assert np.all(om[1:4] == 0)
    h = L // 2
    assert abs(om[0][:h, :h].sum() - 2 * np.pi) < 1e-12        # (L/4, L/4): winding +1 in m=+2
    assert abs(om[0][:h, h:].sum() + 2 * np.pi) < 1e-12
    assert abs(om[0][h:, :h].sum() + 2 * np.pi) < 1e-12
    assert abs(om[0][h:, h:].sum() - 2 * np.pi) < 1e-12
    assert abs(om[4][:h, :h].sum() + 2 * np.pi) < 1e-12        # m=-2 holds the conjugate field
    ys, xs = np.nonzero(np.abs(om[0][:h, :h]) > 1.0)
    assert np.all(np.abs(xs - (L / 4 + 0.5)) <= 1.5) and np.all(np.abs(ys - (L / 4 + 0.5)) <= 1.5)
    # config 4 proper (centres on lattice sites, psi == 0 there, arg(0) := 0): the
    # total still vanishes and the windings are still found with the right signs
    w = inputs.config4(L=L, core=4.0)
    om4 = oracle.vorticity(oracle.split_psi(w.psi))
    assert abs(om4.sum()) < 1e-12
    assert om4[0][:h, :h].sum() > 1.0 and om4[0][:h, h:].sum() < -1.0


def test_vorticity_plane_wave_and_zero_field(oracle):
    L = 16
    X, Y = np.meshgrid(np.arange(L), np.arange(L), indexing="xy")
    psi = np.zeros((5, L, L), complex)
    psi[0] = np.exp(2j * np.pi * (3 * X - 2 * Y) / L)
    om = oracle.vorticity(oracle.split_psi(psi))
    assert np.abs(om).max() < 1e-13          # plane wave -> omega == 0; arg(0) := 0 for empty channels


def test_vorticity_bruteforce_definition(oracle):
    # brute force of eq. (102)-(104) with wrapped phase differences on a random field
    L = 9
    psi = inputs.random_field((L, L), seed=31)
    om = oracle.vorticity(oracle.split_psi(psi))
    wrap = lambda a: (a + np.pi) % (2 * np.pi) - np.pi
    for j in (0, 3):
        S = np.angle(psi[j])
        vx = wrap(np.roll(S, -1, 1) - np.roll(S, 1, 1)) / 2
        vy = wrap(np.roll(S, -1, 0) - np.roll(S, 1, 0)) / 2
        ref = (np.roll(vy, -1, 1) - np.roll(vy, 1, 1) - np.roll(vx, -1, 0) + np.roll(vx, 1, 0)) / 2
        assert np.allclose(om[j], ref, atol=1e-12)
