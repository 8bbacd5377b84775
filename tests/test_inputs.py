"""Checks of the seeded input generators (paper_1907_12834_b200/inputs.py)
against the paper's closed forms.  CPU only."""
import numpy as np

from paper_1907_12834_b200 import inputs
from conftest import table1_coeffs, load_golden


def test_table1_helper_matches_golden_fixture():
    c = (1.0, 0.3, -0.1)
    for row in range(1, 17):
        a = inputs.table1_state(row, 0.02, c, free=(0.03, 0.02))
        b = table1_coeffs(row, 0.02, c, free=(0.03, 0.02))
        assert np.allclose(a, b, atol=1e-16)


def test_pade_default_coefficients_are_table3_at_E_equal_g():
    # Table III row m_f = 2 at E = g := g0 + 4 g1 and the "+" root:
    #   a1 = (19E^3 - 12 g E^2 + gamma_2) / (64 g (2E - g)),
    #   gamma_2 = E^2 sqrt(361 E^2 - 8 g (4 g + 13 E)),
    #   b1 = (16 a1 (g - 3E) + 5 E^2) / (48 (E - 4 a1)),   a2 = a1 (b1 - E/4).
    g = 1.0; E = 1.0
    gamma2 = E**2 * np.sqrt(361 * E**2 - 8 * g * (4 * g + 13 * E))
    a1 = (19 * E**3 - 12 * g * E**2 + gamma2) / (64 * g * (2 * E - g))
    b1 = (16 * a1 * (g - 3 * E) + 5 * E**2) / (48 * (E - 4 * a1))
    a2 = a1 * (b1 - E / 4)
    gold = load_golden("printed_numbers.json")["pade_scalar_limit"]
    frac = lambda s: float(s.split("/")[0]) / float(s.split("/")[1])
    assert abs(a1 - frac(gold["a1"])) < 1e-15
    assert abs(b1 - frac(gold["b1"])) < 1e-15
    assert abs(a2 - frac(gold["a2"])) < 1e-15
    s = np.array([0.0, 0.5, 3.0, 50.0])
    ref = np.sqrt((a2 * s**4 + a1 * s**2) / (a2 * s**4 + b1 * s**2 + 1))
    assert np.allclose(inputs.pade_profile(s), ref)
    assert abs(inputs.pade_profile(np.array([1e3]))[0] - 1.0) < 1e-5 and inputs.pade_profile(np.array([0.0]))[0] == 0.0


def test_configs_shapes_seeds_and_structure():
    w1 = inputs.config1()
    assert w1.psi.shape == (5, 1, 1024) and w1.couplings == (-1.0, -0.5, 0.2)
    assert np.count_nonzero(np.abs(w1.psi).sum(axis=(1, 2))) == 1
    assert abs(np.abs(w1.psi[0]).max() - np.sqrt(2 / 3) / 32) < 1e-15
    w2 = inputs.config2(L=4096)
    assert np.argmax(np.abs(w2.psi[1, 0])) == 1024 and np.argmax(np.abs(w2.psi[3, 0])) == 3072
    a = inputs.config3(L=512); b = inputs.config3(L=512)
    assert np.array_equal(a.psi, b.psi)                        # seeded
    assert abs(np.abs(a.psi[0]).mean() - np.sqrt(0.5) / 16) < 1e-3
    w4 = inputs.config4(L=64, core=4.0)
    assert w4.psi.shape == (5, 64, 64)
    assert np.allclose(w4.psi[4], np.conj(w4.psi[0]))
    # mirror symmetry about x = L/2 and y = L/2 (value-continuous across the wrap)
    V = w4.psi[0]
    assert np.allclose(np.abs(V[:, 1:]), np.abs(V[:, 1:][:, ::-1]))
    w5 = inputs.config5(L=128, core=4.0, spacing=16.0, offset=24.0)
    assert w5.psi.shape == (5, 128, 128)
    assert np.allclose(np.abs(w5.psi[0]), 0.25)                # pure phase noise on the background
    assert w5.ndim == 2 and w5.steps == 5000
