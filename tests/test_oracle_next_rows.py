"""Pins of the oracle functions behind SURVEY.md section 8(f) rows 1-2: the density
L2 error of eq. (115) and the plaquette winding detector.  CPU only."""
import numpy as np

from paper_1907_12834_b200 import inputs
from conftest import table1_coeffs


def _offsite_quadrupole(L, core, shift=0.5):
    a = 1.0 / core
    X, Y = np.meshgrid(np.arange(L, dtype=float), np.arange(L, dtype=float), indexing="xy")
    V = np.ones((L, L), complex)
    cs = ((L / 4, L / 4, +1), (3 * L / 4, L / 4, -1), (L / 4, 3 * L / 4, -1), (3 * L / 4, 3 * L / 4, +1))
    for cx, cy, wd in cs:
        V *= inputs.vortex_factor(X, Y, cx + shift, cy + shift, a, wd)
    psi = np.empty((5, L, L), complex)
    psi[0] = a * V; psi[4] = a * np.conj(V); psi[1:4] = a
    return psi, cs


def test_density_and_l2_error_definition(oracle):
    q = inputs.random_spinor_state((7, 5), seed=3)
    rho = oracle.density(q)
    psi = q[:, 0] + q[:, 1]
    assert np.allclose(rho, np.sum(np.abs(psi) ** 2, axis=0), rtol=1e-15)
    assert oracle.density_l2_error(q, rho) == 0.0
    ref = rho + 0.25
    assert abs(oracle.density_l2_error(q, ref) - 0.0625 * 35) < 1e-13
    # a global phase or a spin rotation about z leaves the density, hence eq. (115), unchanged
    ph = np.exp(-1j * np.array([2, 1, 0, -1, -2]) * 0.7)[:, None, None, None]
    assert oracle.density_l2_error(np.exp(0.3j) * ph * q, rho) < 1e-28


def test_l2_error_of_stationary_soliton_falls_with_lattice_size(oracle):
    # Figs. 23-24: for a fixed number of steps the error of a
    # stationary bright soliton falls faster than L^-4 when its width scales with L.
    c = (-1.0, -0.5, 0.2)
    cm = table1_coeffs(1, -2.0, c)
    eps = []
    for L in (128, 256, 512):
        k = 8.0 / L
        x = np.arange(L)
        psi = np.zeros((5, 1, L), complex)
        psi[:, 0, :] = cm[:, None] * k * inputs.sech(k * (x - L / 2))
        q0 = oracle.split_psi(psi)
        rho0 = oracle.density(q0)
        qn = oracle.step(q0, 1, c, 1, 200)
        eps.append(oracle.density_l2_error(qn, rho0) / np.sum(rho0 ** 2))
    slope = np.polyfit(np.log([128, 256, 512]), np.log(eps), 1)[0]
    assert eps[0] > eps[1] > eps[2] and slope < -4.0


def test_winding_finds_the_quadrupole(oracle):
    L = 48
    psi, cs = _offsite_quadrupole(L, 4.0)
    w = oracle.winding(oracle.split_psi(psi))
    assert w.dtype == np.int32 and w.shape == (5, L, L)
    assert np.all(w[1:4] == 0)
    found = {(int(x), int(y)): int(w[0, y, x]) for y, x in np.argwhere(w[0] != 0)}
    assert found == {(int(cx), int(cy)): wd for cx, cy, wd in cs}     # plaquette (x, y) holds centre (x+.5, y+.5)
    assert np.array_equal(w[4], -w[0])                                 # conjugate field
    assert w.sum() == 0                                                # total winding of a periodic lattice


def test_winding_total_is_zero_and_plane_wave_has_none(oracle):
    L = 12
    X, Y = np.meshgrid(np.arange(L), np.arange(L), indexing="xy")
    psi = np.zeros((5, L, L), complex)
    psi[2] = np.exp(2j * np.pi * (2 * X - Y) / L)
    assert np.all(oracle.winding(oracle.split_psi(psi)) == 0)
    r = inputs.random_field((L, L), seed=8)
    w = oracle.winding(oracle.split_psi(r))
    assert np.all(np.abs(w) <= 1)
    for j in range(5):
        assert w[j].sum() == 0
    # brute force with wrapped phase differences
    S = np.angle(r[1])
    wrap = lambda a: (a + np.pi) % (2 * np.pi) - np.pi
    circ = (wrap(np.roll(S, -1, 1) - S) + wrap(np.roll(np.roll(S, -1, 1), -1, 0) - np.roll(S, -1, 1))
            + wrap(np.roll(S, -1, 0) - np.roll(np.roll(S, -1, 1), -1, 0)) + wrap(S - np.roll(S, -1, 0)))
    assert np.array_equal(w[1], np.rint(circ / (2 * np.pi)).astype(np.int32))


# ---- chemical potential (section II.C; eq. 75) ----
def test_chemical_potential_is_a_global_phase_and_zero_is_the_plain_form(oracle):
    import numpy as np
    from paper_1907_12834_b200 import inputs
    from conftest import rel_l2
    c, mu = (1.0, 0.3, -0.1), 0.0375
    for ndim, dims in ((1, (24, 1)), (2, (10, 8))):
        q0 = inputs.random_spinor_state(dims, seed=8, amplitude=0.1)
        for order in (0, 1):
            ref = oracle.step(q0, ndim, c, order, 5)
            assert np.array_equal(oracle.step(q0, ndim, c, order, 5, mu=0.0), ref)      # bit for bit
            got = oracle.step(q0, ndim, c, order, 5, mu=mu)
            assert rel_l2(got, np.exp(-1j * mu * 5) * ref) < 1e-14
    one = oracle.interaction(q0, c, 0.25, mu=mu)
    assert rel_l2(one, np.exp(-1j * mu * 0.25) * oracle.interaction(q0, c, 0.25)) < 1e-15


def test_dispersion_with_chemical_potential_eq75(oracle):
    # eq. (75): E = mu + p^2 - k^2 (bright): E = mu + p^2 + 2 k^2 (dark), by eq. (85)
    import numpy as np
    L, k, n, mu = 512, 1.0 / 16, 4, 0.011
    p = 2 * np.pi * n / L
    for kind, row, c in (("bright", 3, (-1.0, -0.5, 0.2)), ("dark", 5, (1.0, 0.3, -0.1))):
        q0 = oracle.split_psi(inputs.kicked_soliton(kind, row, c, L, k, n))
        qa = oracle.step(q0, 1, c, 1, 10, mu=mu)
        qb = oracle.step(qa, 1, c, 1, 1, mu=mu)
        e = oracle.observables(qb, 1, c, qprev=qa)["e_dt_re"]
        want = mu + inputs.predicted_energy(kind, k, p)
        assert abs(e - want) < 0.02 * (p * p + k * k), (kind, e, want)
        e0 = oracle.observables(oracle.step(qa, 1, c, 1, 1), 1, c, qprev=qa)["e_dt_re"]
        assert abs((e - e0) - mu) < 1e-3 * mu          # the shift is mu (sin mu at this size)


def test_uniform_table1_state_with_chemical_potential(oracle):
    import numpy as np
    from conftest import table1_coeffs
    c, E, mu, n = (1.0, 0.3, -0.1), 0.002, 0.004, 25
    cm = table1_coeffs(13, E, c)
    psi = np.zeros((5, 1, 8), complex); psi[:, 0, :] = cm[:, None]
    out = oracle.psi_of_q(oracle.step(oracle.split_psi(psi), 1, c, 1, n, mu=mu))
    assert np.abs(out - np.exp(-1j * (E + mu) * n) * psi).max() < 1e-14
