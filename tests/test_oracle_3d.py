"""Pins of the oracle's 3D lattice ("in two
and three dimensions ... n = 8, and n = 12").  CPU only."""
import numpy as np
import pytest

from paper_1907_12834_b200 import inputs
from conftest import rel_l2, norm2, table1_coeffs


def test_stream_along_z_and_kinetic_symbol(oracle):
    nx, ny, nz = 4, 3, 8
    q = np.zeros((5, 2, nz, ny, nx), complex)
    q[:, 1, 7, 2, 1] = 1.0 + 2.0j                      # on the z edge: exercises the wrap
    s = oracle.stream(q, 2, 1, transpose=False)
    exp = np.zeros_like(q); exp[:, 1, 0, 2, 1] = 1.0 + 2.0j
    assert np.array_equal(s, exp)
    assert np.array_equal(oracle.stream(s, 2, 1, transpose=True), q)
    # the four z factors equal the DFT symbol along z
    r = inputs.random_spinor_state((nx, ny, nz), seed=3)
    out = r
    for sigma in (1, 1, 0, 0):
        out = oracle.kinetic_factor(out, 2, sigma)
    C = 0.5 * np.array([[1 - 1j, 1 + 1j], [1 + 1j, 1 - 1j]])
    def sym(k, sg):
        S = np.eye(2, dtype=complex); S[sg, sg] = np.exp(-1j * k)
        return S @ C @ S.conj().T @ C
    Q = np.fft.fft(r, axis=2); R = np.empty_like(Q)
    for kk in range(nz):
        k = 2 * np.pi * kk / nz
        M = sym(k, 0) @ sym(k, 0) @ sym(k, 1) @ sym(k, 1)
        R[:, :, kk] = np.einsum("ab,jb...->ja...", M, Q[:, :, kk])
    assert rel_l2(out, np.fft.ifft(R, axis=2)) < 1e-14


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_plain_3d_step_of_a_one_directional_field_is_the_1d_step(oracle, axis):
    # With the plain ordering, kinetic factors along a direction in which the state is
    # uniform reduce to an even number of component swaps, i.e. to the identity: a field
    # that varies along one axis only must evolve exactly as on the 1D lattice.
    c = (1.0, 0.3, -0.1)
    L = 24
    q1 = inputs.random_spinor_state((L, 1), seed=11, amplitude=0.2)           # (5,2,1,L)
    line = q1[:, :, 0, :]                                                       # (5,2,L)
    shape = [3, 4, 5]; shape[2 - axis] = L                                      # (nz, ny, nx)
    idx = [None, None, None]; idx[2 - axis] = slice(None)
    q3 = np.ascontiguousarray(np.broadcast_to(line[(slice(None), slice(None)) + tuple(idx)], (5, 2) + tuple(shape)))
    ref = oracle.step(q1, 1, c, 0, 3)[:, :, 0, :]
    out = oracle.step(q3, 3, c, 0, 3)
    sel = [0, 0, 0]; sel[2 - axis] = slice(None)
    assert rel_l2(out[(slice(None), slice(None)) + tuple(sel)], ref) < 1e-14
    assert np.allclose(out, np.broadcast_to(out[(slice(None), slice(None)) + tuple(sel)][(slice(None), slice(None)) + tuple(idx)], out.shape), atol=1e-15)


def test_3d_reduces_to_2d_and_uses_twelve_substeps(oracle):
    c = (1.0, 0.3, -0.1)
    q2 = inputs.random_spinor_state((6, 5), seed=2, amplitude=0.2)
    q3 = q2[:, :, None]                                                         # nz = 1
    # plain: a z direction of one site contributes four swaps = identity -> the 2D plain step
    assert rel_l2(oracle.step(q3, 3, c, 0, 2)[:, :, 0], oracle.step(q2, 2, c, 0, 2)) < 1e-14
    # interleaved: 12 applications of U^{1/12} (n = 12) instead of 8 of U^{1/8}: a different
    # splitting of the same flow -- close on a smooth field, not equal
    qs = oracle.split_psi(inputs.smooth_random_field((16, 12), seed=4, amplitude=0.1, kmax=1))
    d = rel_l2(oracle.step(qs[:, :, None], 3, c, 1, 2)[:, :, 0], oracle.step(qs, 2, c, 1, 2))
    assert 1e-12 < d < 1e-2


@pytest.mark.parametrize("row", [1, 5, 13, 16])
def test_table1_uniform_states_3d(oracle, row):
    c = (1.0, 0.3, -0.1)
    E = 0.05
    cm = table1_coeffs(row, E, c)
    psi = np.zeros((5, 3, 4, 5), complex); psi[:] = cm[:, None, None, None]
    q0 = oracle.split_psi(psi)
    for order in (0, 1):
        qn = oracle.step(q0, 3, c, order, 3)
        assert rel_l2(qn, np.exp(-1j * E * 3) * q0) < 5e-15


def test_3d_unitarity_translation_and_observables(oracle):
    c = (1.0, 0.3, -0.1)
    q0 = inputs.random_spinor_state((7, 5, 6), seed=5, amplitude=0.15)
    a = oracle.step(q0, 3, c, 1, 20)
    assert abs(norm2(a) / norm2(q0) - 1) < 1e-14
    b = oracle.step(np.roll(q0, (1, 2, 3), axis=(2, 3, 4)), 3, c, 1, 2)
    assert np.array_equal(np.roll(oracle.step(q0, 3, c, 1, 2), (1, 2, 3), axis=(2, 3, 4)), b)
    ob = oracle.observables(q0, 3, c)
    psi = q0[:, 0] + q0[:, 1]
    ekin = sum(np.sum(np.abs(np.roll(psi, -1, ax) - psi) ** 2) for ax in (1, 2, 3))
    assert abs(ob["e_kin"] - ekin) < 1e-12 * ekin
    assert abs(ob["norm_q"] - np.sum(np.abs(q0) ** 2)) < 1e-12
    rho = oracle.density(q0)
    assert rho.shape == (6, 5, 7) and np.allclose(rho, np.sum(np.abs(psi) ** 2, axis=0))
