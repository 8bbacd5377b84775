"""Pins of the oracle's collide / stream / kinetic-factor operators
(§VII.B.1, eq. 107-109).  CPU only."""
import numpy as np
import pytest

from paper_1907_12834_b200 import inputs
from conftest import rel_l2, norm2


def test_collide_is_sqrt_of_swap_and_unitary(oracle):
    # [R1] C = (1/2)[[1-i,1+i],[1+i,1-i]]: C^2 swaps the two spinor components,
    # C is unitary, and q1+q2 is left invariant by C ("approximately
    # the identity operator when acting on the bosonic state psi").
    q = inputs.random_spinor_state((12, 3), seed=11)
    c1 = oracle.collide(q)
    c2 = oracle.collide(c1)
    assert np.allclose(c2[:, 0], q[:, 1], atol=1e-16)
    assert np.allclose(c2[:, 1], q[:, 0], atol=1e-16)
    assert abs(norm2(c1) / norm2(q) - 1) < 1e-15
    assert np.allclose(c1[:, 0] + c1[:, 1], q[:, 0] + q[:, 1], atol=1e-16)
    # explicit matrix entries on a basis vector: (1,0) -> ((1-i)/2, (1+i)/2)
    e = np.zeros((5, 2, 1, 1), complex); e[:, 0] = 1.0
    ce = oracle.collide(e)
    assert np.allclose(ce[:, 0], (1 - 1j) / 2) and np.allclose(ce[:, 1], (1 + 1j) / 2)


@pytest.mark.parametrize("d", [0, 1])
@pytest.mark.parametrize("sigma", [0, 1])
def test_stream_moves_one_component_one_site(oracle, d, sigma):
    # [R2] S_{d,sigma} moves the content of component sigma toward +e_d by one
    # site, periodically; S^T undoes it; the other component is untouched.
    nx, ny = 7, 5
    q = np.zeros((5, 2, ny, nx), complex)
    q[:, sigma, 2, 6] = 1.0 + 2.0j          # on the x edge: exercises the wrap
    q[:, 1 - sigma, 1, 1] = 3.0
    s = oracle.stream(q, d, sigma, transpose=False)
    exp = np.zeros_like(q)
    if d == 0:
        exp[:, sigma, 2, 0] = 1.0 + 2.0j
    else:
        exp[:, sigma, 3, 6] = 1.0 + 2.0j
    exp[:, 1 - sigma, 1, 1] = 3.0
    assert np.array_equal(s, exp)
    assert np.array_equal(oracle.stream(s, d, sigma, transpose=True), q)
    r = inputs.random_spinor_state((nx, ny), seed=5)
    assert np.array_equal(oracle.stream(oracle.stream(r, d, sigma, True), d, sigma, False), r)


def test_uninterleaved_order_is_identity_on_psi(oracle):
    # "if you simply switched the order of the stream and collide
    # operators ... such that there was no interleaving one would exactly recover
    # the identity operator" (on the bosonic state psi = q1 + q2).
    q = inputs.random_spinor_state((16, 1), seed=3)
    out = oracle.stream(oracle.stream(oracle.collide(oracle.collide(q)), 0, 0, True), 0, 0, False)
    assert np.allclose(oracle.psi_of_q(out), oracle.psi_of_q(q), atol=1e-15)
    # ... while the interleaved product is not the identity
    out2 = oracle.kinetic_factor(q, 0, 0)
    assert rel_l2(oracle.psi_of_q(out2), oracle.psi_of_q(q)) > 1e-2


def _symbol(k, sigma):
    """2x2 Fourier symbol of I'_sigma = S C S^T C for wavenumber k, built from the
    definitions: (S q)_sigma(r) = q_sigma(r - e) -> multiplication by exp(-ik)."""
    C = 0.5 * np.array([[1 - 1j, 1 + 1j], [1 + 1j, 1 - 1j]])
    S = np.eye(2, dtype=complex); S[sigma, sigma] = np.exp(-1j * k)
    return S @ C @ S.conj().T @ C


@pytest.mark.parametrize("d,dims", [(0, (16, 1)), (0, (8, 4)), (1, (4, 8))])
def test_kinetic_factors_equal_bruteforce_dft_symbol(oracle, d, dims):
    # Pin 2: real-space operators == inverse DFT of (symbol x DFT), all modes,
    # for the full kinetic product I'_1 I'_1 I'_2 I'_2 along direction d.
    nx, ny = dims
    q = inputs.random_spinor_state(dims, seed=21)
    out = q
    for sigma in (1, 1, 0, 0):
        out = oracle.kinetic_factor(out, d, sigma)
    axis = 3 if d == 0 else 2
    n = q.shape[axis]
    Q = np.fft.fft(q, axis=axis)            # numpy: q(r) = (1/n) sum_k Q_k e^{+2 pi i k r / n}
    R = np.empty_like(Q)
    for kk in range(n):
        k = 2 * np.pi * kk / n
        M = _symbol(k, 0) @ _symbol(k, 0) @ _symbol(k, 1) @ _symbol(k, 1)
        sl = [slice(None)] * 4; sl[axis] = kk
        Qk = Q[tuple(sl)]                    # shape (5, 2, other)
        R[tuple(sl)] = np.einsum("ab,jb...->ja...", M, Qk)
    ref = np.fft.ifft(R, axis=axis)
    assert rel_l2(out, ref) < 1e-14


def test_eq109_kinetic_expansion(oracle):
    # eq. (109): (I'_1 I'_1 I'_2 I'_2) psi = psi - i p^2 psi + O(p^4)
    L = 4096
    x = np.arange(L)
    errs = []
    for n in (2, 4, 8, 16):
        p = 2 * np.pi * n / L
        psi = np.zeros((5, 1, L), complex)
        psi[1, 0] = np.exp(1j * p * x)
        q = oracle.split_psi(psi)
        for sigma in (1, 1, 0, 0):
            q = oracle.kinetic_factor(q, 0, sigma)
        ratio = oracle.psi_of_q(q)[1, 0] / psi[1, 0]
        assert np.allclose(ratio, ratio[0], atol=1e-13)        # plane wave stays a plane wave
        errs.append(abs(ratio[0] - (1 - 1j * p * p)) / p**4)
        # sign of time: phase is -p^2 (forward evolution exp(-i p^2 t)), modulus ~ 1
        assert np.angle(ratio[0]) < 0
        assert abs(abs(ratio[0]) - 1) < 2 * p**4
    # remainder is O(p^4) with a bounded coefficient
    assert max(errs) < 1.0 and max(errs) / min(errs) < 1.5


def test_kinetic_factor_equals_three_point_stencil(oracle):
    # Pin 3 / DESIGN.md: I'_{d,1} as a radius-1 stencil (sigma=2: roles exchanged).
    q = inputs.random_spinor_state((9, 6), seed=8)
    for d in (0, 1):
        ax = 2 if d == 0 else 1                       # axis within q[:, s] (5, ny, nx)
        for sigma in (0, 1):
            out = oracle.kinetic_factor(q, d, sigma)
            qa, qb = q[:, sigma], q[:, 1 - sigma]     # streamed component, other one
            za = 0.5 * (-1j * qa + qb + 1j * np.roll(qa, 1, ax) + np.roll(qb, 1, ax))
            zb = 0.5 * (np.roll(qa, -1, ax) + 1j * np.roll(qb, -1, ax) + qa - 1j * qb)
            assert np.allclose(out[:, sigma], za, atol=1e-15)
            assert np.allclose(out[:, 1 - sigma], zb, atol=1e-15)


def test_grouping_11_22_pinned(oracle):
    # [R7] within one direction the grouping I'_1 I'_1 I'_2 I'_2 (eq. 108 as printed)
    # keeps the symmetric mode unitary to O(k^6); the alternating grouping does not.
    k = 0.1
    M_ok = _symbol(k, 0) @ _symbol(k, 0) @ _symbol(k, 1) @ _symbol(k, 1)
    M_bad = _symbol(k, 0) @ _symbol(k, 1) @ _symbol(k, 0) @ _symbol(k, 1)
    sym = np.array([0.5, 0.5])
    amp_ok = abs(np.ones(2) @ (M_ok @ sym))
    amp_bad = abs(np.ones(2) @ (M_bad @ sym))
    assert abs(amp_ok - 1) < 1e-9 and abs(amp_bad - 1) > 1e-3
