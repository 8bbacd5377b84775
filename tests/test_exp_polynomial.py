"""The interaction polynomial table of the CUDA library (host-side, no GPU): the
economised polynomial P_p(-ix) must reproduce exp(-ix) within the stated tolerance
on the whole interval it is used for.  Checked in 50-digit arithmetic (mpmath)."""
import math

import numpy as np

import mpmath as mp
import pytest

mp.mp.dps = 50


def _poly(b0, r, p, y):
    acc = mp.mpf(1)
    for k in range(p, 0, -1):
        acc = 1 + mp.mpf(r[k]) * y * acc
    return mp.mpf(b0) * acc


@pytest.mark.parametrize("tol_log2", [-56, -27])
def test_polynomial_meets_tolerance_on_its_interval(tol_log2):
    from paper_1907_12834_b200 import qlga
    tol = mp.mpf(2) ** tol_log2
    prev = 0.0
    for p in range(1, 13):
        theta, b0, r = qlga.exp_polynomial(tol_log2, p)
        assert theta > prev                      # thresholds ascend
        prev = theta
        worst = mp.mpf(0)
        for i in range(0, 201):
            x = mp.mpf(theta) * (mp.mpf(i) / 100 - 1)
            err = abs(_poly(b0, r, p, -1j * x) - mp.e ** (-1j * x))
            worst = max(worst, err)
        # (coefficients are doubles: allow their rounding, 2^-53 * theta, on top of the tolerance)
        assert worst <= tol * mp.mpf("1.02") + mp.mpf(2) ** -52 * theta, (p, float(worst / tol))
        # the economised polynomial reaches ~1.5-2x further than the Taylor polynomial of equal degree
        taylor_theta = float((tol * mp.factorial(p + 1)) ** (mp.mpf(1) / (p + 1)))
        assert theta > (1.25 if p >= 2 else 0.99) * taylor_theta
        # coefficients stay close to 1/k and b0 to 1
        assert abs(b0 - 1.0) <= 2.0 * float(tol) + 1e-18
        for k in range(1, p + 1):
            assert abs(r[k] * k - 1.0) < 0.3


def test_polynomial_is_nearly_unitary():
    # |P_p(-ix)| - 1 stays within the tolerance (the norm drift per application)
    from paper_1907_12834_b200 import qlga
    for p in (3, 5, 6, 8):
        theta, b0, r = qlga.exp_polynomial(-56, p)
        for i in range(0, 41):
            x = mp.mpf(theta) * (mp.mpf(i) / 20 - 1)
            assert abs(abs(_poly(b0, r, p, -1j * x)) - 1) <= mp.mpf(2) ** -56 * mp.mpf("1.02") + mp.mpf(2) ** -52 * theta


def test_bad_arguments():
    from paper_1907_12834_b200 import qlga
    for args in ((-56, 0), (-56, 13), (-4, 3), (-200, 3)):
        with pytest.raises(qlga.QlgaError):
            qlga.exp_polynomial(*args)


def test_degree_lookup_table_is_never_below_the_threshold_rule():
    # the kernels pick the degree by a table lookup on the float bits of theta (qlga_exp_degree):
    # never below "smallest p with theta <= theta_max(p)", at most one above, equal away from bucket edges
    import numpy as np
    from paper_1907_12834_b200 import qlga
    rng = np.random.default_rng(5)
    for tol in (-56, -27):
        thr = [qlga.exp_polynomial(tol, p)[0] for p in range(1, 13)]
        top = min(thr[-1], 0.5)
        thetas = np.concatenate([10.0 ** rng.uniform(-15, np.log10(top), 4000),
                                 np.array(thr[:-1]) * (1 - 1e-6), np.array(thr[:-1]) * (1 + 1e-6), [0.0, 1e-30, top]])
        above = 0
        for th in thetas:
            if th > top:
                continue
            rule = 1 + sum(np.float32(th) > np.float32(t) for t in thr)
            got = qlga.exp_degree(tol, float(th))
            assert rule <= got <= min(rule + 1, 12), (tol, th, rule, got)
            above += got > rule
        assert above < 0.05 * len(thetas)          # buckets are 4-6 % wide: few angles pay an extra stage


@pytest.mark.parametrize("tl,shift", [(-56, 5), (-56, 9), (-58, 7)])          # (-58, 7): the fp64 default
def test_modulus_part_of_the_error_is_held_to_its_own_bound(tl, shift):
    # QLGA_OPT_EXP_MOD_SHIFT: |P_p(-ix)| - 1 (the error that repeats as a density error at every application)
    # stays within 2^(tl - shift) on the interval of every degree, the full error within 2^tl
    from paper_1907_12834_b200 import qlga
    tol, tol_mod = mp.mpf(2) ** tl, mp.mpf(2) ** (tl - shift)
    prev = 0.0
    for p in range(1, 13):
        theta, b0, r = qlga.exp_polynomial(tl, p, shift)
        assert theta >= prev and theta <= qlga.exp_polynomial(tl, p, 0)[0]
        prev = theta
        for i in range(0, 81):
            x = mp.mpf(theta) * (mp.mpf(i) / 40 - 1)
            val = _poly(b0, r, p, -1j * x)
            assert abs(val - mp.e ** (-1j * x)) <= tol * mp.mpf("1.02") + mp.mpf(2) ** -52 * theta
            # modulus: coefficient rounding enters as 2^-53 * theta^2 (the even part starts at x^2; b0 = 1 exactly)
            assert abs(abs(val) - 1) <= tol_mod * mp.mpf("1.05") + mp.mpf(2) ** -52 * theta ** 2, (p, float(x))
        assert b0 == 1.0
    # small even degrees (nearly) keep the reach of the plain tolerance: their leading error is odd, a phase error
    for p in (2, 4):
        assert qlga.exp_polynomial(tl, p, shift)[0] >= 0.97 * qlga.exp_polynomial(tl, p, 0)[0]
    # the degree lookup follows the shifted thresholds
    thr = [qlga.exp_polynomial(tl, p, shift)[0] for p in range(1, 13)]
    for th in (5.2e-5, 0.0047, 0.015, 0.05):
        rule = 1 + sum(np.float32(th) > np.float32(t) for t in thr)
        assert rule <= qlga.exp_degree(tl, th, shift) <= rule + 1
