"""qlga_observable_sums_noalloc: the allocation-free observables entry point (static device scratch inside
the library) against the existing path, qlga_observable_sums of a context, on two calls in a row.

Collected last on purpose (the file name sorts after every other test file): the suite runs with
`pytest -x`, and a failure here must not hide the parity tests.  Passes alone in a fresh process and after
the other tests: it shares no state with them (the static array is overwritten by every call)."""
import numpy as np
import pytest

from paper_1907_12834_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qlga():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1907_12834_b200 import qlga as mod      # fails loudly if libqlga.so is missing
    return mod


def _close(a, b):
    # the tolerance of tests/test_gpu_parity.py::test_observables_match_oracle
    return all(abs(x - y) <= 1e-11 * max(1.0, abs(y)) for x, y in zip(a, b))


def test_noalloc_sums_match_the_context_path_on_two_calls_in_a_row(qlga):
    import torch
    c = (1.0, 0.3, -0.1)
    out = torch.full((qlga.NSUMS,), float("nan"), dtype=torch.float64, device="cuda")
    for precision, cdt in (("f64", torch.complex128), ("f32", torch.complex64)):
        for ndim, dims in ((2, (70, 45)), (1, (3000, 1)), (3, (20, 9, 7))):
            q0 = inputs.random_spinor_state(dims[:ndim] if ndim > 1 else dims, seed=9 + ndim, amplitude=0.3)
            sim = qlga.Qlga(ndim, dims, c, order="interleaved", precision=precision, keep_previous=True)
            sim.set_state_q(q0.astype(sim.np_cdtype))
            shape = q0.shape
            # call 1: the initial state, no previous state
            want1 = sim.observable_sums()
            q_dev = torch.empty(shape, dtype=cdt, device="cuda")
            sim.get_state_q(q_dev)
            qlga.observable_sums_noalloc(q_dev, None, ndim, dims, precision, out)
            got1 = out.cpu().numpy()
            assert _close(got1[:15], want1[:15]), (precision, ndim)
            assert got1[15] == 0.0 and got1[16] == 0.0 and np.isnan(want1[15])
            # call 2, straight after, on another state and with the previous state (eq. 85's two sums): the
            # array still holds call 1's partials, which must not leak into the result
            sim.step(2)
            qprev_dev = q_dev.clone()
            sim.get_state_q(qprev_dev)
            sim.step(1)
            sim.get_state_q(q_dev)
            want2 = sim.observable_sums()
            qlga.observable_sums_noalloc(q_dev, qprev_dev, ndim, dims, precision, out)
            got2 = out.cpu().numpy()
            assert _close(got2, want2), (precision, ndim, got2 - want2)
            assert not _close(got2[:15], want1[:15])                   # the state did change between the calls
            # a smaller grid than the context's (fewer partials than the array held before): same sums to rounding
            qlga.observable_sums_noalloc(q_dev, qprev_dev, ndim, dims, precision, out, nblocks=3)
            assert _close(out.cpu().numpy(), want2)
            sim.close()


def test_noalloc_rejects_sizes_beyond_the_static_scratch(qlga):
    import torch
    q = torch.zeros((5, 2, 4, 8), dtype=torch.complex128, device="cuda")
    out = torch.zeros(qlga.NSUMS, dtype=torch.float64, device="cuda")
    with pytest.raises(qlga.QlgaError) as e:
        qlga.observable_sums_noalloc(q, None, 2, (8, 4), "f64", out, nblocks=qlga.NOALLOC_MAX_BLOCKS + 1)
    assert e.value.status == qlga.QLGA_EINVAL and "QLGA_NOALLOC_MAX_BLOCKS" in str(e.value)
    with pytest.raises(qlga.QlgaError) as e:
        qlga.observable_sums_noalloc(q, None, 1, (8, 4), "f64", out)
    assert e.value.status == qlga.QLGA_EINVAL
    qlga.observable_sums_noalloc(q, None, 2, (8, 4), "f64", out, nblocks=qlga.NOALLOC_MAX_BLOCKS)   # the limit itself is fine
    assert float(out.abs().sum()) == 0.0
