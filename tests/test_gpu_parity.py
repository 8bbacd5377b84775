"""Parity of the CUDA path (through the C ABI, libqlga.so) with the CPU oracle,
element by element on the same seeded inputs.  Needs a B200: run with -m gpu.

Bar (BASELINE.json north_star): max relative L2 field error 1e-12 (fp64) and
1e-5 (fp32) over all 10 spinor planes after the stated step counts."""
import numpy as np
import pytest

from paper_1907_12834_b200 import inputs
from conftest import rel_l2, norm2

pytestmark = pytest.mark.gpu

TOL64 = 1e-12
TOL32 = 1e-5
ORDERS = {"plain": 0, "interleaved": 1}


@pytest.fixture(scope="module")
def qlga():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1907_12834_b200 import qlga as mod      # fails loudly if libqlga.so is missing
    return mod


def run_gpu(qlga, q0, ndim, couplings, order, steps, precision="f64", options=(), keep_previous=False):
    dims = tuple(reversed(q0.shape[2:]))                   # (Nx, Ny) or (Nx, Ny, Nz)
    sim = qlga.Qlga(ndim, dims, couplings, order=order, precision=precision, keep_previous=keep_previous)
    for k, v in options:
        sim.set_option(k, v)
    sim.set_state_q(q0)
    sim.step(steps)
    out = sim.get_state_q().astype(np.complex128)
    sim.close()
    return out


# ---------------------------------------------------------------------------
# generic lattices: several tiles and a ragged tail, tiny and degenerate sizes
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("order", ["plain", "interleaved"])
@pytest.mark.parametrize("L", [1, 2, 7, 119, 120, 121, 1000])
def test_1d_random_state_matches_oracle(qlga, oracle, order, L):
    c = (1.0, 0.3, -0.1)
    q0 = inputs.random_spinor_state((L, 1), seed=100 + L, amplitude=0.3)
    ref = oracle.step(q0, 1, c, ORDERS[order], 3)
    out = run_gpu(qlga, q0, 1, c, order, 3)
    assert rel_l2(out, ref) < TOL64


@pytest.mark.parametrize("order", ["plain", "interleaved"])
@pytest.mark.parametrize("dims", [(1, 1), (5, 3), (4, 57), (130, 9), (100, 70), (67, 130)])
def test_2d_random_state_matches_oracle(qlga, oracle, order, dims):
    c = (0.8, -0.25, 0.4)
    q0 = inputs.random_spinor_state(dims, seed=7 + dims[0], amplitude=0.3)
    ref = oracle.step(q0, 2, c, ORDERS[order], 2)
    out = run_gpu(qlga, q0, 2, c, order, 2)
    assert rel_l2(out, ref) < TOL64


@pytest.mark.parametrize("tile_y", [1, 2, 4, 8])
def test_2d_all_y_tilings(qlga, oracle, tile_y):
    c = (1.0, 0.3, -0.1)
    q0 = inputs.random_spinor_state((37, 150), seed=3, amplitude=0.2)
    ref = oracle.step(q0, 2, c, 1, 2)
    out = run_gpu(qlga, q0, 2, c, "interleaved", 2, options=[(qlga.OPT_TILE_Y, tile_y)])
    assert rel_l2(out, ref) < TOL64
    out = run_gpu(qlga, q0, 2, c, "interleaved", 2, options=[(qlga.OPT_TILE_Y, tile_y), (qlga.OPT_THREADS_X, 256)])
    assert rel_l2(out, ref) < TOL64


def test_large_angles_use_the_split_exponential(qlga, oracle):
    # O(1) amplitudes and couplings: interaction angles of several radians
    # (one step only: at these amplitudes every U multiplies rounding differences by
    # ~2 c0 s rho >> 1, so longer runs measure the map's sensitivity, not the kernels)
    c = (0.7, -0.4, 0.9)
    q0 = inputs.random_spinor_state((64, 1), seed=5, amplitude=1.5)
    for order in ("plain", "interleaved"):
        ref = oracle.step(q0, 1, c, ORDERS[order], 1)
        assert rel_l2(run_gpu(qlga, q0, 1, c, order, 1), ref) < TOL64
    q0 = inputs.random_spinor_state((9, 6), seed=6, amplitude=1.2)
    ref = oracle.step(q0, 2, c, 0, 1)
    assert rel_l2(run_gpu(qlga, q0, 2, c, "plain", 1), ref) < TOL64


@pytest.mark.parametrize("order", ["plain", "interleaved"])
def test_per_operator_path_matches_oracle_and_fused(qlga, oracle, order):
    c = (1.0, 0.3, -0.1)
    for ndim, dims in ((1, (333, 1)), (2, (40, 33))):
        q0 = inputs.random_spinor_state(dims, seed=21, amplitude=0.3)
        ref = oracle.step(q0, ndim, c, ORDERS[order], 2)
        a = run_gpu(qlga, q0, ndim, c, order, 2, options=[(qlga.OPT_PATH, 1)])
        b = run_gpu(qlga, q0, ndim, c, order, 2)
        assert rel_l2(a, ref) < TOL64 and rel_l2(b, ref) < TOL64
        assert rel_l2(a, b) < 1e-14


def test_temporal_blocking_matches_single_step_launches(qlga):
    # same arithmetic per site; only the (warp-uniform) polynomial degree can differ
    # where the warp composition differs, i.e. at the 1e-17 level
    c = (1.0, 0.3, -0.1)
    w = inputs.config3(L=5000)
    q0 = np.repeat(w.psi[:, None] / 2, 2, axis=1)
    base = run_gpu(qlga, q0, 1, c, "interleaved", 13, options=[(qlga.OPT_STEPS_PER_LAUNCH, 1)])
    for k in (2, 3, 5, 7):
        out = run_gpu(qlga, q0, 1, c, "interleaved", 13, options=[(qlga.OPT_STEPS_PER_LAUNCH, k)])
        assert rel_l2(out, base) < 1e-15
    out = run_gpu(qlga, q0, 1, c, "interleaved", 13, options=[(qlga.OPT_THREADS_X, 256), (qlga.OPT_STEPS_PER_LAUNCH, 4)])
    assert rel_l2(out, base) < 1e-15


# ---------------------------------------------------------------------------
# the five BASELINE.json configurations (full size where the oracle finishes in
# seconds, reduced step counts / lattices otherwise)
# ---------------------------------------------------------------------------
def _q_of(w):
    return np.repeat(w.psi[:, None] / 2, 2, axis=1)


@pytest.mark.parametrize("order", ["plain", "interleaved"])
def test_config1_full_length(qlga, oracle, order):
    w = inputs.config1()
    q0 = _q_of(w)
    ref = oracle.step(q0, 1, w.couplings, ORDERS[order], w.steps)
    out = run_gpu(qlga, q0, 1, w.couplings, order, w.steps)
    assert rel_l2(out, ref) < TOL64
    assert abs(norm2(out) / norm2(q0) - 1) < 1e-13
    d0 = np.abs(w.psi[0, 0]) ** 2
    dn = np.abs(out[0, 0, 0] + out[0, 1, 0]) ** 2
    assert np.sqrt(np.sum((dn - d0) ** 2) / np.sum(d0 ** 2)) < 5e-3        # stationary profile


def test_config2_reduced_steps_and_collision_variant(qlga, oracle):
    w = inputs.config2()                                  # full L = 65536, 25 of 50000 steps
    q0 = _q_of(w)
    ref = oracle.step(q0, 1, w.couplings, 1, 25)
    assert rel_l2(run_gpu(qlga, q0, 1, w.couplings, "interleaved", 25), ref) < TOL64
    w = inputs.config2(L=8192, centres=(8192 / 2 - 100, 8192 / 2 + 100))   # overlapping solitons
    q0 = _q_of(w)
    ref = oracle.step(q0, 1, w.couplings, 1, 300)
    assert rel_l2(run_gpu(qlga, q0, 1, w.couplings, "interleaved", 300), ref) < TOL64


def test_config3_reduced_fp64_and_fp32(qlga, oracle):
    w = inputs.config3(L=1 << 16)
    q0 = _q_of(w)
    ref = oracle.step(q0, 1, w.couplings, 1, 40)
    assert rel_l2(run_gpu(qlga, q0, 1, w.couplings, "interleaved", 40), ref) < TOL64
    q32 = q0.astype(np.complex64)
    ref32 = oracle.step(q32.astype(np.complex128), 1, w.couplings, 1, 40)
    assert rel_l2(run_gpu(qlga, q32, 1, w.couplings, "interleaved", 40, precision="f32"), ref32) < TOL32


def test_config4_reduced(qlga, oracle):
    w = inputs.config4(L=192, core=8.0)
    q0 = _q_of(w)
    for order in ("plain", "interleaved"):
        ref = oracle.step(q0, 2, w.couplings, ORDERS[order], 12)
        assert rel_l2(run_gpu(qlga, q0, 2, w.couplings, order, 12), ref) < TOL64


def test_config5_reduced_fp64_and_fp32(qlga, oracle):
    w = inputs.config5(L=160, core=6.0, spacing=24.0, offset=32.0)
    q0 = _q_of(w)
    ref = oracle.step(q0, 2, w.couplings, 1, 10)
    assert rel_l2(run_gpu(qlga, q0, 2, w.couplings, "interleaved", 10), ref) < TOL64
    q32 = q0.astype(np.complex64)
    ref32 = oracle.step(q32.astype(np.complex128), 2, w.couplings, 1, 10)
    assert rel_l2(run_gpu(qlga, q32, 2, w.couplings, "interleaved", 10, precision="f32"), ref32) < TOL32


def test_fp32_plain_and_1d_random(qlga, oracle):
    c = (1.0, 0.3, -0.1)
    q32 = inputs.random_spinor_state((777, 1), seed=2, amplitude=0.2).astype(np.complex64)
    for order in ("plain", "interleaved"):
        ref = oracle.step(q32.astype(np.complex128), 1, c, ORDERS[order], 20)
        assert rel_l2(run_gpu(qlga, q32, 1, c, order, 20, precision="f32"), ref) < TOL32


def test_long_run_error_growth(qlga, oracle):
    # 150 interleaved 2D steps (1200 interaction exponentials per site) on a vortex
    # quadrupole stay at rounding level against the oracle, norm conserved.  (Beyond
    # ~200 steps this small, violently evolving lattice amplifies rounding differences
    # exponentially -- the oracle's own double and long-double builds part ways at the
    # same rate, 2.8e-12 at 300 steps; DESIGN.md section 8 -- so a longer comparison
    # would measure the flow's sensitivity, not the kernels.)
    w = inputs.config4(L=96, core=8.0)
    q0 = _q_of(w)
    ref = oracle.step(q0, 2, w.couplings, 1, 150)
    a = run_gpu(qlga, q0, 2, w.couplings, "interleaved", 150)
    assert rel_l2(a, ref) < 1e-13
    assert abs(norm2(a) / norm2(q0) - 1) < 1e-13


# ---------------------------------------------------------------------------
# full-size lattices in the launch configuration bench.py times: windowed parity
# (the domain of dependence of a site is exactly 4 sites per step per direction)
# ---------------------------------------------------------------------------
def _windowed_parity(qlga, oracle, ndim, dims, couplings, q_dev_in, steps, windows, P, precision, tol,
                     order="interleaved"):
    import torch
    nx, ny = dims
    sim = qlga.Qlga(ndim, dims, couplings, order=order, precision=precision)
    sim.set_state_q(q_dev_in)
    sim.step(steps)
    cdt = torch.complex128 if precision == "f64" else torch.complex64
    out_dev = torch.empty((5, 2, ny, nx), dtype=cdt, device="cuda")
    sim.get_state_q(out_dev)
    h = 4 * steps
    worst = 0.0
    for (cx, cy) in windows:
        xs = (np.arange(cx - h, cx + P + h)) % nx
        ys = (np.arange(cy - h, cy + P + h)) % ny if ndim == 2 else np.array([0])
        xi = torch.as_tensor(xs, device="cuda"); yi = torch.as_tensor(ys, device="cuda")
        patch_in = q_dev_in[:, :, yi][:, :, :, xi].cpu().numpy().astype(np.complex128)
        patch_out = out_dev[:, :, yi][:, :, :, xi].cpu().numpy().astype(np.complex128)
        ref = oracle.step(patch_in, ndim, couplings, ORDERS[order], steps)   # periodic patch: only the centre is valid
        if ndim == 2:
            a, b = patch_out[:, :, h:h + P, h:h + P], ref[:, :, h:h + P, h:h + P]
        else:
            a, b = patch_out[:, :, :, h:h + P], ref[:, :, :, h:h + P]
        worst = max(worst, rel_l2(a, b))
    sim.close()
    assert worst < tol, worst


def test_config5_full_size_windowed(qlga, oracle):
    import torch
    L = 8192
    w = inputs.config5(L=L)
    psi = torch.from_numpy(w.psi).cuda()
    q_dev = (psi[:, None] / 2).expand(5, 2, L, L).contiguous()
    del psi
    windows = [(0, 0), (L // 2 + 40, L // 2 - 260), (L - 20, L - 20), (1234, 4321)]   # wrap corners, a vortex core, bulk
    _windowed_parity(qlga, oracle, 2, (L, L), w.couplings, q_dev, 2, windows, 24, "f64", TOL64)
    _windowed_parity(qlga, oracle, 2, (L, L), w.couplings, q_dev, 2, windows[:3], 24, "f64", TOL64, order="plain")
    q32 = q_dev.to(torch.complex64)
    del q_dev
    _windowed_parity(qlga, oracle, 2, (L, L), w.couplings, q32, 2, windows, 24, "f32", TOL32)
    _windowed_parity(qlga, oracle, 2, (L, L), w.couplings, q32, 2, windows[:3], 24, "f32", TOL32, order="plain")


def test_config4_and_config2_full_size_windowed(qlga, oracle):
    import torch
    L = 2048
    w = inputs.config4(L=L)
    q_dev = torch.from_numpy(_q_of(w)).cuda()
    windows = [(0, 0), (L // 4 - 12, L // 4 - 12), (L - 20, L // 2)]            # wrap corner, a vortex core, wrap edge
    for order in ("interleaved", "plain"):
        _windowed_parity(qlga, oracle, 2, (L, L), w.couplings, q_dev, 3, windows, 24, "f64", TOL64, order=order)
    L = 65536                                                                  # temporal blocking: 4 steps per launch
    w = inputs.config2(L=L)
    q_dev = torch.from_numpy(_q_of(w)).cuda()
    windows = [(0, 0), (L // 4 - 60, 0), (3 * L // 4 - 60, 0), (L - 40, 0)]
    for order in ("interleaved", "plain"):
        _windowed_parity(qlga, oracle, 1, (L, 1), w.couplings, q_dev, 9, windows, 120, "f64", TOL64, order=order)


def test_config3_full_size_windowed(qlga, oracle):
    import torch
    L = 1 << 22
    w = inputs.config3(L=L)
    q_dev = torch.from_numpy(_q_of(w)).cuda()
    windows = [(0, 0), (L // 4 - 50, 0), (L - 30, 0), (3 * L // 4, 0)]
    _windowed_parity(qlga, oracle, 1, (L, 1), w.couplings, q_dev, 5, windows, 100, "f64", TOL64)
    # plain ordering and fp32 run two time steps per launch on a lattice of this size
    _windowed_parity(qlga, oracle, 1, (L, 1), w.couplings, q_dev, 5, windows, 100, "f64", TOL64, order="plain")
    q32 = q_dev.to(torch.complex64)
    _windowed_parity(qlga, oracle, 1, (L, 1), w.couplings, q32, 5, windows, 100, "f32", TOL32)
    _windowed_parity(qlga, oracle, 1, (L, 1), w.couplings, q32, 5, windows, 100, "f32", TOL32, order="plain")


# ---------------------------------------------------------------------------
# observables, vorticity, boundary behaviour
# ---------------------------------------------------------------------------
def test_observables_match_oracle(qlga, oracle):
    c = (1.0, 0.3, -0.1)
    for ndim, dims, keep in ((1, (3000, 1), False), (2, (70, 45), True), (2, (70, 45), False)):
        q0 = inputs.random_spinor_state(dims, seed=9, amplitude=0.3)
        sim = qlga.Qlga(ndim, dims, c, order="interleaved", keep_previous=keep)
        sim.set_state_q(q0)
        ob0 = sim.observables()
        ref0 = oracle.observables(q0, ndim, c)
        assert np.isnan(ob0["e_dt_re"]) and ob0["step"] == 0
        for k, v in ref0.items():
            if not k.startswith("e_dt"):
                assert abs(ob0[k] - v) <= 1e-11 * max(1.0, abs(v)), k
        sim.step(3)
        q3 = sim.get_state_q()
        q2 = oracle.step(q0, ndim, c, 1, 2)
        ob = sim.observables()
        ref = oracle.observables(q3, ndim, c, qprev=q2)
        assert ob["step"] == 3
        for k, v in ref.items():
            if k.startswith("e_dt"):
                if ndim == 1 or keep:
                    assert abs(ob[k] - v) < 1e-10, k
                else:
                    assert np.isnan(ob[k])
            else:
                assert abs(ob[k] - v) <= 1e-11 * max(1.0, abs(v)), k
        sim.close()


def test_diagnostics_on_ragged_lattices(qlga, oracle):
    # The shared-memory diagnostics of round 2 -- observables_ring_kernel (units of 128 columns x a segment of rows, loads
    # staged through a cp.async ring, psi handed to the left neighbour) and vorticity_tile_kernel (tiles of 32 x 8
    # sites with a one-site halo) -- on lattices smaller than a unit / tile, with ragged last units and tiles, one
    # row, one column, several segments, in fp64 and fp32, with the previous-state overlap of eq. (85).
    c = (1.0, 0.3, -0.1)
    for dims in ((1, 1), (5, 3), (31, 7), (33, 9), (130, 9), (1, 40), (257, 40), (300, 203), (128, 64), (129, 2100)):
        q0 = inputs.random_spinor_state(dims, seed=17 + dims[0], amplitude=0.3)
        for precision, rtol, vtol in (("f64", 1e-11, 1e-12), ("f32", 2e-6, 1e-6)):
            qin = q0 if precision == "f64" else q0.astype(np.complex64)
            q64 = qin.astype(np.complex128)
            sim = qlga.Qlga(2, dims, c, precision=precision, keep_previous=True)
            sim.set_state_q(qin)
            ob = sim.observables()
            ref = oracle.observables(q64, 2, c)
            for k, v in ref.items():
                if not k.startswith("e_dt"):
                    assert abs(ob[k] - v) <= rtol * max(1.0, abs(v)), (dims, precision, k)
            assert np.abs(sim.vorticity() - oracle.vorticity(q64)).max() < vtol, (dims, precision)
            sim.step(1)
            q1 = sim.get_state_q().astype(np.complex128)
            ob = sim.observables()
            ref = oracle.observables(q1, 2, c, qprev=q64)
            for k, v in ref.items():
                assert abs(ob[k] - v) <= (1e-9 if precision == "f64" else 2e-5) * max(1.0, abs(v)), (dims, precision, k)
            sim.close()


def test_psi_roundtrip_and_device_transfers(qlga, oracle):
    import torch
    c = (1.0, 0.3, -0.1)
    psi = inputs.random_field((50, 20), seed=4)
    sim = qlga.Qlga(2, (50, 20), c)
    sim.set_state_psi(psi)
    q = sim.get_state_q()
    assert np.array_equal(q[:, 0], psi / 2) and np.array_equal(q[:, 1], psi / 2)      # reading R6
    assert np.array_equal(sim.get_state_psi(), psi)
    sim.set_state_psi(torch.from_numpy(psi).cuda())
    out = torch.empty((5, 20, 50), dtype=torch.complex128, device="cuda")
    sim.get_state_psi(out)
    assert np.array_equal(out.cpu().numpy(), psi)
    sim.close()


def test_vorticity_matches_oracle(qlga, oracle):
    c = (1.0, 0.3, -0.1)
    w = inputs.config4(L=96, core=6.0)
    q0 = _q_of(w)
    q0 += inputs.random_spinor_state((96, 96), seed=1, amplitude=1e-3)
    for precision, tol in (("f64", 1e-12), ("f32", 1e-6)):
        sim = qlga.Qlga(2, (96, 96), c, precision=precision)
        qin = q0 if precision == "f64" else q0.astype(np.complex64)
        sim.set_state_q(qin)
        om = sim.vorticity()
        ref = oracle.vorticity(qin.astype(np.complex128))
        assert np.abs(om - ref).max() < tol
        sim.step(5)
        om = sim.vorticity()
        ref = oracle.vorticity(sim.get_state_q().astype(np.complex128))
        assert np.abs(om - ref).max() < tol
        assert abs(om.sum()) < 1e-3
        sim.close()


def test_error_paths(qlga):
    c = (1.0, 0.3, -0.1)
    sim = qlga.Qlga(1, (64, 1), c)
    with pytest.raises(qlga.QlgaError) as e:
        sim.step(1)
    assert e.value.status == qlga.QLGA_ESTATE
    sim.set_state_psi(inputs.random_field((64, 1), seed=1))
    with pytest.raises(qlga.QlgaError) as e:
        sim.vorticity()
    assert e.value.status == qlga.QLGA_EUNSUP
    with pytest.raises(qlga.QlgaError) as e:
        sim.step(-1)
    assert e.value.status == qlga.QLGA_EINVAL
    with pytest.raises(qlga.QlgaError):
        sim.set_option(qlga.OPT_TILE_Y, 3)
    before = sim.get_state_q()
    sim.step(0)
    assert np.array_equal(sim.get_state_q(), before)
    assert sim.launch_count() >= 1
    sim.close()
    with pytest.raises(qlga.QlgaError):
        qlga.Qlga(1, (64, 2), c)


def test_gpu_unitarity_1000_steps(qlga):
    c = (1.0, 0.3, -0.1)
    psi = inputs.smooth_random_field((4096, 1), seed=4, amplitude=0.08)
    q0 = np.repeat(psi[:, None] / 2, 2, axis=1) + inputs.random_spinor_state((4096, 1), seed=6, amplitude=1e-3)
    for order in ("plain", "interleaved"):
        out = run_gpu(qlga, q0, 1, c, order, 1000)
        assert abs(norm2(out) / norm2(q0) - 1) < 1e-13


# ---------------------------------------------------------------------------
# density / eq. (115) and vortex detection
# ---------------------------------------------------------------------------
def test_density_and_l2_error_match_oracle(qlga, oracle):
    c = (1.0, 0.3, -0.1)
    for precision, tol in (("f64", 1e-13), ("f32", 1e-6)):
        for ndim, dims in ((1, (1500, 1)), (2, (90, 70))):
            q0 = inputs.random_spinor_state(dims, seed=5, amplitude=0.3)
            qin = q0 if precision == "f64" else q0.astype(np.complex64)
            sim = qlga.Qlga(ndim, dims, c, precision=precision)
            sim.set_state_q(qin)
            rho0 = sim.density()
            ref0 = oracle.density(qin.astype(np.complex128))
            assert np.abs(rho0 - ref0).max() <= tol * ref0.max()
            assert sim.density_l2_error(rho0) <= (1e-28 if precision == "f64" else 1e-10)   # f32: rho0 itself is rounded
            sim.step(4)
            qn = sim.get_state_q().astype(np.complex128)
            eps = sim.density_l2_error(rho0)
            ref = oracle.density_l2_error(qn, rho0.astype(np.float64))
            assert abs(eps - ref) <= 1e-10 * ref + 1e-20
            import torch
            assert abs(sim.density_l2_error(torch.from_numpy(rho0).cuda()) - eps) <= 1e-14 * eps
            sim.close()


def test_l2_error_convergence_study(qlga):
    # Figs. 23-24: eps of eq. (115) after 1000 steps against the lattice
    # size, soliton width scaled with L.  The paper prints -5.38 for the dark state with the
    # interleaved ordering (run parameters not given: DESIGN.md section 12b); "engineering
    # precision" is a slope below -4.
    from paper_1907_12834_b200 import convergence
    dark = convergence.l2_convergence("dark", 14, (1.0, 0.3, -0.1), sizes=(256, 512, 1024, 2048))
    s_int, e_int = dark["interleaved"]
    s_pl, e_pl = dark["plain"]
    assert -6.2 < s_int < -4.8
    assert all(a > b for a, b in zip(e_int, e_int[1:]))
    assert e_int[0] < 0.6 * e_pl[0]                  # interleaving pays on a background (small lattice)
    bright = convergence.l2_convergence("bright", 14, (-1.0, -0.5, 0.2), sizes=(256, 512, 1024))
    assert bright["interleaved"][0] < -4.0 and bright["plain"][0] < -4.0
    assert bright["interleaved"][1][0] < bright["plain"][1][0]


def test_vortices_match_oracle_winding(qlga, oracle):
    c = (1.0, 0.3, -0.1)
    L = 96
    w = inputs.config4(L=L, core=6.0)
    q0 = _q_of(w) + inputs.random_spinor_state((L, L), seed=2, amplitude=2e-3)
    for precision in ("f64", "f32"):
        sim = qlga.Qlga(2, (L, L), c, precision=precision)
        qin = q0 if precision == "f64" else q0.astype(np.complex64)
        sim.set_state_q(qin)
        sim.step(40)
        rec, count = sim.vortices()
        ref = oracle.winding(sim.get_state_q().astype(np.complex128))
        want = sorted((int(j), int(x), int(y), int(ref[j, y, x])) for j, y, x in np.argwhere(ref != 0))
        got = sorted(tuple(int(v) for v in r) for r in rec)
        assert count == len(want) and got == want
        assert count >= 8 and sum(r[3] for r in got) == 0          # the quadrupoles are there; total winding 0
        rec2, count2 = sim.vortices(max_out=3)                      # truncation keeps the true count
        assert count2 == count and len(rec2) == 3
        sim.close()
    sim = qlga.Qlga(1, (64, 1), c)
    sim.set_state_psi(inputs.random_field((64, 1), seed=1))
    with pytest.raises(qlga.QlgaError) as e:
        sim.vortices()
    assert e.value.status == qlga.QLGA_EUNSUP
    sim.close()


# ---------------------------------------------------------------------------
# the 3D lattice (12 factors, U^(1/12))
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("order", ["plain", "interleaved"])
@pytest.mark.parametrize("dims", [(1, 1, 1), (5, 3, 2), (130, 5, 3), (9, 125, 4), (6, 7, 131), (40, 33, 21)])
def test_3d_random_state_matches_oracle(qlga, oracle, order, dims):
    c = (0.8, -0.25, 0.4)
    q0 = inputs.random_spinor_state(dims, seed=3 + dims[0], amplitude=0.3)
    ref = oracle.step(q0, 3, c, ORDERS[order], 2)
    out = run_gpu(qlga, q0, 3, c, order, 2)
    assert rel_l2(out, ref) < TOL64
    a = run_gpu(qlga, q0, 3, c, order, 2, options=[(qlga.OPT_PATH, 1)])
    assert rel_l2(a, ref) < TOL64


def test_3d_fp32_observables_density_and_previous_state(qlga, oracle):
    c = (1.0, 0.3, -0.1)
    dims = (36, 20, 17)
    q0 = inputs.random_spinor_state(dims, seed=8, amplitude=0.2)
    q32 = q0.astype(np.complex64)
    ref32 = oracle.step(q32.astype(np.complex128), 3, c, 1, 5)
    assert rel_l2(run_gpu(qlga, q32, 3, c, "interleaved", 5, precision="f32"), ref32) < TOL32
    for keep in (True, False):
        sim = qlga.Qlga(3, dims, c, order="interleaved", keep_previous=keep)
        sim.set_state_q(q0)
        sim.step(3)
        q3 = sim.get_state_q()
        ob = sim.observables()
        ref = oracle.observables(q3, 3, c, qprev=oracle.step(q0, 3, c, 1, 2))
        for k, v in ref.items():
            if k.startswith("e_dt"):
                assert (abs(ob[k] - v) < 1e-10) if keep else np.isnan(ob[k])
            else:
                assert abs(ob[k] - v) <= 1e-11 * max(1.0, abs(v)), k
        assert np.abs(sim.density() - oracle.density(q3)).max() < 1e-13
        assert np.array_equal(sim.get_state_psi(), q3[:, 0] + q3[:, 1])
        with pytest.raises(qlga.QlgaError) as e:
            sim.vorticity()
        assert e.value.status == qlga.QLGA_EUNSUP
        sim.close()


def test_dispersion_relation_of_kicked_solitons_fig5(qlga, oracle):
    # SURVEY.md 8(f) row 4 / Fig. 5: energies of kicked solitons measured with
    # eq. (85) on the CUDA path follow E = p^2 - k^2 (eq. 74) and E = p^2 + 2 k^2,
    # and agree with the oracle's eq. (85) on the same input.
    from paper_1907_12834_b200 import dispersion
    L, k = 1024, 1.0 / 16
    for kind, row, c in (("bright", 3, (-1.0, -0.5, 0.2)), ("dark", 5, (1.0, 0.3, -0.1))):
        es = []
        for n in (0, 4, 8):
            p = 2 * np.pi * n / L
            e = dispersion.measured_energy(kind, row, c, L, k, n, steps=21)
            es.append(e)
            assert abs(e - inputs.predicted_energy(kind, k, p)) < 0.02 * (p * p + k * k), (kind, n)
            q0 = oracle.split_psi(inputs.kicked_soliton(kind, row, c, L, k, n))
            qa = oracle.step(q0, 1, c, 1, 20)
            qb = oracle.step(qa, 1, c, 1, 1)
            assert e == pytest.approx(oracle.observables(qb, 1, c, qprev=qa)["e_dt_re"], rel=1e-9, abs=1e-14)
        assert es[0] < es[1] < es[2]                       # parabolic in p


def test_spin_gauge_degenerate_transverse_spin(qlga, oracle):
    # The fp64 kernels evaluate U in the gauge e = F_+/|F_+| (R12b).  Cases where the
    # transverse spin vanishes or is too small to normalise: single-channel and (m, -m) states
    # (F_+ = 0 exactly), amplitudes whose |F_+|^2 falls below the 1e-36 cut-off, and a state that
    # mixes sites of both kinds inside one warp.
    c = (1.0, 0.3, -0.1)
    L = 96
    rng = np.random.default_rng(77)
    base = inputs.random_spinor_state((L, 1), seed=31, amplitude=0.1)
    only2 = np.zeros_like(base); only2[0] = base[0]                       # m = +2 only
    pair = np.zeros_like(base); pair[0] = base[0]; pair[4] = base[4]      # m = +2 and -2: F_+ = 0, A00 != 0
    tiny = base * 1e-10                                                   # |F_+|^2 ~ 1e-42 < 1e-36
    mixed = base.copy(); mixed[1:4, :, :, ::2] = 0.0                      # every other site has F_+ = 0
    for name, q0 in (("only2", only2), ("pair", pair), ("tiny", tiny), ("mixed", mixed)):
        for order in ("plain", "interleaved"):
            ref = oracle.step(q0, 1, c, ORDERS[order], 6)
            assert rel_l2(run_gpu(qlga, q0, 1, c, order, 6), ref) < TOL64, (name, order)
    q2 = inputs.random_spinor_state((24, 20), seed=32, amplitude=0.1)
    q2[1:4, :, ::3, :] = 0.0
    ref = oracle.step(q2, 2, c, 1, 4)
    assert rel_l2(run_gpu(qlga, q2, 2, c, "interleaved", 4), ref) < TOL64


def test_chemical_potential(qlga, oracle):
    # mu psi_m term (eq. 75): parity with the oracle's orc_step_mu, both orderings,
    # 1D with temporal blocking, 2D, fp32, the per-operator path, a phase beyond the fast path's range,
    # and the dispersion relation E = mu + p^2 - k^2 measured with eq. (85).
    c, mu = (1.0, 0.3, -0.1), 0.0375
    def run(q0, ndim, order, steps, precision="f64", options=(), mu_=mu):
        dims = tuple(reversed(q0.shape[2:]))
        sim = qlga.Qlga(ndim, dims, c, order=order, precision=precision)
        for k, v in options:
            sim.set_option(k, v)
        sim.set_chemical_potential(mu_)
        sim.set_state_q(q0)
        sim.step(steps)
        out = sim.get_state_q().astype(np.complex128)
        sim.close()
        return out
    q1 = inputs.random_spinor_state((300, 1), seed=41, amplitude=0.05)
    q2 = inputs.random_spinor_state((40, 33), seed=42, amplitude=0.05)
    for order in ("plain", "interleaved"):
        assert rel_l2(run(q1, 1, order, 9), oracle.step(q1, 1, c, ORDERS[order], 9, mu=mu)) < TOL64
        assert rel_l2(run(q2, 2, order, 5), oracle.step(q2, 2, c, ORDERS[order], 5, mu=mu)) < TOL64
        assert rel_l2(run(q2, 2, order, 3, options=((qlga.OPT_PATH, 1),)),
                      oracle.step(q2, 2, c, ORDERS[order], 3, mu=mu)) < TOL64
    q32 = q2.astype(np.complex64)
    assert rel_l2(run(q32, 2, "interleaved", 5, precision="f32"),
                  oracle.step(q32.astype(np.complex128), 2, c, 1, 5, mu=mu)) < TOL32
    assert rel_l2(run(q1, 1, "plain", 3, mu_=2.5), oracle.step(q1, 1, c, 0, 3, mu=2.5)) < TOL64   # general path
    assert rel_l2(run(q1, 1, "plain", 3, mu_=0.0), oracle.step(q1, 1, c, 0, 3)) < TOL64
    from paper_1907_12834_b200 import dispersion
    cb, L, k, n = (-1.0, -0.5, 0.2), 1024, 1.0 / 16, 4
    sim = qlga.Qlga(1, (L, 1), cb)
    sim.set_chemical_potential(0.011)
    sim.set_state_psi(inputs.kicked_soliton("bright", 3, cb, L, k, n))
    sim.step(21)
    p = 2 * np.pi * n / L
    assert abs(sim.observables()["e_dt_re"] - (0.011 + p * p - k * k)) < 0.02 * (p * p + k * k)
    with pytest.raises(qlga.QlgaError) as e:
        sim.set_chemical_potential(float("nan"))
    assert e.value.status == qlga.QLGA_EINVAL
    sim.close()


def test_vorticity_and_vortices_degenerate_phases(qlga, oracle):
    # The vorticity / vortex kernels count quadrant changes around the loop instead of calling atan2, and
    # fall back to the term-by-term definition when a vertex is exactly zero or two vertices are exactly
    # antiparallel.  Fields built to sit on those cases: real-valued (every phase 0 or pi), values on the
    # axes, exact zeros sprinkled in, and 8th roots of unity (neighbours exactly antiparallel or orthogonal).
    c = (1.0, 0.3, -0.1)
    nx, ny = 37, 29
    rng = np.random.default_rng(91)
    real = rng.standard_normal((5, ny, nx)) + 0j
    axes = np.where(rng.random((5, ny, nx)) < 0.5, 1.0, 1j) * rng.standard_normal((5, ny, nx))
    unit = np.array([1, 1 + 1j, 1j, -1 + 1j, -1, -1 - 1j, -1j, 1 - 1j])          # exact directions, 45 degrees apart
    roots = unit[rng.integers(0, 8, (5, ny, nx))] * 2.0 ** rng.integers(-3, 3, (5, ny, nx))
    zeros = inputs.random_field((nx, ny), seed=92)
    zeros[rng.random((5, ny, nx)) < 0.15] = 0.0
    generic = inputs.random_field((nx, ny), seed=93)
    for name, psi in (("real", real), ("axes", axes), ("roots", roots), ("zeros", zeros), ("generic", generic)):
        q = np.repeat(psi[:, None] / 2, 2, axis=1)
        for precision in ("f64", "f32"):
            sim = qlga.Qlga(2, (nx, ny), c, precision=precision)
            sim.set_state_q(q.astype(sim.np_cdtype))
            state = sim.get_state_q().astype(np.complex128)
            om = sim.vorticity().astype(np.float64)
            rec, count = sim.vortices()
            sim.close()
            tol = 1e-10 if precision == "f64" else 2e-6
            assert np.abs(om - oracle.vorticity(state)).max() < tol, (name, precision)
            wind = oracle.winding(state)
            want = sorted((int(j), int(x), int(y), int(wind[j, y, x])) for j, y, x in np.argwhere(wind != 0))
            assert count == len(want) and sorted(tuple(int(v) for v in r) for r in rec) == want, (name, precision)


def test_plain_ordering_trailing_interaction(qlga, oracle):
    # Plain ordering, 2D/3D: inside one qlga_step call the U of step t+1 rides on the end of step t's x pass
    # (QLGA_OPT_FUSE_PLAIN_U, default on).  Same operator product: parity with the oracle for every split of
    # the steps into calls, with the option off, with a previous-state buffer (eq. 85 needs a true state of
    # the time series in it), and in fp32 / 3D.
    c = (1.0, 0.3, -0.1)
    q0 = inputs.random_spinor_state((45, 38), seed=51, amplitude=0.06)
    refs = {n: oracle.step(q0, 2, c, 0, n) for n in (1, 2, 3, 5, 6)}
    for calls in ((1,), (2,), (3,), (5,), (2, 3), (1, 1, 1), (6,)):
        for fuse in (1, 0):
            for keep in (False, True):
                sim = qlga.Qlga(2, (45, 38), c, order="plain", keep_previous=keep)
                sim.set_option(qlga.OPT_FUSE_PLAIN_U, fuse)
                sim.set_state_q(q0)
                for n in calls:
                    sim.step(n)
                out = sim.get_state_q()
                ob = sim.observables()
                sim.close()
                total = sum(calls)
                assert rel_l2(out, refs[total]) < TOL64, (calls, fuse, keep)
                if keep:
                    prev = oracle.step(q0, 2, c, 0, total - 1) if total > 1 else q0
                    want = oracle.observables(refs[total], 2, c, qprev=prev)
                    assert ob["e_dt_re"] == pytest.approx(want["e_dt_re"], rel=1e-9, abs=1e-13), (calls, fuse)
                    assert ob["e_dt_im"] == pytest.approx(want["e_dt_im"], rel=1e-9, abs=1e-13), (calls, fuse)
    q3 = inputs.random_spinor_state((12, 10, 9), seed=52, amplitude=0.06)
    assert rel_l2(run_gpu(qlga, q3, 3, c, "plain", 4), oracle.step(q3, 3, c, 0, 4)) < TOL64
    q32 = q0.astype(np.complex64)
    assert rel_l2(run_gpu(qlga, q32, 2, c, "plain", 5, precision="f32"),
                  oracle.step(q32.astype(np.complex128), 2, c, 0, 5)) < TOL32


def test_marching_pass_is_bit_identical_to_the_tile_kernel(qlga, oracle):
    # Plain ordering: the interaction-free strided passes run by column marching (QLGA_OPT_MARCH, default on):
    # the same operations in the same order as the tile kernel, so the states agree bit for bit -- lattices
    # smaller than the pipeline's run-in, ragged columns, several segments, 3D (y and z passes), every precision.
    c = (1.0, 0.3, -0.1)
    cases = [(2, (1, 1)), (2, (3, 2)), (2, (130, 7)), (2, (257, 300)), (2, (64, 2100)), (3, (5, 3, 2)), (3, (33, 40, 9)),
             (3, (12, 10, 70))]
    for ndim, dims in cases:
        q0 = inputs.random_spinor_state(dims, seed=61 + dims[0], amplitude=0.05)
        for precision in ("f64", "f32", "f32x"):
            qin = q0 if precision == "f64" else q0.astype(np.complex64)
            outs = []
            for march in (1, 0):
                sim = qlga.Qlga(ndim, dims, c, order="plain", precision=precision)
                sim.set_option(qlga.OPT_MARCH, march)
                sim.set_state_q(qin)
                sim.step(3)
                outs.append(sim.get_state_q())
                sim.close()
            assert np.array_equal(outs[0], outs[1]), (ndim, dims, precision)
        ref32 = oracle.step(q0.astype(np.complex64).astype(np.complex128), ndim, c, 0, 3)
        assert rel_l2(outs[0].astype(np.complex128), ref32) < TOL32            # f32x, marching off: the last run
        assert rel_l2(run_gpu(qlga, q0, ndim, c, "plain", 3), oracle.step(q0, ndim, c, 0, 3)) < TOL64


def test_band_mode_is_bit_identical_and_matches_the_oracle(qlga, oracle):
    # QLGA_OPT_BAND: the plain 2D step pipelined band by band (marching y pass -> ring in L2 -> x pass with the next
    # step's U), issued on the library's own streams (1) or replayed as a CUDA graph (2).  Same kernels, same
    # arithmetic: bit-identical to the two-launch step -- ragged last band, bands of one row, more slots than bands
    # would need, lattices with fewer than four bands (falls back), every precision, with and without the
    # previous-state buffer, every split of the steps into calls, options and the chemical potential changed
    # between calls (the instantiated graphs hold kernel arguments and must be dropped).  And against the oracle.
    c = (1.0, 0.3, -0.1)
    cases = [((300, 203), 16, 3), ((130, 64), 8, 2), ((257, 100), 25, 4), ((64, 40), 1, 8), ((96, 33), 0, 0), ((50, 20), 8, 3)]
    for dims, rows, slots in cases:
        q0 = inputs.random_spinor_state(dims, seed=71 + dims[0], amplitude=0.05)
        for precision in ("f64", "f32", "f32x"):
            qin = q0 if precision == "f64" else q0.astype(np.complex64)
            for keep in (False, True):
                outs, obs, launches = [], [], []
                for band in (0, 1, 2):
                    sim = qlga.Qlga(2, dims, c, order="plain", precision=precision, keep_previous=keep)
                    sim.set_option(qlga.OPT_BAND, band)
                    sim.set_option(qlga.OPT_BAND_ROWS, rows)
                    sim.set_option(qlga.OPT_BAND_SLOTS, slots)
                    sim.set_state_q(qin)
                    n0 = sim.launch_count()
                    sim.step(6)
                    launches.append(sim.launch_count() - n0)
                    outs.append(sim.get_state_q())
                    obs.append(sim.observables())
                    sim.close()
                assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2]), (dims, precision, keep)
                assert launches[1] == launches[2], (dims, launches)       # the graph replays what mode 1 launches
                if rows and dims[1] >= 4 * rows:
                    assert launches[1] > launches[0], (dims, launches)    # band mode really ran
                if keep:
                    for k in (1, 2):
                        assert obs[k]["e_dt_re"] == obs[0]["e_dt_re"] and obs[k]["e_dt_im"] == obs[0]["e_dt_im"]
        assert rel_l2(outs[2].astype(np.complex128),
                      oracle.step(q0.astype(np.complex64).astype(np.complex128), 2, c, 0, 6)) < TOL32      # f32x
    # several calls, an option and the chemical potential changed in between; against the oracle
    dims = (300, 203)
    q0 = inputs.random_spinor_state(dims, seed=77, amplitude=0.05)
    sim = qlga.Qlga(2, dims, c, order="plain")
    sim.set_option(qlga.OPT_BAND, 2)
    sim.set_option(qlga.OPT_BAND_ROWS, 16)
    sim.set_state_q(q0)
    sim.step(4)
    sim.step(3)
    assert rel_l2(sim.get_state_q(), oracle.step(q0, 2, c, 0, 7)) < TOL64
    q7 = sim.get_state_q()
    sim.set_chemical_potential(0.37)
    sim.set_option(qlga.OPT_BAND_ROWS, 24)
    sim.step(4)
    out = sim.get_state_q()
    sim.close()
    assert rel_l2(out, oracle.step(q7, 2, c, 0, 4, mu=0.37)) < TOL64
    ref = qlga.Qlga(2, dims, c, order="plain")
    ref.set_chemical_potential(0.37)
    ref.set_state_q(q7)
    ref.step(4)
    assert np.array_equal(out, ref.get_state_q())
    ref.close()
    # the options are validated
    sim = qlga.Qlga(2, dims, c, order="plain")
    for key, bad in ((qlga.OPT_BAND, 3), (qlga.OPT_BAND, -2), (qlga.OPT_BAND_ROWS, -2), (qlga.OPT_BAND_SLOTS, 1), (qlga.OPT_BAND_SLOTS, 9)):
        with pytest.raises(qlga.QlgaError):
            sim.set_option(key, bad)
    sim.close()


def test_option_validation_and_the_device_error_word(qlga):
    # (TILE_Y, THREADS_Y) are validated as a pair (only built kernels), STEPS_PER_LAUNCH against what the kernels support;
    # a state with a non-finite amplitude does not hang the sub-angle loop: the kernels raise the context's error word
    # and the next synchronising call reports QLGA_ESTATE (once), after which the context is usable again.
    c = (1.0, 0.3, -0.1)
    sim = qlga.Qlga(2, (40, 33), c)
    sim.set_option(qlga.OPT_TILE_Y, 4)
    with pytest.raises(qlga.QlgaError) as e:
        sim.set_option(qlga.OPT_THREADS_Y, 128)                 # 4 columns x 128 threads: no such kernel
    assert e.value.status == qlga.QLGA_EINVAL
    sim.set_option(qlga.OPT_THREADS_Y, 256)
    with pytest.raises(qlga.QlgaError):
        sim.set_option(qlga.OPT_TILE_Y, 1)                      # 1 x 256: no such kernel either
    sim.set_option(qlga.OPT_THREADS_Y, 0); sim.set_option(qlga.OPT_TILE_Y, 0)
    for key, bad in ((qlga.OPT_STEPS_PER_LAUNCH, 16), (qlga.OPT_EXP_MOD_SHIFT, 17), (qlga.OPT_F32_PHASE, 3), (qlga.OPT_MARCH, 2)):
        with pytest.raises(qlga.QlgaError) as e:
            sim.set_option(key, bad)
        assert e.value.status == qlga.QLGA_EINVAL
    q0 = inputs.random_spinor_state((40, 33), seed=71, amplitude=0.1)
    for poison in (np.inf, np.nan, 1e200):
        q = q0.copy()
        q[2, 0, 5, 7] = poison
        sim.set_state_q(q)
        sim.step(1)
        with pytest.raises(qlga.QlgaError) as e:
            sim.observables()
        assert e.value.status == qlga.QLGA_ESTATE and "interaction angle" in str(e.value)
        sim.set_state_q(q0)                                     # a good state: the word was cleared by the report
        sim.step(1)
        assert abs(sim.observables()["norm_q"] / norm2(q0) - 1) < 1e-13
    sim.close()


def test_angle_stats_match_the_definition(qlga):
    # qlga_angle_stats (diagnostic): theta = s (2|c1||F| + |c2| rho / 5), phase = |s c0 rho| per site of one application of U,
    # and the histogram of the degrees the kernels' lookup assigns to them
    c = (0.9, -0.35, 0.6)
    q0 = inputs.random_spinor_state((64, 48), seed=81, amplitude=0.2)
    psi = q0[:, 0] + q0[:, 1]
    n = np.abs(psi) ** 2
    rho = n.sum(0)
    fz = 2 * (n[0] - n[4]) + n[1] - n[3]
    fp = 2 * (np.conj(psi[0]) * psi[1] + np.conj(psi[3]) * psi[4]) + np.sqrt(6.0) * (np.conj(psi[1]) * psi[2] + np.conj(psi[2]) * psi[3])
    fabs = np.sqrt(fz ** 2 + np.abs(fp) ** 2)
    for order, s in (("interleaved", 1 / 8), ("plain", 1.0)):
        sim = qlga.Qlga(2, (64, 48), c, order=order)
        sim.set_state_q(q0)
        st = sim.angle_stats()
        theta = s * (2 * abs(c[1]) * fabs + abs(c[2]) / 5 * rho)
        assert st["theta_max"] == pytest.approx(theta.max(), rel=1e-6)
        assert st["theta_mean"] == pytest.approx(theta.mean(), rel=1e-10)
        assert st["phase_max"] == pytest.approx((s * abs(c[0]) * rho).max(), rel=1e-6)
        hist = st["degree_hist"]
        assert sum(hist) == 64 * 48
        split = min(qlga.exp_polynomial(-58, 12, 7)[0], 0.5)
        want = np.zeros(13, dtype=np.int64)
        for th in theta.ravel():
            want[0 if np.float32(th) > np.float32(split) else qlga.exp_degree(-58, float(np.float32(th) * np.float32(1.0009765625)), 7)] += 1
        assert np.abs(np.array(hist) - want).sum() <= 4            # sites on a bucket edge may land on either side (fp32 angle)
        sim.close()
