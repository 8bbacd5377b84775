"""Slab decomposition on the CUDA path: several slab contexts on one
GPU, stepped in turn and exchanged through qlga_slab_edge_get / qlga_slab_ghost_set, against
the oracle on the undivided lattice.  Needs a B200: run with -m gpu.  (The transport between
GPUs -- torch.distributed P2P -- is covered on the CPU by tests/test_slab.py with gloo.)"""
import numpy as np
import pytest

from paper_1907_12834_b200 import inputs
from conftest import rel_l2

pytestmark = pytest.mark.gpu

TOL64 = 1e-12
TOL32 = 1e-5
C = (1.0, 0.3, -0.1)


@pytest.fixture(scope="module")
def mods():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1907_12834_b200 import qlga, slab          # fails loudly if libqlga.so is missing
    return qlga, slab


@pytest.mark.parametrize("ndim,dims,nslabs", [(2, (40, 50), 3), (2, (33, 24), 2), (2, (16, 200), 1),
                                              (1, (119,), 2), (1, (1000,), 4), (3, (10, 6, 27), 2)])
@pytest.mark.parametrize("order", [0, 1])
def test_slabs_reproduce_the_undivided_lattice(mods, oracle, ndim, dims, nslabs, order):
    qlga, slab = mods
    q0 = inputs.random_spinor_state(dims if ndim > 1 else (dims[0], 1), seed=21, amplitude=0.05)
    steps = 5
    ref = oracle.step(q0, ndim, C, order, steps)
    g = slab.SlabGroup(ndim, dims, C, order=("plain", "interleaved")[order], nslabs=nslabs)
    g.set_state_q(q0)
    g.step(steps)
    out = g.get_state_q()
    obs = g.observables()
    g.close()
    assert out.shape == ref.shape
    assert rel_l2(out, ref) < TOL64
    ref_obs = oracle.observables(ref, ndim, C)
    for k in ("norm_q", "norm_psi", "e_kin", "e_total", "F_z", "A00_abs2"):
        assert obs[k] == pytest.approx(ref_obs[k], rel=1e-11, abs=1e-13), k


def test_slabs_fp32_and_single_process_self_exchange(mods, oracle):
    qlga, slab = mods
    dims = (48, 36)
    q32 = inputs.random_spinor_state(dims, seed=22, amplitude=0.05).astype(np.complex64)
    ref = oracle.step(q32.astype(np.complex128), 2, C, 1, 6)
    g = slab.SlabGroup(2, dims, C, precision="f32", nslabs=2)
    g.set_state_q(q32)
    g.step(6)
    assert rel_l2(g.get_state_q().astype(np.complex128), ref) < TOL32
    g.close()
    # world = 1 through SlabQlga.exchange (its own edges wrap around)
    s = slab.SlabQlga(2, dims, C, rank=0, world=1, device="cuda:0")
    q0 = q32.astype(np.complex128)
    s.set_state_q(q0)
    s.step(6)
    assert rel_l2(s.get_state_q(), oracle.step(q0, 2, C, 1, 6)) < TOL64
    assert s.observables()["norm_q"] == pytest.approx(float(np.sum(np.abs(q0) ** 2)), rel=1e-12)
    s.close()


def test_slab_vorticity_vortices_and_energy_of_a_quadrupole(mods, oracle):
    qlga, slab = mods
    w = inputs.config4(L=96, core=6.0)
    q0 = np.repeat(w.psi[:, None] / 2, 2, axis=1)
    steps = 4
    ref = oracle.step(q0, 2, w.couplings, 1, steps)
    prev = oracle.step(q0, 2, w.couplings, 1, steps - 1)
    g = slab.SlabGroup(2, w.dims, w.couplings, nslabs=3, keep_previous=True)
    g.set_state_q(q0)
    g.step(steps)
    om, (rec, cnt), obs, out = g.vorticity(), g.vortices(), g.observables(), g.get_state_q()
    g.close()
    assert rel_l2(out, ref) < TOL64
    assert np.abs(om - oracle.vorticity(out)).max() < 1e-10
    wind = oracle.winding(out)                   # the detector on the same (GPU) state, undivided
    want = sorted((int(j), int(x), int(y), int(wind[j, y, x])) for j, y, x in np.argwhere(wind != 0))
    assert cnt == len(want) >= 8
    assert sorted(tuple(int(v) for v in r) for r in rec) == want
    ref_obs = oracle.observables(ref, 2, w.couplings, qprev=prev)
    for k in ("e_total", "e_dt_re", "e_dt_im", "norm_q"):       # eq. (85) needs the summed overlaps
        assert obs[k] == pytest.approx(ref_obs[k], rel=1e-9, abs=1e-12), k


def test_slab_call_errors(mods):
    qlga, slab = mods
    import torch
    sim = qlga.Qlga(2, (16, 16), C)
    buf = torch.empty(10 * 4 * 16 * 2, dtype=torch.float64, device="cuda:0")
    with pytest.raises(qlga.QlgaError) as e:
        sim.slab_configure(6)                    # 3 * ghost > extent
    assert e.value.status == qlga.QLGA_EINVAL
    sim.slab_configure(4)
    with pytest.raises(qlga.QlgaError) as e:
        sim.slab_edge_get(0, buf)                # no state yet
    assert e.value.status == qlga.QLGA_ESTATE
    sim.set_state_q(inputs.random_spinor_state((16, 16), seed=1))
    with pytest.raises(qlga.QlgaError) as e:
        sim.slab_edge_get(2, buf)
    assert e.value.status == qlga.QLGA_EINVAL
    sim.slab_configure(0)
    with pytest.raises(qlga.QlgaError) as e:
        sim.slab_ghost_set(0, buf)               # not a slab
    assert e.value.status == qlga.QLGA_ESTATE
    sim.close()
