"""Thin Python binding of the C ABI in include/qlga.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of libqlga.so; torch is used for
device memory and streams.  Importing this module fails loudly if the shared
library has not been built (python -m paper_1907_12834_b200.build): there is no
CPU fallback.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libqlga.so")

QLGA_OK, QLGA_EINVAL, QLGA_ENOMEM, QLGA_ECUDA, QLGA_ESTATE, QLGA_EUNSUP = range(6)
QLGA_F64, QLGA_F32, QLGA_F32X = 0, 1, 2
QLGA_PLAIN, QLGA_INTERLEAVED = 0, 1
(OPT_PATH, OPT_STEPS_PER_LAUNCH, OPT_EXP_TOL_LOG2, OPT_THREADS_X, OPT_TILE_Y, OPT_THREADS_Y, OPT_FUSE_PLAIN_U,
 OPT_F32_PHASE, OPT_EXP_POLY, OPT_EXP_MOD_SHIFT, OPT_MARCH, OPT_BAND, OPT_BAND_ROWS, OPT_BAND_SLOTS) = range(14)
_PRECISIONS = {"f64": QLGA_F64, "fp64": QLGA_F64, "double": QLGA_F64, "f32": QLGA_F32, "fp32": QLGA_F32,
               "float": QLGA_F32, "f32x": QLGA_F32X}

ABI_SYMBOLS = (
    "qlga_init", "qlga_state_bytes", "qlga_set_option", "qlga_set_state_psi", "qlga_set_state_q",
    "qlga_get_state_q", "qlga_get_state_psi", "qlga_step", "qlga_observables", "qlga_vorticity",
    "qlga_launch_count", "qlga_last_error", "qlga_destroy", "qlga_version",
    "qlga_profile_enable", "qlga_profile_read", "qlga_exp_polynomial",
    "qlga_density", "qlga_density_l2_error", "qlga_vortices",
    "qlga_slab_configure", "qlga_slab_edge_get", "qlga_slab_ghost_set",
    "qlga_observable_sums", "qlga_observables_from_sums", "qlga_exp_degree", "qlga_set_chemical_potential",
    "qlga_angle_stats", "qlga_issue_peak", "qlga_observable_sums_noalloc", "qlga_noalloc_last_error",
    "qlga_vortex_match",
)
NSUMS = 17


class QlgaObs(ctypes.Structure):
    _fields_ = [("n_m", ctypes.c_double * 5), ("norm_psi", ctypes.c_double), ("norm_q", ctypes.c_double),
                ("F", ctypes.c_double * 3), ("A00_re", ctypes.c_double), ("A00_im", ctypes.c_double),
                ("A00_abs2", ctypes.c_double), ("e_kin", ctypes.c_double), ("e_c0", ctypes.c_double),
                ("e_c1", ctypes.c_double), ("e_c2", ctypes.c_double), ("e_total", ctypes.c_double),
                ("e_dt_re", ctypes.c_double), ("e_dt_im", ctypes.c_double), ("step", ctypes.c_int64)]


class QlgaAngles(ctypes.Structure):
    _fields_ = [("theta_max", ctypes.c_double), ("theta_mean", ctypes.c_double), ("phase_max", ctypes.c_double),
                ("degree_hist", ctypes.c_int64 * 13)]


class QlgaProfile(ctypes.Structure):
    _fields_ = [("ms", ctypes.c_double * 4), ("launches", ctypes.c_int64 * 4)]


class QlgaError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"qlga status {status}: {text}")
        self.status = status


def load_library():
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: build it with "
                          "`python -m paper_1907_12834_b200.build` (needs nvcc); there is no CPU fallback")
    lib = ctypes.CDLL(_LIB_PATH)
    P, I, I64, D, SZ = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double, ctypes.c_size_t
    lib.qlga_init.argtypes = [ctypes.POINTER(P), I, ctypes.POINTER(I64), D, D, D, I, I, P, P, P, SZ, P]
    lib.qlga_init.restype = I
    lib.qlga_state_bytes.argtypes = [I, ctypes.POINTER(I64), I]
    lib.qlga_state_bytes.restype = SZ
    lib.qlga_set_option.argtypes = [P, I, I64]
    lib.qlga_set_option.restype = I
    for name in ("qlga_set_state_psi", "qlga_set_state_q", "qlga_get_state_q", "qlga_get_state_psi",
                 "qlga_vorticity"):
        fn = getattr(lib, name)
        fn.argtypes = [P, P, I]
        fn.restype = I
    lib.qlga_set_chemical_potential.argtypes = [P, D]
    lib.qlga_set_chemical_potential.restype = I
    lib.qlga_step.argtypes = [P, I64]
    lib.qlga_step.restype = I
    lib.qlga_observables.argtypes = [P, ctypes.POINTER(QlgaObs)]
    lib.qlga_observables.restype = I
    lib.qlga_launch_count.argtypes = [P]
    lib.qlga_launch_count.restype = I64
    lib.qlga_last_error.argtypes = [P]
    lib.qlga_last_error.restype = ctypes.c_char_p
    lib.qlga_destroy.argtypes = [P]
    lib.qlga_destroy.restype = I
    lib.qlga_profile_enable.argtypes = [P, I]
    lib.qlga_profile_enable.restype = I
    lib.qlga_profile_read.argtypes = [P, ctypes.POINTER(QlgaProfile)]
    lib.qlga_profile_read.restype = I
    lib.qlga_density.argtypes = [P, P, I]
    lib.qlga_density.restype = I
    lib.qlga_density_l2_error.argtypes = [P, P, I, ctypes.POINTER(D)]
    lib.qlga_density_l2_error.restype = I
    lib.qlga_vortices.argtypes = [P, P, I64, ctypes.POINTER(I64)]
    lib.qlga_vortices.restype = I
    lib.qlga_slab_configure.argtypes = [P, I64]
    lib.qlga_slab_configure.restype = I
    lib.qlga_slab_edge_get.argtypes = [P, I, P]
    lib.qlga_slab_edge_get.restype = I
    lib.qlga_slab_ghost_set.argtypes = [P, I, P]
    lib.qlga_slab_ghost_set.restype = I
    lib.qlga_observable_sums.argtypes = [P, ctypes.POINTER(D)]
    lib.qlga_observable_sums.restype = I
    lib.qlga_observables_from_sums.argtypes = [P, ctypes.POINTER(D), ctypes.POINTER(QlgaObs)]
    lib.qlga_observables_from_sums.restype = I
    lib.qlga_exp_polynomial.argtypes = [I, I, I, ctypes.POINTER(D), ctypes.POINTER(D), ctypes.POINTER(D)]
    lib.qlga_exp_polynomial.restype = I
    lib.qlga_exp_degree.argtypes = [I, I, D, ctypes.POINTER(I)]
    lib.qlga_exp_degree.restype = I
    lib.qlga_angle_stats.argtypes = [P, ctypes.POINTER(QlgaAngles)]
    lib.qlga_angle_stats.restype = I
    lib.qlga_issue_peak.argtypes = [I, P, ctypes.POINTER(D), ctypes.POINTER(D), ctypes.POINTER(D)]
    lib.qlga_issue_peak.restype = I
    lib.qlga_observable_sums_noalloc.argtypes = [P, P, I, ctypes.POINTER(I64), I, I, P, P]
    lib.qlga_observable_sums_noalloc.restype = I
    lib.qlga_noalloc_last_error.argtypes = []
    lib.qlga_noalloc_last_error.restype = ctypes.c_char_p
    lib.qlga_vortex_match.argtypes = [P, P, I64, P, I64, I64, P, P]
    lib.qlga_vortex_match.restype = I
    lib.qlga_version.argtypes = []
    lib.qlga_version.restype = ctypes.c_char_p
    return lib


_lib = load_library()


def version() -> str:
    return _lib.qlga_version().decode()


def exp_polynomial(tol_log2, p, mod_shift=0):
    """(theta_max, b0, r[0..p]) of the degree-p interaction polynomial (host only); mod_shift: the even
    (modulus) part of its error is held to 2^(tol_log2 - mod_shift) (QLGA_OPT_EXP_MOD_SHIFT)."""
    th, b0 = ctypes.c_double(), ctypes.c_double()
    r = (ctypes.c_double * (p + 1))()
    st = _lib.qlga_exp_polynomial(int(tol_log2), int(mod_shift), int(p), ctypes.byref(th), ctypes.byref(b0), r)
    if st != QLGA_OK:
        raise QlgaError(st, "qlga_exp_polynomial: bad arguments")
    return th.value, b0.value, list(r)


def exp_degree(tol_log2, theta, mod_shift=0):
    """Degree the kernels' lookup table picks for the angle theta (host only)."""
    p = ctypes.c_int()
    st = _lib.qlga_exp_degree(int(tol_log2), int(mod_shift), float(theta), ctypes.byref(p))
    if st != QLGA_OK:
        raise QlgaError(st, "qlga_exp_degree: bad arguments")
    return p.value


def issue_peak(kind, stream=None):
    """Measured issue rate of the DFMA / FFMA / FFMA2 pipes on the current device (qlga_issue_peak):
    {'instr_per_s', 'instr_per_clk_per_sm', 'ms'}; kind = "dfma" | "ffma" | "ffma2"."""
    k = {"dfma": 0, "ffma": 1, "ffma2": 2}[kind]
    a, b, c = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    st = _lib.qlga_issue_peak(k, ctypes.c_void_p(stream.cuda_stream) if stream is not None else None,
                              ctypes.byref(a), ctypes.byref(b), ctypes.byref(c))
    if st != QLGA_OK:
        raise QlgaError(st, "qlga_issue_peak failed")
    return {"instr_per_s": a.value, "instr_per_clk_per_sm": b.value, "ms": c.value}


NOALLOC_MAX_BLOCKS = 2048


def observable_sums_noalloc(q, qprev, ndim, dims, precision, out, nblocks=0, stream=None):
    """qlga_observable_sums_noalloc: the NSUMS lattice sums of the device state `q` (torch tensor, layout
    [5][2][..lattice..] complex) into the device tensor `out` (float64, >= NSUMS elements), with no context
    and no device allocation (static scratch inside the library; calls that overlap on the GPU race).
    Asynchronous on `stream` (default: torch's current stream)."""
    import torch
    assert q.is_cuda and q.is_contiguous() and out.is_cuda and out.is_contiguous()
    assert out.dtype == torch.float64 and out.numel() >= NSUMS
    if stream is None:
        stream = torch.cuda.current_stream(q.device)
    d = (ctypes.c_int64 * 3)(*_dims3(ndim, dims))
    st = _lib.qlga_observable_sums_noalloc(q.data_ptr(), qprev.data_ptr() if qprev is not None else None, int(ndim), d,
                                           _PRECISIONS[precision], int(nblocks), out.data_ptr(),
                                           ctypes.c_void_p(stream.cuda_stream))
    if st != QLGA_OK:
        raise QlgaError(st, _lib.qlga_noalloc_last_error().decode())


def _dims3(ndim, dims):
    dims = tuple(int(v) for v in dims)
    if int(ndim) == 3:
        return (dims + (0, 0, 0))[:3]          # a missing extent is reported by the library (EINVAL)
    return (dims[0], dims[1] if len(dims) > 1 else 1, 1)


def state_bytes(ndim, dims, prec) -> int:
    d = (ctypes.c_int64 * 3)(*_dims3(ndim, dims))
    return int(_lib.qlga_state_bytes(int(ndim), d, int(prec)))


class Qlga:
    """One lattice on one GPU.  dims = (Nx, Ny) (Ny = 1 in 1D) or (Nx, Ny, Nz) in 3D; arrays
    are q[5][2][Ny][Nx] / psi[5][Ny][Nx] (3D: [..][Nz][Ny][Nx]); couplings = (c0, c1, c2)
    = the paper's (g0, g1, g2); order "plain" (eq. 108) or "interleaved" (eq. 112);
    precision "f64", "f32" or "f32x" (fp32 storage, fp64 arithmetic in registers).  `keep_previous=True` allocates the third buffer that
    eq. (85)'s energy needs in 2D."""

    def __init__(self, ndim, dims, couplings, order="interleaved", precision="f64",
                 device="cuda:0", stream=None, keep_previous=False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("qlga needs a CUDA device (B200, sm_100a); there is no CPU fallback")
        self.torch = torch
        self.ndim = int(ndim)
        self.nx, self.ny, self.nz = _dims3(ndim, dims)
        self.lat = (self.ny, self.nx) if self.ndim < 3 else (self.nz, self.ny, self.nx)
        self.prec = _PRECISIONS[precision]
        self.order = QLGA_INTERLEAVED if order in ("interleaved", 1) else QLGA_PLAIN
        self.device = torch.device(device)
        self.rdtype = torch.float64 if self.prec == QLGA_F64 else torch.float32
        self.np_cdtype = np.complex128 if self.prec == QLGA_F64 else np.complex64
        self.np_rdtype = np.float64 if self.prec == QLGA_F64 else np.float32
        nbytes = state_bytes(self.ndim, (self.nx, self.ny, self.nz), self.prec)
        if nbytes == 0:
            raise QlgaError(QLGA_EINVAL, "bad ndim/dims")
        nreal = nbytes // (8 if self.prec == QLGA_F64 else 4)
        with torch.cuda.device(self.device):
            nbuf = 3 if (keep_previous and self.ndim >= 2) else 2
            self.bufs = [torch.empty(nreal, dtype=self.rdtype, device=self.device) for _ in range(nbuf)]
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            dims_c = (ctypes.c_int64 * 3)(self.nx, self.ny, self.nz)
            ctx = ctypes.c_void_p()
            c0, c1, c2 = (float(v) for v in couplings)
            st = _lib.qlga_init(ctypes.byref(ctx), self.ndim, dims_c, c0, c1, c2, self.order, self.prec,
                                self.bufs[0].data_ptr(), self.bufs[1].data_ptr(),
                                self.bufs[2].data_ptr() if nbuf == 3 else None, nbytes,
                                ctypes.c_void_p(self.stream.cuda_stream))
        if st != QLGA_OK:
            raise QlgaError(st, _lib.qlga_last_error(None).decode())
        self.ctx = ctx

    # -- plumbing ----------------------------------------------------------
    def _check(self, st):
        if st != QLGA_OK:
            raise QlgaError(st, _lib.qlga_last_error(self.ctx).decode())

    def _ptr(self, a):
        """(pointer, on_device) of a numpy array or torch tensor."""
        if isinstance(a, np.ndarray):
            assert a.flags["C_CONTIGUOUS"]
            return a.ctypes.data, 0
        assert a.is_contiguous()
        return a.data_ptr(), int(a.is_cuda)

    def close(self):
        if getattr(self, "ctx", None):
            _lib.qlga_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key, value):
        self._check(_lib.qlga_set_option(self.ctx, int(key), int(value)))

    # -- state -------------------------------------------------------------
    def set_state_psi(self, psi):
        if isinstance(psi, np.ndarray):
            psi = np.ascontiguousarray(psi, dtype=self.np_cdtype)
            assert psi.shape == (5,) + self.lat, psi.shape
        p, dev = self._ptr(psi)
        self._check(_lib.qlga_set_state_psi(self.ctx, p, dev))

    def set_state_q(self, q):
        if isinstance(q, np.ndarray):
            q = np.ascontiguousarray(q, dtype=self.np_cdtype)
            assert q.shape == (5, 2) + self.lat, q.shape
        p, dev = self._ptr(q)
        self._check(_lib.qlga_set_state_q(self.ctx, p, dev))

    def get_state_q(self, out=None):
        if out is None:
            out = np.empty((5, 2) + self.lat, dtype=self.np_cdtype)
        p, dev = self._ptr(out)
        self._check(_lib.qlga_get_state_q(self.ctx, p, dev))
        return out

    def get_state_psi(self, out=None):
        if out is None:
            out = np.empty((5,) + self.lat, dtype=self.np_cdtype)
        p, dev = self._ptr(out)
        self._check(_lib.qlga_get_state_psi(self.ctx, p, dev))
        return out

    # -- evolution and diagnostics -----------------------------------------
    def set_chemical_potential(self, mu):
        """mu psi_m term of the equation of motion (eq. 75); default 0."""
        self._check(_lib.qlga_set_chemical_potential(self.ctx, float(mu)))

    def step(self, n=1):
        self._check(_lib.qlga_step(self.ctx, int(n)))

    @staticmethod
    def _obs_dict(ob):
        return {"n_p2": ob.n_m[0], "n_p1": ob.n_m[1], "n_0": ob.n_m[2], "n_m1": ob.n_m[3], "n_m2": ob.n_m[4],
                "norm_psi": ob.norm_psi, "norm_q": ob.norm_q, "F_x": ob.F[0], "F_y": ob.F[1], "F_z": ob.F[2],
                "A00_re": ob.A00_re, "A00_im": ob.A00_im, "A00_abs2": ob.A00_abs2, "e_kin": ob.e_kin,
                "e_c0": ob.e_c0, "e_c1": ob.e_c1, "e_c2": ob.e_c2, "e_total": ob.e_total,
                "e_dt_re": ob.e_dt_re, "e_dt_im": ob.e_dt_im, "step": ob.step}

    def observables(self):
        ob = QlgaObs()
        self._check(_lib.qlga_observables(self.ctx, ctypes.byref(ob)))
        return self._obs_dict(ob)

    def observable_sums(self):
        """The NSUMS additive lattice sums behind observables() (owned layers of a slab)."""
        h = (ctypes.c_double * NSUMS)()
        self._check(_lib.qlga_observable_sums(self.ctx, h))
        return np.array(h, dtype=np.float64)

    def observables_from_sums(self, sums):
        h = (ctypes.c_double * NSUMS)(*[float(v) for v in sums])
        ob = QlgaObs()
        self._check(_lib.qlga_observables_from_sums(self.ctx, h, ctypes.byref(ob)))
        return self._obs_dict(ob)

    # -- slab decomposition (include/qlga.h "Slab decomposition"; driver in slab.py) --------
    def slab_configure(self, ghost):
        self._check(_lib.qlga_slab_configure(self.ctx, int(ghost)))

    def slab_edge_get(self, side, dev_out):
        assert dev_out.is_cuda and dev_out.is_contiguous()
        self._check(_lib.qlga_slab_edge_get(self.ctx, int(side), dev_out.data_ptr()))

    def slab_ghost_set(self, side, dev_in):
        assert dev_in.is_cuda and dev_in.is_contiguous()
        self._check(_lib.qlga_slab_ghost_set(self.ctx, int(side), dev_in.data_ptr()))

    def vorticity(self, out=None):
        if out is None:
            out = np.empty((5, self.ny, self.nx), dtype=self.np_rdtype)
        p, dev = self._ptr(out)
        self._check(_lib.qlga_vorticity(self.ctx, p, dev))
        return out

    def angle_stats(self):
        """{'theta_max', 'theta_mean', 'phase_max', 'degree_hist'} of one application of U on the current
        state (qlga_angle_stats): which polynomial degrees the state exercises."""
        a = QlgaAngles()
        self._check(_lib.qlga_angle_stats(self.ctx, ctypes.byref(a)))
        return {"theta_max": a.theta_max, "theta_mean": a.theta_mean, "phase_max": a.phase_max,
                "degree_hist": [int(v) for v in a.degree_hist]}

    def density(self, out=None):
        if out is None:
            out = np.empty(self.lat, dtype=self.np_rdtype)
        p, dev = self._ptr(out)
        self._check(_lib.qlga_density(self.ctx, p, dev))
        return out

    def density_l2_error(self, rho_ref):
        """eq. (115): sum_r (rho_ref - rho)^2 against a reference density (numpy or torch)."""
        if isinstance(rho_ref, np.ndarray):
            rho_ref = np.ascontiguousarray(rho_ref, dtype=self.np_rdtype)
            assert rho_ref.shape == self.lat
        p, dev = self._ptr(rho_ref)
        eps = ctypes.c_double()
        self._check(_lib.qlga_density_l2_error(self.ctx, p, dev, ctypes.byref(eps)))
        return eps.value

    def vortices(self, max_out=65536):
        """(records, count): records int32 (k, 4) = (j, x, y, winding) of the plaquettes with
        non-zero winding (order unspecified), count = total number found."""
        out = np.empty((max_out, 4), dtype=np.int32)
        cnt = ctypes.c_int64()
        self._check(_lib.qlga_vortices(self.ctx, out.ctypes.data, int(max_out), ctypes.byref(cnt)))
        return out[:min(cnt.value, max_out)].copy(), cnt.value

    def vortex_match(self, prev, cur, max_dist2):
        """(match_cur, match_prev) of two detections (int32 (n, 4) records of vortices()): mutual nearest
        neighbours with the same channel and winding under the periodic metric (qlga_vortex_match)."""
        prev = np.ascontiguousarray(prev, dtype=np.int32).reshape(-1, 4)
        cur = np.ascontiguousarray(cur, dtype=np.int32).reshape(-1, 4)
        mc = np.full(len(cur), -1, dtype=np.int32)
        mp = np.full(len(prev), -1, dtype=np.int32)
        self._check(_lib.qlga_vortex_match(self.ctx, prev.ctypes.data if len(prev) else None, len(prev),
                                           cur.ctypes.data if len(cur) else None, len(cur), int(max_dist2),
                                           mc.ctypes.data if len(cur) else None, mp.ctypes.data if len(prev) else None))
        return mc, mp

    def profile_enable(self, on=True):
        self._check(_lib.qlga_profile_enable(self.ctx, int(bool(on))))

    def profile_read(self):
        """{'x_pass': (ms, launches), 'y_pass': ..., 'per_operator': ..., 'band_step': ...} since the last read."""
        pr = QlgaProfile()
        self._check(_lib.qlga_profile_read(self.ctx, ctypes.byref(pr)))
        names = ("x_pass", "y_pass", "per_operator", "band_step")
        return {n: (pr.ms[k], int(pr.launches[k])) for k, n in enumerate(names)}

    def launch_count(self):
        return int(_lib.qlga_launch_count(self.ctx))
