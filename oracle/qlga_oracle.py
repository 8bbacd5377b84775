"""ctypes front-end of the CPU oracle (oracle/qlga_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It never
imports the CUDA package and the CUDA package never imports it.

`Oracle(precision="double" | "longdouble")` wraps one build of the C file;
arrays are numpy complex128 (or clongdouble) in the layout q[5][2][Ny][Nx]
(1D, 2D) or q[5][2][Nz][Ny][Nx] (3D).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qlga_oracle.c")
_LIBS = {"double": ("libqlga_oracle.so", []),
         "longdouble": ("libqlga_oracle_ld.so", ['-DREAL=long double'])}

OBS_FIELDS = ("n_p2", "n_p1", "n_0", "n_m1", "n_m2", "norm_psi", "norm_q",
              "F_x", "F_y", "F_z", "A00_re", "A00_im", "A00_abs2",
              "e_kin", "e_c0", "e_c1", "e_c2", "e_total", "e_dt_re", "e_dt_im")


def build(force: bool = False) -> None:
    """Compile the oracle's C file (both precisions) with gcc; no FMA contraction."""
    for lib, defs in _LIBS.values():
        out = os.path.join(_HERE, lib)
        if (not force and os.path.exists(out)
                and os.path.getmtime(out) >= os.path.getmtime(_SRC)):
            continue
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fcx-limited-range", "-fPIC", "-shared",
               *defs, _SRC, "-o", out, "-lm"]
        subprocess.run(cmd, check=True)


class Oracle:
    def __init__(self, precision: str = "double"):
        build()
        self.precision = precision
        self.lib = ctypes.CDLL(os.path.join(_HERE, _LIBS[precision][0]))
        if precision == "double":
            self.ctype, self.rtype, self.creal = np.complex128, np.float64, ctypes.c_double
        else:
            self.ctype, self.rtype, self.creal = np.clongdouble, np.longdouble, ctypes.c_longdouble
        self.lib.orc_sizeof_real.restype = ctypes.c_size_t
        assert self.lib.orc_sizeof_real() == np.dtype(self.rtype).itemsize
        L, I, P, R = ctypes.c_long, ctypes.c_int, ctypes.c_void_p, self.creal
        sig = {
            "orc_split_psi": [P, P, L, L, L],
            "orc_psi_of_q": [P, P, L, L, L],
            "orc_collide": [P, L, L, L],
            "orc_stream": [P, L, L, L, I, I, I],
            "orc_kinetic_factor": [P, L, L, L, I, I],
            "orc_spin_matrices": [P, P, P],
            "orc_site_hamiltonian": [P, R, R, R, P],
            "orc_interaction": [P, L, L, L, R, R, R, R],
            "orc_interaction_mu": [P, L, L, L, R, R, R, R, R],
            "orc_step": [P, L, L, L, I, R, R, R, I, L],
            "orc_step_mu": [P, L, L, L, I, R, R, R, R, I, L],
            "orc_observables": [P, P, L, L, L, I, R, R, R, P],
            "orc_vorticity": [P, L, L, P],
            "orc_density": [P, L, L, L, P],
            "orc_winding": [P, L, L, P],
        }
        for name, args in sig.items():
            fn = getattr(self.lib, name)
            fn.argtypes = args
            fn.restype = None

        self.lib.orc_vortex_match.argtypes = [P, L, P, L, L, L, L, P, P]
        self.lib.orc_vortex_match.restype = None
        self.lib.orc_density_l2_error.argtypes = [P, P, L, L, L]
        self.lib.orc_density_l2_error.restype = ctypes.c_double

    # -- helpers ---------------------------------------------------------
    def _c(self, a, shape=None):
        a = np.ascontiguousarray(a, dtype=self.ctype)
        if shape is not None:
            assert a.shape == tuple(shape), (a.shape, shape)
        return a

    @staticmethod
    def _p(a):
        return a.ctypes.data_as(ctypes.c_void_p)

    @staticmethod
    def _dims(q):
        """(nx, ny, nz) of a state q[5][2][Ny][Nx] (1D/2D) or q[5][2][Nz][Ny][Nx] (3D)."""
        assert q.ndim in (4, 5) and q.shape[0] == 5 and q.shape[1] == 2, q.shape
        if q.ndim == 4:
            return q.shape[3], q.shape[2], 1
        return q.shape[4], q.shape[3], q.shape[2]

    @staticmethod
    def _dims2(q):
        assert q.ndim == 4, "2D-only operation"
        return q.shape[3], q.shape[2]

    # -- operators (each returns a new array) ------------------------------
    def split_psi(self, psi):
        psi = self._c(psi)
        sp = psi.shape[1:]
        nz, ny, nx = ((1,) + sp) if len(sp) == 2 else sp
        q = np.empty((5, 2) + sp, dtype=self.ctype)
        self.lib.orc_split_psi(self._p(psi), self._p(q), nx, ny, nz)
        return q

    def psi_of_q(self, q):
        q = self._c(q)
        nx, ny, nz = self._dims(q)
        psi = np.empty((5,) + q.shape[2:], dtype=self.ctype)
        self.lib.orc_psi_of_q(self._p(q), self._p(psi), nx, ny, nz)
        return psi

    def collide(self, q):
        q = self._c(q).copy()
        nx, ny, nz = self._dims(q)
        self.lib.orc_collide(self._p(q), nx, ny, nz)
        return q

    def stream(self, q, d, sigma, transpose=False):
        q = self._c(q).copy()
        nx, ny, nz = self._dims(q)
        self.lib.orc_stream(self._p(q), nx, ny, nz, int(d), int(sigma), int(bool(transpose)))
        return q

    def kinetic_factor(self, q, d, sigma):
        q = self._c(q).copy()
        nx, ny, nz = self._dims(q)
        self.lib.orc_kinetic_factor(self._p(q), nx, ny, nz, int(d), int(sigma))
        return q

    def spin_matrices(self):
        f = [np.empty((5, 5), dtype=self.ctype) for _ in range(3)]
        self.lib.orc_spin_matrices(*(self._p(a) for a in f))
        return f

    def site_hamiltonian(self, psi5, couplings):
        psi5 = self._c(psi5, (5,))
        H = np.empty((5, 5), dtype=self.ctype)
        c0, c1, c2 = couplings
        self.lib.orc_site_hamiltonian(self._p(psi5), self.creal(c0), self.creal(c1),
                                      self.creal(c2), self._p(H))
        return H

    def interaction(self, q, couplings, s, mu=None):
        """mu: chemical potential (eq. 75); None = the form without it."""
        q = self._c(q).copy()
        nx, ny, nz = self._dims(q)
        c0, c1, c2 = couplings
        if mu is None:
            self.lib.orc_interaction(self._p(q), nx, ny, nz, self.creal(c0), self.creal(c1),
                                     self.creal(c2), self.creal(s))
        else:
            self.lib.orc_interaction_mu(self._p(q), nx, ny, nz, self.creal(c0), self.creal(c1),
                                        self.creal(c2), self.creal(mu), self.creal(s))
        return q

    def step(self, q, ndim, couplings, order, nsteps=1, mu=None):
        """order: 0 = plain (eq. 108), 1 = interleaved (eq. 112); mu: chemical potential or None."""
        q = self._c(q).copy()
        nx, ny, nz = self._dims(q)
        assert ndim in (1, 2, 3) and (ndim >= 2 or ny == 1) and (ndim == 3 or nz == 1)
        c0, c1, c2 = couplings
        if mu is None:
            self.lib.orc_step(self._p(q), nx, ny, nz, int(ndim), self.creal(c0), self.creal(c1),
                              self.creal(c2), int(order), int(nsteps))
        else:
            self.lib.orc_step_mu(self._p(q), nx, ny, nz, int(ndim), self.creal(c0), self.creal(c1),
                                 self.creal(c2), self.creal(mu), int(order), int(nsteps))
        return q

    def observables(self, q, ndim, couplings, qprev=None):
        q = self._c(q)
        nx, ny, nz = self._dims(q)
        out = np.empty(20, dtype=np.float64)
        c0, c1, c2 = couplings
        if qprev is not None:
            qprev = self._c(qprev, q.shape)
        self.lib.orc_observables(self._p(q), None if qprev is None else self._p(qprev),
                                 nx, ny, nz, int(ndim), self.creal(c0), self.creal(c1),
                                 self.creal(c2), self._p(out))
        return dict(zip(OBS_FIELDS, out.tolist()))

    def vorticity(self, q):
        q = self._c(q)
        nx, ny = self._dims2(q)
        om = np.empty((5, ny, nx), dtype=self.rtype)
        self.lib.orc_vorticity(self._p(q), nx, ny, self._p(om))
        return om

    def density(self, q):
        """rho(r) = sum_m |psi_m|^2, shape (Ny, Nx)."""
        q = self._c(q)
        nx, ny, nz = self._dims(q)
        rho = np.empty(q.shape[2:], dtype=self.rtype)
        self.lib.orc_density(self._p(q), nx, ny, nz, self._p(rho))
        return rho

    def density_l2_error(self, q, rho_ref):
        """eq. (115): sum_r (rho_ref - rho)^2."""
        q = self._c(q)
        nx, ny, nz = self._dims(q)
        rho_ref = np.ascontiguousarray(rho_ref, dtype=self.rtype)
        assert rho_ref.shape == q.shape[2:]
        return float(self.lib.orc_density_l2_error(self._p(q), self._p(rho_ref), nx, ny, nz))

    def winding(self, q):
        """Plaquette winding numbers, int32 (5, Ny, Nx)."""
        q = self._c(q)
        nx, ny = self._dims2(q)
        w = np.empty((5, ny, nx), dtype=np.int32)
        self.lib.orc_winding(self._p(q), nx, ny, self._p(w))
        return w

    def vortex_match(self, prev, cur, dims, max_dist2):
        """(match_cur, match_prev): mutual nearest neighbours of equal channel and winding under the periodic
        metric of the (Nx, Ny) lattice; records are int32 rows (j, x, y, w)."""
        prev = np.ascontiguousarray(prev, dtype=np.int32).reshape(-1, 4)
        cur = np.ascontiguousarray(cur, dtype=np.int32).reshape(-1, 4)
        mc = np.full(max(len(cur), 1), -1, dtype=np.int32)
        mp = np.full(max(len(prev), 1), -1, dtype=np.int32)
        self.lib.orc_vortex_match(self._p(prev), len(prev), self._p(cur), len(cur), int(dims[0]), int(dims[1]),
                                  int(max_dist2), self._p(mc), self._p(mp))
        return mc[:len(cur)], mp[:len(prev)]
