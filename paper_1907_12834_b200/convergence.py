"""Convergence study of the QLGA step (PAPER.md:1066-1088,
Figs. 23-24): the L2 error of eq. (115), epsilon = sum_r (rho_0 - rho_sim)^2, of a 1D
energy eigenstate after a fixed number of steps, against the lattice size L, with the
soliton width scaled with L, for the plain (eq. 108) and interleaved (eq. 112) orderings.

    python -m paper_1907_12834_b200.convergence            # prints the table and the slopes

Everything runs in the CUDA library (qlga_step, qlga_density, qlga_density_l2_error)."""
from __future__ import annotations

import numpy as np

from . import inputs


def eigenstate_profile(kind, L, widths_per_lattice=16.0):
    """k sech(k(x - L/2)) (bright, eq. 67) or the periodic dark pair of eq. (84) with
    k = widths_per_lattice / L (the paper scales the soliton with the lattice)."""
    x = np.arange(L, dtype=np.float64)
    k = widths_per_lattice / L
    if kind == "bright":
        return k * inputs.sech(k * (x - L / 2))
    if kind == "dark":
        return k * np.tanh(k * (x - L / 4)) * np.tanh(k * (3 * L / 4 - x))
    raise ValueError(kind)


def l2_convergence(kind, row, couplings, sizes=(256, 512, 1024, 2048, 4096), steps=1000,
                   precision="f64"):
    """{order: (slope, [eps(L) ...])} for order in ("plain", "interleaved")."""
    from . import qlga
    E = -2.0 if kind == "bright" else 2.0                     # Table I
    cm = inputs.table1_state(row, E, couplings)
    out = {}
    for order in ("plain", "interleaved"):
        eps = []
        for L in sizes:
            psi = np.zeros((5, 1, L), dtype=np.complex128)
            psi[:, 0, :] = cm[:, None] * eigenstate_profile(kind, L)
            sim = qlga.Qlga(1, (L, 1), couplings, order=order, precision=precision)
            sim.set_state_psi(psi)
            rho0 = sim.density()
            sim.step(steps)
            eps.append(sim.density_l2_error(rho0))
            sim.close()
        slope = float(np.polyfit(np.log(np.asarray(sizes, dtype=np.float64)), np.log(eps), 1)[0])
        out[order] = (slope, eps)
    return out


def main():
    cases = (("dark", 14, (1.0, 0.3, -0.1)), ("dark", 5, (1.0, 0.3, -0.1)),
             ("bright", 14, (-1.0, -0.5, 0.2)), ("bright", 1, (-1.0, -0.5, 0.2)))
    print("paper (Figs. 23-24, state 14, 1000 steps): bright -4.77 plain / -5.67 interleaved; "
          "dark -2.34 plain / -5.38 interleaved (run parameters not printed)")
    for kind, row, c in cases:
        r = l2_convergence(kind, row, c)
        for order in ("plain", "interleaved"):
            slope, eps = r[order]
            print(f"{kind:6s} state {row:2d} {order:11s} slope {slope:6.2f}  eps(L) = "
                  + " ".join(f"{e:.2e}" for e in eps))


if __name__ == "__main__":
    main()
