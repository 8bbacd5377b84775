"""Dispersion relation of kicked solitons (Fig. 5):
a 1D bright soliton (eq. 71) or periodic dark-soliton pair (eq. 81, 84) is given the momentum
p = 2 pi n / L by the factor exp(i p x), evolved, and its energy measured from two successive
states with eq. (85),

    E = i (<psi(t)|psi(t)> - <psi(t)|psi(t - tau)>) / <psi(t)|psi(t)>,

against the predictions E = p^2 - k^2 (eq. 74) and E = p^2 + 2 k^2.

    python -m paper_1907_12834_b200.dispersion            # prints the table of Fig. 5

Everything runs in the CUDA library (qlga_step, qlga_observables: e_dt_re is Re E of eq. 85)."""
from __future__ import annotations

import numpy as np

from . import inputs


def measured_energy(kind, row, couplings, L, k, n_kick, steps=50, order="interleaved", precision="f64"):
    """Re E of eq. (85) after `steps` time steps on the CUDA path."""
    from . import qlga
    sim = qlga.Qlga(1, (L, 1), couplings, order=order, precision=precision)
    sim.set_state_psi(inputs.kicked_soliton(kind, row, couplings, L, k, n_kick))
    sim.step(steps)
    ob = sim.observables()
    sim.close()
    return ob["e_dt_re"]


def dispersion_table(kind, row, couplings, L=2048, k=1.0 / 16, kicks=(0, 2, 4, 8, 12, 16, 24), **kw):
    """[(p, E measured, E predicted) ...]"""
    rows = []
    for n in kicks:
        p = 2.0 * np.pi * n / L
        rows.append((p, measured_energy(kind, row, couplings, L, k, n, **kw), inputs.predicted_energy(kind, k, p)))
    return rows


def main():
    for kind, row, c in (("bright", 3, (-1.0, -0.5, 0.2)), ("bright", 1, (-1.0, -0.5, 0.2)),
                         ("dark", 5, (1.0, 0.3, -0.1)), ("dark", 14, (1.0, 0.3, -0.1))):
        print(f"{kind} soliton, Table I state {row}, k = 1/16, L = 2048, eq. (85) after 50 interleaved steps")
        for p, em, ep in dispersion_table(kind, row, c):
            print(f"  p = {p:.5f}   E measured {em:+.6e}   predicted {ep:+.6e}   diff {em - ep:+.1e}")


if __name__ == "__main__":
    main()
