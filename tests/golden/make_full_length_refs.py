"""Writes the full-length reference states used by tests/test_gpu_full_length.py:

    python tests/golden/make_full_length_refs.py [cfg3|cfg2]

  cfg3_L1024_20000_longdouble.npz   config 3's recipe (inputs.config3(L=1024)) after its 20 000 interleaved steps
  cfg2_L2048_50000_longdouble.npz   config 2's recipe (inputs.config2(L=2048)) after its 50 000 interleaved steps

both evolved by the LONG-DOUBLE build of the CPU oracle (oracle/qlga_oracle.c, -DREAL="long double") and rounded
once to complex128 at the end.  The full-size lattices (2^22, 65 536 sites) are out of the oracle's reach at these
step counts (days); these reduced lattices take 10 and 40 minutes.  Calls only oracle/ and the seeded input
generators; nothing here comes from the CUDA path.  The double build of the oracle agrees with these states to
9.8e-14 (cfg3) and 8.2e-14 (cfg2): the arbiter of SURVEY.md 8(c) "parity procedure"."""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from paper_1907_12834_b200 import inputs          # noqa: E402  (seeded generators: no method arithmetic)
from oracle.qlga_oracle import Oracle             # noqa: E402

CASES = {"cfg3": (lambda: inputs.config3(L=1024), "cfg3_L1024_20000_longdouble.npz"),
         "cfg2": (lambda: inputs.config2(L=2048), "cfg2_L2048_50000_longdouble.npz")}


def main():
    which = sys.argv[1:] or list(CASES)
    orc = Oracle("longdouble")
    for name in which:
        gen, fname = CASES[name]
        w = gen()
        q = np.repeat(w.psi[:, None] / 2, 2, axis=1).astype(orc.ctype)          # q1 = q2 = psi/2 (reading R6)
        t0 = time.time()
        q = orc.step(q, 1, w.couplings, 1, w.steps)
        out = os.path.join(os.path.dirname(os.path.abspath(__file__)), fname)
        np.savez_compressed(out, q=q.astype(np.complex128), steps=w.steps, lattice=w.dims[0])
        print(f"{name}: {w.steps} steps on L = {w.dims[0]} in {time.time() - t0:.0f} s -> {out}")


if __name__ == "__main__":
    main()
