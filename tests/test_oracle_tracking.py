"""Pins of the oracle's vortex association (orc_vortex_match, reading R18) and of the tracks built on it:
hand-made cases, order independence, and the drift speed 2p = 4 pi n / L of a kicked Pade quadrupole
(eq. 71; the units are those the printed drift times fix)."""
import numpy as np

from paper_1907_12834_b200 import inputs


def test_hand_made_cases(oracle):
    dims = (10, 8)
    # wrap-around: (9, 0) and (0, 7) are one site apart in x and one in y on a 10 x 8 torus
    mc, mp = oracle.vortex_match([[0, 9, 0, 1]], [[0, 0, 7, 1]], dims, 2)
    assert mc.tolist() == [0] and mp.tolist() == [0]
    mc, mp = oracle.vortex_match([[0, 9, 0, 1]], [[0, 0, 7, 1]], dims, 1)          # d2 = 2 > cut-off
    assert mc.tolist() == [-1] and mp.tolist() == [-1]
    # winding and channel must agree
    mc, mp = oracle.vortex_match([[0, 3, 3, 1]], [[0, 3, 3, -1], [1, 3, 3, 1]], dims, 100)
    assert mc.tolist() == [-1, -1] and mp.tolist() == [-1]
    # a non-mutual pair: cur[1] prefers prev[0], but prev[0]'s nearest is cur[0]: cur[1] is a birth
    mc, mp = oracle.vortex_match([[2, 4, 4, 1]], [[2, 4, 5, 1], [2, 4, 2, 1]], dims, 100)
    assert mc.tolist() == [0, -1] and mp.tolist() == [0]
    # a tie in distance goes to the smaller (y, x), whatever the order of the list
    for cur in ([[0, 5, 4, 1], [0, 3, 4, 1]], [[0, 3, 4, 1], [0, 5, 4, 1]]):
        mc, mp = oracle.vortex_match([[0, 4, 4, 1]], cur, dims, 100)
        assert cur[mp[0]] == [0, 3, 4, 1]
    # empty lists
    mc, mp = oracle.vortex_match(np.zeros((0, 4)), [[0, 1, 1, 1]], dims, 4)
    assert mc.tolist() == [-1] and len(mp) == 0
    mc, mp = oracle.vortex_match([[0, 1, 1, 1]], np.zeros((0, 4)), dims, 4)
    assert len(mc) == 0 and mp.tolist() == [-1]


def test_matching_is_a_partial_bijection_and_order_independent(oracle):
    rng = np.random.default_rng(11)
    dims = (40, 30)

    def cloud(n):
        xy = rng.permutation(dims[0] * dims[1])[:n]
        return np.stack([rng.integers(0, 5, n), xy % dims[0], xy // dims[0], rng.choice([-1, 1], n)], axis=1)

    prev, cur = cloud(150), cloud(170)
    mc, mp = oracle.vortex_match(prev, cur, dims, 25)
    assert (mc >= 0).sum() == (mp >= 0).sum() > 20
    for i, k in enumerate(mc):
        if k >= 0:
            assert mp[k] == i and prev[k, 0] == cur[i, 0] and prev[k, 3] == cur[i, 3]
    pp, pc = rng.permutation(len(prev)), rng.permutation(len(cur))
    mc2, mp2 = oracle.vortex_match(prev[pp], cur[pc], dims, 25)
    pairs = {(tuple(prev[k]), tuple(cur[i])) for i, k in enumerate(mc) if k >= 0}
    pairs2 = {(tuple(prev[pp][k]), tuple(cur[pc][i])) for i, k in enumerate(mc2) if k >= 0}
    assert pairs == pairs2
    # brute force of the definition in numpy
    def nearest(a, b):
        out = []
        for r in a:
            best = None
            for k, s in enumerate(b):
                if s[0] != r[0] or s[3] != r[3]:
                    continue
                dx = abs(int(r[1]) - int(s[1])); dy = abs(int(r[2]) - int(s[2]))
                d2 = min(dx, dims[0] - dx) ** 2 + min(dy, dims[1] - dy) ** 2
                if d2 <= 25 and (best is None or (d2, s[2], s[1]) < best[0]):
                    best = ((d2, s[2], s[1]), k)
            out.append(-1 if best is None else best[1])
        return out
    nc, npv = nearest(cur, prev), nearest(prev, cur)
    assert mc.tolist() == [k if k >= 0 and npv[k] == i else -1 for i, k in enumerate(nc)]


def _records(wind):
    return np.array(sorted((int(j), int(x), int(y), int(wind[j, y, x])) for j, y, x in np.argwhere(wind != 0)),
                    dtype=np.int32).reshape(-1, 4)


def test_tracked_drift_speed_of_a_kicked_quadrupole(oracle):
    # a kicked single-channel Pade quadrupole drifts as a whole at 2p = 4 pi n / L sites per step
    L, n, steps, every = 96, 1, 200, 10
    w = inputs.kicked_quadrupole(L, core=6.0, n_kick=n, axis="x")
    q = oracle.split_psi(w.psi)
    prev = _records(oracle.winding(q))
    assert len(prev) == 4 and prev[:, 3].sum() == 0 and set(prev[:, 0]) == {0}
    pos = {i: [float(prev[i, 1]), float(prev[i, 2])] for i in range(4)}        # unwrapped positions per track
    ids = list(range(4))
    for _ in range(steps // every):
        q = oracle.step(q, 2, w.couplings, 1, every)
        cur = _records(oracle.winding(q))
        mc, mp = oracle.vortex_match(prev, cur, (L, L), 16)
        assert len(cur) == 4 and (mc >= 0).all() and (mp >= 0).all()          # no births, no deaths
        new_ids = []
        for i, k in enumerate(mc):
            assert cur[i, 3] == prev[k, 3]
            dx = (int(cur[i, 1]) - int(prev[k, 1]) + L // 2) % L - L // 2
            dy = (int(cur[i, 2]) - int(prev[k, 2]) + L // 2) % L - L // 2
            pos[ids[k]][0] += dx; pos[ids[k]][1] += dy
            new_ids.append(ids[k])
        prev, ids = cur, new_ids
    start = _records(oracle.winding(oracle.split_psi(w.psi)))
    want = 2 * (2 * np.pi * n / L) * steps                                     # 26.2 sites
    for i in range(4):
        assert abs(pos[i][0] - start[i, 1] - want) <= 2.5, (i, pos[i][0] - start[i, 1], want)
        assert abs(pos[i][1] - start[i, 2]) <= 1.5
