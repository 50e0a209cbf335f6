"""Shared helpers of the parity tests: drive both implementations from one seeded System, compare
them under BASELINE.json `north_star`'s rules, and compute the 1000-step observables in double."""
from __future__ import annotations

import numpy as np

import oracle
import scmf_inputs as si


def gpu_system(s, path: int = 0, options=None, **kw):
    import paper_2606_09356_b200 as soma
    g = soma.Soma.from_system(s, **kw)
    for name, value in (options or {}).items():
        g.set_option(name, value)
    if path:
        g.set_option("path", path)
    return g


def assert_same_state(g, o, what=""):
    """Bit equality of positions, densities and omega (north_star: densities bit-exact, positions
    within 1e-6 b -- below one fp32 ulp at |r| >= 16 b, so equality is what is asserted)."""
    gx, gy, gz = g.positions()
    ox, oy, oz = o.positions()
    for name, a, b in (("x", gx, ox), ("y", gy, oy), ("z", gz, oz)):
        bad = np.nonzero(a != b)[0]
        assert bad.size == 0, f"{what}: {bad.size} beads differ in {name}, first {bad[:5]}: gpu {a[bad[:5]]} oracle {b[bad[:5]]}"
    gd, od = g.density(), o.density()
    assert np.array_equal(gd, od), f"{what}: density grids differ in {(gd != od).sum()} cells"
    go, oo = g.omega(), o.omega()
    assert np.array_equal(go.view(np.uint32), oo.view(np.uint32)), f"{what}: omega differs in {(go != oo).sum()} cells"


def lockstep(s, steps: int, path_for_finish: int = 1):
    """north_star comparison protocol, per half-sweep.

    GPU (generic path, one half-sweep per call) and oracle advance together; beads whose positions
    differ after a half-sweep are decision flips.  A flip is legal only if the oracle's double
    margin |dE + ln u| < 1e-4; the oracle is then resynchronised to the GPU's positions for exactly
    those beads.  Returns (n_moves, n_flips, max |margin| over flips).
    """
    g = gpu_system(s, path=1)
    o = oracle.Oracle.from_system(s)
    g.load_state(s.x, s.y, s.z)
    o.load_state(s.x, s.y, s.z)
    n_moves = n_flips = 0
    worst = 0.0
    for _ in range(steps):
        for parity in (0, 1):
            acc_g = g.debug_half_sweep(parity)
            acc_o, mask, marg = o.half_sweep(parity, want_mask=True, want_margins=True)
            gx, gy, gz = g.positions()
            ox, oy, oz = o.positions()
            diff = np.nonzero((gx != ox) | (gy != oy) | (gz != oz))[0]
            n_moves += (s.workload.N + 1 - parity) // 2 * s.workload.n_chains
            if diff.size:
                assert np.all(diff % s.workload.N % 2 == parity), "a bead of the other parity moved"
                assert np.all(np.abs(marg[diff]) < 1e-4), f"illegal flips: margins {marg[diff][:8]}"
                worst = max(worst, float(np.abs(marg[diff]).max()))
                n_flips += diff.size
                o.set_beads(diff, gx[diff], gy[diff], gz[diff])
            else:
                assert acc_g == acc_o
        g.debug_finish_step()
        o.finish_step()
        assert np.array_equal(g.density(), o.density())
        assert np.array_equal(g.omega().view(np.uint32), o.omega().view(np.uint32))
    g.close()
    return n_moves, n_flips, worst


# ---- observables of the 1000-step statistical check, double precision -----------

def mean_sq_end_to_end(x, y, z, n_chains, N):
    x, y, z = (np.asarray(v, dtype=np.float64).reshape(n_chains, N) for v in (x, y, z))
    r2 = (x[:, -1] - x[:, 0]) ** 2 + (y[:, -1] - y[:, 0]) ** 2 + (z[:, -1] - z[:, 0]) ** 2
    return float(r2.mean()), float(r2.std(ddof=1) / np.sqrt(n_chains))


def structure_factor_AB(x, y, z, types, box, n_shells=3):
    """S_AB(q) = |sum_j sigma_j exp(-i q.r_j)|^2 / B, sigma = +1 (type 0) / -1 (others), averaged
    over the q-vectors of each of the `n_shells` smallest non-zero |q| shells of a cubic box."""
    x, y, z = (np.asarray(v, dtype=np.float64) for v in (x, y, z))
    sigma = np.where(np.asarray(types) == 0, 1.0, -1.0)
    L = np.asarray(box, dtype=np.float64)
    m = np.array([(a, b, c) for a in range(-2, 3) for b in range(-2, 3) for c in range(-2, 3) if (a, b, c) != (0, 0, 0)])
    q = 2 * np.pi * m / L
    qn = np.round(np.sqrt((q ** 2).sum(axis=1)), 9)
    shells = np.unique(qn)[:n_shells]
    out = []
    for qs in shells:
        vals = []
        for qv in q[qn == qs]:
            ph = qv[0] * x + qv[1] * y + qv[2] * z
            vals.append(((sigma * np.cos(ph)).sum() ** 2 + (sigma * np.sin(ph)).sum() ** 2) / x.size)
        out.append((float(qs), float(np.mean(vals)), float(np.std(vals, ddof=1) / np.sqrt(len(vals)))))
    return out
