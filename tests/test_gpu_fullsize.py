"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (sfh_advance on the
whole problem, one persistent CTA per SM).

* C2 (256^3), C4 (128^3 + 3 levels, all 10 coarse steps) and C5 (1.8e5 blocks on 5 levels, all 5 coarse steps;
  the oracle's three ghosted copies take 38 GB of host memory) are compared with the oracle in every cell.
* C3 (512^3): every cell after one step, and every cell outside the reach of the oracle's non-positive cells after the
  configured ten; besides, the oracle recomputes sampled outputs.  One step of the scheme reaches 3 cells (1 for the
  predictor, 2 for the corrector), so the inner 2^3 blocks of a sub-box cut out of the full initial state
  with a margin of 3 cells per step (outflow on the cut faces), stepped with the full problem's dt
  sequence, are exactly the full problem's values there: one step on 4^3-block boxes, the configured ten
  steps on 10^3-block boxes.  The Mach-10 input develops non-positive pressures (R28); a box
  whose oracle values are not finite is counted and reported, never skipped silently.
* C5 additionally: conservation over leaf cells to round-off on the periodic box across refinement
  boundaries, and sub-step counts that are powers of two (eq. 14-15).
"""
import numpy as np
import pytest

import paper_2604_21438_b200 as sfh
from helpers import oracle_for, parity_errors
from sfh_inputs import make_config
from sfh_inputs.configs import Problem

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

TOL1, TOL10, TOLDT = 1e-12, 1e-10, 1e-14


def gpu_for(p):
    g = sfh.Mesh.from_problem(p)
    g.set_state(p.U)
    g.restrict_all(0)
    return g


def test_c2_full_size_every_cell():
    p = make_config("C2")
    o = oracle_for(p)
    g = gpu_for(p)
    o.advance(1, 0)
    g.advance(1, 0)
    assert abs(g.t.value - o.t.value) <= TOLDT * o.t.value
    err = parity_errors(g.get_state().cpu().numpy(), o.get_state(), p.gamma)
    assert (err <= TOL1).all(), err
    o.advance(9, 0)
    g.advance(9, 0)
    assert abs(g.t.value - o.t.value) <= 1e-13 * o.t.value
    assert o.status() == 0 and g.status() == 0
    err = parity_errors(g.get_state().cpu().numpy(), o.get_state(), p.gamma)
    assert (err <= TOL10).all(), err


def test_c4_full_size_adaptive_every_cell():
    p = make_config("C4")
    o = oracle_for(p)
    o.restrict_all(0)
    g = gpu_for(p)
    assert np.array_equal(g.get_state().cpu().numpy(), o.get_state())
    o.advance(1, 1)
    g.advance(1, 1)
    assert np.array_equal(o.nupd, g.nupd), (o.nupd, g.nupd)
    assert abs(g.t.value - o.t.value) <= TOLDT * o.t.value
    err = parity_errors(g.get_state().cpu().numpy(), o.get_state(), p.gamma)
    assert (err <= TOL1).all(), err
    o.advance(p.nsteps - 1, 1)                 # all 10 coarse steps of the config
    g.advance(p.nsteps - 1, 1)
    assert p.nsteps == 10 and np.array_equal(o.nupd, g.nupd), (o.nupd, g.nupd)
    assert abs(g.t.value - o.t.value) <= 1e-13 * o.t.value
    assert o.status() == 0 and g.status() == 0
    err = parity_errors(g.get_state().cpu().numpy(), o.get_state(), p.gamma)
    assert (err <= TOL10).all(), err


def sub_box_problem(p, where, o0, S):
    """The S^3 blocks at block offset o0 of the uniform problem p as a problem of its own (outflow cut faces)."""
    nb = p.nb0[0]
    sub_ijk = np.array([(i, j, k) for k in range(S) for j in range(S) for i in range(S)], dtype=np.int32)
    idx = where[(o0[0] + sub_ijk[:, 0]) % nb, (o0[1] + sub_ijk[:, 1]) % nb, (o0[2] + sub_ijk[:, 2]) % nb]
    sub = Problem("C3-sub", (S, S, S), 0, ((1, 1),) * 3, (S / nb,) * 3, p.gamma, p.cfl, 0, 1,
                  np.zeros(S ** 3, dtype=np.int32), sub_ijk, np.ascontiguousarray(p.U[idx]))
    return sub, sub_ijk, idx


def test_c3_full_size_sampled_sub_boxes():
    p = make_config("C3")
    nb = p.nb0[0]
    g = gpu_for(p)
    where = np.full((nb, nb, nb), -1, dtype=np.int64)
    where[p.ijk[:, 0], p.ijk[:, 1], p.ijk[:, 2]] = np.arange(p.nblocks)
    dts, states = [], {}
    for step in range(1, p.nsteps + 1):
        dts.append(g.cfl_dt())
        g.advance(1, 0, dts[-1])
        if step in (1, p.nsteps):
            states[step] = g.get_state().cpu().numpy()
    rng = np.random.default_rng(3)
    report = {}
    for nsteps, S, margin, nbox, tol in ((1, 4, 1, 6, TOL1), (p.nsteps, 10, 4, 5, TOL10)):
        Ug = states[nsteps]
        compared = nonfinite = 0
        for _ in range(nbox):
            o0 = rng.integers(0, nb, size=3)                      # periodic box: any offset, wrapped
            sub, sub_ijk, idx = sub_box_problem(p, where, o0, S)
            inner = ((sub_ijk >= margin) & (sub_ijk < S - margin)).all(axis=1)
            o = oracle_for(sub)
            assert o.cell_width(0) == g.cell_width(0)
            for dt in dts[:nsteps]:
                o.advance(1, 0, dt)
            Uo, Ua = o.get_state()[inner], Ug[idx[inner]]
            if not np.isfinite(Uo).all():
                # a non-positive pressure of the Mach-10 input inside the box (R28): the CUDA path must be non-finite
                # in the same cells at least; no tolerance can be stated there
                nonfinite += 1
                assert (~np.isfinite(Ua)).any(), "oracle not finite where the CUDA path is"
                continue
            err = parity_errors(Ua, Uo, p.gamma)
            assert (err <= tol).all(), (nsteps, o0, err)
            compared += 1
        report[nsteps] = (compared, nonfinite)
    print("C3 sub-boxes (steps: compared, non-finite):", report, "bad cells after %d steps: %d" % (p.nsteps, g.status()))
    # every box whose oracle values stayed finite was compared above; at least two of the ten-step boxes must have been
    assert report[1][0] >= 4 and report[p.nsteps][0] >= 2, report


def leaf_mask(level, ijk):
    key = lambda l, c: (l.astype(np.int64) << 48) | (c[:, 0].astype(np.int64) << 32) | (c[:, 1].astype(np.int64) << 16) | c[:, 2]
    parents = set(key(level[level > 0] - 1, ijk[level > 0] >> 1).tolist())
    return np.array([k not in parents for k in key(level, ijk).tolist()])


def totals(U, level, leaf, max_level):
    tot = np.zeros(5, dtype=np.longdouble)
    for l in range(max_level + 1):
        sel = leaf & (level == l)
        if sel.any():
            tot += U[sel].sum(axis=(0, 2, 3, 4), dtype=np.longdouble) * np.longdouble(8.0) ** (-l)
    return tot


def test_c5_full_size_conservation_and_subcycling():
    p = make_config("C5")
    assert 1.5e5 < p.nblocks < 2.2e5, p.census()
    g = gpu_for(p)
    leaf = leaf_mask(p.level, p.ijk)
    U0 = g.get_state().cpu().numpy()
    t0 = totals(U0, p.level, leaf, p.max_level)
    del U0
    assert p.nsteps == 5
    g.advance(p.nsteps, 1)                     # the configured 5 coarse steps
    U1 = g.get_state().cpu().numpy()
    assert np.isfinite(U1).all()
    t1 = totals(U1, p.level, leaf, p.max_level)
    # momentum components nearly cancel over the box: their scale is the sum of the magnitudes
    mscale = totals(np.abs(U1), p.level, leaf, p.max_level)[1:4].max()
    assert abs(t1[0] - t0[0]) <= 1e-12 * abs(t0[0]), (t0, t1)
    assert abs(t1[4] - t0[4]) <= 1e-12 * abs(t0[4]), (t0, t1)
    assert (np.abs(t1[1:4] - t0[1:4]) <= 1e-12 * mscale).all(), (t0, t1)
    # eq. (14)-(15): each level takes 2^n sub-steps of its parent, n >= 0
    n = g.nupd
    assert n[0] == p.nsteps
    for l in range(1, p.max_level + 1):
        # per coarse step the ratio is a power of two (checked step by step in test_gpu_parity); over several steps the
        # counts add up, so only "a whole number of sub-steps per parent update, at least one" holds for the totals
        assert n[l] >= n[l - 1], n
    assert g.status() == 0


def test_c5_full_size_every_cell_all_coarse_steps():
    """The whole 182 008-block hierarchy against the oracle in every cell: after one adaptive coarse step (1e-12) and
    after the configured 5 (BASELINE.json configs[4]; 1e-10), every level sub-cycling, equal update counts per level
    (a few minutes of oracle time on 16 cores; 38 GB of host memory for its ghosted copies)."""
    import os
    ram_gb = os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_PHYS_PAGES") / 2 ** 30
    print("host RAM %.0f GB, %d cores" % (ram_gb, len(os.sched_getaffinity(0))))
    if ram_gb < 80:
        pytest.skip("the oracle's three ghosted copies of C5 need 38 GB (+ inputs): host has %.0f GB" % ram_gb)
    p = make_config("C5")
    o = oracle_for(p)
    o.restrict_all(0)
    g = gpu_for(p)
    assert np.array_equal(g.get_state().cpu().numpy(), o.get_state())
    g.advance(1, 1)
    o.advance(1, 1)
    assert np.array_equal(o.nupd, g.nupd), (o.nupd, g.nupd)
    assert abs(g.t.value - o.t.value) <= TOLDT * o.t.value
    assert o.status() == 0 and g.status() == 0
    err = parity_errors(g.get_state().cpu().numpy(), o.get_state(), p.gamma)
    print("C5 full size, 1 coarse step: updates/level", list(g.nupd), "parity", err)
    assert (err <= TOL1).all(), err
    assert p.nsteps == 5
    g.advance(p.nsteps - 1, 1)
    o.advance(p.nsteps - 1, 1)
    assert np.array_equal(o.nupd, g.nupd), (o.nupd, g.nupd)
    assert abs(g.t.value - o.t.value) <= 1e-13 * o.t.value
    assert o.status() == 0 and g.status() == 0
    err = parity_errors(g.get_state().cpu().numpy(), o.get_state(), p.gamma)
    print("C5 full size, %d coarse steps: updates/level" % p.nsteps, list(g.nupd), "parity", err)
    assert (err <= TOL10).all(), err


def test_c3_full_size_every_cell_one_step():
    """All 1.3e8 cells of C3 against the oracle after one step (the oracle's three ghosted copies take 54 GB of host
    memory).  The Mach-10 input puts a few cells at non-positive pressure in this very step (R28: no floors on
    either side; what such a cell holds is undefined, and its neighbours read it only in the NEXT step), so the
    comparison covers every cell whose oracle value is finite with positive density and pressure, and the number of
    cells left out is reported and bounded."""
    import os
    ram_gb = os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_PHYS_PAGES") / 2 ** 30
    if ram_gb < 110:
        pytest.skip("the oracle's three ghosted copies of C3 need 54 GB (+ inputs): host has %.0f GB" % ram_gb)
    p = make_config("C3")
    o = oracle_for(p)
    g = gpu_for(p)
    o.advance(1, 0)
    g.advance(1, 0)
    assert abs(g.t.value - o.t.value) <= TOLDT * o.t.value
    Uo = o.get_state()
    Ug = g.get_state().cpu().numpy()
    rho, E = Uo[:, 0], Uo[:, 4]
    P = (p.gamma - 1.0) * (E - 0.5 * (Uo[:, 1] ** 2 + Uo[:, 2] ** 2 + Uo[:, 3] ** 2) / rho)
    good = np.isfinite(Uo).all(axis=1) & (rho > 0.0) & (P > 0.0)
    nbad = int((~good).sum())
    print("C3 full size, one step: %d of %d cells left out (oracle not positive), oracle status %d, CUDA status %d"
          % (nbad, good.size, o.status(), g.status()))
    assert nbad <= 100 and nbad == o.status() and g.status() == nbad
    scale = np.array([np.abs(Uo[:, 0][good]).max(), 0.0, 0.0, 0.0, np.abs(Uo[:, 4][good]).max()])
    cs = np.sqrt(p.gamma * P[good] / rho[good])
    mscale = max((np.abs(Uo[:, v][good]) + rho[good] * cs).max() for v in (1, 2, 3))
    scale[1:4] = mscale
    for v in range(5):
        d = np.abs(Ug[:, v][good] - Uo[:, v][good]).max() / scale[v]
        assert d <= TOL1, (v, d)


def global_grid(p, A):
    """Per-cell block array A[nb][8][8][8] of the uniform problem p on the global grid [z][y][x]."""
    nb = p.nb0[0]
    order = np.lexsort((p.ijk[:, 0], p.ijk[:, 1], p.ijk[:, 2]))          # z slowest
    G = A[order].reshape(nb, nb, nb, 8, 8, 8)                            # [bz][by][bx][k][j][i]
    return np.ascontiguousarray(G.transpose(0, 3, 1, 4, 2, 5)).reshape(nb * 8, nb * 8, nb * 8)


def dilate_periodic(mask, r):
    """Every cell within r cells (per axis: a cube, which contains one step's stencil reach) of a marked cell."""
    for ax in range(3):
        acc = mask.copy()
        for s in range(1, r + 1):
            acc |= np.roll(mask, s, axis=ax)
            acc |= np.roll(mask, -s, axis=ax)
        mask = acc
    return mask


def not_positive(U, gamma):
    rho, E = U[:, 0], U[:, 4]
    with np.errstate(all="ignore"):
        P = (gamma - 1.0) * (E - 0.5 * (U[:, 1] ** 2 + U[:, 2] ** 2 + U[:, 3] ** 2) / rho)
        return ~(np.isfinite(U).all(axis=1) & (rho > 0.0) & (P > 0.0))


def test_c3_full_size_every_cell_ten_steps_outside_the_reach_of_bad_cells():
    """All of C3's configured 10 steps against the oracle in every cell that the oracle's non-positive cells cannot
    have reached.  The Mach-10 input leaves a few cells at non-positive pressure from the first step on (DESIGN.md
    R28: no floors on either side; such a cell's content is undefined and spreads 3 cells per step: 1 through the
    predictor, 2 through the corrector).  A cell is left out when, at any step, it lay within 3 cells per later step
    of a cell that was not positive and finite on either side; everything else (the fraction is printed and must be
    >= 0.9) is compared at 1e-10.  Both sides step with the oracle's CFL steps."""
    import os
    ram_gb = os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_PHYS_PAGES") / 2 ** 30
    if ram_gb < 110:
        pytest.skip("the oracle's three ghosted copies of C3 need 54 GB (+ inputs): host has %.0f GB" % ram_gb)
    p = make_config("C3")
    assert p.nsteps == 10
    o = oracle_for(p)
    g = gpu_for(p)
    reach, n_only_g = 3, 0
    mask = np.zeros((p.nb0[0] * 8,) * 3, dtype=bool)
    for step in range(1, p.nsteps + 1):
        dt = o.cfl_dt()
        if step == 1:
            assert abs(g.cfl_dt() - dt) <= TOLDT * dt
        o.advance(1, 0, dt)
        g.advance(1, 0, dt)
        if step > 1:
            mask = dilate_periodic(mask, reach)                  # what the marked cells reached in this step
        Uo = o.get_state()
        bad = not_positive(Uo, p.gamma)
        if step < p.nsteps:
            # a cell that goes bad on the CUDA side only, OUTSIDE the reach of earlier bad cells (where the two sides
            # agreed to round-off a step ago), can only be a pressure within round-off of zero: left out too, but
            # counted and bounded, so that this mask cannot hide a fault of the CUDA path
            only_g = global_grid(p, not_positive(g.get_state().cpu().numpy(), p.gamma) & ~bad) & ~mask
            n_only_g += int(only_g.sum())
            mask |= only_g
        mask |= global_grid(p, bad)
        print("C3 step %d: %d oracle cells not positive, %d cells left out so far, %d bad on the CUDA side only"
              % (step, int(bad.sum()), int(mask.sum()), n_only_g))
    assert n_only_g <= 10
    Ug = g.get_state().cpu().numpy()
    keep = ~mask
    frac = keep.mean()
    print("C3 full size, %d steps: compared %.4f of %d cells; oracle status %d, CUDA status %d"
          % (p.nsteps, frac, keep.size, o.status(), g.status()))
    assert frac >= 0.9
    Go = [global_grid(p, Uo[:, v])[keep] for v in range(5)]
    Gg = [global_grid(p, Ug[:, v])[keep] for v in range(5)]
    assert all(np.isfinite(a).all() for a in Gg)
    rho, E = Go[0], Go[4]
    P = (p.gamma - 1.0) * (E - 0.5 * (Go[1] ** 2 + Go[2] ** 2 + Go[3] ** 2) / rho)
    cs = np.sqrt(p.gamma * P / rho)
    mscale = max((np.abs(Go[v]) + rho * cs).max() for v in (1, 2, 3))
    scale = [np.abs(rho).max(), mscale, mscale, mscale, np.abs(E).max()]
    err = [float(np.abs(Gg[v] - Go[v]).max() / scale[v]) for v in range(5)]
    print("C3 full size, %d steps: parity" % p.nsteps, err)
    assert max(err) <= TOL10, err
