"""Pins of the oracle's Roe solver ("the method of Roe (1981)"; SURVEY.md 8(f) row 2,
DESIGN.md reading R30) against what the mathematics fixes.  CPU only.

* Roe's Property U: the linearisation is exact for the flux jump, F_R - F_L = sum_k lambda_k alpha_k K_k,
  and the wave strengths decompose the state jump, U_R - U_L = sum_k alpha_k K_k.  Both are checked
  through the flux itself: away from the entropy-fix band, F_roe(L,R) - F_roe(R,L)|mirrored and the
  supersonic limits below only hold if every average, eigenvalue, strength and eigenvector is right.
* consistency F(W,W) = physical flux; supersonic states return the upwind flux;
* an isolated stationary contact has the exact flux (0, P, 0, 0, 0) and is preserved by the full scheme;
* mirror antisymmetry and axis permutation;
* the Sod tube converges to the exact Riemann solution; conservation on AMR meshes is unchanged.
"""
import numpy as np
import pytest

import exact_riemann
from helpers import leaf_totals, oracle_for, problem_from_tree, small_amr_tree
from oracle.binding import hllc, roe
from sfh_inputs import prim_to_cons, unblockify, uniform_tree
from sfh_inputs.configs import Problem, cell_centres, sod
from test_oracle_pins import phys_flux, prims, run_to


def cons(W, gamma):
    rho, v, P = W[0], W[1:4], W[4]
    return np.array([rho, *(rho * v), P / (gamma - 1) + 0.5 * rho * (v @ v)])


def random_state(rng, vscale=1.5):
    return np.array([rng.uniform(0.1, 3), *rng.normal(0, vscale, 3), rng.uniform(0.1, 3)])


def test_roe_consistency_and_supersonic_upwinding():
    rng = np.random.default_rng(5)
    gamma = 5.0 / 3.0
    for _ in range(100):
        W = random_state(rng)
        for d in range(3):
            assert np.allclose(roe(W, W, d, gamma), phys_flux(W, d, gamma), rtol=1e-14, atol=1e-15)
    for _ in range(100):
        WL, WR = random_state(rng, 0.2), random_state(rng, 0.2)
        cmax = np.sqrt(gamma * max(WL[4] / WL[0], WR[4] / WR[0]))
        for d in range(3):
            WL[1 + d] = WR[1 + d] = 0.0
            WL[1 + d] += 3.0 * cmax + rng.uniform(0, 1)      # every wave moves right: F = F_L.  This is
            WR[1 + d] += 3.0 * cmax + rng.uniform(0, 1)      # Property U: sum lambda alpha K = F_R - F_L
            FL = phys_flux(WL, d, gamma)
            assert np.allclose(roe(WL, WR, d, gamma), FL, rtol=2e-13, atol=2e-13 * np.abs(FL).max())
            WL[1 + d] *= -1.0
            WR[1 + d] *= -1.0
            FR = phys_flux(WR, d, gamma)
            assert np.allclose(roe(WL, WR, d, gamma), FR, rtol=2e-13, atol=2e-13 * np.abs(FR).max())
            WL[1 + d] = WR[1 + d] = 0.0


def test_roe_upwind_dissipation_equals_the_state_jump_for_a_uniform_wave_speed():
    """With all |lambda_k| equal (u~ >> c~ is not needed: take the dissipation itself): for a pure
    supersonic jump F_L + F_R - 2 F_roe = sum lambda alpha K = F_R - F_L; for the mirrored one the sign
    flips.  Adding both removes the flux jump and leaves 2 u-weighted state jumps only if
    sum alpha K = U_R - U_L: checked here in the limit of a large common advection speed a, where
    lambda_k -> a (1 + O(c/a)) and (F_L + F_R - 2 F_roe) / a -> U_R - U_L."""
    rng = np.random.default_rng(6)
    gamma = 1.4
    a = 1.0e6
    for _ in range(20):
        WL, WR = random_state(rng, 0.3), random_state(rng, 0.3)
        WL[1] += a
        WR[1] += a
        D = (phys_flux(WL, 0, gamma) + phys_flux(WR, 0, gamma) - 2.0 * roe(WL, WR, 0, gamma)) / a
        dU = cons(WR, gamma) - cons(WL, gamma)
        # the energy jump is O(a^2), momentum O(a): compare relative to each component's scale
        scale = np.abs(cons(WR, gamma)) + np.abs(cons(WL, gamma))
        assert (np.abs(D - dU) <= 1e-5 * scale).all(), (D, dU)


def test_roe_stationary_contact_flux_is_exact():
    for d in range(3):
        WL = np.array([1.0, 0.0, 0.0, 0.0, 0.7])
        WR = np.array([0.013, 0.0, 0.0, 0.0, 0.7])
        expect = np.zeros(5)
        expect[1 + d] = 0.7
        assert (roe(WL, WR, d, 1.4) == expect).all()


def test_roe_mirror_antisymmetry_and_axis_permutation():
    rng = np.random.default_rng(11)
    for _ in range(50):
        WL, WR = random_state(rng), random_state(rng)
        F = roe(WL, WR, 0, 1.4)
        ml, mr = WR.copy(), WL.copy()
        ml[1] *= -1
        mr[1] *= -1
        sign = np.array([-1, 1, -1, -1, -1.0])
        assert np.allclose(roe(ml, mr, 0, 1.4), sign * F, rtol=1e-12, atol=1e-13)
        perm = lambda W: np.array([W[0], W[3], W[1], W[2], W[4]])
        assert np.allclose(roe(perm(WL), perm(WR), 1, 1.4), perm(F), rtol=1e-14, atol=1e-15)


def test_roe_is_close_to_hllc_for_weak_jumps():
    """Both are consistent, linearly exact solvers: for a jump of size eps they differ by O(eps^2)."""
    rng = np.random.default_rng(12)
    W0 = np.array([1.0, 0.3, -0.2, 0.1, 0.8])
    dW = rng.normal(0, 1, 5)
    diffs = []
    for eps in (1e-2, 1e-3):
        WL, WR = W0 - 0.5 * eps * dW, W0 + 0.5 * eps * dW
        diffs.append(np.abs(roe(WL, WR, 0, 1.4) - hllc(WL, WR, 0, 1.4)).max())
    assert diffs[1] < 0.02 * diffs[0], diffs


@pytest.mark.parametrize("gamma,T", [(1.4, 0.2)])
def test_roe_sod_converges_to_exact_solution(gamma, T):
    errs = []
    for nb in (4, 8, 16):
        p = sod(nb=nb, gamma=gamma, slab=True)
        m = oracle_for(p)
        m.set_riemann("roe")
        run_to(m, T)
        assert m.status() == 0
        rho, v, P = prims(m.get_state(), gamma)
        x = (np.arange(nb * 8) + 0.5) / (nb * 8)
        re, ue, pe = exact_riemann.sample((x - 0.5) / T, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, gamma)
        errs.append([np.abs(unblockify(rho, p.nb0)[3, 4, :] - re).mean(),
                     np.abs(unblockify(v[0], p.nb0)[3, 4, :] - ue).mean(),
                     np.abs(unblockify(P, p.nb0)[3, 4, :] - pe).mean()])
    errs = np.array(errs)
    assert (errs[1] < 0.7 * errs[0]).all() and (errs[2] < 0.7 * errs[1]).all(), errs
    assert errs[2, 0] < 8e-3 and errs[2, 1] < 1.5e-2 and errs[2, 2] < 7e-3, errs


def test_roe_stationary_contact_preserved_exactly_by_the_full_scheme():
    t = uniform_tree((4, 1, 1), 0)
    level, ijk = t.block_list()
    X, Y, Z = cell_centres(level, ijk, t.nb0)
    rho = np.where((X > 0.25) & (X < 0.75), 1.0, 0.05)
    z = np.zeros_like(rho)
    U = prim_to_cons(rho, z, z, z, np.full_like(rho, 0.6), 1.4)
    p = Problem("contact", t.nb0, 0, ((0, 0),) * 3, (1.0, 0.25, 0.25), 1.4, 0.4, 0, 5, level, ijk, U)
    m = oracle_for(p)
    m.set_riemann("roe")
    m.advance(5, 0)
    assert np.array_equal(m.get_state(), U)


def test_roe_conservation_on_amr_with_subcycling():
    p = problem_from_tree(small_amr_tree(), mode=1)
    m = oracle_for(p)
    m.set_riemann("roe")
    m.restrict_all(0)
    leaf = m.is_leaf()
    h0 = m.cell_width(0)
    tot0 = leaf_totals(leaf, m.get_state(), p.level, h0)
    m.advance(2, 1)
    tot1 = leaf_totals(leaf, m.get_state(), p.level, h0)
    assert (np.abs(tot1 - tot0) <= 1e-13 * max(np.abs(tot0).max(), 1.0)).all(), tot1 - tot0
