"""Shared test helpers: re-exports of the small-mesh generators (sfh_inputs.small), the oracle constructor and the
parity norm (oracle/), plus exact leaf totals.  No method arithmetic."""
import math

import numpy as np

from sfh_inputs import Tree, prim_to_cons  # noqa: F401
from sfh_inputs.configs import Problem, cell_centres  # noqa: F401
from sfh_inputs.small import problem_from_tree, small_amr_tree, smooth_fields  # noqa: F401

N = 8


def oracle_for(p, U=None):
    from oracle import oracle_for as f
    return f(p, U)


def parity_errors(Ua, Ub, gamma):
    from oracle.norms import parity_errors as f
    return f(Ua, Ub, gamma)


def leaf_totals(m_or_leaf, U, level, h0):
    """Exact (fsum) totals of the conserved variables over leaf cells: sum U * h_l^3."""
    leaf = m_or_leaf
    tot = []
    for v in range(5):
        terms = []
        for l in np.unique(level):
            sel = leaf & (level == l)
            if sel.any():
                vol = (h0 / 2.0 ** l) ** 3
                terms.append(math.fsum(U[sel, v].ravel().tolist()) * vol)
        tot.append(math.fsum(terms))
    return np.array(tot)
