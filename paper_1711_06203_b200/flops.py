"""Algorithmic flop model of one burn.

Counts the method's own arithmetic from the per-call counters the kernel reports
(nrhs, njac, nlu, nsolve, nst), so redundant work inside a kernel cannot inflate the figure.
Conventions: FMA = 2, + - * / = 1 each, exp = 32 (13-term Horner + range reduction),
log = 40.  n = N + 1 unknowns, K reactions, m_k reactant particles, s_k stoichiometry entries,
c_k distinct reactant species of reaction k.
"""
from __future__ import annotations

import numpy as np

EXP_FLOPS = 32
LOG_FLOPS = 40


def flop_model(net) -> dict:
    n = net.nspec + 1
    K = net.nreac
    m = (np.asarray(net.reactant) >= 0).sum(axis=1)
    s = (np.asarray(net.stoich_id) >= 0).sum(axis=1)
    c = np.array([len(set(int(r) for r in row if r >= 0)) for row in np.asarray(net.reactant)])
    # RHS: per reaction the exponent (2 fma), exp, prefactor (2 mul), product (m mul),
    # scatter (s fma) and the energy sum (1 fma); per call T9, log, t13 = exp, 1/T, rho^2, f_T
    rhs = int(np.sum(4 + EXP_FLOPS + 2 + m + 2 * s + 2)) + (LOG_FLOPS + EXP_FLOPS + 6)
    # Jacobian extra: per reaction the partials (<= m(m-1)+1 mul/add each), the T-derivative
    # (fma + 2 mul), scatter of (c + 1) columns into (s + 1) rows by fma
    jac = int(np.sum(c * np.maximum(m, 1) + 4 + 2 * (c + 1) * (s + 1))) + n
    newton_matrix = 2 * n * n                                  # P = I - gamma J, one fma per entry
    lu = n * (n - 1) // 2 + (n - 1) * n * (2 * n - 1) // 3 + n  # multipliers + rank-1 fmas + n reciprocals
    solve = 2 * n * (n - 1) + n
    nordsieck = 37 * n                                          # predict, correct, norms, weights, residual
    return dict(n=n, K=K, rhs=rhs, jac=jac, newton_matrix=newton_matrix, lu=lu, solve=solve,
                nordsieck=nordsieck)


def algorithmic_flops(net, counters: dict) -> float:
    """Total algorithmic flops of a burn whose counters are `counters`."""
    fm = flop_model(net)
    return float(counters["nrhs"] * fm["rhs"] + counters["njac"] * fm["jac"]
                 + counters["nlu"] * (fm["newton_matrix"] + fm["lu"])
                 + counters["nsolve"] * fm["solve"] + counters["nst"] * fm["nordsieck"])


def state_bytes_per_zone(nspec: int) -> int:
    """Algorithmic HBM bytes per zone: in 8(N+2), out 8(N+1)+4."""
    return 8 * (nspec + 2) + 8 * (nspec + 1) + 4
