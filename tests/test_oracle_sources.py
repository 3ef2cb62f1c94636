"""Pins of the oracle's constant-source burn (burn_zones_src): the system
dy/dt = f(rho, y) + s with dT/dt += src_T, dY_i/dt += src_X_i / A_i (SDC-style coupling,
PAPER.md:L71).  None of these re-types the oracle: closed forms, an exactness property of BDF,
a linear invariant and scipy's Radau on an independent right-hand side (tests/_refmodel.py)."""
import math

import numpy as np
import pytest
import scipy.integrate

import oracle
from workloads import first_order_decay_network, make_workload
from _refmodel import RefModel

RTOL, ATOL = 1e-8, 1e-12


def _burn1(net, rho, T, X, sT, sX, dt, rtol=RTOL, atol=ATOL):
    To, Xo, ns, cnt = oracle.burn(net, np.array([rho]), np.array([T]), np.array(X, dtype=float)[:, None], dt, rtol, atol,
                                  src_T=np.array([sT], dtype=float), src_X=np.array(sX, dtype=float)[:, None])
    return To[0], Xo[:, 0], int(ns[0]), cnt


def test_zero_sources_change_nothing():
    """s = 0 must reproduce the plain burn bit for bit (f + 0.0 == f for every f that is not -0)."""
    for cfg, zones in ((1, 64), (3, 65536), (5, 262144)):
        w = make_workload(cfg, zones=zones)
        a = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL)
        b = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL, src_T=np.zeros(w.nz), src_X=np.zeros_like(w.X))
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


def test_pure_source_is_integrated_exactly():
    """With a negligible reaction rate the solution is the straight line y0 + s t.  Every BDF order
    integrates a linear function exactly, so the result is exact up to rounding, in very few steps."""
    net = first_order_decay_network(1e-250)
    dt = 1e-6
    sT, sX = 3.0e13, [2.0e4, -1.0e4]
    T, X, ns, _ = _burn1(net, 1e6, 2e9, [0.5, 0.25], sT, sX, dt)
    assert 0 < ns <= 12
    assert abs(T - (2e9 + sT * dt)) <= 1e-14 * T
    assert abs(X[0] - (0.5 + sX[0] * dt)) <= 1e-14
    assert abs(X[1] - (0.25 + sX[1] * dt)) <= 1e-14


@pytest.mark.parametrize("lamdt", [0.1, 1.0, 5.0, 20.0])
def test_decay_with_constant_source_closed_form(lamdt):
    """Y_P' = -lam Y_P + s:  Y_P(t) = s/lam + (Y0 - s/lam) e^{-lam t};  Y_P + Y_D grows by s t
    (only the parent is fed).  Q = 0 and no T source: T is exactly constant."""
    dt = 1e-6
    lam = lamdt / dt
    net = first_order_decay_network(lam)
    Y0, D0 = 0.7 / 4, 0.1 / 4
    s = 0.05 / 4 / dt                       # feeds 0.05 of mass fraction over the step
    T, X, ns, _ = _burn1(net, 1e6, 2e9, [0.7, 0.1], 0.0, [4 * s, 0.0], dt)
    assert ns > 0 and T == 2e9
    YP = s / lam + (Y0 - s / lam) * math.exp(-lamdt)
    YD = (Y0 + D0 + s * dt) - YP            # total Y_P + Y_D = Y0 + D0 + s dt
    assert abs(X[0] / 4 - YP) <= 100 * (RTOL * abs(YP) + ATOL)
    assert abs(X[1] / 4 - YD) <= 100 * (RTOL * abs(YD) + ATOL)


def test_temperature_source_only_moves_T_when_rates_ignore_T():
    """first_order_decay_network has a temperature-independent rate (n = B = 0) and Q = 0, so a pure
    T source leaves the abundances exactly on the source-free trajectory and T = T0 + s_T dt."""
    dt, lam = 1e-6, 3.0e6
    net = first_order_decay_network(lam)
    T0, X0 = 1.5e9, [0.6, 0.2]
    Ta, Xa, _, _ = _burn1(net, 1e6, T0, X0, 0.0, [0.0, 0.0], dt)
    Tb, Xb, _, _ = _burn1(net, 1e6, T0, X0, 4.0e14, [0.0, 0.0], dt)
    assert Ta == T0
    assert abs(Tb - (T0 + 4.0e14 * dt)) <= 1e-13 * Tb
    ref = 0.6 / 4 * math.exp(-lam * dt)
    for X in (Xa, Xb):
        assert abs(X[0] / 4 - ref) <= 100 * (RTOL * ref + ATOL)


@pytest.mark.parametrize("config", [1, 2, 3, 5])
def test_mass_invariant_with_sources(config):
    """sum_i A_i Y_i obeys d/dt = sum_i src_X_i exactly (the network conserves it; BDF + Newton with
    an exact-column-sum Jacobian preserves linear invariants to rounding)."""
    w = make_workload(config, zones={1: 64, 2: 4096, 3: 32768, 5: 131072}[config])
    rng = np.random.default_rng(100 + config)
    sX = (rng.random(w.X.shape) - 0.5) * 2e-3 / w.dt * np.maximum(w.X, 1e-3)
    sT = (rng.random(w.nz) - 0.5) * 2e-2 * w.T / w.dt
    To, Xo, ns, _ = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL, src_T=sT, src_X=sX)
    ok = ns > 0
    assert ok.mean() > 0.95
    lhs = Xo.sum(axis=0) - w.X.sum(axis=0)
    rhs = sX.sum(axis=0) * w.dt
    assert np.all(np.abs(lhs - rhs)[ok] <= 1e-10)


@pytest.mark.parametrize("config,zones", [(1, [3, 700, 2500]), (2, [11, 90000]), (3, [1000, 1900000])])
def test_sources_against_scipy_radau(config, zones):
    """Library cross-check on an independent right-hand side (tests/_refmodel.py) plus the source."""
    w = make_workload(config, zones=zones)
    ref = RefModel(w.net)
    rng = np.random.default_rng(7 + config)
    sX = (rng.random(w.X.shape) - 0.3) * 1e-2 / w.dt * np.maximum(w.X, 1e-2)
    sT = (rng.random(w.nz) - 0.5) * 0.1 * w.T / w.dt
    To, Xo, ns, _ = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL, src_T=sT, src_X=sX)
    for z in range(w.nz):
        assert ns[z] > 0
        s = np.append(sX[:, z] / w.net.aion, sT[z])
        y0 = np.append(w.X[:, z] / w.net.aion, w.T[z])
        sol = scipy.integrate.solve_ivp(lambda t, y: ref.f(w.rho[z], y) + s, (0, w.dt), y0, method="Radau",
                                        rtol=1e-11, atol=1e-16, jac=lambda t, y: ref.jac_fd(w.rho[z], y))
        assert sol.success
        yr = sol.y[:, -1]
        Xr = yr[:-1] * w.net.aion
        assert abs(To[z] - yr[-1]) <= 1e-7 * yr[-1]
        dom = Xr > 1e-3
        assert np.all(np.abs(Xo[dom, z] - Xr[dom]) <= 1e-6 * Xr[dom])
        assert np.all(np.abs(Xo[:, z] - Xr) / w.net.aion <= 2e-7 * np.abs(yr[:-1]) + 300 * ATOL)


def test_non_finite_source_is_an_invalid_zone():
    w = make_workload(1, zones=[1, 2, 3])
    sT = np.array([0.0, np.nan, 0.0])
    sX = np.zeros_like(w.X)
    sX[0, 2] = np.inf
    To, Xo, ns, _ = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL, src_T=sT, src_X=sX)
    assert ns[0] > 0 and ns[1] == -4 and ns[2] == -4
    assert np.array_equal(To[1:], w.T[1:]) and np.array_equal(Xo[:, 1:], w.X[:, 1:])
