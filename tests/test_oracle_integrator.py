"""Pins of the oracle's integrator (BZ-BDF v1) against closed forms,
invariants, brute-force implicit Euler, scipy's Radau, and its own tolerance ladder."""
import math

import numpy as np
import pytest
import scipy.integrate
import scipy.optimize

import oracle
from workloads import (first_order_decay_network, make_workload, network_for_config)
from _refmodel import RefModel, NA_MEV

RTOL, ATOL = 1e-8, 1e-12


def _burn1(net, rho, T, X, dt, rtol=RTOL, atol=ATOL, **kw):
    To, Xo, ns, cnt = oracle.burn(net, np.array([rho]), np.array([T]), np.array(X)[:, None], dt, rtol, atol, **kw)
    return To[0], Xo[:, 0], int(ns[0]), cnt


# ------------------------------------------------------------------ closed form 1 (north_star)
@pytest.mark.parametrize("lamdt", [0.1, 1.0, 5.0, 20.0, 100.0])
def test_first_order_decay_closed_form(lamdt):
    """One first-order reaction at fixed T (Q = 0): Y_i(dt) = Y_i(0) exp(-lambda dt)."""
    dt = 1e-6
    lam = lamdt / dt
    net = first_order_decay_network(lam)
    X0 = [0.7, 0.1]
    T, X, ns, _ = _burn1(net, 1e6, 2e9, X0, dt)
    assert ns > 0
    assert T == 2e9                                     # T drift exactly 0
    Yi = 0.7 / 4 * math.exp(-lamdt)
    Yk = 0.1 / 4 + 0.7 / 4 * (1 - math.exp(-lamdt))
    for got, ref in ((X[0] / 4, Yi), (X[1] / 4, Yk)):
        assert abs(got - ref) <= 100 * (RTOL * abs(ref) + ATOL)


# ------------------------------------------------------------------ closed form 2
def test_second_order_closed_form():
    """Config-1 reaction with Q = 0: dY/dt = -rho lam Y^2  =>  Y = Y0/(1 + rho lam Y0 dt)."""
    net = network_for_config(1)
    net.q_mev = np.array([0.0])
    for rho, T in ((1e8, 2.0e9), (1e9, 2.6e9)):
        lam = 4.27e26 * (T * 1e-9) ** (-2 / 3) * math.exp(-84.165 / (T * 1e-9) ** (1 / 3))
        Y0 = 0.4 / 12
        To, X, ns, _ = _burn1(net, rho, T, [0.4, 0.0], 1e-6)
        ref = Y0 / (1 + rho * lam * Y0 * 1e-6)
        assert To == T
        assert abs(X[0] / 12 - ref) <= 3e-7 * ref
        assert abs(X[1] / 24 - (Y0 - ref) / 2) <= 3e-7 * (Y0 - ref) / 2 + 1e-11


# ------------------------------------------------------------------ reduced quadrature
def test_config1_reduced_quadrature():
    """With Q != 0, T = T0 + (N_A MeV Q/cv)(Y0 - Y)/2 exactly, so
    dt = int_Y^Y0 dY' / (rho lam(T(Y')) Y'^2); invert with quad + brentq."""
    net = network_for_config(1)
    A, en, B, Q = 4.27e26, -2 / 3, 84.165, 13.93
    k = NA_MEV * Q / 1e8 / 2
    for rho, T0, X0 in ((2e7, 1.8e9, 0.45), (3e8, 2.2e9, 0.35), (8e8, 1.6e9, 0.5)):
        Y0 = X0 / 12

        def tof(Y):
            # in u = ln Y':  dt = int du / (rho lam(T(Y')) Y')
            def g(u):
                y = math.exp(u)
                T9 = (T0 + k * (Y0 - y)) * 1e-9
                return 1.0 / (rho * A * T9 ** en * math.exp(-B / T9 ** (1 / 3)) * y)
            return scipy.integrate.quad(g, math.log(Y), math.log(Y0), epsabs=0, epsrel=1e-13, limit=400)[0]

        lo = Y0
        for fr in (0.999, 0.99, 0.9, 0.5, 0.1, 1e-2, 1e-3, 1e-4, 1e-6):
            lo = Y0 * fr
            if tof(lo) > 1e-6:
                break
        Yref = scipy.optimize.brentq(lambda Y: tof(Y) - 1e-6, lo, Y0, xtol=1e-18, rtol=1e-14)
        T, X, ns, _ = _burn1(net, rho, T0, [X0, 0.0], 1e-6)
        if 12 * Yref > 1e-4:
            assert abs(X[0] / 12 - Yref) <= 1e-6 * Yref
        assert abs(T - (T0 + k * (Y0 - X[0] / 12))) <= 1e-9 * T        # energy invariant


# ------------------------------------------------------------------ invariants (north_star)
@pytest.mark.parametrize("config,zones", [(1, None), (2, 509), (3, 8191), (4, 32771), (5, 65521)])
def test_mass_invariant_1e10(config, zones):
    if config == 4:   # a strided sample plus the x-line through one hotspot centre
        c = make_workload(4, zones=[0]).meta["centres"][0].astype(int)
        line = np.arange(256) + 256 * (c[1] + 256 * c[2])
        zones = np.unique(np.concatenate([np.arange(0, 256 ** 3, zones), line]))
    w = make_workload(config, zones=zones)
    To, Xo, ns, cnt = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol)
    ok = ns > 0
    assert ok.mean() > 0.99
    drift = np.abs(Xo.sum(axis=0) - w.X.sum(axis=0))       # sum_i A_i Y_i (reading s24)
    assert drift[ok].max() <= 1e-10
    assert np.isfinite(To).all() and (To > 0).all()
    if config == 1:
        dT = NA_MEV * 13.93 / 1e8 * (Xo[1] / 24)
        assert np.abs(To - w.T - dT).max() <= 1e-9 * To.max()
    if config == 4:                                           # >100x spread in step counts
        assert ns.min() == 1 and ns.max() > 100


# ------------------------------------------------------------------ order of accuracy
def test_fixed_order_convergence_slopes():
    """Fixed-q fixed-h hook on y' = -lam y (exact Nordsieck start): error ~ h^q."""
    lam, dt = 1.0e6, 1e-6
    net = first_order_decay_network(lam)
    y0 = 0.7 / 4
    for q in range(1, 6):
        errs = []
        for M in (20, 40, 80):
            h = dt / M
            z = np.zeros((q + 1, 3))
            for j in range(q + 1):
                c = (h ** j) * ((-lam) ** j) / math.factorial(j) * y0
                z[j, 0] = c
                z[j, 1] = -c if j > 0 else 0.1 / 4
            z[0, 2] = 2e9
            T, X, ns, _ = _burn1(net, 1e6, 2e9, [0.7, 0.1], dt, rtol=1e-14, atol=1e-30,
                                 fixed_q=q, fixed_h=h, z_init=z)
            assert ns == M
            errs.append(abs(X[0] / 4 - y0 * math.exp(-lam * dt)))
        s1 = math.log2(errs[0] / errs[1])
        s2 = math.log2(errs[1] / errs[2])
        assert abs(s2 - q) < 0.25 and abs(s1 - q) < 0.45, (q, errs)


# ------------------------------------------------------------------ brute force (north_star)
def _implicit_euler(ref, rho, y0, dt, M):
    """Fixed-step backward Euler; modified Newton (J frozen per step) iterated to roundoff."""
    y = y0.copy()
    h = dt / M
    n = len(y0)
    for _ in range(M):
        Ji = np.linalg.inv(np.eye(n) - h * ref.jac_fd(rho, y))
        yn = y.copy()
        for _it in range(40):
            d = -Ji @ (yn - y - h * ref.f(rho, yn))
            yn = yn + d
            if np.all(np.abs(d) <= 1e-14 * np.abs(yn) + 1e-26):
                break
        y = yn
    return y


@pytest.mark.parametrize("config,zone", [(1, 427), (2, 2560), (2, 8960), (3, 4608)])
def test_brute_force_implicit_euler(config, zone):
    """Tiny-step implicit Euler (first order in 1/M), Richardson (M, 2M), on single mild zones
    (25-50 BDF steps, T rising by <= 10 %) over the config's full dt."""
    w = make_workload(config, zones=[zone])
    ref = RefModel(w.net)
    y0 = np.append(w.X[:, 0] / w.net.aion, w.T[0])
    rho = w.rho[0]
    a = _implicit_euler(ref, rho, y0, w.dt, 1500)
    b = _implicit_euler(ref, rho, y0, w.dt, 3000)
    rich = 2 * b - a                                    # O(1/M^2); |b - a| ~ first-order error of b
    To, Xo, ns, _ = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL)
    assert ns[0] >= 2
    Y = Xo[:, 0] / w.net.aion
    big = np.abs(rich[:-1] * w.net.aion) > 1e-6
    assert big.any()
    tol = 1e-6 * np.abs(rich) + 0.02 * np.abs(b - a)    # 0.02|b-a| ~ 10x the Richardson remainder
    assert np.all(np.abs(Y - rich[:-1])[big] <= tol[:-1][big])
    assert abs(To[0] - rich[-1]) <= tol[-1]


# ------------------------------------------------------------------ library cross-check
@pytest.mark.parametrize("config,zones", [(1, [5, 300, 2000]), (2, [11, 70000]), (3, [123, 1500000]),
                                          (4, None), (5, [77])])
def test_against_scipy_radau(config, zones):
    if config == 4:
        c = make_workload(4, zones=[0]).meta["centres"][3].astype(int)
        zones = [int(c[0] + 3 + 256 * (c[1] + 256 * c[2]))]       # 3 zones off a hotspot centre
    w = make_workload(config, zones=zones)
    ref = RefModel(w.net)
    To, Xo, ns, _ = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL)
    for z in range(w.nz):
        y0 = np.append(w.X[:, z] / w.net.aion, w.T[z])
        sol = scipy.integrate.solve_ivp(lambda t, y: ref.f(w.rho[z], y), (0, w.dt), y0, method="Radau",
                                        rtol=1e-11, atol=1e-16, jac=lambda t, y: ref.jac_fd(w.rho[z], y))
        assert sol.success
        yr = sol.y[:, -1]
        Xr = yr[:-1] * w.net.aion
        assert abs(To[z] - yr[-1]) <= 1e-7 * yr[-1]
        dom = Xr > 1e-3
        assert np.all(np.abs(Xo[dom, z] - Xr[dom]) <= 1e-6 * Xr[dom])
        # trace species: only the integrator's own accuracy (~atol absolute on Y) can be asked
        assert np.all(np.abs(Xo[:, z] - Xr) / w.net.aion <= 2e-7 * np.abs(yr[:-1]) + 300 * ATOL)


# ------------------------------------------------------------------ self-convergence
def test_tolerance_ladder():
    w = make_workload(3, zones=[1000, 600000, 1900000])
    res = []
    for rt in (1e-6, 1e-8, 1e-10):
        To, Xo, ns, _ = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, rt, rt * 1e-4)
        res.append((To, Xo))
    ref = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, 1e-12, 1e-16)
    e = [np.abs(r[0] - ref[0]).max() / ref[0].max() + np.abs(r[1] - ref[1]).max() for r in res]
    assert e[0] > e[1] > e[2]
    assert e[2] < 1e-7 and e[1] < 1e-5


# ------------------------------------------------------------------ plausibility and edge cases
def test_step_counts_comparable_to_scipy_bdf():
    w = make_workload(1, zones=[5])
    ref = RefModel(w.net)
    _, _, ns, _ = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL)
    y0 = np.append(w.X[:, 0] / w.net.aion, w.T[0])
    sol = scipy.integrate.solve_ivp(lambda t, y: ref.f(w.rho[0], y), (0, w.dt), y0, method="BDF",
                                    rtol=RTOL, atol=ATOL, jac=lambda t, y: ref.jac_fd(w.rho[0], y))
    assert 0.5 * len(sol.t) <= ns[0] <= 1.5 * len(sol.t)


def test_failure_codes_and_edge_inputs():
    net = network_for_config(1)
    rho = np.array([1e8, -1.0, 1e8, 1e8, np.nan])
    T = np.array([2e9, 2e9, 0.0, np.inf, 2e9])
    X = np.array([[0.4] * 5, [0.0] * 5])
    To, Xo, ns, cnt = oracle.burn(net, rho, T, X, 1e-6, RTOL, ATOL)
    assert ns[0] > 0 and list(ns[1:]) == [-4] * 4
    assert np.array_equal(Xo[:, 1:], X[:, 1:]) and To[2] == 0.0
    assert cnt["nfailzones"] == 4
    # nz = 0 is a no-op; bad scalars are call-level errors
    out = oracle.burn(net, np.zeros(0), np.zeros(0), np.zeros((2, 0)), 1e-6, RTOL, ATOL)
    assert out[2].shape == (0,)
    with pytest.raises(ValueError):
        oracle.burn(net, rho, T, X, -1.0, RTOL, ATOL)
    # a cold zone takes a single step and changes nothing measurable
    To, Xo, ns, _ = oracle.burn(net, np.array([1e7]), np.array([3e8]), np.array([[0.4], [0.0]]), 1e-6, RTOL, ATOL)
    assert ns[0] == 1 and abs(Xo[0, 0] - 0.4) < 1e-15


def test_norm_lanes_changes_only_rounding():
    """The norm association is a declared parameter of the CUDA path; it may
    move results by rounding only."""
    w = make_workload(3, zones=[17, 4242, 999999])
    a = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL, norm_lanes=1)
    b = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL, norm_lanes=16)
    assert np.abs(a[0] - b[0]).max() <= 1e-9 * a[0].max()
    big = a[1] > 1e-6
    assert np.all(np.abs(a[1] - b[1])[big] <= 1e-7 * a[1][big])
