"""Pins of the oracle's pieces (rate law, RHS, Jacobian, LU/solve, exp/log, BDF coefficients,
norm) against things other than the oracle itself: worked values, invariants, finite
differences, numpy/scipy routines, textbook BDF numbers.  DESIGN.md section 4 lists them."""
import math
import os

import numpy as np
import pytest
import scipy.linalg

import oracle
from workloads import make_workload, network_for_config
from _refmodel import RefModel, NA_MEV

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


# ------------------------------------------------------------------ inputs / RNG reading s13
def test_rng_first_draws():
    for seed, val in _rows("rng_first_draws.txt"):
        assert np.random.default_rng(int(seed)).random() == float(val)


def test_workload_shapes_and_mass():
    for c, zones in ((1, None), (2, 997), (3, 4099), (4, 65537), (5, 16411)):
        w = make_workload(c, zones=zones)
        assert w.X.shape == (w.net.nspec, w.nz)
        s = w.X.sum(axis=0)
        if c == 1:
            assert (s >= 0.3).all() and (s <= 0.5).all()      # remainder is inert O16
        else:
            assert np.abs(s - 1).max() < 1e-14
        # every reaction conserves sum A_i Y_i
        net = w.net
        for k in range(net.nreac):
            m = net.stoich_id[k] >= 0
            assert abs(np.sum(net.aion[net.stoich_id[k][m]] * net.stoich_dy[k][m])) == 0.0


def test_config4_structure():
    """Divergence stress: hot zones are rare and clustered (BASELINE.json configs[3])."""
    w = make_workload(4, zones=np.arange(0, 256 ** 3, 37))
    assert w.T.min() == 3e8 and w.T.max() <= 3e9
    frac_hot = np.mean(w.T > 1.2e9)
    assert 0.001 < frac_hot < 0.01
    centres = w.meta["centres"]
    c = centres[0].astype(int)
    z = c[0] + 256 * (c[1] + 256 * c[2])
    wc = make_workload(4, zones=[z])
    assert abs(wc.T[0] - 3e9) < 1.0            # peak is exactly 3e9 at a hotspot centre


# ------------------------------------------------------------------ rate law: worked values
def test_rate_law_worked_values():
    net = network_for_config(1)
    for what, T9, rho, X, val in _rows("config1_rate_values.txt"):
        T9, rho, X, val = float(T9), float(rho), float(X), float(val)
        if what == "lambda":
            # R = lambda * rho * Y^2 / 2 with rho = 1, Y = sqrt(2): R = lambda
            f = oracle.rates(net, 1.0, np.array([math.sqrt(2.0), 0.0, T9 * 1e9]), jac=False)
            got = f[1]
            tol = 2e-9
        else:
            f = oracle.rates(net, rho, np.array([X / 12.0, 0.0, T9 * 1e9]), jac=False)
            got = {"r": f[1], "dYC12dt": f[0], "dTdt": f[2]}[what]
            tol = 1e-9 if what != "dYC12dt" else 2e-7   # that golden value has 7 digits
        assert abs(got - val) <= tol * abs(val), (what, T9, got, val)


def test_rhs_against_second_implementation():
    rng = np.random.default_rng(11)
    for c in (1, 2, 3, 5):
        net = network_for_config(c)
        ref = RefModel(net)
        for _ in range(5):
            y = np.append(rng.random(net.nspec) * 0.05, 1e9 * (0.8 + 2.5 * rng.random()))
            rho = 10 ** (5 + 4 * rng.random())
            f = oracle.rates(net, rho, y, jac=False)
            g = ref.f(rho, y)
            scale = np.abs(g).max()
            assert np.abs(f - g).max() <= 1e-11 * scale


def test_rhs_mass_invariant():
    rng = np.random.default_rng(5)
    for c in (1, 2, 3, 5):
        net = network_for_config(c)
        for _ in range(10):
            y = np.append(rng.random(net.nspec) * 0.05, 1e9 * (0.5 + 3 * rng.random()))
            f, J = oracle.rates(net, 10 ** (5 + 4 * rng.random()), y)
            a = net.aion
            assert abs(a @ f[:-1]) <= 1e-13 * np.sum(np.abs(a * f[:-1])) + 1e-300
            col = a @ J[:-1, :]
            assert np.all(np.abs(col) <= 1e-13 * (np.abs(a)[:, None] * np.abs(J[:-1, :])).sum(axis=0) + 1e-300)


def test_jacobian_finite_differences():
    rng = np.random.default_rng(7)
    for c in (1, 2, 3, 5):
        net = network_for_config(c)
        n = net.neq
        y = np.append(0.002 + rng.random(net.nspec) * 0.03, 2.1e9)
        rho = 3e6
        f0, J = oracle.rates(net, rho, y)
        Jfd = np.zeros((n, n))
        for j in range(n):
            h = 1e-6 * y[j]
            yp, ym = y.copy(), y.copy()
            yp[j] += h
            ym[j] -= h
            Jfd[:, j] = (oracle.rates(net, rho, yp, jac=False) - oracle.rates(net, rho, ym, jac=False)) / (2 * h)
        # entries above the finite-difference noise floor
        noise = 1e-9 * np.abs(f0)[:, None] / (1e-6 * y)[None, :]
        big = np.abs(J) > 1e3 * noise
        assert big.sum() > n
        assert np.all(np.abs(J - Jfd)[big] <= 2e-7 * np.abs(J)[big])
        assert np.all(np.abs(Jfd)[~big] <= 1e4 * noise[~big] + 1e-7 * np.abs(J).max())
        # structural zeros are exact zeros
        ref = RefModel(net)
        dep = np.zeros((n, n), dtype=bool)
        for k in range(net.nreac):
            for i, _ in ref.sto[k]:
                dep[i, ref.reac[k]] = True
                dep[i, n - 1] = True
            dep[n - 1, ref.reac[k]] = True
            dep[n - 1, n - 1] = True
        assert np.all(J[~dep] == 0.0)


def test_negative_abundance_extension_is_odd_and_restoring():
    """Reading s19: R = -pref*prod|Y| when any reactant abundance is negative, so a species
    that dipped below zero is pushed back up and the implicit equations stay monotone."""
    net = network_for_config(3)
    y = np.append(np.full(13, 0.01), 2e9)
    for j in (0, 1, 2):
        yn = y.copy()
        yn[j] = -1e-9
        f, J = oracle.rates(net, 1e7, yn)
        assert f[j] > 0.0
        assert J[j, j] < 0.0
    # identical pair: R(-Y) = -R(Y)
    net1 = network_for_config(1)
    fp = oracle.rates(net1, 1e8, np.array([0.02, 0.0, 2e9]), jac=False)
    fm = oracle.rates(net1, 1e8, np.array([-0.02, 0.0, 2e9]), jac=False)
    assert fm[1] == -fp[1] and fm[0] == -fp[0]


# ------------------------------------------------------------------ own exp / log (C.5 item 3)
def _ulps(a, b):
    return abs(a - b) / math.ulp(b)


def test_exp_log_within_2ulp():
    rng = np.random.default_rng(3)
    for x in np.concatenate([rng.uniform(-300, 100, 4000), rng.uniform(-2, 2, 2000), [0.0, -700.0, 700.0]]):
        assert _ulps(oracle.oexp(float(x)), math.exp(float(x))) <= 2.0
    for x in np.concatenate([10 ** rng.uniform(-3, 2, 4000), 10 ** rng.uniform(-290, 290, 1000), [1.0, 0.5, 2.0]]):
        got, ref = oracle.olog(float(x)), math.log(float(x))
        assert abs(got - ref) <= 2.0 * math.ulp(ref) + 1e-17
    assert oracle.oexp(-701.0) == 0.0 and oracle.oexp(701.0) == math.inf
    assert oracle.oexp(0.0) == 1.0 and oracle.olog(1.0) == 0.0


# ------------------------------------------------------------------ LU / solve (dgefa/dgesl)
def test_lu_solve_against_lapack():
    rng = np.random.default_rng(9)
    for n in list(range(1, 32)):
        A = rng.standard_normal((n, n))
        b = rng.standard_normal(n)
        lu, ipvt, inv, info = oracle.lu_factor(A)
        assert info == 0
        x = oracle.lu_solve(lu, ipvt, inv, b)
        xr = np.linalg.solve(A, b)
        cond = np.linalg.cond(A)
        assert np.abs(x - xr).max() <= 1e-13 * cond * np.abs(xr).max()
        assert np.abs(A @ x - b).max() <= 1e-12 * cond * np.abs(b).max()
        # same pivot sequence as LAPACK's partial pivoting (first maximal element)
        _, piv = scipy.linalg.lu_factor(A)
        assert np.array_equal(ipvt, piv.astype(np.int32))
        np.testing.assert_allclose(inv, 1.0 / np.diag(lu), rtol=0, atol=0)


def test_lu_on_newton_matrices_and_ties():
    net = network_for_config(3)
    y = np.append(np.full(13, 0.01), 2e9)
    _, J = oracle.rates(net, 1e7, y)
    for gamma in (1e-12, 1e-9, 1e-6):
        P = np.eye(14) - gamma * J
        lu, ipvt, inv, info = oracle.lu_factor(P)
        b = np.arange(1.0, 15.0)
        x = oracle.lu_solve(lu, ipvt, inv, b)
        assert np.abs(P @ x - b).max() <= 1e-12 * np.linalg.cond(P) * 14
    # ties: the FIRST maximal entry wins; exact zero pivot is reported
    A = np.array([[1.0, 2.0, 3.0], [-1.0, 5.0, 1.0], [1.0, 0.0, 7.0]])
    _, ipvt, _, info = oracle.lu_factor(A)
    assert ipvt[0] == 0 and info == 0
    _, _, _, info = oracle.lu_factor(np.array([[0.0, 1.0], [0.0, 2.0]]))
    assert info == 1


# ------------------------------------------------------------------ BDF coefficients (C.2-B.1)
def test_bdf_coefficients_constant_step():
    H = [1.0, 3 / 2, 11 / 6, 25 / 12, 137 / 60]
    for q in range(1, 6):
        l = oracle.bdf_coeffs(q, 0.37, [0.37] * 5)
        assert l[0] == 1.0
        assert abs(l[1] - H[q - 1]) <= 4e-16 * H[q - 1]
        fact = math.factorial(q)
        assert abs(l[q] - 1.0 / fact) <= 4e-16 / fact
    np.testing.assert_allclose(oracle.bdf_coeffs(2, 1.0, [1.0] * 5), [1, 1.5, 0.5], rtol=1e-15)
    np.testing.assert_allclose(oracle.bdf_coeffs(3, 1.0, [1.0] * 5), [1, 11 / 6, 1, 1 / 6], rtol=1e-15)


def test_bdf_coefficients_variable_step_are_the_interpolation_polynomial():
    """l(x) = prod (1 + x/xi_i) must vanish at the previous q mesh points."""
    h, tau = 0.3, [0.2, 0.5, 0.1, 0.4, 0.25]
    for q in range(1, 6):
        l = oracle.bdf_coeffs(q, h, tau)
        back = h
        for i in range(1, q + 1):
            x = -back / h                    # t_{n-i} in units of h from t_n
            assert abs(np.polyval(l[::-1], x)) < 1e-13
            back += tau[i - 1]


# ------------------------------------------------------------------ norm association
def test_wrms_association():
    rng = np.random.default_rng(2)
    v, w = rng.standard_normal(14), rng.random(14) + 0.5
    d2 = (v * w) ** 2
    ref = math.sqrt(d2.sum() / 14)
    for lanes in (1, 2, 4, 8, 16, 32):
        assert abs(oracle.wrms(v, w, lanes) - ref) <= 4e-16 * ref
    # lanes=4: four interleaved partial sums then ((p0+p2)+(p1+p3))
    p = [0.0] * 4
    for i in range(14):
        d = v[i] * w[i]
        p[i % 4] = math.fma(d, d, p[i % 4]) if hasattr(math, "fma") else p[i % 4] + d * d
    if hasattr(math, "fma"):
        s = (p[0] + p[2]) + (p[1] + p[3])
        assert oracle.wrms(v, w, 4) == math.sqrt(s * (1.0 / 14))
