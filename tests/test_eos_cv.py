"""the specific heat from an analytic equation of state evaluated inside the right-hand
side (bz_net_desc.zion):  c_v = 1.5 R (extra + sum_i (1+Z_i) Y_i) + 4 a T^3 / rho.
Oracle pins first (an exact energy integral, the independent numpy model, centred differences, Radau),
GPU parity last."""
import math

import numpy as np
import pytest
import scipy.integrate
import scipy.optimize

import oracle
from workloads import first_order_decay_network, make_workload, make_urca9_like_workload
from _refmodel import RefModel, NA_MEV, RGAS, ARAD
from _parity import compare

RTOL, ATOL = 1e-8, 1e-12
Z13 = np.array([2, 6, 8, 10, 12, 14, 16, 18, 20, 22, 24, 26, 28.0])


@pytest.mark.parametrize("rho", [1e5, 1e6, 1e8])
def test_energy_integral_closed_form(rho):
    """A -> B at a temperature-independent rate, Z_A = Z_B, so the ion/electron part c0 of c_v is
    constant and c_v dT = N_A MeV Q dY_B integrates exactly:
        c0 (T - T0) + (a/rho) (T^4 - T0^4) = N_A MeV Q Y_A0 (1 - exp(-lambda dt)).
    rho = 1e5: radiation dominates c_v; 1e8: the gas does; 1e6: both matter.  A wrong constant, T^3 for
    T^4, a missing electron term or c_v frozen at its initial value misses by far more than the bound."""
    dt, lamdt, Q, Z, extra = 1e-6, 1.5, 5.0, 6.0, 0.01
    net = first_order_decay_network(lamdt / dt, q_mev=Q)
    net.zion = np.array([Z, Z])
    net.eos_extra = extra
    T0, XA, XB = 2e9, 0.7, 0.1
    To, Xo, ns, _ = oracle.burn(net, np.array([rho]), np.array([T0]), np.array([[XA], [XB]]), dt, RTOL, ATOL)
    assert ns[0] > 5
    YA0 = XA / 4
    assert abs(Xo[0, 0] / 4 - YA0 * math.exp(-lamdt)) <= 100 * (RTOL * YA0 + ATOL)
    c0 = 1.5 * RGAS * (extra + (1 + Z) * (XA + XB) / 4)
    E = NA_MEV * Q * YA0 * (1 - math.exp(-lamdt))
    Tref = scipy.optimize.brentq(lambda T: c0 * (T - T0) + ARAD / rho * (T ** 4 - T0 ** 4) - E, T0, 1e12, xtol=1e-3, rtol=1e-15)
    assert Tref - T0 > 1e7                                   # the burn heats visibly
    assert abs(To[0] - Tref) <= 3e-7 * Tref, (rho, To[0], Tref)
    # and it is NOT what a c_v frozen at its initial value gives
    cv0 = c0 + 4 * ARAD * T0 ** 3 / rho
    assert abs((T0 + E / cv0) - Tref) > 1e-3 * (Tref - T0)


@pytest.mark.parametrize("config", [2, 3, 5])
def test_rhs_and_jacobian_with_eos(config):
    w = make_workload(config, zones=[0])
    net = w.net
    net.zion = np.round(net.aion / 2)
    net.eos_extra = 0.003
    ref = RefModel(net)
    rng = np.random.default_rng(31 + config)
    N = net.nspec
    for _ in range(6):
        y = np.append((0.02 + rng.random(N)) / net.aion, 8e8 + 2e9 * rng.random())
        rho = 10 ** (4 + 4 * rng.random())
        f, J = oracle.rates(net, rho, y)
        fr = ref.f(rho, y)
        assert np.allclose(f, fr, rtol=1e-11, atol=1e-12 * np.abs(fr).max())
        Jfd = ref.jac_fd(rho, y)
        term = np.abs(Jfd * y[None, :]).max(axis=1, keepdims=True)
        assert np.all(np.abs(J - Jfd) <= 3e-6 * np.abs(Jfd) + 1e-8 * term / np.abs(y)[None, :])
        # the species rows do not know about the EOS
        net0 = make_workload(config, zones=[0]).net
        f0, J0 = oracle.rates(net0, rho, y)
        assert np.array_equal(f[:N], f0[:N]) and np.array_equal(J[:N, :], J0[:N, :])


def test_integrated_against_radau_and_invariant():
    w = make_workload(3, zones=[123, 1000, 1500000, 600000])
    w.net.zion = Z13
    To, Xo, ns, cnt = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL)
    assert (ns > 3).all()
    assert np.abs(Xo.sum(axis=0) - w.X.sum(axis=0)).max() <= 1e-10
    ref = RefModel(w.net)
    for z in range(w.nz):
        y0 = np.append(w.X[:, z] / w.net.aion, w.T[z])
        sol = scipy.integrate.solve_ivp(lambda t, y: ref.f(w.rho[z], y), (0, w.dt), y0, method="Radau", rtol=1e-11,
                                        atol=1e-16, jac=lambda t, y: ref.jac_fd(w.rho[z], y))
        assert sol.success
        yr = sol.y[:, -1]
        Xr = yr[:-1] * w.net.aion
        assert abs(To[z] - yr[-1]) <= 2e-7 * yr[-1]
        dom = Xr > 1e-3
        assert np.all(np.abs(Xo[dom, z] - Xr[dom]) <= 1e-6 * Xr[dom])
        assert np.all(np.abs(Xo[:, z] - Xr) / w.net.aion <= 2e-7 * np.abs(yr[:-1]) + 300 * ATOL)
    # with the EOS the same zones heat less than with the configs' constant 1e8 (c_v is 2-4x larger here)
    w0 = make_workload(3, zones=[123, 1000, 1500000, 600000])
    T0 = oracle.burn(w0.net, w0.rho, w0.T, w0.X, w0.dt, RTOL, ATOL)[0]
    assert ((To - w.T) <= (T0 - w.T) + 1.0).all()


def test_bad_eos_descriptors_are_refused():
    w = make_workload(1, zones=[0])
    w.net.zion = np.array([6.0, np.nan])
    with pytest.raises(ValueError):
        oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL)
    import paper_1711_06203_b200 as bz
    with pytest.raises(bz.BurnError) as e:
        bz.net_create(w.net)
    assert e.value.code == -3
    w.net.zion = np.array([6.0, 12.0])
    w.net.eos_extra = -1.0
    with pytest.raises(bz.BurnError) as e:
        bz.net_create(w.net)
    assert e.value.code == -3


@pytest.mark.gpu
@pytest.mark.parametrize("case", ["config3", "config5", "urca", "config2+src"])
def test_eos_gpu_parity(case):
    import torch
    import paper_1711_06203_b200 as bz
    dev = torch.device("cuda:0")
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    src = None
    if case == "config3":
        w = make_workload(3, zones=1021)
        w.net.zion = Z13
    elif case == "config5":
        w = make_workload(5, zones=8191)
        w.net.zion = np.round(w.net.aion / 2)
        w.net.eos_extra = 0.001
    elif case == "urca":
        w = make_urca9_like_workload(2053)                   # density exponents AND the EOS together
        w.net.zion = np.array([0, 1, 2, 6, 8, 10, 10, 11, 12.0])
    else:
        w = make_workload(2, zones=127)
        w.net.zion = np.array([2, 6, 8, 10, 12, 14, 28.0])
        rng = np.random.default_rng(8)
        src = ((rng.random(w.nz) - 0.5) * 2e-2 * w.T / w.dt, (rng.random(w.X.shape) - 0.5) * 2e-3 / w.dt * np.maximum(w.X, 1e-3))
    net = bz.net_create(w.net)
    assert net.kernel_name.startswith("burn_coop")           # the generated kernels have no EOS
    if src is None:
        To, Xo, ns = bz.burn_zones(net, d(w.rho), d(w.T), d(w.X), w.dt, w.rtol, w.atol)
        kw = {}
    else:
        To, Xo, ns = bz.burn_zones_src(net, d(w.rho), d(w.T), d(w.X), d(src[0]), d(src[1]), w.dt, w.rtol, w.atol)
        kw = dict(src_T=src[0], src_X=src[1])
    torch.cuda.synchronize()
    cnt = bz.get_counters(net)
    Tr, Xr, nr, cr = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol, norm_lanes=net.norm_lanes, **kw)
    stats = compare(To.cpu().numpy(), Xo.cpu().numpy(), ns.cpu().numpy(), Tr, Xr, nr)
    assert stats["nsteps_equal"] == 1.0 and stats["bitexact_X"] == 1.0 and stats["bitexact_T"] == 1.0, stats
    assert all(cnt[k] == cr[k] for k in cnt)
    bz.net_destroy(net)
