"""Second half of SURVEY.md 8(f)-4: a 9-species Urca-like network with weak, first-order reactions
whose rates depend on density and temperature ("the 9-isotope Urca network is used for our Urca
simulations").  The real rate tables are not available and are not reproduced; the
stand-in (workloads.urca9_like_network) brings ONE new thing to the model: per-reaction density exponents
(bz_net_desc.rate_rho_exp, lambda_k *= rho^e_k inside the exponent).  Pins of the oracle first, GPU
parity last."""
import math

import numpy as np
import pytest
import scipy.integrate

import oracle
from workloads import make_urca9_like_workload, urca9_like_network, first_order_decay_network
from _refmodel import RefModel
from _parity import compare

RTOL, ATOL = 1e-8, 1e-12


def test_topology_conserves_mass_and_has_the_new_features():
    net = urca9_like_network()
    assert net.nspec == 9 and net.nreac == 12
    for k in range(net.nreac):
        ids = net.stoich_id[k][net.stoich_id[k] >= 0]
        assert abs(sum(net.aion[i] * net.stoich_dy[k][m] for m, i in enumerate(ids))) < 1e-12
    e = net.rate_rho_exp
    first_order = (net.reactant >= 0).sum(axis=1) == 1
    assert np.array_equal(e != 0.0, first_order)                 # exactly the weak links carry an exponent
    assert (e > 1).sum() == 3 and (e < 0).sum() == 2             # captures grow with rho, decays are blocked
    assert (net.q_mev < 0).any() and ((net.stoich_id >= 0).sum(axis=1) == 4).any()


@pytest.mark.parametrize("e", [-0.75, 0.0, 1.5])
def test_density_exponent_closed_form(e):
    """One first-order reaction with lambda = A rho^e at fixed T: Y(dt) = Y0 exp(-A rho^e dt), for three
    densities a factor 10 apart -- a dropped exponent, a wrong sign or log10 for ln fails by factors."""
    dt = 1e-6
    for rho in (1e8, 1e9, 1e10):
        lamdt = 2.0
        net = first_order_decay_network(lamdt / dt / rho ** e)        # A such that lambda dt = 2 at this rho
        net.rate_rho_exp = np.array([e])
        To, Xo, ns, _ = oracle.burn(net, np.array([rho, 10 * rho]), np.array([2e9, 2e9]), np.array([[0.7, 0.7], [0.1, 0.1]]),
                                    dt, RTOL, ATOL)
        for z, ld in ((0, lamdt), (1, lamdt * 10.0 ** e)):              # the second zone is 10x denser
            ref = 0.7 / 4 * math.exp(-ld)
            assert abs(Xo[0, z] / 4 - ref) <= 100 * (RTOL * ref + ATOL), (e, rho, z)
        assert To[0] == 2e9


def test_rhs_and_jacobian_against_the_independent_model():
    net = urca9_like_network()
    ref = RefModel(net)
    rng = np.random.default_rng(77)
    for _ in range(10):
        y = np.append((0.01 + rng.random(9)) / net.aion, 5e8 + 2.5e9 * rng.random())
        rho = 10 ** (8 + 2 * rng.random())
        f, J = oracle.rates(net, rho, y)
        fr = ref.f(rho, y)
        assert np.allclose(f, fr, rtol=1e-11, atol=1e-12 * np.abs(fr).max())
        assert abs(np.dot(net.aion, f[:9])) <= 1e-12 * np.abs(net.aion * f[:9]).sum()      # sum A_i f_i = 0
        Jfd = ref.jac_fd(rho, y)
        term = np.abs(Jfd * y[None, :]).max(axis=1, keepdims=True)
        assert np.all(np.abs(J - Jfd) <= 2e-6 * np.abs(Jfd) + 1e-8 * term / np.abs(y)[None, :])
        assert np.abs(net.aion @ J[:9, :]).max() <= 1e-10 * np.abs(net.aion[:, None] * J[:9, :]).sum(axis=0).max()


def test_integrated_invariant_and_radau():
    w = make_urca9_like_workload(96)
    To, Xo, ns, cnt = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL)
    assert (ns > 20).all() and np.median(ns) > 300
    assert np.abs(Xo.sum(axis=0) - w.X.sum(axis=0)).max() <= 1e-10
    moved = np.abs(Xo[6] - w.X[6]) + np.abs(Xo[7] - w.X[7])          # the Urca pair is active
    assert (moved > 1e-3).mean() > 0.5
    ref = RefModel(w.net)

    def radau(z):
        y0 = np.append(w.X[:, z] / w.net.aion, w.T[z])
        sol = scipy.integrate.solve_ivp(lambda t, y: ref.f(w.rho[z], y), (0, w.dt), y0, method="Radau", rtol=1e-11,
                                        atol=1e-16, jac=lambda t, y: ref.jac_fd(w.rho[z], y))
        assert sol.success
        return sol.y[:, -1]

    for z in (3, 40):
        yr = radau(z)
        Xr = yr[:-1] * w.net.aion
        assert abs(To[z] - yr[-1]) <= 1e-7 * yr[-1]
        dom = Xr > 1e-3
        assert np.all(np.abs(Xo[dom, z] - Xr[dom]) <= 1e-6 * Xr[dom])
        assert np.all(np.abs(Xo[:, z] - Xr) / w.net.aion <= 2e-7 * np.abs(yr[:-1]) + 300 * ATOL)
    # zone 77 is caught in mid-runaway at t = dt (T: 5.8e8 -> 9.8e8 and rising), which amplifies the
    # tolerance: pinned as convergence to Radau under tolerance tightening instead of a fixed bound
    z, errs = 77, []
    yr = radau(z)
    for rt in (1e-8, 1e-10, 1e-12):
        o = oracle.burn(w.net, w.rho[z:z + 1], w.T[z:z + 1], w.X[:, z:z + 1], w.dt, rt, rt * 1e-4)
        errs.append(abs(o[0][0] - yr[-1]) / yr[-1])
    assert errs[0] <= 1e-5 and errs[1] <= errs[0] / 30 and errs[2] <= 3e-9, errs


def test_exponents_of_zero_change_no_bit():
    """fma(0, ln rho, x) = x exactly: a network handed an all-zero exponent array is the plain network."""
    from workloads import make_workload
    w = make_workload(3, zones=8191)
    a = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol)
    w.net.rate_rho_exp = np.zeros(w.net.nreac)
    b = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


@pytest.mark.gpu
def test_urca9_like_gpu_parity():
    import torch
    import paper_1711_06203_b200 as bz
    w = make_urca9_like_workload(4099)
    dev = torch.device("cuda:0")
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    net = bz.net_create(w.net)
    assert net.kernel_name == "burn_coop<16,16>"
    To, Xo, ns = bz.burn_zones(net, d(w.rho), d(w.T), d(w.X), w.dt, w.rtol, w.atol)
    torch.cuda.synchronize()
    cnt = bz.get_counters(net)
    Tr, Xr, nr, cr = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol, norm_lanes=net.norm_lanes)
    stats = compare(To.cpu().numpy(), Xo.cpu().numpy(), ns.cpu().numpy(), Tr, Xr, nr)
    assert stats["nsteps_equal"] == 1.0 and stats["bitexact_X"] == 1.0 and stats["bitexact_T"] == 1.0
    assert all(cnt[k] == cr[k] for k in cnt)
    # the no-allocation entry point takes the exponents too
    To2, Xo2, ns2 = torch.empty_like(To), torch.empty_like(Xo), torch.empty_like(ns)
    bz.burn_zones_static(w.net, d(w.rho), d(w.T), d(w.X), w.dt, w.rtol, w.atol, To2, Xo2, ns2)
    torch.cuda.synchronize()
    assert torch.equal(To, To2) and torch.equal(Xo, Xo2) and torch.equal(ns, ns2)
    bz.net_destroy(net)
    # a known topology that carries exponents must leave the generated kernel
    from workloads import make_workload
    w3 = make_workload(3, zones=4099)
    w3.net.rate_rho_exp = np.full(w3.net.nreac, 0.01)
    net = bz.net_create(w3.net)
    assert net.kernel_name.startswith("burn_coop")
    To, Xo, ns = bz.burn_zones(net, d(w3.rho), d(w3.T), d(w3.X), w3.dt, w3.rtol, w3.atol)
    torch.cuda.synchronize()
    Tr, Xr, nr, _ = oracle.burn(w3.net, w3.rho, w3.T, w3.X, w3.dt, w3.rtol, w3.atol, norm_lanes=net.norm_lanes)
    assert np.array_equal(Xo.cpu().numpy(), Xr) and np.array_equal(ns.cpu().numpy(), nr)
    bz.net_destroy(net)
