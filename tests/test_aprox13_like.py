"""A second 13-isotope workload: the alpha chain with
alpha-emitting heavy-ion channels and reverse (photodisintegration) links, synthetic rate data
(workloads.aprox13_like_network).  It has first-order reactions, four-entry stoichiometry and
negative Q-values, none of which the five BASELINE configs contain; and it runs on the generic
cooperative kernel.  CPU part: the oracle on this network against an independent right-hand side,
invariants, finite differences and scipy's Radau.  GPU part: parity with the oracle."""
import numpy as np
import pytest
import scipy.integrate

import oracle
from workloads import aprox13_like_network, make_aprox13_like_workload
from _refmodel import RefModel
from _parity import compare

RTOL, ATOL = 1e-8, 1e-12


def test_topology_conserves_mass_and_has_the_new_features():
    net = aprox13_like_network()
    assert net.nspec == 13 and net.nreac == 26
    for k in range(net.nreac):
        assert abs(sum(net.aion[i] * d for i, d in zip(net.stoich_id[k], net.stoich_dy[k]) if i >= 0)) < 1e-12
    nreact = (np.asarray(net.reactant) >= 0).sum(axis=1)
    assert (nreact == 1).sum() == 11                      # first-order reverse links
    assert ((np.asarray(net.stoich_id) >= 0).sum(axis=1) == 4).sum() == 1   # C12+O16 -> Mg24 + a
    assert (np.asarray(net.q_mev) < 0).sum() == 11        # endothermic


def test_rhs_and_jacobian():
    net = aprox13_like_network()
    ref = RefModel(net)
    rng = np.random.default_rng(3)
    n = net.neq
    for _ in range(6):
        y = np.append(0.002 + rng.random(13) * 0.03, 1e9 * (1.0 + 3.0 * rng.random()))
        rho = 10 ** (6 + 2 * rng.random())
        f, J = oracle.rates(net, rho, y)
        g = ref.f(rho, y)
        assert np.abs(f - g).max() <= 1e-11 * np.abs(g).max()
        a = net.aion
        assert abs(a @ f[:-1]) <= 1e-13 * np.sum(np.abs(a * f[:-1]))
        assert np.all(np.abs(a @ J[:-1, :]) <= 1e-13 * (np.abs(a)[:, None] * np.abs(J[:-1, :])).sum(axis=0) + 1e-300)
        Jfd = np.zeros((n, n))
        for j in range(n):
            h = 1e-6 * y[j]
            yp, ym = y.copy(), y.copy()
            yp[j] += h
            ym[j] -= h
            Jfd[:, j] = (oracle.rates(net, rho, yp, jac=False) - oracle.rates(net, rho, ym, jac=False)) / (2 * h)
        noise = 1e-9 * np.abs(f)[:, None] / (1e-6 * y)[None, :]
        big = np.abs(J) > 1e3 * noise
        assert big.sum() > n
        assert np.all(np.abs(J - Jfd)[big] <= 2e-7 * np.abs(J)[big])


def test_burn_invariant_and_scipy():
    w = make_aprox13_like_workload(96)
    To, Xo, ns, cnt = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, RTOL, ATOL)
    assert (ns > 0).all() and ns.max() > 50 * ns.min()           # lively and divergent
    assert np.abs(Xo.sum(axis=0) - w.X.sum(axis=0)).max() <= 1e-10
    ref = RefModel(w.net)
    # Library cross-check in two steps: the oracle at rtol 1e-11 against scipy's Radau on the
    # independent right-hand side (model + integrator agree to 1e-8), then the rtol 1e-8 run against
    # the tight one (global error of a BDF run: some tens of rtol; a zone with ~25 large steps shows
    # 2e-7 relative here).  (The hottest zones reach T > 1e10, where Radau takes minutes: skipped.)
    for z in np.flatnonzero(To < 6e9)[:4]:
        y0 = np.append(w.X[:, z] / w.net.aion, w.T[z])
        sol = scipy.integrate.solve_ivp(lambda t, y: ref.f(w.rho[z], y), (0, w.dt), y0, method="Radau",
                                        rtol=1e-11, atol=1e-16, jac=lambda t, y: ref.jac_fd(w.rho[z], y))
        assert sol.success
        yr = sol.y[:, -1]
        Tt, Xt, nt, _ = oracle.burn(w.net, w.rho[z:z + 1], w.T[z:z + 1], w.X[:, z:z + 1], w.dt, 1e-11, 1e-15)
        Yt = Xt[:, 0] / w.net.aion
        assert nt[0] > 0 and abs(Tt[0] - yr[-1]) <= 1e-8 * yr[-1]
        assert np.all(np.abs(Yt - yr[:-1]) <= 1e-8 * np.abs(yr[:-1]) + 1e-14)
        assert abs(To[z] - Tt[0]) <= 1e-6 * Tt[0]
        assert np.all(np.abs(Xo[:, z] / w.net.aion - Yt) <= 1e-6 * np.abs(Yt) + 300 * ATOL)


@pytest.mark.gpu
@pytest.mark.parametrize("with_sources", [False, True])
def test_gpu_parity(with_sources):
    """Runs on the generic cooperative kernel: this topology gets no generated kernel, on purpose.
    Its Newton matrices need 0.77 row interchanges per factorisation (the reverse links pair large
    off-diagonal entries; config 3 needs none), so the quad kernel's no-interchange LU would fall to
    its general path almost every step -- measured 14x slower than the cooperative kernel, which
    pivots natively."""
    import torch
    import paper_1711_06203_b200 as bz
    w = make_aprox13_like_workload(2053)
    net = bz.net_create(w.net)
    assert net.kernel_name.startswith("burn_coop<14,16>"), net.kernel_name
    dev = torch.device("cuda:0")
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    kw = {}
    if with_sources:
        rng = np.random.default_rng(77)
        kw = dict(src_T=(rng.random(w.nz) - 0.5) * 2e-2 * w.T / w.dt,
                  src_X=(rng.random(w.X.shape) - 0.5) * 2e-3 / w.dt * np.maximum(w.X, 1e-3))
        To, Xo, ns = bz.burn_zones_src(net, d(w.rho), d(w.T), d(w.X), d(kw["src_T"]), d(kw["src_X"]), w.dt, w.rtol, w.atol)
    else:
        To, Xo, ns = bz.burn_zones(net, d(w.rho), d(w.T), d(w.X), w.dt, w.rtol, w.atol)
    torch.cuda.synchronize()
    cnt = bz.get_counters(net)
    Tr, Xr, nr, cr = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol, norm_lanes=net.norm_lanes, **kw)
    stats = compare(To.cpu().numpy(), Xo.cpu().numpy(), ns.cpu().numpy(), Tr, Xr, nr)
    assert stats["bitexact_X"] == 1.0 and stats["bitexact_T"] == 1.0 and stats["nsteps_equal"] == 1.0, stats
    assert all(cnt[k] == cr[k] for k in cnt), (cnt, cr)
    bz.net_destroy(net)
