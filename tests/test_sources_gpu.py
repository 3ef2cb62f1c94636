"""GPU parity of burn_zones_src (constant source terms) and of the Strang
driver against the CPU oracle: same seeded inputs, element by element; expected bit-identical."""
import numpy as np
import pytest

import oracle
from workloads import make_workload, first_order_decay_network
from _parity import compare

pytestmark = pytest.mark.gpu


def _sources(w, seed, scale_x=2e-3, scale_t=2e-2):
    """Synthetic advective sources: a few per mille of the composition and a few per cent of T per
    burn interval, either sign (what a hydro update over one step typically moves)."""
    rng = np.random.default_rng(seed)
    sX = (rng.random(w.X.shape) - 0.5) * scale_x / w.dt * np.maximum(w.X, 1e-3)
    sT = (rng.random(w.nz) - 0.5) * scale_t * w.T / w.dt
    return sT, sX


def _gpu_burn_src(w, sT, sX, kind="auto"):
    import torch
    import paper_1711_06203_b200 as bz
    net = bz.net_create(w.net)
    net.select_kernel(kind)
    dev = torch.device("cuda:0")
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    To, Xo, ns = bz.burn_zones_src(net, d(w.rho), d(w.T), d(w.X), d(sT), d(sX), w.dt, w.rtol, w.atol)
    torch.cuda.synchronize()
    cnt = bz.get_counters(net)
    out = To.cpu().numpy(), Xo.cpu().numpy(), ns.cpu().numpy(), cnt, net.norm_lanes, net.kernel_name
    bz.net_destroy(net)
    return out


@pytest.mark.parametrize("kind", ["auto", "coop"])
@pytest.mark.parametrize("config,zones", [(1, None), (2, 61), (3, 509), (5, 4099)])
def test_parity_with_sources(config, zones, kind):
    if kind == "coop" and config == 5:
        pytest.skip("config 5: auto already is the cooperative kernel")
    w = make_workload(config, zones=zones)
    sT, sX = _sources(w, 40 + config)
    To, Xo, ns, cnt, lanes, name = _gpu_burn_src(w, sT, sX, kind)
    assert name.startswith("burn_coop" if (kind == "coop" or config == 5) else "burn_quad"), name
    Tr, Xr, nr, cr = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol, norm_lanes=lanes, src_T=sT, src_X=sX)
    stats = compare(To, Xo, ns, Tr, Xr, nr)
    assert stats["bitexact_X"] == 1.0 and stats["bitexact_T"] == 1.0 and stats["nsteps_equal"] == 1.0, stats
    assert all(cnt[k] == cr[k] for k in cnt), (cnt, cr)
    # the sources really did something: the plain burn differs
    Tp, Xp, _, _ = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol, norm_lanes=lanes)
    assert np.abs(Tp - Tr).max() > 1e-4 * Tr.max()
    # linear invariant with sources, on the GPU result itself
    ok = ns > 0
    assert np.abs((Xo.sum(axis=0) - w.X.sum(axis=0)) - sX.sum(axis=0) * w.dt)[ok].max() <= 1e-10


def test_zero_sources_equal_plain_burn_on_gpu():
    import torch
    import paper_1711_06203_b200 as bz
    w = make_workload(3, zones=2039)
    net = bz.net_create(w.net)
    dev = torch.device("cuda:0")
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    a = bz.burn_zones(net, d(w.rho), d(w.T), d(w.X), w.dt, w.rtol, w.atol)
    b = bz.burn_zones_src(net, d(w.rho), d(w.T), d(w.X), d(np.zeros(w.nz)), d(np.zeros_like(w.X)), w.dt, w.rtol, w.atol)
    torch.cuda.synchronize()
    for x, y in zip(a, b):
        assert torch.equal(x, y)
    bz.net_destroy(net)


def test_closed_form_with_source_on_gpu():
    """Y_P' = -lam Y_P + s evaluated on the CUDA path directly (generic cooperative kernel)."""
    import math
    dt, lamdt = 1e-6, 5.0
    lam = lamdt / dt
    w = make_workload(1, zones=[0])
    w.net, w.dt = first_order_decay_network(lam), dt
    w.rho, w.T, w.X = np.array([1e6]), np.array([2e9]), np.array([[0.7], [0.1]])
    s = 0.05 / 4 / dt
    To, Xo, ns, *_ = _gpu_burn_src(w, np.array([0.0]), np.array([[4 * s], [0.0]]))
    YP = s / lam + (0.7 / 4 - s / lam) * math.exp(-lamdt)
    assert ns[0] > 0 and To[0] == 2e9
    assert abs(Xo[0, 0] / 4 - YP) <= 100 * (1e-8 * YP + 1e-12)


def test_invalid_sources():
    import torch
    import paper_1711_06203_b200 as bz
    w = make_workload(1, zones=[1, 2, 3, 4])
    dev = torch.device("cuda:0")
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    sT = np.array([0.0, np.nan, 0.0, 0.0])
    sX = np.zeros_like(w.X)
    sX[1, 2] = -np.inf
    for kind in ("auto", "coop"):
        net = bz.net_create(w.net)
        net.select_kernel(kind)
        To, Xo, ns = bz.burn_zones_src(net, d(w.rho), d(w.T), d(w.X), d(sT), d(sX), w.dt, w.rtol, w.atol)
        torch.cuda.synchronize()
        ns = ns.cpu().numpy()
        assert ns[0] > 0 and ns[3] > 0 and ns[1] == -4 and ns[2] == -4, (kind, ns)
        assert np.array_equal(To.cpu().numpy()[1:3], w.T[1:3]) and np.array_equal(Xo.cpu().numpy()[:, 1:3], w.X[:, 1:3])
        bz.net_destroy(net)


def test_strang_step_matches_two_oracle_half_burns():
    """burn(dt/2) - update - burn(dt/2): the driver is two burn_zones calls around the
    caller's update; compare with the oracle run the same way."""
    import torch
    import paper_1711_06203_b200 as bz
    w = make_workload(3, zones=4099)
    net = bz.net_create(w.net)
    lanes = net.norm_lanes
    dev = torch.device("cuda:0")
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)

    def update_np(rho, T, X):                 # a stand-in "hydro" update: compress and heat a little
        return rho * 1.01, T * 1.002, X

    def update_t(rho, T, X):
        return rho * 1.01, T * 1.002, X

    rho2, T2, X2, ns1, ns2 = bz.strang_step(net, d(w.rho), d(w.T), d(w.X), w.dt, w.rtol, w.atol, update=update_t)
    torch.cuda.synchronize()
    Ta, Xa, na, _ = oracle.burn(w.net, w.rho, w.T, w.X, 0.5 * w.dt, w.rtol, w.atol, norm_lanes=lanes)
    rb, Tb, Xb = update_np(w.rho, Ta, Xa)
    Tc, Xc, nc, _ = oracle.burn(w.net, rb, Tb, Xb, 0.5 * w.dt, w.rtol, w.atol, norm_lanes=lanes)
    assert np.array_equal(ns1.cpu().numpy(), na)
    stats = compare(T2.cpu().numpy(), X2.cpu().numpy(), ns2.cpu().numpy(), Tc, Xc, nc)
    assert stats["bitexact_X"] == 1.0 and stats["bitexact_T"] == 1.0 and stats["nsteps_equal"] == 1.0, stats
    bz.net_destroy(net)
