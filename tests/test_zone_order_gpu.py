"""bz_set_zone_order (step a2, second half: the order in which the work queue hands the zones out,
include/burnzones.h).  Zones are independent, so the order may change the time and nothing else: every
test here burns a batch in some order and demands the SAME BITS as in index order (which the parity tests
compare with the oracle), at the zone's own index; one test goes to the oracle directly."""
import numpy as np
import pytest

import oracle
from workloads import make_workload
from _parity import compare

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).to(torch.device("cuda:0"))


def _burn(net, w, order=None, validate=True, fill=None):
    import torch
    import paper_1711_06203_b200 as bz
    net.set_zone_order(order, validate=validate) if order is not None else net.set_zone_order(None)
    kw = {}
    if fill is not None:  # pre-filled outputs show which zones the call touched
        kw = dict(T_out=torch.full((w.nz,), fill, dtype=torch.float64, device="cuda:0"),
                  X_out=torch.full(w.X.shape, fill, dtype=torch.float64, device="cuda:0"),
                  nsteps=torch.full((w.nz,), -99, dtype=torch.int32, device="cuda:0"))
    To, Xo, ns = bz.burn_zones(net, _dev(w.rho), _dev(w.T), _dev(w.X), w.dt, w.rtol, w.atol, **kw)
    torch.cuda.synchronize()
    return To.cpu().numpy(), Xo.cpu().numpy(), ns.cpu().numpy(), bz.get_counters(net)


@pytest.mark.parametrize("config,zones,kind", [(3, 257, "quad"), (3, 1021, "coop"), (2, 61, "quad"), (5, 4099, "auto"),
                                               (1, None, "coop")])
def test_results_do_not_depend_on_the_order(config, zones, kind):
    import torch
    import paper_1711_06203_b200 as bz
    w = make_workload(config, zones=zones)
    net = bz.net_create(w.net)
    net.select_kernel(kind)
    T0, X0, n0, c0 = _burn(net, w)
    rng = np.random.default_rng(config)
    orders = {"reversed": np.arange(w.nz)[::-1].copy(), "random": rng.permutation(w.nz),
              "dearest first": np.argsort(-n0, kind="stable"), "identity": np.arange(w.nz)}
    for tag, o in orders.items():
        T1, X1, n1, c1 = _burn(net, w, torch.from_numpy(o.astype(np.int64)).to("cuda:0"))
        assert np.array_equal(n1, n0), tag
        assert np.array_equal(T1.view(np.uint64), T0.view(np.uint64)), tag
        assert np.array_equal(X1.view(np.uint64), X0.view(np.uint64)), tag
        assert c1 == c0, tag                       # every event counter too: the same work was done
    T2, X2, n2, c2 = _burn(net, w)                 # None switches it off again
    assert np.array_equal(X2.view(np.uint64), X0.view(np.uint64)) and c2 == c0
    bz.net_destroy(net)


def test_ordered_burn_against_the_oracle():
    import torch
    import paper_1711_06203_b200 as bz
    w = make_workload(3, zones=2039)
    net = bz.net_create(w.net)
    o = np.random.default_rng(11).permutation(w.nz).astype(np.int64)
    To, Xo, ns, cnt = _burn(net, w, torch.from_numpy(o).to("cuda:0"))
    Tr, Xr, nr, cr = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol, norm_lanes=net.norm_lanes)
    stats = compare(To, Xo, ns, Tr, Xr, nr)
    assert stats["bitexact_X"] == 1.0 and stats["bitexact_T"] == 1.0 and stats["nsteps_equal"] == 1.0
    assert all(cnt[k] == cr[k] for k in cnt)
    bz.net_destroy(net)


@pytest.mark.parametrize("kind", ["quad", "coop"])
def test_entries_that_are_no_zone_are_ignored_and_unnamed_zones_untouched(kind):
    import torch
    import paper_1711_06203_b200 as bz
    w = make_workload(3, zones=4093)             # 513 zones
    net = bz.net_create(w.net)
    net.select_kernel(kind)
    T0, X0, n0, _ = _burn(net, w)
    o = np.arange(w.nz, dtype=np.int64)
    o[5] = w.nz + 7                              # beyond the batch
    o[17] = -3                                   # negative
    o[40] = 41                                   # zone 41 named twice, zone 40 by nobody
    with pytest.raises(ValueError):
        net.set_zone_order(torch.from_numpy(o).to("cuda:0"))           # the binding's check
    T1, X1, n1, _ = _burn(net, w, torch.from_numpy(o).to("cuda:0"), validate=False, fill=-7.0)
    skipped = np.array([5, 17, 40])
    burned = np.setdiff1d(np.arange(w.nz), skipped)
    assert np.array_equal(n1[skipped], [-99, -99, -99]) and np.all(T1[skipped] == -7.0) and np.all(X1[:, skipped] == -7.0)
    assert np.array_equal(n1[burned], n0[burned])
    assert np.array_equal(T1[burned].view(np.uint64), T0[burned].view(np.uint64))
    assert np.array_equal(X1[:, burned].view(np.uint64), X0[:, burned].view(np.uint64))
    bz.net_destroy(net)


def test_order_errors():
    import torch
    import paper_1711_06203_b200 as bz
    from paper_1711_06203_b200.binding import BurnError
    w = make_workload(3, zones=4093)
    net = bz.net_create(w.net)
    perm = torch.arange(w.nz, dtype=torch.int64, device="cuda:0")
    for bad in (perm.to(torch.int32), perm.cpu(), perm.reshape(1, -1), perm[::2]):
        with pytest.raises(ValueError):
            net.set_zone_order(bad)
    net.set_zone_order(perm[:-1].contiguous())                    # an order for another batch size
    with pytest.raises(BurnError) as e:
        bz.burn_zones(net, _dev(w.rho), _dev(w.T), _dev(w.X), w.dt, w.rtol, w.atol)
    assert e.value.code == -2
    net.set_zone_order(perm)
    net.set_schedule("static")                                    # the order belongs to the queue
    with pytest.raises(BurnError) as e:
        bz.burn_zones(net, _dev(w.rho), _dev(w.T), _dev(w.X), w.dt, w.rtol, w.atol)
    assert e.value.code == -7
    net.set_schedule("queue")
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    with pytest.raises(BurnError) as e:                           # the host path burns in chunks
        bz.burn_zones_host(net, pin(w.rho), pin(w.T), pin(w.X), w.dt, w.rtol, w.atol,
                           torch.empty(w.nz, dtype=torch.float64).pin_memory(),
                           torch.empty(w.X.shape, dtype=torch.float64).pin_memory(),
                           torch.empty(w.nz, dtype=torch.int32).pin_memory())
    assert e.value.code == -7
    net.set_zone_order(None)
    bz.burn_zones(net, _dev(w.rho), _dev(w.T), _dev(w.X), w.dt, w.rtol, w.atol)
    torch.cuda.synchronize()
    bz.net_destroy(net)


@pytest.mark.parametrize("config,zones,kind", [(3, 64, "quad"), (3, 128, "coop"), (2, None, "quad"), (4, 16, "quad"),
                                               (5, 256, "auto"), (1, None, "quad")])
def test_cost_schedule_gives_the_same_bits(config, zones, kind):
    """bz_set_schedule(net, 2), the default: the library orders the queue itself (cost key kernel + radix sort).
    Batches larger than the grid holds at once, or the library skips the ordering (config 1 here: that path)."""
    import torch
    import paper_1711_06203_b200 as bz
    w = make_workload(config, zones=zones)
    net = bz.net_create(w.net)
    net.select_kernel(kind)
    net.set_schedule("queue")
    T0, X0, n0, c0 = _burn(net, w)
    net.set_schedule("cost")
    for _ in range(2):                                       # twice: the second call reuses the buffers
        T1, X1, n1, c1 = _burn(net, w)
        assert np.array_equal(n1, n0) and c1 == c0
        assert np.array_equal(T1.view(np.uint64), T0.view(np.uint64))
        assert np.array_equal(X1.view(np.uint64), X0.view(np.uint64))
    # a caller's order wins over the library's
    T2, X2, n2, c2 = _burn(net, w, torch.arange(w.nz - 1, -1, -1, dtype=torch.int64, device="cuda:0"))
    assert np.array_equal(X2.view(np.uint64), X0.view(np.uint64)) and c2 == c0
    bz.net_destroy(net)


def test_cost_schedule_batches_of_changing_size_sources_and_host_path():
    import torch
    import paper_1711_06203_b200 as bz
    net_d = make_workload(3, zones=4093).net
    net = bz.net_create(net_d)
    ref = bz.net_create(net_d)
    net.set_schedule("cost")
    ref.set_schedule("queue")
    rng = np.random.default_rng(3)
    for stride in (64, 16, 128, 32):                         # 32768, 131072, 16384, 65536 zones: buffers grow and are reused
        w = make_workload(3, zones=stride)
        sT = (rng.random(w.nz) - 0.5) * 2e-2 * w.T / w.dt
        sX = (rng.random(w.X.shape) - 0.5) * 2e-3 / w.dt * np.maximum(w.X, 1e-3)
        a = bz.burn_zones_src(net, _dev(w.rho), _dev(w.T), _dev(w.X), _dev(sT), _dev(sX), w.dt, w.rtol, w.atol)
        b = bz.burn_zones_src(ref, _dev(w.rho), _dev(w.T), _dev(w.X), _dev(sT), _dev(sX), w.dt, w.rtol, w.atol)
        torch.cuda.synchronize()
        for x, y in zip(a, b):
            assert torch.equal(x, y)
        assert bz.get_counters(net) == bz.get_counters(ref)
    w = make_workload(3, zones=61)                          # 34380 zones through the host path
    pin = lambda t: torch.from_numpy(np.ascontiguousarray(t)).pin_memory()
    outs = []
    for h in (net, ref):
        To = torch.empty(w.nz, dtype=torch.float64).pin_memory()
        Xo = torch.empty(w.X.shape, dtype=torch.float64).pin_memory()
        ns = torch.empty(w.nz, dtype=torch.int32).pin_memory()
        bz.burn_zones_host(h, pin(w.rho), pin(w.T), pin(w.X), w.dt, w.rtol, w.atol, To, Xo, ns)
        torch.cuda.synchronize()
        outs.append((To.clone(), Xo.clone(), ns.clone()))
    for x, y in zip(*outs):
        assert torch.equal(x, y)
    bz.net_destroy(net)
    bz.net_destroy(ref)


def test_cost_key_puts_the_dear_zones_first():
    """Config 4 at full size (256^3 zones: a cold background that takes one step, hot spots that take up to ~400):
    the key must send the dear zones out early.  Checked through its effect, the only thing visible at the
    boundary: the burn is much shorter than in index order (measured 46 ms against 79 ms; the bar is 0.8)."""
    import torch
    import paper_1711_06203_b200 as bz
    w = make_workload(4)
    net = bz.net_create(w.net)
    rho, T, X = _dev(w.rho), _dev(w.T), _dev(w.X)
    To, Xo = torch.empty_like(T), torch.empty_like(X)
    ns = torch.empty(w.nz, dtype=torch.int32, device="cuda:0")

    def timed():
        ts = []
        for _ in range(4):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            bz.burn_zones(net, rho, T, X, w.dt, w.rtol, w.atol, T_out=To, X_out=Xo, nsteps=ns)
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return min(ts[1:])

    net.set_schedule("queue")
    t_index = timed()
    ref = (To.clone(), Xo.clone(), ns.clone())
    net.set_schedule("cost")
    t_cost = timed()
    assert int((ns > 50).sum()) > 1000                       # there are dear zones
    assert torch.equal(To, ref[0]) and torch.equal(Xo, ref[1]) and torch.equal(ns, ref[2])
    assert t_cost < 0.8 * t_index, (t_cost, t_index)
    bz.net_destroy(net)
