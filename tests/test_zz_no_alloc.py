"""burn_zones_static (include/burnzones.h): the burn for callers that may not allocate device
memory.  Its scratch -- work-queue head, counters, network tables -- is a static 32 KiB device
array shared by every call, so the test makes TWO calls in a row with DIFFERENT networks (the second
must not see the first one's tables, queue position or counters) and compares each with the existing
path (net_create + the cooperative kernel + burn_zones) at the parity tolerance of tests/_parity.py;
the two run the same kernel, so the results are in fact bit-identical, which is asserted too.

Collected last on purpose (file name): the suite runs with pytest -x.  Passes alone in a fresh
process and after the other tests (nothing here depends on earlier state; the static array is
re-initialised by every call)."""
import ctypes as C

import numpy as np
import pytest

from _parity import compare
from workloads import make_workload


def _existing_path(bz, torch, w, dev):
    net = bz.net_create(w.net)
    net.select_kernel("coop")
    To, Xo, ns = bz.burn_zones(net, torch.from_numpy(w.rho).to(dev), torch.from_numpy(w.T).to(dev),
                               torch.from_numpy(w.X).to(dev), w.dt, w.rtol, w.atol)
    torch.cuda.synchronize()
    out = To.cpu().numpy(), Xo.cpu().numpy(), ns.cpu().numpy()
    bz.net_destroy(net)
    return out


@pytest.mark.gpu
def test_static_entry_matches_existing_path_on_two_calls_in_a_row():
    import torch
    import paper_1711_06203_b200 as bz
    dev = torch.device("cuda:0")
    cases = [make_workload(3, zones=4099), make_workload(5, zones=16411), make_workload(1, zones=8)]
    refs = [_existing_path(bz, torch, w, dev) for w in cases]
    # inputs and outputs are the caller's: allocate them all BEFORE the calls under test
    bufs = []
    for w in cases:
        rho, T, X = (torch.from_numpy(a).to(dev) for a in (w.rho, w.T, w.X))
        bufs.append((rho, T, X, torch.empty_like(T), torch.empty_like(X),
                     torch.empty(w.nz, dtype=torch.int32, device=dev)))
    torch.cuda.synchronize()
    mem0 = torch.cuda.mem_get_info()[0]
    for w, b in zip(cases, bufs):                     # back to back on one stream, no sync in between
        bz.burn_zones_static(w.net, b[0], b[1], b[2], w.dt, w.rtol, w.atol, b[3], b[4], b[5])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= mem0       # the calls took no device memory
    for w, b, (Tr, Xr, nr) in zip(cases, bufs, refs):
        To, Xo, ns = b[3].cpu().numpy(), b[4].cpu().numpy(), b[5].cpu().numpy()
        stats = compare(To, Xo, ns, Tr, Xr, nr)       # the tolerance the parity tests use
        assert stats["nsteps_equal"] == 1.0 and stats["bitexact_X"] == 1.0 and stats["bitexact_T"] == 1.0
        assert (nr > 0).mean() > 0.99 and nr.max() > 100
    # a second round over the same array (it now holds the config-1 tables): same answers again
    w, b, (Tr, Xr, nr) = cases[0], bufs[0], refs[0]
    b[3].zero_(), b[4].zero_(), b[5].zero_()
    bz.burn_zones_static(w.net, b[0], b[1], b[2], w.dt, w.rtol, w.atol, b[3], b[4], b[5])
    torch.cuda.synchronize()
    assert np.array_equal(b[4].cpu().numpy(), Xr) and np.array_equal(b[3].cpu().numpy(), Tr)
    assert np.array_equal(b[5].cpu().numpy(), nr)


@pytest.mark.gpu
def test_static_entry_rejects_what_does_not_fit_and_bad_arguments():
    import torch
    import paper_1711_06203_b200 as bz
    from workloads.configs import Network
    dev = torch.device("cuda:0")
    w = make_workload(1, zones=64)
    rho, T, X = (torch.from_numpy(a).to(dev) for a in (w.rho, w.T, w.X))
    To, Xo, ns = torch.empty_like(T), torch.empty_like(X), torch.empty(w.nz, dtype=torch.int32, device=dev)
    K = 257                                           # one reaction more than the static tables hold
    big = Network("big", ["a", "b"], np.array([12.0, 24.0]), np.tile(np.array([[0, 0, -1]], dtype=np.int32), (K, 1)),
                  np.tile(np.array([[0, 1, -1, -1]], dtype=np.int32), (K, 1)), np.tile(np.array([[-2.0, 1.0, 0, 0]]), (K, 1)),
                  np.full(K, 1e10), np.zeros(K), np.full(K, 30.0), np.ones(K))
    with pytest.raises(bz.BurnError) as e:
        bz.burn_zones_static(big, rho, T, X, w.dt, w.rtol, w.atol, To, Xo, ns)
    assert e.value.code == -2                         # BZ_ERR_SIZE, nothing enqueued
    with pytest.raises(bz.BurnError) as e:
        bz.burn_zones_static(w.net, rho, T, X, -1.0, w.rtol, w.atol, To, Xo, ns)
    assert e.value.code == -4
    bad = make_workload(1, zones=64).net
    bad.rate_A = np.array([np.inf])
    with pytest.raises(bz.BurnError) as e:
        bz.burn_zones_static(bad, rho, T, X, w.dt, w.rtol, w.atol, To, Xo, ns)
    assert e.value.code == -3
    # and the array is still usable afterwards
    bz.burn_zones_static(w.net, rho, T, X, w.dt, w.rtol, w.atol, To, Xo, ns)
    torch.cuda.synchronize()
    assert (ns.cpu().numpy() > 0).all()


def test_static_entry_validates_before_cuda():
    """No GPU needed: sizes beyond the static array and NULL descriptors are refused up front."""
    import paper_1711_06203_b200 as bz
    from paper_1711_06203_b200 import build as bzbuild
    bzbuild.build()
    lib = C.CDLL(bz.library_path())
    lib.burn_zones_static.restype = C.c_int
    assert lib.burn_zones_static(None, C.c_int64(0), None, None, None, C.c_double(1e-6), C.c_double(1e-8),
                                 C.c_double(1e-12), None, None, None, None) == -1
    assert bz.STATIC_SCRATCH_BYTES == 32768
