"""ctypes wrapper of liboracle.so: numpy in, numpy out.  No arithmetic of the method here."""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

COUNTER_NAMES = ("nst", "nrhs", "njac", "nlu", "nsolve", "netf", "ncfn", "nfailzones")

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class _Desc(C.Structure):
    _fields_ = [("nspec", C.c_int32), ("nreac", C.c_int32), ("aion", _dp), ("reactant", _ip),
                ("stoich_id", _ip), ("stoich_dy", _dp), ("rate_A", _dp), ("rate_n", _dp),
                ("rate_B", _dp), ("q_mev", _dp), ("cv", C.c_double), ("rate_rho_exp", _dp),
                ("zion", _dp), ("eos_extra", C.c_double)]


class _Opts(C.Structure):
    _fields_ = [("norm_lanes", C.c_int32), ("fixed_q", C.c_int32), ("fixed_h", C.c_double),
                ("z_init", _dp), ("nthreads", C.c_int32), ("src_T", _dp), ("src_X", _dp),
                ("trace", _dp), ("trace_cap", C.c_int32), ("trace_n", _ip),
                ("mxstep", C.c_int32), ("mxnef", C.c_int32), ("mxncf", C.c_int32),
                ("inject_step", C.c_int32), ("inject_nef", C.c_int32),
                ("policy", C.c_int32), ("nstale", C.POINTER(C.c_uint64))]


TRACE_HEAD = 16
TRACE_FIELDS = ("kind", "t", "h_used", "q_used", "dsm", "eta_q", "eta_qm1", "eta_qp1", "E_minus", "E_plus",
                "action", "eta", "h_next", "q_next", "nef", "ncf")


_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        lib.orc_burn.restype = C.c_int
        lib.orc_burn.argtypes = [C.POINTER(_Desc), C.c_int64, _dp, _dp, _dp, C.c_double, C.c_double,
                                 C.c_double, _dp, _dp, _ip, C.POINTER(_Opts), C.POINTER(C.c_uint64)]
        lib.orc_rates.restype = C.c_int
        lib.orc_rates.argtypes = [C.POINTER(_Desc), C.c_double, _dp, _dp, _dp]
        lib.orc_exp.restype = C.c_double
        lib.orc_exp.argtypes = [C.c_double]
        lib.orc_log.restype = C.c_double
        lib.orc_log.argtypes = [C.c_double]
        lib.orc_lu_factor.restype = C.c_int
        lib.orc_lu_factor.argtypes = [C.c_int, _dp, _ip, _dp]
        lib.orc_lu_solve.restype = None
        lib.orc_lu_solve.argtypes = [C.c_int, _dp, _ip, _dp, _dp]
        lib.orc_bdf_coeffs.restype = None
        lib.orc_bdf_coeffs.argtypes = [C.c_int, C.c_double, _dp, _dp]
        lib.orc_wrms.restype = C.c_double
        lib.orc_wrms.argtypes = [C.c_int, _dp, _dp, C.c_int]
        lib.orc_max_threads.restype = C.c_int
        lib.orc_event_counts.restype = None
        lib.orc_event_counts.argtypes = [C.c_int, C.POINTER(C.c_uint64)]
        lib.orc_interchanges.restype = C.c_uint64
        lib.orc_interchanges.argtypes = [C.c_int]
        lib.orc_build_d.restype = None
        lib.orc_build_d.argtypes = [C.c_int, _dp, _dp]
        _lib = lib
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def _desc(net):
    """net: any object with the fields of workloads.Network.  Returns (struct, keepalive)."""
    keep = dict(
        aion=np.ascontiguousarray(net.aion, dtype=np.float64),
        reactant=np.ascontiguousarray(net.reactant, dtype=np.int32),
        stoich_id=np.ascontiguousarray(net.stoich_id, dtype=np.int32),
        stoich_dy=np.ascontiguousarray(net.stoich_dy, dtype=np.float64),
        rate_A=np.ascontiguousarray(net.rate_A, dtype=np.float64),
        rate_n=np.ascontiguousarray(net.rate_n, dtype=np.float64),
        rate_B=np.ascontiguousarray(net.rate_B, dtype=np.float64),
        q_mev=np.ascontiguousarray(net.q_mev, dtype=np.float64),
    )
    zion = getattr(net, "zion", None)
    if zion is not None:
        keep["zion"] = np.ascontiguousarray(zion, dtype=np.float64)
        assert keep["zion"].shape == keep["aion"].shape
    rexp = getattr(net, "rate_rho_exp", None)
    if rexp is not None:
        keep["rate_rho_exp"] = np.ascontiguousarray(rexp, dtype=np.float64)
        assert keep["rate_rho_exp"].shape == keep["rate_A"].shape
    d = _Desc(int(keep["aion"].shape[0]), int(keep["rate_A"].shape[0]), _d(keep["aion"]),
              _i(keep["reactant"]), _i(keep["stoich_id"]), _d(keep["stoich_dy"]), _d(keep["rate_A"]),
              _d(keep["rate_n"]), _d(keep["rate_B"]), _d(keep["q_mev"]), float(net.cv),
              _d(keep["rate_rho_exp"]) if rexp is not None else None,
              _d(keep["zion"]) if zion is not None else None, float(getattr(net, "eos_extra", 0.0) or 0.0))
    return d, keep


def interchanges(reset: bool = False) -> int:
    """Row interchanges performed by the LU since the last reset (test aid)."""
    return int(_L().orc_interchanges(1 if reset else 0))


def event_counts(reset: bool = False) -> dict:
    """How often rarely taken paths ran since the last reset (test aid)."""
    out = (C.c_uint64 * 3)()
    _L().orc_event_counts(1 if reset else 0, out)
    return dict(interchanges=int(out[0]), etf_lower_order=int(out[1]), etf_restart_order1=int(out[2]))


def max_threads() -> int:
    return int(_L().orc_max_threads())


def burn(net, rho, T, X, dt, rtol, atol, norm_lanes=1, nthreads=0, fixed_q=0, fixed_h=0.0, z_init=None,
         src_T=None, src_X=None, trace=0, mxstep=0, mxnef=0, mxncf=0, inject=(0, 0), policy=0):
    """Integrate every zone over dt.  X: [nspec, nz].  Returns (T_out, X_out, nsteps, counters).
    src_T [nz] (K/s) and src_X [nspec, nz] (mass-fraction rate, 1/s): optional constant source terms
    (dy/dt = f + s, bz_oracle.h); give both or neither.
    mxstep / mxnef / mxncf: the limits behind the failure codes -3 / -2 / -1 (0 = defaults 20000 / 7 / 10).
    policy: 0 = fresh Jacobian and LU on every attempt (v1, default); 1 = VODE-style reuse of the Newton
    matrix (v2, bz_oracle.h); with policy 1 the counters dict also holds 'nstale'.
    inject = (step, nef): test hook, the attempts of accepted step `step` fail the error test nef times.
    trace = capacity in events: zone 0's event records (bz_oracle.h, orc_opts.trace) are returned as a
    fifth value, a list of dicts with the TRACE_FIELDS plus 'Zacc', 'Zend' ([6, n] arrays, API order)."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    T = np.ascontiguousarray(T, dtype=np.float64)
    X = np.ascontiguousarray(X, dtype=np.float64)
    nz = rho.shape[0]
    d, keep = _desc(net)
    assert X.shape == (d.nspec, nz) and T.shape == (nz,)
    T_out = np.empty(nz)
    X_out = np.empty((d.nspec, nz))
    nsteps = np.empty(nz, dtype=np.int32)
    cnt = (C.c_uint64 * 8)()
    zi = None
    if z_init is not None:
        zi = np.ascontiguousarray(z_init, dtype=np.float64)
    assert (src_T is None) == (src_X is None)
    sT = sX = None
    if src_T is not None:
        sT = np.ascontiguousarray(src_T, dtype=np.float64)
        sX = np.ascontiguousarray(src_X, dtype=np.float64)
        assert sT.shape == (nz,) and sX.shape == (d.nspec, nz)
    n = d.nspec + 1
    tbuf = np.zeros((int(trace), TRACE_HEAD + 12 * n)) if trace else None
    tn = np.zeros(1, dtype=np.int32)
    stale = C.c_uint64(0)
    opts = _Opts(int(norm_lanes), int(fixed_q), float(fixed_h), _d(zi) if zi is not None else None,
                 int(nthreads), _d(sT) if sT is not None else None, _d(sX) if sX is not None else None,
                 _d(tbuf) if trace else None, int(trace), _i(tn), int(mxstep), int(mxnef), int(mxncf), int(inject[0]), int(inject[1]),
                 int(policy), C.cast(C.pointer(stale), C.POINTER(C.c_uint64)))
    rc = _L().orc_burn(C.byref(d), nz, _d(rho), _d(T), _d(X), dt, rtol, atol, _d(T_out), _d(X_out),
                       _i(nsteps), C.byref(opts), cnt)
    if rc != 0:
        raise ValueError(f"orc_burn failed with code {rc}")
    out = (T_out, X_out, nsteps, dict(zip(COUNTER_NAMES, (int(c) for c in cnt))))
    if policy:
        out[3]["nstale"] = int(stale.value)
    if not trace:
        return out
    if int(tn[0]) > int(trace):
        raise ValueError(f"trace capacity {trace} too small for {int(tn[0])} events")
    recs = []
    for r in tbuf[: int(tn[0])]:
        e = dict(zip(TRACE_FIELDS, r[:TRACE_HEAD]))
        for k in ("kind", "q_used", "action", "q_next", "nef", "ncf"):
            e[k] = int(e[k])
        e["Zacc"] = r[TRACE_HEAD:TRACE_HEAD + 6 * n].reshape(6, n).copy()
        e["Zend"] = r[TRACE_HEAD + 6 * n:].reshape(6, n).copy()
        recs.append(e)
    return out + (recs,)


def rates(net, rho, y, jac=True):
    d, keep = _desc(net)
    y = np.ascontiguousarray(y, dtype=np.float64)
    n = d.nspec + 1
    assert y.shape == (n,)
    f = np.empty(n)
    J = np.empty((n, n)) if jac else None
    rc = _L().orc_rates(C.byref(d), float(rho), _d(y), _d(f), _d(J) if jac else None)
    if rc != 0:
        raise ValueError(f"orc_rates failed with code {rc}")
    return (f, J) if jac else f


def oexp(x: float) -> float:
    return float(_L().orc_exp(float(x)))


def olog(x: float) -> float:
    return float(_L().orc_log(float(x)))


def lu_factor(a):
    a = np.array(a, dtype=np.float64, order="C")
    n = a.shape[0]
    ipvt = np.empty(n, dtype=np.int32)
    inv = np.empty(n)
    info = _L().orc_lu_factor(n, _d(a), _i(ipvt), _d(inv))
    return a, ipvt, inv, int(info)


def lu_solve(lu, ipvt, inv, b):
    b = np.array(b, dtype=np.float64)
    lu = np.ascontiguousarray(lu)
    _L().orc_lu_solve(lu.shape[0], _d(lu), _i(ipvt), _d(inv), _d(b))
    return b


def bdf_coeffs(q, h, tau):
    """tau: [tau_1 .. tau_5] most recent first.  Returns l[0..q]."""
    t = np.zeros(8)
    t[1:1 + len(tau)] = tau
    out = np.zeros(8)
    _L().orc_bdf_coeffs(int(q), float(h), _d(t), _d(out))
    return out[: q + 1].copy()


def build_d(xi):
    """Coefficients d_0..d_7 of d(x) = x^2 prod_i (x + xi_i) (C.2-E), xi = [xi_1, xi_2, ...]."""
    x = np.zeros(8)
    x[1:1 + len(xi)] = xi
    d = np.zeros(8)
    _L().orc_build_d(len(xi), _d(x), _d(d))
    return d


def wrms(v, w, lanes=1):
    v = np.ascontiguousarray(v, dtype=np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64)
    return float(_L().orc_wrms(v.shape[0], _d(v), _d(w), int(lanes)))
