"""ctypes binding of libburn.so -- argument marshalling only; every step of the burn runs in the
CUDA kernels behind the C ABI (include/burnzones.h)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
COUNTER_NAMES = ("nst", "nrhs", "njac", "nlu", "nsolve", "netf", "ncfn", "nfailzones")
EXPORTED_SYMBOLS = ("net_create", "burn_zones", "burn_zones_src", "burn_zones_host", "burn_zones_static", "net_destroy",
                    "bz_get_counters",
                    "bz_norm_lanes", "bz_select_kernel", "bz_set_schedule", "bz_set_zone_order", "bz_set_limits", "bz_set_policy",
                    "bz_kernel_name",
                    "bz_last_cuda_error", "bz_fp64_peak_probe")
_STATUS = {-1: "null pointer", -2: "bad size", -3: "bad network", -4: "bad scalar",
           -5: "CUDA runtime error", -6: "out of memory", -7: "unsupported", -8: "handle belongs to another device"}

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class BurnError(RuntimeError):
    def __init__(self, code, what, cuda_error=0):
        self.code = code
        self.cuda_error = cuda_error
        extra = f" (cudaError_t {cuda_error})" if code == -5 else ""
        super().__init__(f"{what} failed: {_STATUS.get(code, 'unknown')} [{code}]{extra}")


class _Desc(C.Structure):
    _fields_ = [("nspec", C.c_int32), ("nreac", C.c_int32), ("aion", _dp), ("reactant", _ip),
                ("stoich_id", _ip), ("stoich_dy", _dp), ("rate_A", _dp), ("rate_n", _dp),
                ("rate_B", _dp), ("q_mev", _dp), ("cv", C.c_double), ("rate_rho_exp", _dp),
                ("zion", _dp), ("eos_extra", C.c_double)]


def library_path() -> str:
    """The in-tree build (python -m paper_1711_06203_b200.build)."""
    return os.path.join(_HERE, "libburn.so")


_lib = None


def _L():
    """Load libburn.so.  It must have been built (python -m paper_1711_06203_b200.build or
    __graft_entry__.build()); a missing library is an error, never a fallback."""
    global _lib
    if _lib is None:
        path = library_path()
        if not os.path.exists(path):
            raise ImportError(f"{path} is missing: build it with __graft_entry__.build(); "
                              "there is no CPU fallback for the burn")
        lib = C.CDLL(path)
        vp = C.c_void_p
        lib.net_create.restype = C.c_int
        lib.net_create.argtypes = [C.POINTER(_Desc), C.POINTER(vp)]
        lib.net_destroy.restype = C.c_int
        lib.net_destroy.argtypes = [vp]
        sig = [vp, C.c_int64, vp, vp, vp, C.c_double, C.c_double, C.c_double, vp, vp, vp, vp]
        lib.burn_zones.restype = C.c_int
        lib.burn_zones.argtypes = sig
        lib.burn_zones_host.restype = C.c_int
        lib.burn_zones_host.argtypes = sig
        lib.burn_zones_src.restype = C.c_int
        lib.burn_zones_src.argtypes = [vp, C.c_int64, vp, vp, vp, vp, vp, C.c_double, C.c_double, C.c_double,
                                       vp, vp, vp, vp]
        lib.burn_zones_static.restype = C.c_int
        lib.burn_zones_static.argtypes = [C.POINTER(_Desc)] + sig[1:]
        lib.bz_get_counters.restype = C.c_int
        lib.bz_get_counters.argtypes = [vp, vp, C.POINTER(C.c_uint64)]
        lib.bz_norm_lanes.restype = C.c_int
        lib.bz_norm_lanes.argtypes = [vp]
        lib.bz_select_kernel.restype = C.c_int
        lib.bz_select_kernel.argtypes = [vp, C.c_int]
        lib.bz_set_schedule.restype = C.c_int
        lib.bz_set_schedule.argtypes = [vp, C.c_int]
        lib.bz_set_zone_order.restype = C.c_int
        lib.bz_set_zone_order.argtypes = [vp, C.c_void_p, C.c_int64]
        lib.bz_set_policy.restype = C.c_int
        lib.bz_set_policy.argtypes = [vp, C.c_int]
        lib.bz_set_limits.restype = C.c_int
        lib.bz_set_limits.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32]
        lib.bz_kernel_name.restype = C.c_char_p
        lib.bz_kernel_name.argtypes = [vp]
        lib.bz_last_cuda_error.restype = C.c_int
        lib.bz_fp64_peak_probe.restype = C.c_int
        lib.bz_fp64_peak_probe.argtypes = [C.c_int64, vp, _dp, _dp]
        _lib = lib
    return _lib


def _check(rc, what):
    if rc != 0:
        raise BurnError(rc, what, _L().bz_last_cuda_error())


class Net:
    """Handle returned by net_create (owns the library-side bz_net)."""

    def __init__(self, handle, nspec, nreac):
        self._h = handle
        self.nspec = nspec
        self.nreac = nreac

    @property
    def norm_lanes(self) -> int:
        return int(_L().bz_norm_lanes(self._h))

    @property
    def kernel_name(self) -> str:
        return _L().bz_kernel_name(self._h).decode()

    def select_kernel(self, kind: str = "auto") -> None:
        """'auto' (specialised quad kernel when available), 'coop' (generic), 'quad'."""
        _check(_L().bz_select_kernel(self._h, {"auto": 0, "coop": 1, "quad": 3}[kind]), "bz_select_kernel")

    def set_schedule(self, kind: str = "cost") -> None:
        """'cost' (work queue, zones handed out dearest first by the library's a-priori cost key; the default of
        a new handle), 'queue' (work queue in index order) or 'static' (round-robin assignment; for measuring a2)."""
        _check(_L().bz_set_schedule(self._h, {"queue": 0, "static": 1, "cost": 2}[kind]), "bz_set_schedule")

    def set_zone_order(self, order=None, validate: bool = True) -> None:
        """The order in which the work queue hands the zones out: a CUDA int64 tensor holding a permutation
        of 0..nz-1 (e.g. ``torch.argsort(nsteps_of_the_previous_burn, descending=True)``), or None for
        index order.  Applies to the later burn_zones / burn_zones_src calls of this handle on batches of
        exactly that many zones.  Results do not depend on it, only the time does (include/burnzones.h).
        The tensor is kept alive by the handle; do not modify it while burns that use it are in flight."""
        if order is None:
            _check(_L().bz_set_zone_order(self._h, None, 0), "bz_set_zone_order")
            self._order = None
            return
        import torch
        if not (isinstance(order, torch.Tensor) and order.is_cuda and order.dtype == torch.int64 and order.dim() == 1
                and order.is_contiguous()):
            raise ValueError("order: a contiguous 1-d CUDA int64 tensor")
        nz = order.numel()
        if validate and nz > 0:
            seen = torch.zeros(nz, dtype=torch.bool, device=order.device)
            if int(order.min()) < 0 or int(order.max()) >= nz:
                raise ValueError("order: entries outside 0..nz-1")
            seen[order] = True
            if not bool(seen.all()):
                raise ValueError("order: not a permutation of 0..nz-1")
        _check(_L().bz_set_zone_order(self._h, order.data_ptr(), nz), "bz_set_zone_order")
        self._order = order

    def set_policy(self, kind: str = "fresh") -> None:
        """'fresh' (Jacobian + LU on every attempt, default) or 'reuse' (VODE-style kept Newton matrix;
        specialised kernels only)."""
        _check(_L().bz_set_policy(self._h, {"fresh": 0, "reuse": 1}[kind]), "bz_set_policy")

    def set_limits(self, mxstep: int = 0, mxnef: int = 0, mxncf: int = 0) -> None:
        """Limits behind the failure codes -3 / -2 / -1; 0 = default (20000 / 7 / 10)."""
        _check(_L().bz_set_limits(self._h, int(mxstep), int(mxnef), int(mxncf)), "bz_set_limits")

    def close(self):
        if self._h is not None:
            _L().net_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def net_create(net=None, *, aion=None, reactant=None, stoich_id=None, stoich_dy=None, rate_A=None,
               rate_n=None, rate_B=None, q_mev=None, cv=None, rate_rho_exp=None, zion=None, eos_extra=None) -> Net:
    """net_create(rates, Q-values, isotope masses): `net` is any object with those fields
    (e.g. workloads.Network), or pass them as keywords."""
    g = (lambda k, v: v if v is not None else getattr(net, k))
    keep = dict(aion=_f64(g("aion", aion)), reactant=_i32(g("reactant", reactant)),
                stoich_id=_i32(g("stoich_id", stoich_id)), stoich_dy=_f64(g("stoich_dy", stoich_dy)),
                rate_A=_f64(g("rate_A", rate_A)), rate_n=_f64(g("rate_n", rate_n)),
                rate_B=_f64(g("rate_B", rate_B)), q_mev=_f64(g("q_mev", q_mev)))
    N, K = keep["aion"].shape[0], keep["rate_A"].shape[0]
    if keep["reactant"].shape != (K, 3) or keep["stoich_id"].shape != (K, 4) or keep["stoich_dy"].shape != (K, 4):
        raise ValueError("reactant must be [K,3], stoich_id/stoich_dy [K,4]")
    for k in ("rate_n", "rate_B", "q_mev"):
        if keep[k].shape != (K,):
            raise ValueError(f"{k} must be [K]")
    rexp = rate_rho_exp if rate_rho_exp is not None else getattr(net, "rate_rho_exp", None)
    d = _Desc(N, K, keep["aion"].ctypes.data_as(_dp), keep["reactant"].ctypes.data_as(_ip),
              keep["stoich_id"].ctypes.data_as(_ip), keep["stoich_dy"].ctypes.data_as(_dp),
              keep["rate_A"].ctypes.data_as(_dp), keep["rate_n"].ctypes.data_as(_dp),
              keep["rate_B"].ctypes.data_as(_dp), keep["q_mev"].ctypes.data_as(_dp),
              float(g("cv", cv)), _rexp_ptr(rexp, K, keep),
              _zion_ptr(zion if zion is not None else getattr(net, "zion", None), N, keep),
              float(eos_extra if eos_extra is not None else (getattr(net, "eos_extra", 0.0) or 0.0)))
    h = C.c_void_p()
    _check(_L().net_create(C.byref(d), C.byref(h)), "net_create")
    return Net(h, N, K)


def _rexp_ptr(rexp, K, keep):
    """Optional density exponents [K] -> pointer (NULL when absent); the array is kept alive in `keep`."""
    if rexp is None:
        return None
    keep["rate_rho_exp"] = _f64(rexp)
    if keep["rate_rho_exp"].shape != (K,):
        raise ValueError("rate_rho_exp must be [K]")
    return keep["rate_rho_exp"].ctypes.data_as(_dp)


def _zion_ptr(zion, N, keep):
    """Optional charges [N] (select the analytic EOS for c_v) -> pointer, NULL when absent."""
    if zion is None:
        return None
    keep["zion"] = _f64(zion)
    if keep["zion"].shape != (N,):
        raise ValueError("zion must be [N]")
    return keep["zion"].ctypes.data_as(_dp)


def net_destroy(net: Net) -> None:
    net.close()


def _stream_ptr(stream):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _device_args(nspec, rho, T, X, extra_in=(), T_out=None, X_out=None, nsteps=None):
    """Check the device tensors of a burn call (float64 / int32, contiguous, CUDA, right shapes) and
    create the outputs the caller did not pass.  Marshalling only."""
    import torch
    nz = rho.shape[0]
    ins = [("rho", rho, (nz,)), ("T", T, (nz,)), ("X", X, (nspec, nz))] + list(extra_in)
    for name, t, shape in ins:
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == shape):
            raise ValueError(f"{name} must be a contiguous float64 CUDA tensor of shape {shape}")
    if T_out is None:
        T_out = torch.empty_like(T)
    if X_out is None:
        X_out = torch.empty_like(X)
    if nsteps is None:
        nsteps = torch.empty(nz, dtype=torch.int32, device=rho.device)
    for name, t, dt_, shape in (("T_out", T_out, torch.float64, (nz,)), ("X_out", X_out, torch.float64, (nspec, nz)),
                                ("nsteps", nsteps, torch.int32, (nz,))):
        if not (t.is_cuda and t.dtype == dt_ and t.is_contiguous() and tuple(t.shape) == shape):
            raise ValueError(f"{name} must be a contiguous CUDA tensor of shape {shape}")
    return nz, T_out, X_out, nsteps


def _p(t):
    return C.c_void_p(t.data_ptr())


def burn_zones(net: Net, rho, T, X, dt, rtol, atol, T_out=None, X_out=None, nsteps=None, stream=None):
    """Device tensors in, device tensors out (torch, float64, contiguous; X is [nspec, nz]).
    Enqueues on `stream` (default: torch's current stream) and returns without synchronising."""
    nz, T_out, X_out, nsteps = _device_args(net.nspec, rho, T, X, (), T_out, X_out, nsteps)
    _check(_L().burn_zones(net._h, nz, _p(rho), _p(T), _p(X), float(dt), float(rtol), float(atol),
                           _p(T_out), _p(X_out), _p(nsteps), _stream_ptr(stream)), "burn_zones")
    return T_out, X_out, nsteps


def burn_zones_src(net: Net, rho, T, X, src_T, src_X, dt, rtol, atol, T_out=None, X_out=None, nsteps=None,
                   stream=None):
    """burn_zones with constant per-zone source terms (include/burnzones.h: burn_zones_src):
    dT/dt += src_T [nz] (K/s), dX_i/dt += src_X [nspec, nz] (1/s).  Device tensors like burn_zones."""
    nz0 = rho.shape[0]
    extra = (("src_T", src_T, (nz0,)), ("src_X", src_X, (net.nspec, nz0)))
    nz, T_out, X_out, nsteps = _device_args(net.nspec, rho, T, X, extra, T_out, X_out, nsteps)
    _check(_L().burn_zones_src(net._h, nz, _p(rho), _p(T), _p(X), _p(src_T), _p(src_X), float(dt), float(rtol),
                               float(atol), _p(T_out), _p(X_out), _p(nsteps), _stream_ptr(stream)), "burn_zones_src")
    return T_out, X_out, nsteps


def strang_step(net: Net, rho, T, X, dt, rtol, atol, update=None, stream=None):
    """One Strang-split step of an operator-split code ("reactions are incorporated via operator
    splitting", section 3.1): burn(dt/2), the caller's `update` (hydro/advection of
    the state, any function (rho, T, X) -> (rho, T, X) of device tensors enqueued on the same
    stream; None = identity), burn(dt/2).  Marshalling only: both halves are burn_zones calls.
    Returns (rho, T, X, nsteps_first_half, nsteps_second_half); nothing is synchronised."""
    T1, X1, ns1 = burn_zones(net, rho, T, X, 0.5 * dt, rtol, atol, stream=stream)
    if update is not None:
        rho, T1, X1 = update(rho, T1, X1)
    T2, X2, ns2 = burn_zones(net, rho, T1, X1, 0.5 * dt, rtol, atol, stream=stream)
    return rho, T2, X2, ns1, ns2


def _host_ptr(name, a, dtype_name, shape):
    """Address of a host array (numpy, or a CPU torch tensor) after checking dtype, C-contiguity and
    shape: the library copies exactly prod(shape) elements from/to this address."""
    if hasattr(a, "data_ptr"):                      # torch tensor
        if a.is_cuda or str(a.dtype) != f"torch.{dtype_name}" or not a.is_contiguous() or tuple(a.shape) != shape:
            raise ValueError(f"{name} must be a contiguous CPU {dtype_name} tensor of shape {shape}")
        return C.c_void_p(a.data_ptr())
    if not isinstance(a, np.ndarray) or a.dtype != np.dtype(dtype_name) or not a.flags.c_contiguous \
            or a.shape != shape:
        raise ValueError(f"{name} must be a C-contiguous {dtype_name} array of shape {shape}")
    return C.c_void_p(a.ctypes.data)


def burn_zones_host(net: Net, rho, T, X, dt, rtol, atol, T_out, X_out, nsteps, stream=None):
    """Host arrays in and out (numpy or CPU torch tensors; float64, nsteps int32; C-contiguous; X and
    X_out [nspec, nz]).  H2D + burn + D2H are enqueued on `stream` and the call returns; with PINNED
    memory it returns without waiting for the copies, with pageable memory the runtime stages each copy
    before returning.  The caller synchronises the stream before reading the outputs."""
    nz = rho.shape[0]
    args = [_host_ptr("rho", rho, "float64", (nz,)), _host_ptr("T", T, "float64", (nz,)),
            _host_ptr("X", X, "float64", (net.nspec, nz))]
    outs = [_host_ptr("T_out", T_out, "float64", (nz,)), _host_ptr("X_out", X_out, "float64", (net.nspec, nz)),
            _host_ptr("nsteps", nsteps, "int32", (nz,))]
    _check(_L().burn_zones_host(net._h, nz, *args, float(dt), float(rtol), float(atol), *outs, _stream_ptr(stream)),
           "burn_zones_host")
    return T_out, X_out, nsteps


STATIC_SCRATCH_BYTES = 32768      # include/burnzones.h: BZ_STATIC_SCRATCH_BYTES


def burn_zones_static(desc, rho, T, X, dt, rtol, atol, T_out, X_out, nsteps, stream=None):
    """The burn without a handle and without any device allocation (include/burnzones.h:
    burn_zones_static): `desc` is any object with the fields of workloads.Network; the library keeps
    its tables and work queue in a static 32 KiB device array shared by all calls, so calls must be
    ordered on the GPU (one stream).  The caller passes all six device tensors; nothing is allocated
    here either.  Runs the generic cooperative kernel; returns without synchronising."""
    import torch
    keep = dict(aion=_f64(desc.aion), reactant=_i32(desc.reactant), stoich_id=_i32(desc.stoich_id),
                stoich_dy=_f64(desc.stoich_dy), rate_A=_f64(desc.rate_A), rate_n=_f64(desc.rate_n),
                rate_B=_f64(desc.rate_B), q_mev=_f64(desc.q_mev))
    N, K = keep["aion"].shape[0], keep["rate_A"].shape[0]
    if keep["reactant"].shape != (K, 3) or keep["stoich_id"].shape != (K, 4) or keep["stoich_dy"].shape != (K, 4):
        raise ValueError("reactant must be [K,3], stoich_id/stoich_dy [K,4]")
    for k in ("rate_n", "rate_B", "q_mev"):
        if keep[k].shape != (K,):
            raise ValueError(f"{k} must be [K]")
    nz = rho.shape[0]
    for name, t, dt_, shape in (("rho", rho, torch.float64, (nz,)), ("T", T, torch.float64, (nz,)),
                                ("X", X, torch.float64, (N, nz)), ("T_out", T_out, torch.float64, (nz,)),
                                ("X_out", X_out, torch.float64, (N, nz)), ("nsteps", nsteps, torch.int32, (nz,))):
        if not (t.is_cuda and t.dtype == dt_ and t.is_contiguous() and tuple(t.shape) == shape):
            raise ValueError(f"{name} must be a contiguous CUDA tensor of shape {shape}")
    d = _Desc(N, K, keep["aion"].ctypes.data_as(_dp), keep["reactant"].ctypes.data_as(_ip),
              keep["stoich_id"].ctypes.data_as(_ip), keep["stoich_dy"].ctypes.data_as(_dp),
              keep["rate_A"].ctypes.data_as(_dp), keep["rate_n"].ctypes.data_as(_dp),
              keep["rate_B"].ctypes.data_as(_dp), keep["q_mev"].ctypes.data_as(_dp), float(desc.cv),
              _rexp_ptr(getattr(desc, "rate_rho_exp", None), K, keep),
              _zion_ptr(getattr(desc, "zion", None), N, keep), float(getattr(desc, "eos_extra", 0.0) or 0.0))
    p = lambda t: C.c_void_p(t.data_ptr())
    _check(_L().burn_zones_static(C.byref(d), nz, p(rho), p(T), p(X), float(dt), float(rtol), float(atol),
                                  p(T_out), p(X_out), p(nsteps), _stream_ptr(stream)), "burn_zones_static")
    return T_out, X_out, nsteps


def get_counters(net: Net, stream=None) -> dict:
    out = (C.c_uint64 * 8)()
    _check(_L().bz_get_counters(net._h, _stream_ptr(stream), out), "bz_get_counters")
    return dict(zip(COUNTER_NAMES, (int(v) for v in out)))


def fp64_peak_probe(iters: int = 4000, stream=None):
    """Measured DFMA throughput of this GPU: returns (TFLOP/s, milliseconds)."""
    tf, ms = C.c_double(), C.c_double()
    _check(_L().bz_fp64_peak_probe(int(iters), _stream_ptr(stream), C.byref(tf), C.byref(ms)), "bz_fp64_peak_probe")
    return tf.value, ms.value
