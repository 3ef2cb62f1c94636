"""Shared comparison of a CUDA burn against the oracle (north_star's parity bar)."""
import numpy as np

X_FLOOR, X_RTOL, T_RTOL = 1e-10, 1e-5, 1e-6


def compare(T_gpu, X_gpu, ns_gpu, T_ref, X_ref, ns_ref):
    """Returns a dict of statistics; raises AssertionError if the bar is missed.
    Bar: |X_gpu - X_ref| <= 1e-5 X_ref wherever X_ref > 1e-10; |T_gpu - T_ref| <= 1e-6 T_ref;
    failure codes (nsteps < 0) identical."""
    T_gpu, X_gpu, ns_gpu = np.asarray(T_gpu), np.asarray(X_gpu), np.asarray(ns_gpu)
    assert T_gpu.shape == T_ref.shape and X_gpu.shape == X_ref.shape
    big = X_ref > X_FLOOR
    relX = np.zeros_like(X_ref)
    relX[big] = np.abs(X_gpu[big] - X_ref[big]) / X_ref[big]
    relT = np.abs(T_gpu - T_ref) / np.abs(T_ref)
    stats = dict(
        nz=int(T_ref.shape[0]),
        max_rel_X=float(relX.max()) if relX.size else 0.0,
        max_rel_T=float(relT.max()) if relT.size else 0.0,
        bitexact_X=float(np.mean(X_gpu == X_ref)) if X_ref.size else 1.0,
        bitexact_T=float(np.mean(T_gpu == T_ref)) if T_ref.size else 1.0,
        nsteps_equal=float(np.mean(ns_gpu == ns_ref)) if ns_ref.size else 1.0,
        nfail_ref=int((ns_ref < 0).sum()),
    )
    assert np.array_equal(ns_gpu < 0, ns_ref < 0), "failure masks differ"
    assert np.array_equal(ns_gpu[ns_ref < 0], ns_ref[ns_ref < 0]), "failure codes differ"
    assert np.isfinite(X_gpu).all() and np.isfinite(T_gpu).all()
    assert stats["max_rel_X"] <= X_RTOL, stats
    assert stats["max_rel_T"] <= T_RTOL, stats
    return stats
