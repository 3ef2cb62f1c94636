"""Generators for the five synthetic burn workloads (BASELINE.json:configs[0..4]).

Recipe = SURVEY.md section 8(d) table, restated in DESIGN.md "Input recipe":
``rng = numpy.random.default_rng(seed)``, only ``rng.random(shape)`` calls, in a
fixed order.  Zone index z = i + nx*(j + ny*k) (x fastest).  Nothing here
evaluates a reaction rate or touches the integrator; the arrays produced are
handed unchanged to both the CPU oracle and the CUDA library.

Why synthetic: the paper's burn benchmark (Fig. 5) used real
networks on 16^3..128^3 grids cut from application states; neither is available,
so these stand in for them with the paper's shapes (3-/13-isotope networks,
64^3/128^3 grids, XRB-like and SN Ia-like rho/T ranges).
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

CONFIG_NZ = {1: 4096, 2: 64 ** 3, 3: 128 ** 3, 4: 256 ** 3, 5: 128 ** 3}
CONFIG_DT = {1: 1e-6, 2: 1e-7, 3: 1e-6, 4: 1e-6, 5: 1e-7}
CONFIG_SEED = {1: 0, 2: 1, 3: 2, 4: 3, 5: 4}
RTOL = 1e-8
ATOL = 1e-12
CV = 1e8


@dataclass
class Network:
    """A reaction-network description: the argument of ``net_create``.

    reactant[k]  : species id of each reactant particle (-1 = unused; identical
                   particles repeated, e.g. triple-alpha = (0, 0, 0)).
    stoich_id/dy : species whose abundance changes and the change per event.
    rate_A/n/B   : lambda = A * T9^n * exp(-B / T9^(1/3)).
    q_mev        : MeV released per reaction event.  cv: erg/g/K (constant).
    """

    name: str
    species: Sequence[str]
    aion: np.ndarray
    reactant: np.ndarray
    stoich_id: np.ndarray
    stoich_dy: np.ndarray
    rate_A: np.ndarray
    rate_n: np.ndarray
    rate_B: np.ndarray
    q_mev: np.ndarray
    cv: float = CV
    rate_rho_exp: Optional[np.ndarray] = None    # [K] density exponents of weak rates (None = none)
    zion: Optional[np.ndarray] = None            # [N] charges Z_i: selects the analytic EOS for c_v (None = constant cv)
    eos_extra: float = 0.0                       # mol/g: sum (1 + Z_i) Y_i over species that are not evolved

    @property
    def nspec(self) -> int:
        return int(self.aion.shape[0])

    @property
    def nreac(self) -> int:
        return int(self.rate_A.shape[0])

    @property
    def neq(self) -> int:
        return self.nspec + 1


@dataclass
class Workload:
    config: int
    net: Network
    rho: np.ndarray          # [nz]
    T: np.ndarray            # [nz]
    X: np.ndarray            # [nspec, nz]  (species-major, zone fastest)
    dt: float
    rtol: float = RTOL
    atol: float = ATOL
    zone_index: Optional[np.ndarray] = None   # global zone ids of this (sub)set
    nz_full: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def nz(self) -> int:
        return int(self.rho.shape[0])


def sha256_of(*arrays: np.ndarray) -> str:
    h = hashlib.sha256()
    for a in arrays:
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


# --------------------------------------------------------------------------
# network topologies
# --------------------------------------------------------------------------
def _pack(n_reac, reactants, stoich):
    reactant = -np.ones((n_reac, 3), dtype=np.int32)
    sid = -np.ones((n_reac, 4), dtype=np.int32)
    sdy = np.zeros((n_reac, 4), dtype=np.float64)
    for k, (r, s) in enumerate(zip(reactants, stoich)):
        reactant[k, : len(r)] = r
        for m, (i, d) in enumerate(s):
            sid[k, m] = i
            sdy[k, m] = d
    return reactant, sid, sdy


def _coeffs(rng, K):
    """uA, un, uB, uQ = rng.random(K) x4 -> A log-uniform [1e5,1e25], n in [-1,1],
    B in [20,90], Q in [5,10] MeV (uniform; reading s12)."""
    uA = rng.random(K)
    un = rng.random(K)
    uB = rng.random(K)
    uQ = rng.random(K)
    return 10.0 ** (5.0 + 20.0 * uA), -1.0 + 2.0 * un, 20.0 + 70.0 * uB, 5.0 + 5.0 * uQ


def _net1() -> Network:
    # config 1: C12 + C12 -> Mg24; O16 inert, not passed (reading (iii) of 8(b))
    reactant, sid, sdy = _pack(1, [[0, 0]], [[(0, -2.0), (1, +1.0)]])
    return Network(
        "carbon3", ["C12", "Mg24"], np.array([12.0, 24.0]), reactant, sid, sdy,
        np.array([4.27e26]), np.array([-2.0 / 3.0]), np.array([84.165]), np.array([13.93]))


def _net2(rng) -> Network:
    sp = ["He4", "C12", "O16", "Ne20", "Mg24", "Si28", "Ni56"]
    aion = np.array([4.0, 12.0, 16.0, 20.0, 24.0, 28.0, 56.0])
    reactants = [[0, 0, 0]]
    stoich = [[(0, -3.0), (1, +1.0)]]
    for x in range(1, 5):          # C12,O16,Ne20,Mg24 (a,g)
        reactants.append([x, 0])
        stoich.append([(x, -1.0), (0, -1.0), (x + 1, +1.0)])
    reactants.append([5, 0])        # Si28 + a (+6a) -> Ni56, two-body law (reading s4)
    stoich.append([(5, -1.0), (0, -7.0), (6, +1.0)])
    reactant, sid, sdy = _pack(6, reactants, stoich)
    A, n, B, Q = _coeffs(rng, 6)
    return Network("alpha7", sp, aion, reactant, sid, sdy, A, n, B, Q)


def _net3(rng) -> Network:
    sp = ["He4", "C12", "O16", "Ne20", "Mg24", "Si28", "S32", "Ar36", "Ca40",
          "Ti44", "Cr48", "Fe52", "Ni56"]
    aion = np.array([4.0 * (i + 1) if i else 4.0 for i in range(13)])
    aion[1:] = 12.0 + 4.0 * np.arange(12)
    reactants = [[0, 0, 0]]
    stoich = [[(0, -3.0), (1, +1.0)]]
    for x in range(1, 12):         # eleven (a,g) captures C12->O16 ... Fe52->Ni56
        reactants.append([x, 0])
        stoich.append([(x, -1.0), (0, -1.0), (x + 1, +1.0)])
    reactants.append([1, 1]); stoich.append([(1, -2.0), (4, +1.0)])             # C12+C12->Mg24
    reactants.append([1, 2]); stoich.append([(1, -1.0), (2, -1.0), (5, +1.0)])  # C12+O16->Si28
    reactants.append([2, 2]); stoich.append([(2, -2.0), (6, +1.0)])             # O16+O16->S32
    reactant, sid, sdy = _pack(15, reactants, stoich)
    A, n, B, Q = _coeffs(rng, 15)
    return Network("alpha13", sp, aion, reactant, sid, sdy, A, n, B, Q)


def _net5(rng) -> Network:
    N = 30
    aion = 4.0 * (np.arange(N) + 1.0)
    A, n, B, Q = _coeffs(rng, 96)
    keys = rng.random(225)
    triples = [(i, j, i + j + 1) for i in range(N) for j in range(i, N) if i + j + 1 <= N - 1]
    assert len(triples) == 225
    chosen = np.sort(np.argsort(keys, kind="stable")[:96])   # 96 smallest keys, enumeration order
    reactants, stoich = [], []
    for t in chosen:
        i, j, k = triples[int(t)]
        reactants.append([i, j])
        if i == j:
            stoich.append([(i, -2.0), (k, +1.0)])
        else:
            stoich.append([(i, -1.0), (j, -1.0), (k, +1.0)])
    reactant, sid, sdy = _pack(96, reactants, stoich)
    sp = [f"A{int(a)}" for a in aion]
    return Network("synth30", sp, aion, reactant, sid, sdy, A, n, B, Q)


def network_for_config(config: int) -> Network:
    """The network of a config only (consumes exactly the coefficient draws)."""
    if config == 1:
        return _net1()
    if config == 2:
        return _net2(np.random.default_rng(1))
    if config in (3, 4):
        return _net3(np.random.default_rng(2))     # config 4 = config 3's network (seed 2)
    if config == 5:
        return _net5(np.random.default_rng(4))
    raise ValueError(f"unknown config {config}")


def aprox13_like_network(seed: int = 6) -> Network:
    """A second 13-isotope workload in the style of the networks the paper's Fig. 5 ran
    (SURVEY.md 8(f)-4): the alpha chain of config 3 with ALPHA-EMITTING heavy-ion
    channels (C12+C12 -> Ne20 + a, C12+O16 -> Mg24 + a, O16+O16 -> Si28 + a) and the eleven REVERSE
    (photodisintegration) links X_{m+1} -> X_m + a as first-order reactions.  The rate data are
    synthetic (the real fits are not available and are not reproduced): forward coefficients as in
    config 2 from ``default_rng(seed)``; reverse links A = 10^(10 u), n in [-1,1], B in [60,120]
    (they switch on at high temperature) and Q = -Q of the matching capture.  26 reactions; runs on
    the generic cooperative kernel (no generated code for this topology: its LU needs interchanges)."""
    rng = np.random.default_rng(seed)
    sp = ["He4", "C12", "O16", "Ne20", "Mg24", "Si28", "S32", "Ar36", "Ca40",
          "Ti44", "Cr48", "Fe52", "Ni56"]
    aion = np.empty(13)
    aion[0] = 4.0
    aion[1:] = 12.0 + 4.0 * np.arange(12)
    reactants = [[0, 0, 0]]
    stoich = [[(0, -3.0), (1, +1.0)]]
    for x in range(1, 12):         # eleven (a,g) captures
        reactants.append([x, 0])
        stoich.append([(x, -1.0), (0, -1.0), (x + 1, +1.0)])
    reactants.append([1, 1]); stoich.append([(1, -2.0), (3, +1.0), (0, +1.0)])             # C12+C12 -> Ne20 + a
    reactants.append([1, 2]); stoich.append([(1, -1.0), (2, -1.0), (4, +1.0), (0, +1.0)])  # C12+O16 -> Mg24 + a
    reactants.append([2, 2]); stoich.append([(2, -2.0), (5, +1.0), (0, +1.0)])             # O16+O16 -> Si28 + a
    A, n, B, Q = _coeffs(rng, 15)
    uA, un, uB = rng.random(11), rng.random(11), rng.random(11)
    for x in range(1, 12):         # reverse links X_{x+1} -> X_x + a
        reactants.append([x + 1])
        stoich.append([(x + 1, -1.0), (x, +1.0), (0, +1.0)])
    A = np.concatenate([A, 10.0 ** (10.0 * uA)])
    n = np.concatenate([n, -1.0 + 2.0 * un])
    B = np.concatenate([B, 60.0 + 60.0 * uB])
    Q = np.concatenate([Q, -Q[1:12]])
    reactant, sid, sdy = _pack(26, reactants, stoich)
    return Network("aprox13like", sp, aion, reactant, sid, sdy, A, n, B, Q)


def make_aprox13_like_workload(nz: int, seed: int = 6, dt: float = 1e-6) -> Workload:
    """``nz`` zones for ``aprox13_like_network``: rho log-uniform [1e6, 1e8], T uniform [1e9, 4e9]
    (hot enough for the reverse links to matter), X = Dirichlet(1) over He4/C12/O16/Si28/Ni56."""
    net = aprox13_like_network(seed)
    rng = np.random.default_rng(seed + 1000)
    u_rho, u_T = rng.random(nz), rng.random(nz)
    g = -np.log1p(-rng.random((5, nz)))
    X = np.zeros((13, nz))
    X[[0, 1, 2, 5, 12]] = g / g.sum(axis=0)
    return Workload(6, net, 10.0 ** (6.0 + 2.0 * u_rho), 1e9 + 3e9 * u_T, X, dt, nz_full=nz)


def urca9_like_network(seed: int = 9) -> Network:
    """A 9-species network in the style of the Urca network the paper's Fig. 5 ran ("the 9-isotope Urca
    network is used for our Urca simulations"): free neutrons and
    protons, the carbon-burning channels that emit alpha / p / n, and an A = 23 Urca pair linked by
    WEAK, first-order reactions whose rates depend on density and temperature (electron capture grows
    with rho, beta decay is blocked by it).  The real network takes those rates from tables in
    (rho Y_e, T), which are not available and are not reproduced: here lambda = A T9^n exp(-B/T9^(1/3))
    rho^e with synthetic coefficients from ``default_rng(seed)`` -- capture-like links e in [1, 2] and
    A = 10^(-21+3u)... chosen so that lambda ~ 1e5..1e7 /s around rho = 1e9; decay-like links e in
    [-1, -0.3].  12 reactions, four-entry stoichiometry, reactions with negative Q.  Runs on the generic
    cooperative kernel."""
    rng = np.random.default_rng(seed)
    sp = ["n", "p", "He4", "C12", "O16", "Ne20", "Ne23", "Na23", "Mg23"]
    aion = np.array([1.0, 1.0, 4.0, 12.0, 16.0, 20.0, 23.0, 23.0, 23.0])
    n_, p_, he, c12, o16, ne20, ne23, na23, mg23 = range(9)
    strong = [
        ([c12, c12], [(c12, -2.0), (ne20, +1.0), (he, +1.0)]),               # C12 + C12 -> Ne20 + a
        ([c12, c12], [(c12, -2.0), (na23, +1.0), (p_, +1.0)]),               # C12 + C12 -> Na23 + p
        ([c12, c12], [(c12, -2.0), (mg23, +1.0), (n_, +1.0)]),               # C12 + C12 -> Mg23 + n
        ([c12, he], [(c12, -1.0), (he, -1.0), (o16, +1.0)]),                 # C12 (a,g) O16
        ([o16, he], [(o16, -1.0), (he, -1.0), (ne20, +1.0)]),                # O16 (a,g) Ne20
        ([na23, p_], [(na23, -1.0), (p_, -1.0), (ne20, +1.0), (he, +1.0)]),  # Na23 (p,a) Ne20
        ([mg23, n_], [(mg23, -1.0), (n_, -1.0), (na23, +1.0), (p_, +1.0)]),  # Mg23 (n,p) Na23
    ]
    weak = [   # (reactant, product, capture-like?)
        (ne23, na23, False),   # beta decay of the Urca pair
        (na23, ne23, True),    # electron capture of the Urca pair
        (mg23, na23, True),
        (n_, p_, False),
        (p_, n_, True),
    ]
    reactants = [r for r, _ in strong] + [[a] for a, _, _ in weak]
    stoich = [s for _, s in strong] + [[(a, -1.0), (b, +1.0)] for a, b, _ in weak]
    K = len(reactants)
    A, n, B, Q = _coeffs(rng, len(strong))
    u = rng.random((4, len(weak)))
    cap = np.array([c for _, _, c in weak])
    e_w = np.where(cap, 1.0 + u[0], -1.0 + 0.7 * u[0])
    # lambda ~ 10^(5..7) /s at rho = 1e9, T9 = 1:  A = 10^(5 + 2u - 9 e)
    A_w = 10.0 ** (5.0 + 2.0 * u[1] - 9.0 * e_w)
    n_w = -1.0 + 2.0 * u[2]
    B_w = 5.0 * u[3]
    Q_w = np.where(cap, -1.0, +1.0) * (0.5 + 4.0 * rng.random(len(weak)))
    reactant, sid, sdy = _pack(K, reactants, stoich)
    return Network("urca9like", sp, aion, reactant, sid, sdy, np.concatenate([A, A_w]), np.concatenate([n, n_w]),
                   np.concatenate([B, B_w]), np.concatenate([Q, Q_w]),
                   rate_rho_exp=np.concatenate([np.zeros(len(strong)), e_w]))


def make_urca9_like_workload(nz: int, seed: int = 9, dt: float = 1e-6) -> Workload:
    """``nz`` zones for ``urca9_like_network``: rho log-uniform [1e8, 1e10] (around an Urca threshold),
    T uniform [5e8, 3e9], X = Dirichlet(1) over C12, O16, Ne23, Na23 with 1e-3 of free n and p each."""
    net = urca9_like_network(seed)
    rng = np.random.default_rng(seed + 1000)
    u_rho, u_T = rng.random(nz), rng.random(nz)
    g = -np.log1p(-rng.random((4, nz)))
    X = np.zeros((9, nz))
    X[[3, 4, 6, 7]] = 0.998 * g / g.sum(axis=0)
    X[0] = 1e-3
    X[1] = 1e-3
    return Workload(7, net, 10.0 ** (8.0 + 2.0 * u_rho), 5e8 + 2.5e9 * u_T, X, dt, nz_full=nz)


def first_order_decay_network(lam: float, q_mev: float = 0.0) -> Network:
    """i -> k, one first-order reaction with a temperature-independent rate
    (n = 0, B = 0): the closed-form pin named by north_star."""
    reactant, sid, sdy = _pack(1, [[0]], [[(0, -1.0), (1, +1.0)]])
    return Network("decay", ["P", "D"], np.array([4.0, 4.0]), reactant, sid, sdy,
                   np.array([lam]), np.array([0.0]), np.array([0.0]), np.array([q_mev]))


# --------------------------------------------------------------------------
# zone states
# --------------------------------------------------------------------------
def _resolve_zones(nz_full: int, zones) -> Optional[np.ndarray]:
    if zones is None:
        return None
    if isinstance(zones, (int, np.integer)):       # stride
        return np.arange(0, nz_full, int(zones), dtype=np.int64)
    idx = np.asarray(zones, dtype=np.int64)
    if idx.size and (idx.min() < 0 or idx.max() >= nz_full):
        raise ValueError("zone index out of range")
    return idx


def _take(a: np.ndarray, idx: Optional[np.ndarray]) -> np.ndarray:
    return np.ascontiguousarray(a if idx is None else a[..., idx])


def _config4_fields(idx: Optional[np.ndarray]):
    n = 256
    centres = np.floor(256.0 * np.random.default_rng(3).random((64, 3)))
    if idx is None:
        idx = np.arange(n ** 3, dtype=np.int64)
    ix = (idx % n).astype(np.float64)
    iy = ((idx // n) % n).astype(np.float64)
    iz = (idx // (n * n)).astype(np.float64)
    r = np.sqrt((ix - 127.5) ** 2 + (iy - 127.5) ** 2 + (iz - 127.5) ** 2)
    rho = 2e9 * np.exp(-r / 64.0)
    g = np.zeros(idx.shape[0], dtype=np.float64)
    # exp(-d2/32) below 1.1e-17 cannot change 3e8 + 2.7e9*g in fp64 (half an ulp of
    # 3e8 is 3e-8), so zones farther than 40 zones from a centre are skipped exactly.
    for c in centres:
        d2 = (ix - c[0]) ** 2 + (iy - c[1]) ** 2 + (iz - c[2]) ** 2
        near = d2 < 1600.0
        if near.any():
            g[near] = np.maximum(g[near], np.exp(-d2[near] / 32.0))
    T = 3e8 + 2.7e9 * g
    return rho, T, centres


def make_workload(config: int, zones=None, nz_full: Optional[int] = None) -> Workload:
    """Build config ``config``.  ``zones``: None = every zone; an int s = every
    s-th zone; an index array = those zones.  Random configs always draw the full
    arrays (stream order is part of the recipe) and then subset.  ``nz_full``
    overrides the grid size (tests only; changes the stream for configs 2,3,5)."""
    nzf = int(nz_full) if nz_full is not None else CONFIG_NZ[config]
    idx = _resolve_zones(nzf, zones)
    dt = CONFIG_DT[config]
    if config == 1:
        rng = np.random.default_rng(0)
        u_rho, u_T, u_X = rng.random(nzf), rng.random(nzf), rng.random(nzf)
        net = _net1()
        rho = 10.0 ** (7.0 + 2.0 * u_rho)
        T = 1.5e9 + 1.5e9 * u_T
        X = np.stack([0.3 + 0.2 * u_X, np.zeros(nzf)])
    elif config == 2:
        rng = np.random.default_rng(1)
        net = _net2(rng)
        u_rho, u_T = rng.random(nzf), rng.random(nzf)
        uX = rng.random((3, nzf))
        rho = 10.0 ** (6.0 + 2.0 * u_rho)
        T = 1e9 + 2e9 * u_T
        g = -np.log1p(-uX)
        X = np.zeros((7, nzf))
        X[:3] = g / g.sum(axis=0)
    elif config == 3:
        rng = np.random.default_rng(2)
        net = _net3(rng)
        u_rho, u_T = rng.random(nzf), rng.random(nzf)
        rho = 10.0 ** (5.0 + 2.0 * u_rho)
        T = 5e8 + 1.5e9 * u_T
        X = np.zeros((13, nzf))
        X[0] = 0.99
        X[1] = 0.01
    elif config == 4:
        if nz_full is not None and nz_full != 256 ** 3:
            raise ValueError("config 4 is defined on the 256^3 grid only")
        net = _net3(np.random.default_rng(2))
        rho, T, centres = _config4_fields(idx)
        X = np.zeros((13, rho.shape[0]))
        X[1] = 0.5
        X[2] = 0.5
        return Workload(4, net, np.ascontiguousarray(rho), np.ascontiguousarray(T), X, dt,
                        zone_index=idx, nz_full=nzf, meta={"centres": centres})
    elif config == 5:
        rng = np.random.default_rng(4)
        net = _net5(rng)
        u_rho, u_T = rng.random(nzf), rng.random(nzf)
        rho = 10.0 ** (6.0 + 3.0 * u_rho)
        T = 1e9 + 3e9 * u_T
        nsel = nzf if idx is None else idx.shape[0]
        # rng.random((30, nz)) fills row-major, so one species row at a time is the same stream
        g = np.empty((30, nsel))
        for i in range(30):
            g[i] = -np.log1p(-_take(rng.random(nzf), idx))
        for i in range(30):
            g[i] *= np.cos(2.0 * np.pi * _take(rng.random(nzf), idx)) ** 2
        X = g / g.sum(axis=0)
        return Workload(5, net, _take(rho, idx), _take(T, idx), np.ascontiguousarray(X), dt,
                        zone_index=idx, nz_full=nzf)
    else:
        raise ValueError(f"unknown config {config}")
    return Workload(config, net, _take(rho, idx), _take(T, idx), _take(X, idx), dt,
                    zone_index=idx, nz_full=nzf)
