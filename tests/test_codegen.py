"""Host-side checks of the build-time generator (paper_1711_06203_b200/codegen.py): the emitted
Jacobian sparsity must equal the structural non-zeros the oracle's Jacobian shows, topology
hashes must separate the networks, and the generated headers in csrc/gen must be current."""
import os
import re

import numpy as np

import oracle
from paper_1711_06203_b200 import codegen
from workloads import network_for_config, first_order_decay_network

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TAGS = {1: "carbon3", 2: "alpha7", 3: "alpha13"}


def _mask_from_source(src, n):
    body = re.search(r"jmask\(int i\) \{\s*return (.*?);\s*\}", src, re.S).group(1)
    vals = [int(v, 16) for v in re.findall(r"\? (0x[0-9a-f]+)u", body)]
    assert len(vals) == n
    return np.array([[(vals[i] >> j) & 1 for j in range(n)] for i in range(n)], dtype=bool)


def test_generated_sparsity_matches_oracle_jacobian():
    rng = np.random.default_rng(3)
    for cfg, tag in TAGS.items():
        net = network_for_config(cfg)
        n = net.neq
        src = codegen.emit(net, tag)
        mask = _mask_from_source(src, n)                       # internal order: T first
        y = np.append(0.01 + 0.05 * rng.random(net.nspec), 2.2e9)
        _, J = oracle.rates(net, 3e7, y)                        # API order: T last
        perm = [n - 1] + list(range(n - 1))                     # internal index -> API index
        Ji = J[np.ix_(perm, perm)]
        assert np.array_equal(mask, Ji != 0.0), tag
        assert f"NEQ = {n}" in src and "eval_quad" in src


def test_topology_hash_separates_networks_and_ignores_coefficients():
    hs = {codegen.topology_hash(network_for_config(c)) for c in (1, 2, 3, 5)}
    hs.add(codegen.topology_hash(first_order_decay_network(1e6)))
    assert len(hs) == 5
    a = network_for_config(3)
    b = network_for_config(3)
    b.rate_A = b.rate_A * 3.0
    b.q_mev = b.q_mev + 1.0
    assert codegen.topology_hash(a) == codegen.topology_hash(b)
    c = network_for_config(3)
    c.stoich_dy = c.stoich_dy.copy()
    c.stoich_dy[5, 0] = -2.0
    assert codegen.topology_hash(a) != codegen.topology_hash(c)


def test_committed_generated_headers_are_current():
    gen = os.path.join(ROOT, "paper_1711_06203_b200", "csrc", "gen")
    for cfg, tag in TAGS.items():
        want = codegen.emit(network_for_config(cfg), tag)
        have = open(os.path.join(gen, f"net_{tag}.cuh")).read()
        assert have == want, f"csrc/gen/net_{tag}.cuh is stale: run python -m paper_1711_06203_b200.build"
