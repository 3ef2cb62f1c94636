"""Host-side checks of the C ABI that need no GPU: the library loads, exports every symbol that
include/burnzones.h declares, validates descriptors before touching CUDA, and there is no CPU
fallback behind the binding."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_1711_06203_b200 as bz
from paper_1711_06203_b200 import build as bzbuild
from workloads import network_for_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    bzbuild.build()
    return C.CDLL(bz.library_path())


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "burnzones.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(?:int|const char \*)\s*(\w+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    decl = _declared_functions()
    assert set(decl) == set(bz.EXPORTED_SYMBOLS)
    for name in decl:
        assert hasattr(lib, name), name


def test_descriptor_validation_happens_before_cuda():
    """Bad descriptors are rejected with their own codes even on a box without a GPU."""
    net = network_for_config(2)
    bad = dict(aion=net.aion.copy(), reactant=net.reactant.copy(), stoich_id=net.stoich_id.copy(),
               stoich_dy=net.stoich_dy.copy(), rate_A=net.rate_A.copy(), rate_n=net.rate_n.copy(),
               rate_B=net.rate_B.copy(), q_mev=net.q_mev.copy(), cv=net.cv)

    def code(**kw):
        d = dict(bad)
        d.update(kw)
        with pytest.raises(bz.BurnError) as e:
            bz.net_create(**d)
        return e.value.code

    r = net.reactant.copy(); r[2, 0] = 7
    assert code(reactant=r) == -3                       # species id out of range
    r = net.reactant.copy(); r[1, :] = -1
    assert code(reactant=r) == -3                       # reaction without reactant
    a = net.aion.copy(); a[3] = 0.0
    assert code(aion=a) == -3
    assert code(cv=0.0) == -3
    A = net.rate_A.copy(); A[0] = np.inf
    assert code(rate_A=A) == -3
    s = net.stoich_id.copy(); s[1, 1] = s[1, 0]
    assert code(stoich_id=s) == -3                      # repeated stoichiometry id
    assert code(aion=np.ones(40), reactant=net.reactant) == -2   # nspec out of range


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(bz.BurnError) as e:
        bz.net_create(network_for_config(1))
    assert e.value.code == -5 and e.value.cuda_error != 0


def test_product_does_not_import_oracle():
    """The oracle is test infrastructure: nothing under the package or bench's product path may
    import it."""
    pkg = os.path.join(ROOT, "paper_1711_06203_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "bz_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1711_06203_b200" not in txt.replace("It never imports paper_1711_06203_b200", "") \
                .replace("shares no code with the CUDA path (paper_1711_06203_b200/)", ""), f


def test_shard_ranges_cover_and_balance():
    for nz in (0, 1, 7, 4096, 2097152):
        for world in (1, 2, 3, 8):
            spans = [bz.shard_range(nz, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == nz
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
