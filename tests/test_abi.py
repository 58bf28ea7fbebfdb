"""The C-ABI library loads without a GPU and exports every symbol include/oscnet.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_2410_19075_b200 import build
    return build.build()


def _declared():
    txt = open(os.path.join(ROOT, "include", "oscnet.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(net_[a-z_]+)\s*\(", txt)))


def test_exports_every_declared_symbol(built_lib):
    L = ctypes.CDLL(built_lib)
    names = _declared()
    assert len(names) >= 19
    for n in names:
        assert hasattr(L, n), n
    from paper_2410_19075_b200 import binding
    assert sorted(binding.ABI_SYMBOLS) == names


def test_version_and_pure_host_calls(built_lib):
    from paper_2410_19075_b200 import binding as B
    assert B.net_version().endswith("sm_100a")
    d = B.Desc()
    d.model, d.dtype, d.n, d.batch, d.method = B.MODEL_FHN, B.F32, 64 ** 3, 1, B.METHOD_AUTO
    d.topo.kind, d.topo.ndim, d.topo.radius = B.TOPO_LATTICE, 3, 2
    for q in range(3):
        d.topo.extent[q] = 64
    nbytes = B.net_workspace_bytes(d)          # pure function: no GPU needed
    assert nbytes > 4 * 2 * 4 * 64 ** 3
    d.topo.radius = 40                         # 2P >= extent
    with pytest.raises(B.OscnetError) as e:
        B.net_workspace_bytes(d)
    assert e.value.code == -1 and "radius" in str(e.value)
    d.topo.radius, d.batch = 2, 4
    with pytest.raises(B.OscnetError) as e:
        B.net_workspace_bytes(d)
    assert e.value.code == -5
    d.batch, d.model = 1, 7
    with pytest.raises(B.OscnetError):
        B.net_workspace_bytes(d)
    # batches of rings: the workspace grows with the number of replicas; batch < 1 is invalid
    r = B.Desc()
    r.model, r.dtype, r.n, r.batch, r.method = B.MODEL_KS, B.F64, 256, 1, B.METHOD_AUTO
    r.topo.kind, r.topo.ndim, r.topo.radius = B.TOPO_RING, 1, 64
    one = B.net_workspace_bytes(r)
    r.batch = 1184
    many = B.net_workspace_bytes(r)
    assert many >= one + 4 * 8 * 256 * 1183
    r.batch = 0
    with pytest.raises(B.OscnetError) as e:
        B.net_workspace_bytes(r)
    assert e.value.code == -1
    r.batch, r.n = 1 << 20, 1 << 12           # n * batch > 2^31 - 1
    with pytest.raises(B.OscnetError) as e:
        B.net_workspace_bytes(r)
    assert e.value.code == -1


def test_product_path_does_not_import_oracle():
    import subprocess, sys
    code = ("import sys; import paper_2410_19075_b200.binding, paper_2410_19075_b200.configs, "
            "paper_2410_19075_b200.inputs, paper_2410_19075_b200.replicas; "
            "assert not any(m.startswith('oracle') for m in sys.modules), 'oracle imported'")
    subprocess.check_call([sys.executable, "-c", code], cwd=ROOT)
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2410_19075_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "oscnet_oracle" not in src, f
