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
    d.topo.radius, d.batch = 2, 4                # batches of lattices: the block-diagonal per-link form
    assert B.net_workspace_bytes(d) > nbytes
    d.batch, d.delay_steps = 1, 3              # only NET_MODEL_FHN2 has a delay
    with pytest.raises(B.OscnetError) as e:
        B.net_workspace_bytes(d)
    assert e.value.code == -1
    d.delay_steps, d.model = 0, 7
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


def test_python_structs_match_the_header(tmp_path):
    """sizeof / offsetof of every struct of include/oscnet.h as gcc lays them out against the ctypes
    mirrors in binding.py (a field added on one side only would silently shift every later one)."""
    import subprocess
    from paper_2410_19075_b200 import binding as B
    fields = {
        "net_ks_params": (B.KSParams, ["K", "alpha", "omega0"]),
        "net_ksi_params": (B.KSIParams, ["K", "alpha", "m", "eps", "omega0"]),
        "net_fhn_params": (B.FHNParams, ["eps", "a", "sigma", "phi"]),
        "net_fhn2_params": (B.FHN2Params, ["eps", "a", "sigma", "I_app", "D", "seed"]),
        "net_hh_params": (B.HHParams, ["gNa", "k_syn", "I_ext0", "V_c", "V_s"]),
        "net_hhs_params": (B.HHSParams, ["hh", "a_s", "b_s"]),
        "net_compressed": (B.Compressed, ["n", "v_len", "v_pos", "k", "d_ptr", "d_pos", "c"]),
        "net_topology": (B.Topology, ["kind", "ndim", "extent", "radius", "include_self", "row_ptr", "col_idx",
                                      "nnz", "ptrs_are_device", "in_degree", "seed", "compressed"]),
        "net_desc": (B.Desc, ["model", "dtype", "n", "batch", "method", "topo", "delay_steps"]),
    }
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "oscnet.h"', "int main(void) {"]
    for name, (_, fs) in fields.items():
        lines.append('printf("%s %%zu\\n", sizeof(%s));' % (name, name))
        for f in fs:
            lines.append('printf("%s.%s %%zu\\n", offsetof(%s, %s));' % (name, f, name, f))
    lines.append("return 0; }")
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    got = dict(l.split() for l in subprocess.check_output([str(exe)], text=True).splitlines())
    for name, (cls, fs) in fields.items():
        assert int(got[name]) == ctypes.sizeof(cls), name
        for f in fs:
            assert int(got["%s.%s" % (name, f)]) == getattr(cls, f).offset, (name, f)
