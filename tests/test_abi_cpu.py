"""-m "not gpu": the C-ABI library loads without a GPU, exports every symbol include/hyb.h declares,
and its pure-host entry points (workspace size, parameter validation) behave as documented."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    import __graft_entry__
    __graft_entry__.build()
    import paper_1406_6158_b200 as pkg
    return pkg.lib()


def test_exports_every_declared_symbol(L):
    hdr = open(os.path.join(ROOT, "include", "hyb.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(hyb_[a-z_0-9]+)\s*\(", hdr))
    assert {"hyb_init", "hyb_build_tree", "hyb_soft_force", "hyb_hard_force", "hyb_step", "hyb_free"} <= names
    for n in names:
        assert hasattr(L, n), n


def test_header_compiles_as_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "hyb.h"\nint main(void){hyb_params p; (void)p; return sizeof(hyb_float4)==16?0:1;}\n')
    import subprocess
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o",
                    str(tmp_path / "t")], check=True)
    assert subprocess.run([str(tmp_path / "t")]).returncode == 0


def test_workspace_bytes_and_validation(L):
    from paper_1406_6158_b200 import HybParams, hyb_workspace_bytes
    from workloads import CONFIGS
    sizes = [hyb_workspace_bytes(c.n, HybParams.from_config(c)) for c in CONFIGS]
    assert all(s > 0 and s % 256 == 0 for s in sizes) and sizes == sorted(sizes)
    assert sizes[-1] < 16 * 2 ** 30                    # 2^24 particles fit comfortably in 180 GB
    good = HybParams.from_config(CONFIGS[0])
    bad = [dict(eps=0.0), dict(n_sub=0), dict(leaf_max=0), dict(group_max=4), dict(group_max=65), dict(mac=2),
           dict(kfunc=2), dict(split=2), dict(r_in=0.2), dict(theta=-1.0), dict(mac=1, a_err=0.0)]
    for kw in bad:
        assert hyb_workspace_bytes(4096, HybParams.from_config(CONFIGS[0], **kw)) == 0, kw
    assert hyb_workspace_bytes(0, good) == 0 and hyb_workspace_bytes(1 << 30, good) == 0
    # hyb_init rejects bad arguments before touching CUDA
    h = C.c_void_p()
    rc = L.hyb_init(C.byref(h), C.byref(good), 4096, None, None, None, None, None, None, 0, 0, None)
    assert rc == -1 and b"NULL" in L.hyb_last_error(None)
    rc = L.hyb_init(C.byref(h), C.byref(HybParams.from_config(CONFIGS[0], eps=-1.0)), 4096, 256, 256, 256, 256, 256,
                    256, 1 << 40, 0, None)
    assert rc == -1 and b"eps" in L.hyb_last_error(None)
    rc = L.hyb_init(C.byref(h), C.byref(good), 4096, 256, 256, 256, 256, 256, 256, 1024, 0, None)
    assert rc == -2


def test_missing_library_fails_loudly(monkeypatch):
    import paper_1406_6158_b200.binding as b
    monkeypatch.setattr(b, "_lib", None)
    monkeypatch.setattr(b, "LIBPATH", "/nonexistent/libhyb.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        b.lib()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1406_6158_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("shares nothing with oracle/", ""), f
