"""The C-ABI library loads and exports every symbol include/autoddl.h declares; host-only calls work and
compute calls fail loudly (no CPU fallback) when there is no CUDA device.  No GPU needed."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2301_06813_b200 import configs as cf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def adl():
    from paper_2301_06813_b200 import build
    build.build()                                    # nvcc cross-compiles sm_100a without a GPU
    from paper_2301_06813_b200 import binding
    return binding


def _declared():
    text = open(os.path.join(ROOT, "include", "autoddl.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(autoddl_[a-z_]+)\s*\(", text)))


def test_header_symbols_exported(adl):
    names = _declared()
    assert set(names) == set(adl.EXPORTS)
    lib = C.CDLL(adl.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n


def test_struct_layouts_match_header(adl):
    assert cf.LAYER_DTYPE.itemsize == 64
    assert [cf.LAYER_DTYPE.fields[k][1] for k in ("M", "Kd", "N", "in_rows", "in_cols", "kind", "act_bytes",
            "wgrad_bytes", "wstate_bytes", "max_split_rows", "max_split_cols")] == [0, 8, 16, 24, 32, 40, 44, 48, 52, 56, 60]
    assert C.sizeof(adl.CMesh) == 68 and C.sizeof(adl.CNet) == 48


def test_host_only_calls(adl):
    assert adl.num_signatures(cf.Mesh((2, 2), (1, 0))) == 36
    assert adl.num_signatures(cf.Mesh((8, 8, 8), (1, 1, 0))) == 216
    assert adl.num_signatures(cf.Mesh((4,), (1,))) == 6
    with pytest.raises(adl.AutoddlError, match="256"):                       # 6^4 signatures: rows must be restricted (R26)
        adl.num_signatures(cf.Mesh((2, 2, 2, 2), (0, 0, 0, 0)))
    with pytest.raises(adl.AutoddlError, match="ndim"):
        adl.num_signatures(cf.Mesh((2,) * 6, (0x07 << 8,) * 6))
    assert adl.num_signatures(cf.Mesh((2, 2, 2, 2), (0x07 << 8,) * 4)) == 81
    assert adl.num_signatures(cf.CONFIGS[7]().mesh) == 243 == cf.CONFIGS[7]().K
    w = cf.config4_batched(Bp=2)
    assert adl.workspace_bytes(4096, 64, 1, w.mesh) >= 4096 * 64 * 36 * 36 * 8 + 4096 * 64 * 64
    w5 = cf.config5_transformer96()
    assert adl.workspace_bytes(1, 480, 1024, w5.mesh) >= 480 * 216 * 216 * 8 + 480 * 216


def test_validation_errors_without_gpu(adl):
    lib = adl.lib()
    w = cf.config1_tiny()
    m, n = adl.c_mesh(w.mesh), adl.c_net(w.net)
    buf = np.zeros(4096, np.uint8)
    ptr = buf.ctypes.data // 256 * 256 + 256
    assert lib.autoddl_build_tables(None, 1, 4, C.addressof(m), C.addressof(n), None, None, None, None) == -1
    assert lib.autoddl_build_tables(ptr, 0, 4, C.addressof(m), C.addressof(n), ptr, None, None, None) == -1
    assert lib.autoddl_build_tables(ptr, 1, 4, C.addressof(m), C.addressof(n), ptr + 8, None, None, None) == -1   # misaligned T
    n.beta_ps_per_byte[0] = -1
    assert lib.autoddl_build_tables(ptr, 1, 4, C.addressof(m), C.addressof(n), ptr, None, None, None) == -1
    assert b"beta" in lib.autoddl_last_error()
    # workspace too small is reported before any device work
    w5 = cf.config5_transformer96()
    m5 = adl.c_mesh(w5.mesh)
    assert lib.autoddl_chain_dp(None, 1, 480, C.addressof(m5), None, ptr, ptr, 16, ptr, ptr, None) == -3


def test_no_cpu_fallback(adl):
    """without a device the compute entry points return ECUDA; with one this test is skipped"""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    lib = adl.lib()
    w = cf.config1_tiny()
    m, n = adl.c_mesh(w.mesh), adl.c_net(w.net)
    buf = np.zeros(1 << 16, np.uint8)
    ptr = buf.ctypes.data // 256 * 256 + 256
    assert lib.autoddl_build_tables(ptr, 1, 4, C.addressof(m), C.addressof(n), ptr, None, None, None) == -2
    assert b"no CPU fallback" in lib.autoddl_last_error()
    assert lib.autoddl_chain_dp(None, 1, 4, C.addressof(m), None, ptr, None, 0, ptr, ptr, None) == -2
    assert lib.autoddl_copy_probe(ptr, ptr + 4096, 4096, None) == -2


def test_product_does_not_import_oracle():
    """the product path shares nothing with oracle/ (neither imports the other)"""
    pkg = os.path.join(ROOT, "paper_2301_06813_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "autoddl_ref" not in text and "import oracle" not in text and "from oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "binding" not in text and "libautoddl.so" not in text and "include/autoddl.h" not in text, f


def test_header_is_plain_c(tmp_path):
    """the boundary is a C ABI: include/autoddl.h compiles as C99 with no torch / C++ types"""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no gcc")
    src = tmp_path / "h.c"
    src.write_text('#include "include/autoddl.h"\nint main(void) { return (int)sizeof(autoddl_layer) - 64; }\n')
    r = subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", ROOT, "-c", str(src), "-o", str(tmp_path / "h.o")],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
