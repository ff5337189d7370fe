"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/stag.h declares (no compute calls: there is no GPU here), and the binding agrees with it."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "stag.h")


@pytest.fixture(scope="module")
def so_path():
    from paper_1010_5433_b200 import _build
    return _build.build()


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(stag_[a-z0-9_]+)\s*\(", text)))


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "stag.h"\nint main(void){ stag_cg_info i; (void)i; return STAG_OK; }\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                           "-c", str(src), "-o", str(tmp_path / "t.o")])


def test_library_exports_every_declared_symbol(so_path):
    names = declared_symbols()
    assert len(names) >= 20
    lib = ctypes.CDLL(so_path)
    for n in names:
        assert hasattr(lib, n), "missing export: " + n


def test_binding_symbol_list_matches_header():
    from paper_1010_5433_b200 import SYMBOLS
    assert sorted(SYMBOLS) == declared_symbols()


def test_strerror_and_info_struct_layout(so_path, tmp_path):
    import paper_1010_5433_b200 as stag
    assert stag.strerror(0) == "ok"
    assert "converge" in stag.strerror(stag.ERR_NOTCONV)
    # sizeof(stag_cg_info) as the C compiler sees it == ctypes mirror
    src = tmp_path / "s.c"
    src.write_text('#include <stdio.h>\n#include "stag.h"\nint main(void){printf("%zu %zu %zu", sizeof(stag_cg_info), '
                   'sizeof(stag_polish_info), sizeof(stag_mixed_info));return 0;}\n')
    exe = tmp_path / "s"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    sizes = [int(v) for v in subprocess.check_output([str(exe)]).split()]
    assert sizes == [ctypes.sizeof(stag.CgInfo), ctypes.sizeof(stag.PolishInfo), ctypes.sizeof(stag.MixedInfo)]


def test_no_cpu_fallback_without_gpu():
    import torch
    import paper_1010_5433_b200 as stag
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        stag.Stag((4, 4, 4, 4))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1010_5433_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text
                assert "stag_oracle" not in text


def test_host_side_argument_checks_need_no_gpu(so_path):
    """The error behaviour include/stag.h states for stag_ctx_create and the *_bytes calls is decided on the host,
    before any CUDA call: bad extents -> BADARG, V >= 2^31 -> UNSUPPORTED, null handles -> 0 bytes."""
    import ctypes as C
    from paper_1010_5433_b200 import binding as b
    l = b.lib()
    h = C.c_void_p()
    for L in ((4, 4, 4, 3), (4, 4, 4, 0), (4, -2, 4, 4), (1, 4, 4, 4)):
        assert l.stag_ctx_create((C.c_int * 4)(*L), C.byref(h)) == b.ERR_BADARG, L
    assert l.stag_ctx_create((C.c_int * 4)(256, 256, 256, 256), C.byref(h)) == b.ERR_UNSUPPORTED      # V = 2^32
    assert l.stag_ctx_create(None, C.byref(h)) == b.ERR_BADARG
    assert l.stag_ctx_create((C.c_int * 4)(4, 4, 4, 4), None) == b.ERR_BADARG
    assert l.stag_gauge_canonical_bytes(None) == 0 and l.stag_vector_bytes(None, 0) == 0
    assert l.stag_cg_workspace_bytes(None, 0, 4) == 0 and l.stag_force_workspace_bytes(None, 0, 4) == 0
    for code, word in ((0, "ok"), (b.ERR_BADARG, "bad argument"), (b.ERR_UNSUPPORTED, "unsupported"),
                       (b.ERR_NOT_SU3, "SU(3)"), (b.ERR_NOTCONV, "converge"), (b.ERR_BREAKDOWN, "breakdown")):
        assert word in b.strerror(code)
