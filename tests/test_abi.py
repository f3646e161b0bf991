"""CPU-side checks of the boundary: liboo.so builds, loads, and exports every symbol include/oo.h declares; the Python
binding mirrors the same names; the product path fails loudly without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "oo.h")).read()
    return re.findall(r"^OO_API\s+[\w\s\*]+?\b(oo_\w+)\s*\(", src, flags=re.M)


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2606_08469_b200 import build as B
    path = B.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    names = _declared()
    assert len(names) >= 13 and {"oo_upload_tree", "oo_upload_mlp", "oo_encode", "oo_query"} <= set(names)
    for n in names:
        assert hasattr(lib, n), "liboo.so does not export %s" % n


def test_binding_mirrors_the_abi():
    import paper_2606_08469_b200 as P
    assert sorted(P.EXPORTED_SYMBOLS) == sorted(_declared())
    for n in ("oo_upload_tree", "oo_upload_mlp", "oo_encode", "oo_query", "oo_sort_queries", "oo_query_host", "oo_reserve",
              "oo_set_path", "oo_get_info", "oo_read_padded_map"):
        assert callable(getattr(P.OctaOctree, n))


def test_static_sort_refuses_oversize_batches_before_touching_cuda():
    """oo_sort_queries_static checks n against its built-in scratch before any CUDA call, so the refusal (status, message that names
    the limit) can be checked without a GPU; the header's constant, the binding's and the library's agree."""
    import paper_2606_08469_b200 as P
    hdr = open(os.path.join(ROOT, "include", "oo.h")).read()
    limit = int(re.search(r"#define\s+OO_SORT_STATIC_MAX_QUERIES\s+(\d+)u", hdr).group(1))
    assert limit == P.SORT_STATIC_MAX_QUERIES == 1 << 20
    L = P.load_library()
    err = ctypes.create_string_buffer(256)
    st = L.oo_sort_queries_static(None, limit + 1, None, None, err, len(err))
    assert st == 3 and b"OO_SORT_STATIC_MAX_QUERIES" in err.value and str(limit).encode() in err.value
    assert L.oo_sort_queries_static(None, 1 << 40, None, None, None, 0) == 3          # no message buffer: status only
    short = ctypes.create_string_buffer(8)                                              # a short buffer is filled and terminated, not overrun
    assert L.oo_sort_queries_static(None, limit + 1, None, None, short, len(short)) == 3 and len(short.value) == 7


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_08469_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dp, f)).read()
                assert "oracle" not in s.lower().replace("no cpu fallback", ""), "%s mentions the oracle" % f
    for f in sorted(os.listdir(os.path.join(ROOT, "oracle"))):
        if not f.endswith((".py", ".c")):
            continue
        s = open(os.path.join(ROOT, "oracle", f)).read()
        assert "import paper_2606_08469_b200" not in s and "from paper_2606_08469_b200" not in s and "liboo.so" not in s


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present: covered by the gpu tests")
    import paper_2606_08469_b200 as P
    with pytest.raises(P.OOError):
        P.OctaOctree(0)
