"""Host-side checks (no GPU): the C-ABI library loads and exports every symbol include/vog.h declares,
the binding's structs match the header, and the build step is wired.  No compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libvog():
    from paper_1301_5892_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def _declared():
    src = open(os.path.join(ROOT, "include", "vog.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(vog_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for need in ("vog_plan", "vog_advect_x", "vog_advect_v", "vog_field", "vog_step"):
        assert need in names


def test_library_exports_every_declared_symbol(libvog):
    for name in _declared():
        assert hasattr(libvog, name), name


def test_binding_lists_the_same_symbols():
    from paper_1301_5892_b200 import vog
    assert set(_declared()) <= set(vog.EXPORTS)


def test_struct_layout_matches_header():
    from paper_1301_5892_b200 import vog
    assert ctypes.sizeof(vog.vog_feq_t) == 8 + 3 * 4 * 8          # int + pad, 3 x double[4]
    assert ctypes.sizeof(vog.vog_params_t) == 8 + 3 * 8 + 8 + ctypes.sizeof(vog.vog_feq_t) + 8
    assert vog.vog_params_t.feq.offset == 40


def test_strerror_is_callable_without_a_gpu(libvog):
    libvog.vog_strerror.restype = ctypes.c_char_p
    assert libvog.vog_strerror(0) == b"ok"
    assert b"invalid" in libvog.vog_strerror(-1)


def test_product_path_does_not_import_the_oracle():
    """The binding and the CUDA sources must not reference oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1301_5892_b200")
    for root, _d, files in os.walk(pkg):
        if "build" in root.split(os.sep)[-1:]:
            continue
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(root, fn)).read()
                assert "vog_oracle" not in txt and "import oracle" not in txt and "from oracle" not in txt, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_1301_5892_b200" not in txt.replace("paper_1301_5892_b200/csrc/", ""), fn
            assert "libvog.so" not in txt
