"""The C-ABI library loads and exports every symbol include/vr.h declares (no compute calls)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "vr.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vr_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import __graft_entry__
    __graft_entry__.build()
    from paper_1012_2909_b200 import vr
    lib = vr.load()
    names = declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/vr.h but not exported"
    assert sorted(vr.EXPORTS) == names


def test_layout_and_status_strings_need_no_gpu():
    from paper_1012_2909_b200 import vr
    lib = vr.load()
    assert lib.vr_status_string(0) == b"VR_OK" and lib.vr_status_string(-4) == b"VR_ERR_STATE"
    cb, mb = vr.cube_layout((512, 512, 1024), (64, 64, 64))
    # 1024 bricks with a one-sided halo: rows layout 68 x 65 x 65 floats (x pitch padded to 4), blocks
    # layout 17 x 17 x 33 micro-blocks of 32 floats; the caller's buffer must hold either (VR_OPT_LAYOUT)
    assert cb == 1024 * max((68 * 65 * 65 + 31) // 32 * 32, 32 * 17 * 17 * 33) * 4
    assert mb > 1024 * 8
    # C5: 128 GiB cube with halos must fit the 180 GB of one B200 (hard part 4)
    cb5, mb5 = vr.cube_layout((4096, 4096, 2048), (256, 256, 256))
    assert cb5 + mb5 < 160e9 and cb5 >= 4096 * 4096 * 2048 * 4
    try:
        vr.cube_layout((0, 1, 1), (1, 1, 1))
        assert False
    except vr.VRError as e:
        assert e.status == vr.ERR_INVALID_ARG


def test_no_oracle_in_product_path():
    """The product package never imports oracle/ (and the oracle never imports the binding)."""
    pkg = os.path.join(ROOT, "paper_1012_2909_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "ovr.h" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1012_2909_b200", src, flags=re.M), f
            assert not re.search(r"#include\s+\"[^\"]*(?<!o)vr[_a-z]*\.(h|cuh)\"", src), f


def test_binding_constants_match_the_header():
    """Constants the binding repeats (ctypes cannot read macros) are the header's."""
    from paper_1012_2909_b200 import vr
    text = open(os.path.join(ROOT, "include", "vr.h")).read()
    m = re.search(r"#define\s+VR_STATIC_MAX_PARTIALS\s+(\d+)", text)
    assert m and int(m.group(1)) == vr.STATIC_MAX_PARTIALS
    opts = dict(re.findall(r"(VR_OPT_[A-Z0-9_]+)\s*=\s*(\d+)", text))
    for name, value in opts.items():
        assert getattr(vr, name[3:]) == int(value), name
