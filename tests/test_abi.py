"""CPU-only checks of the boundary: libosog.so builds / loads without a GPU, exports every symbol that
include/osog.h declares, the ctypes structs match the header's field order, and the entry points that can run
without a device fail cleanly (no compute call is made here)."""
import ctypes as C
import os
import re

import pytest

import paper_2606_21381_b200 as og

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "osog.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(osog_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported():
    names = _declared()
    assert {"osog_create", "osog_render_opd", "osog_render_field", "osog_render_intensity", "osog_destroy"} <= set(names)
    lib = C.CDLL(og.lib_path()) if os.path.exists(og.lib_path()) else og.lib()
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/osog.h but not exported by libosog.so"
    assert set(names) == set(og.EXPORTS), "binding and header disagree on the entry points"


def test_struct_layouts_follow_the_header():
    src = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)
    bodies = {m.group(2): m.group(1) for m in re.finditer(r"typedef struct \{([^}]*)\} (\w+);", src)}
    for name, st in (("osog_config", og.osog_config), ("osog_particles", og.osog_particles), ("osog_optics", og.osog_optics),
                     ("osog_dic", og.osog_dic)):
        body = bodies[name]
        fields = []
        for decl in body.split(";"):
            decl = decl.strip()
            if not decl:
                continue
            tail = decl.split(None, 1)[1] if not decl.startswith("const") else decl.split(None, 2)[2]
            fields += [f.strip().lstrip("*").strip() for f in tail.split(",")]
        assert fields == [f[0] for f in st._fields_], name
    assert C.sizeof(og.osog_config) == 48
    assert C.sizeof(og.osog_particles) == 8 + 13 * 8
    assert C.sizeof(og.osog_optics) == 104
    assert C.sizeof(og.osog_dic) == 24


def test_calls_that_need_no_device():
    lib = og.lib()
    assert lib.osog_tile_size() == 32
    assert lib.osog_strerror(0) == b"ok"
    assert b"overflow" in lib.osog_strerror(og.OSOG_ECAPACITY)
    assert lib.osog_destroy(None) == og.OSOG_EINVAL
    assert lib.osog_status(None, None, None) == og.OSOG_EINVAL
    ctx = C.c_void_p()
    assert lib.osog_create(C.byref(ctx), None) == og.OSOG_EINVAL
    cfg = og.osog_config()
    cfg.struct_size = 4                                  # wrong ABI size
    assert lib.osog_create(C.byref(ctx), C.byref(cfg)) == og.OSOG_EINVAL
    cfg.struct_size = C.sizeof(og.osog_config)
    cfg.H, cfg.W, cfg.max_frames, cfg.max_particles = 0, 64, 1, 10
    assert lib.osog_create(C.byref(ctx), C.byref(cfg)) == og.OSOG_EINVAL
    assert not ctx.value


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    with pytest.raises(RuntimeError):
        og.Context(64, 64, 10)
    lib = og.lib()
    ctx = C.c_void_p()
    cfg = og.osog_config()
    cfg.struct_size = C.sizeof(og.osog_config)
    cfg.H, cfg.W, cfg.max_frames, cfg.max_particles = 64, 64, 1, 10
    assert lib.osog_create(C.byref(ctx), C.byref(cfg)) == og.OSOG_ECUDA
    assert not ctx.value


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_21381_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("the oracle", "").replace("oracle's", "").replace("oracle/", "") \
                    or f in ("binding.py", "__init__.py") and "import oracle" not in text and "from oracle" not in text, f
                assert "import oracle" not in text and "from oracle" not in text, f
