"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol that
include/sp2.h declares, and its host-side logic (sizes, status strings, argument checks that
need no device) behaves.  No compute call is made here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "sp2.h")


@pytest.fixture(scope="module")
def sp2():
    from paper_2107_02737_b200 import build

    build.build()                       # nvcc cross-compiles without a GPU
    from paper_2107_02737_b200 import sp2 as mod

    return mod


def _declared_symbols():
    text = open(HEADER).read()
    return sorted(set(re.findall(r"SP2_API\s+[\w\s\*]+?\b(sp2_\w+)\s*\(", text)))


def test_header_declares_the_calls_north_star_names():
    names = _declared_symbols()
    for must in ("sp2_density", "sp2_response", "sp2_sequence_begin", "sp2_sequence_step", "sp2_sequence_end",
                 "sp2_workspace_bytes", "sp2_create", "sp2_destroy"):
        assert must in names


def test_library_exports_every_declared_symbol(sp2):
    names = _declared_symbols()
    assert len(names) >= 18
    for n in names:
        assert hasattr(sp2.lib, n), f"{n} declared in include/sp2.h but not exported"
    assert sorted(sp2.EXPORTS) == names          # the Python binding covers the whole header


def test_struct_layouts_match_the_header(sp2):
    # sizes implied by the C declarations (natural alignment, LP64)
    assert ctypes.sizeof(sp2.Sp2Options) == 80   # 2 int, 2 double, 2 int, u64, 10 int
    assert ctypes.sizeof(sp2.Sp2Result) == 96
    assert sp2.Sp2Result.tr_d.offset == 32 and sp2.Sp2Result.gpu_ms.offset == 80


def test_workspace_bytes_and_status_strings(sp2):
    assert sp2.workspace_bytes(0) == 0 and sp2.workspace_bytes(-5) == 0
    b1 = sp2.workspace_bytes(1024)
    b2 = sp2.workspace_bytes(1024, sp2.SP2_WITH_RESPONSE)
    b3 = sp2.workspace_bytes(1024, sp2.SP2_WITH_RESPONSE | sp2.SP2_WITH_HOST_STAGING)
    plane = 1024 * 1024 * 2
    assert b1 >= 4 * plane and b2 - b1 >= 4 * plane - 4096
    assert b3 - b2 >= 4 * 1024 * 1024 * 8
    # padding to the 256-wide tile: N = 6000 needs 6144^2 planes
    assert sp2.workspace_bytes(6000) >= 4 * 6144 * 6144 * 2
    # memory claim of DESIGN.md: N = 16384 density-only fits in ~2.2 GB of workspace
    assert sp2.workspace_bytes(16384) < 2.3 * 2 ** 30
    # SP2_MAX_N = 32768 is the largest supported (and GPU-tested) dimension
    assert sp2.workspace_bytes(32768) > 0 and sp2.workspace_bytes(32769) == 0
    # batched response: 4 more planes per extra perturbation
    b4 = sp2.workspace_bytes(1024, sp2.SP2_WITH_BATCH(4))
    assert b4 - b2 >= 3 * 4 * plane and sp2.workspace_bytes(1024, sp2.SP2_WITH_BATCH(1)) == b2
    assert sp2.status_string(sp2.SP2_OK) == "ok"
    assert "degenerate" in sp2.status_string(sp2.SP2_ERR_DEGENERATE)
    assert "unknown" in sp2.status_string(99)


def test_calls_fail_loudly_without_a_handle_or_device(sp2):
    lib = sp2.lib
    h = ctypes.c_void_p()
    assert lib.sp2_create(ctypes.byref(h), 128, 0, None, 0) == sp2.SP2_ERR_WORKSPACE
    assert lib.sp2_create(None, 128, 0, None, 0) == sp2.SP2_ERR_INVALID_ARG
    assert lib.sp2_destroy(None) == sp2.SP2_ERR_INVALID_ARG
    assert lib.sp2_set_options(None, None) == sp2.SP2_ERR_INVALID_ARG
    assert lib.sp2_launch_count(None) == 0
    import torch

    if not torch.cuda.is_available():
        with pytest.raises(RuntimeError):          # the product path has no CPU fallback
            sp2.Sp2Handle(128)


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2107_02737_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2107_02737_b200" not in src and "from paper_2107_02737_b200" not in src


@pytest.mark.parametrize("n_tiles, resp, segs, ncl", [(528, False, 32, 74), (528, True, 32, 74), (36, True, 4, 148),
                                                      (10, False, 4, 74), (3, True, 1, 3), (300, False, 24, 74),
                                                      (2080, False, 64, 74), (1, False, 1, 1), (528, 4, 16, 74),
                                                      (45, 8, 2, 148)])
def test_work_schedule_covers_every_segment_once_and_is_balanced(sp2, n_tiles, resp, segs, ncl):
    lists = sp2.debug_schedule(n_tiles, resp, segs, ncl)
    n_units = n_tiles * (1 + int(resp))                          # resp = number of perturbations carried
    cost = lambda u: 2 * segs if u < int(resp) * n_tiles else segs
    cover = {u: [0] * cost(u) for u in range(n_units)}
    loads, owners, contribs = [], {}, {}
    for items in lists:
        load, seen_owner = 0, False
        for it in items:
            assert 0 <= it["seg0"] < it["seg1"] <= cost(it["unit"])
            for sgm in range(it["seg0"], it["seg1"]):
                cover[it["unit"]][sgm] += 1
            load += it["seg1"] - it["seg0"]
            if it["kind"] == 2:
                seen_owner = True
                owners[it["unit"]] = it
            else:
                assert not seen_owner              # owners (which wait) come last: no wait cycles
            if it["kind"] == 1:
                contribs.setdefault(it["unit"], []).append(it)
            if it["kind"] == 0:
                assert (it["seg0"], it["seg1"]) == (0, cost(it["unit"]))
        loads.append(load)
    assert all(v == 1 for u in cover for v in cover[u])           # every segment exactly once
    total = sum(cost(u) for u in range(n_units))
    assert max(loads) == -(-total // ncl)                         # optimal makespan, in segments
    assert sum(loads) == total and max(loads) - min(loads) < ncl
    assert set(owners) == set(contribs)
    slots = []
    for u, own in owners.items():
        cs = contribs[u]
        assert own["nparts"] == len(cs) and all(c["flag_id"] == own["flag_id"] for c in cs)
        assert sorted(c["slot"] for c in cs) == list(range(own["slot"], own["slot"] + own["nparts"]))
        slots += [c["slot"] for c in cs]
    assert len(set(slots)) == len(slots) and len(slots) <= 2 * ncl
    assert len({o["flag_id"] for o in owners.values()}) == len(owners)


def test_header_is_plain_c_and_links_from_c(sp2, tmp_path):
    """include/sp2.h must be usable from C (no C++ / torch types): compile a C99 program against it, link the
    shared library, and call the two entry points that need no device."""
    import shutil
    import subprocess

    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("gcc not available")
    src = tmp_path / "use_sp2.c"
    src.write_text(
        '#include <stdio.h>\n#include "sp2.h"\n'
        "int main(void) {\n"
        "  sp2_options_t o; sp2_result_t r; (void)o; (void)r;\n"
        "  size_t b = sp2_workspace_bytes(1024, SP2_WITH_RESPONSE);\n"
        '  printf("%zu %s %d\\n", b, sp2_status_string(SP2_ERR_DEGENERATE), (int)sizeof(sp2_result_t));\n'
        "  return sp2_create(NULL, 8, 0, NULL, 0) == SP2_ERR_INVALID_ARG ? 0 : 1;\n"
        "}\n")
    exe = tmp_path / "use_sp2"
    libdir = os.path.join(ROOT, "paper_2107_02737_b200")
    subprocess.run([gcc, "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"), str(src),
                    "-o", str(exe), "-L", libdir, "-l:libsp2_b200.so", f"-Wl,-rpath,{libdir}"], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()
    assert int(out[0]) == sp2.workspace_bytes(1024, sp2.SP2_WITH_RESPONSE)
    assert "degenerate" in " ".join(out[1:-1]) and int(out[-1]) == 96
