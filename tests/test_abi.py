"""The C-ABI boundary without a GPU: the library loads, exports every symbol include/flod.h declares, the
ctypes mirrors of its structs have the C compiler's layout, and host-side argument checks work."""
import ctypes as C
import os
import subprocess
import sys
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2408_12894_b200 import build
    build.build()
    import paper_2408_12894_b200 as pkg
    return pkg.load_library()


def test_library_exports_every_declared_symbol(lib):
    import paper_2408_12894_b200 as pkg
    names = pkg.abi_symbols()
    assert len(names) >= 15 and "flod_upload_levels" in names and "flod_render" in names
    for n in names:
        assert hasattr(lib, n), f"libflod.so does not export {n}"
    assert lib.flod_abi_version() == 10


def test_struct_layouts_match_the_c_compiler(lib):
    from paper_2408_12894_b200 import binding as b
    src = r'''
    #include <stdio.h>
    #include <stddef.h>
    #include "flod.h"
    int main(void) {
        printf("%zu %zu %zu %zu %zu %zu\n", sizeof(flod_level_desc), sizeof(flod_camera), sizeof(flod_level_mode),
               sizeof(flod_stats), sizeof(flod_dbg_projected), sizeof(flod_dbg_pair));
        printf("%zu %zu %zu %zu\n", offsetof(flod_level_desc, mean), offsetof(flod_camera, width),
               offsetof(flod_stats, evals), offsetof(flod_stats, ms_stage));
        return 0;
    }'''
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "t.c"), "w").write(src)
        subprocess.run(["gcc", "-std=c11", "-I", os.path.join(ROOT, "include"), os.path.join(d, "t.c"), "-o",
                        os.path.join(d, "t")], check=True)
        out = subprocess.run([os.path.join(d, "t")], check=True, capture_output=True, text=True).stdout.split()
    sizes = list(map(int, out))
    assert sizes[:6] == [C.sizeof(b.LevelDesc), C.sizeof(b.CameraStruct), C.sizeof(b.LevelMode), C.sizeof(b.Stats),
                         b.DBG_PROJECTED_DTYPE.itemsize, b.DBG_PAIR_DTYPE.itemsize]
    assert sizes[6:] == [b.LevelDesc.mean.offset, b.CameraStruct.width.offset, b.Stats.evals.offset,
                         b.Stats.ms_stage.offset]


def test_host_side_argument_checks_need_no_gpu(lib):
    from paper_2408_12894_b200 import binding as b
    assert lib.flod_scene_bytes(0, None, 0) == 0
    d = (b.LevelDesc * 2)()
    d[0].n, d[1].n = 1000, 4000
    assert lib.flod_scene_bytes(2, d, 4) == 0
    n0 = lib.flod_scene_bytes(2, d, 0)
    n3 = lib.flod_scene_bytes(2, d, 3)
    assert n0 >= 5000 * (12 + 24 + 4 + 4 + 12) and n3 >= 5000 * (12 + 24 + 4 + 4 + 192) and n3 > n0
    assert lib.flod_workspace_bytes(None, 128, 128, 1 << 20) == 0
    assert lib.flod_destroy(None) < 0 and lib.flod_render(None, None, b.LevelMode(1, 1), 1.0, None, None) < 0
    assert lib.flod_last_error(None) == b"null context"


def test_create_fails_loudly_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    assert lib.flod_create(C.byref(h), 0) < 0 and not h.value
    import paper_2408_12894_b200 as pkg
    with pytest.raises(RuntimeError):
        pkg.Renderer(0)


def test_product_does_not_import_the_oracle():
    """The CUDA path and the oracle share no code: the package never imports oracle/ (and vice versa)."""
    code = "import sys, paper_2408_12894_b200, flod_synth; assert 'oracle' not in sys.modules"
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)
    code = "import sys, oracle; assert not any(m.startswith('paper_2408_12894_b200') for m in sys.modules)"
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)
    import re
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2408_12894_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(root, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, re.M), f
                assert not re.search(r"#include\s+[<\"].*oracle", text), f
