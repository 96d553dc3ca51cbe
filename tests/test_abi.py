"""CPU-side checks of the boundary: libtpmc.so builds, loads without a GPU and exports every
symbol include/tpmc.h declares; struct layouts of the binding match the header; the product
package does not import the oracle.  No compute calls here."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1312_3691_b200 import build
    return build.build()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "tpmc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(tpmc_[a-z_0-9]+)\s*\(", src)
    return sorted(set(names))


def test_header_declares_the_expected_entry_points():
    names = declared_functions()
    for n in ("tpmc_mesh_create", "tpmc_mesh_destroy", "tpmc_mesh_info", "tpmc_run", "tpmc_run_host",
              "tpmc_seed", "tpmc_trace", "tpmc_strerror"):
        assert n in names


def test_library_exports_every_declared_symbol(libpath):
    L = C.CDLL(libpath)
    for n in declared_functions():
        assert hasattr(L, n), n
    import paper_1312_3691_b200 as t
    assert sorted(t.EXPORTS) == declared_functions()
    assert "sm_100a" in t.tpmc_version()


def test_sass_is_sm100a(libpath):
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_struct_layouts_match_header(libpath, tmp_path):
    import paper_1312_3691_b200 as t
    prog = tmp_path / "sz.c"
    prog.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "tpmc.h"\nint main(){printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n",'
                    "sizeof(tpmc_params),sizeof(tpmc_stats),sizeof(tpmc_debug),sizeof(tpmc_mesh_info_t),"
                    "offsetof(tpmc_params,N),offsetof(tpmc_params,x_ref),offsetof(tpmc_mesh_info_t,nt),"
                    "offsetof(tpmc_params,flags),offsetof(tpmc_params,control_volume),offsetof(tpmc_stats,ret_precull_a),"
                    "offsetof(tpmc_stats,ms_sort));return 0;}\n")
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(prog), "-o", str(exe)], check=True)
    got = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    want = [C.sizeof(t.tpmc_params), C.sizeof(t.tpmc_stats), C.sizeof(t.tpmc_debug), C.sizeof(t.tpmc_mesh_info_t),
            t.tpmc_params.N.offset, t.tpmc_params.x_ref.offset, t.tpmc_mesh_info_t.nt.offset,
            t.tpmc_params.flags.offset, t.tpmc_params.control_volume.offset, t.tpmc_stats.ret_precull_a.offset,
            t.tpmc_stats.ms_sort.offset]
    assert got == want
    assert (t.TPMC_FLAG_NO_PRECULL, t.TPMC_FLAG_NO_HORIZON, t.TPMC_FLAG_ALIGN_OFF, t.TPMC_FLAG_ALIGN_ON,
            t.TPMC_FLAG_EXACT_TRACE, t.TPMC_FLAG_SORT_RAYS) == (1, 2, 4, 8, 16, 32)


def test_library_reads_no_environment_variable():
    """Behaviour is selected through tpmc_params only (include/tpmc.h conventions)."""
    csrc = os.path.join(ROOT, "paper_1312_3691_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f


def test_error_strings_and_null_arguments(libpath):
    import paper_1312_3691_b200 as t
    L = t.lib()
    assert L.tpmc_strerror(0) == b"ok"
    assert L.tpmc_strerror(t.TPMC_EINVAL) == b"invalid argument"
    # argument validation happens before any CUDA call
    h = C.c_void_p()
    assert L.tpmc_mesh_create(None, 0, None, 0, None, 0, None, C.byref(h)) == t.TPMC_EINVAL
    assert L.tpmc_run(None, None, None, None, None, None, None, None) == t.TPMC_EINVAL
    assert L.tpmc_mesh_info(None, None) == t.TPMC_EINVAL


def test_product_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_1312_3691_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "tpmc_oracle" not in txt, f
    code = "import sys; import paper_1312_3691_b200; assert 'oracle' not in sys.modules"
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)


def test_compute_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("has a GPU")
    import numpy as np
    import paper_1312_3691_b200 as t
    with pytest.raises(t.TpmcError):
        t.Mesh(np.zeros((3, 3), np.float32), np.array([[0, 1, 2]], np.int32))
