"""-m "not gpu": the C-ABI library loads, exports every symbol include/nsfrb.h declares, and its
host-side validation behaves as the header says.  No compute calls (there is no GPU here)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    from paper_2510_18136_b200 import build, nsfrb
    build.build()
    return nsfrb


def test_header_symbols_are_exported():
    nsfrb = _lib()
    hdr = open(os.path.join(ROOT, "include", "nsfrb.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(nsfrb_[a-z_]+)\s*\(", hdr))
    assert declared == set(nsfrb.EXPORTS), declared ^ set(nsfrb.EXPORTS)
    L = nsfrb.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert b"sm_100a" in L.nsfrb_version()
    assert ctypes.sizeof(nsfrb.nsfrb_cand) == 20


def test_library_holds_sm100a_code_only():
    import subprocess
    nsfrb = _lib()
    out = subprocess.run(["cuobjdump", "--list-elf", nsfrb.LIB_PATH], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    archs = set(re.findall(r"sm_\d+a?", out.stdout))
    assert archs == {"sm_100a"}, archs


def _create(nsfrb, **kw):
    a = dict(nx=4, ny=4, nchan=4, nt=64, freqs=np.linspace(1.3, 1.5, 4), tsamp=0.1342,
             dms=np.asarray([0.0, 100.0]), widths=np.asarray([1, 2], np.int32), thr=6.0)
    a.update(kw)
    h = ctypes.c_void_p()
    f = np.ascontiguousarray(a["freqs"], np.float64)
    dm = np.ascontiguousarray(a["dms"], np.float64)
    w = np.ascontiguousarray(a["widths"], np.int32)
    rc = nsfrb.lib().nsfrb_plan_create(
        ctypes.byref(h), a["nx"], a["ny"], a["nchan"], a["nt"], f.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
        a["tsamp"], dm.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), dm.size,
        w.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), w.size, a["thr"])
    return rc, h


@pytest.mark.parametrize("kw", [
    dict(nx=0), dict(nt=0), dict(nchan=4, freqs=np.asarray([1.3, 1.4, -1.0, 1.5])),
    dict(freqs=np.asarray([1.3, np.nan, 1.4, 1.5])), dict(tsamp=0.0), dict(tsamp=float("inf")),
    dict(dms=np.asarray([0.0, -5.0])), dict(widths=np.asarray([1, 0], np.int32)),
    dict(widths=np.asarray([3, 3], np.int32)),
    dict(dms=np.asarray([0.0, 1e7])),   # delay reaches nt: no valid sample left
])
def test_plan_create_rejects_bad_arguments(kw):
    nsfrb = _lib()
    rc, h = _create(nsfrb, **kw)
    assert rc == nsfrb.NSFRB_EINVAL and not h.value
    assert len(nsfrb.last_error()) > 0


def test_null_arguments_and_destroy_null():
    nsfrb = _lib()
    L = nsfrb.lib()
    assert L.nsfrb_plan_destroy(None) == 0
    assert L.nsfrb_search(None, None, None, None, None, None, 0, None) == nsfrb.NSFRB_EINVAL
    assert L.nsfrb_stream_push(None, None, 1, None, None, None, None, 0, None) == nsfrb.NSFRB_EINVAL
    assert L.nsfrb_plan_get_delays(None, None) == nsfrb.NSFRB_EINVAL
    assert L.nsfrb_plan_last_launches(None) == 0
    assert L.nsfrb_psf_mask(None, 3, 3, 90.0, None, None, None) == nsfrb.NSFRB_EINVAL
    assert L.nsfrb_cluster(None, None, None, None, None, 3, 3, 10, None, None, None, None, None) == nsfrb.NSFRB_EINVAL
    buf = (ctypes.c_float * 9)()
    m = (ctypes.c_uint8 * 9)()      # host memory: the argument checks come before any launch
    addr = ctypes.addressof
    assert L.nsfrb_psf_mask(addr(buf), 0, 3, 90.0, addr(m), None, None) == nsfrb.NSFRB_EINVAL
    assert L.nsfrb_psf_mask(addr(buf), 3, 3, 101.0, addr(m), None, None) == nsfrb.NSFRB_EINVAL
    assert L.nsfrb_psf_mask(addr(buf), 3, 3, float("nan"), addr(m), None, None) == nsfrb.NSFRB_EINVAL


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    nsfrb = _lib()
    rc, h = _create(nsfrb)   # valid arguments, but no device: must fail loudly, not fall back
    assert rc in (nsfrb.NSFRB_ECUDA, nsfrb.NSFRB_ENOMEM) and not h.value
    assert "plan device setup" in nsfrb.last_error()


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2510_18136_b200")
    for dp, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dp, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), fn
                assert "nsfrb_oracle" not in src, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_2510_18136_b200" not in src and "libnsfrb.so" not in src, fn


def test_header_is_valid_c99_and_a_c_caller_links(tmp_path):
    """include/nsfrb.h must be usable from plain C: compile a C99 caller of the four main entry points against the
    header and link it with the library (no GPU needed to link; the program is not run here)."""
    import shutil
    import subprocess
    nsfrb = _lib()
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("gcc not available")
    src = tmp_path / "caller.c"
    src.write_text(r'''
#include <stdio.h>
#include "nsfrb.h"
int main(void)
{
    nsfrb_plan *plan = NULL;
    const double f[2] = {1.3, 1.5}, dm[1] = {0.0};
    const int32_t w[1] = {1};
    int rc = nsfrb_plan_create(&plan, 4, 4, 2, 64, f, 0.1342, dm, 1, w, 1, 6.0f);
    if (rc != NSFRB_OK) { printf("%s\n", nsfrb_last_error()); return 1; }
    rc = nsfrb_search(plan, NULL, NULL, NULL, NULL, NULL, 0, NULL);          /* EINVAL: null cube */
    rc = nsfrb_stream_push(plan, NULL, 25, NULL, NULL, NULL, NULL, 0, NULL); /* EINVAL: null chunk */
    (void)sizeof(nsfrb_cand);
    return nsfrb_plan_destroy(plan);
}
''')
    inc = os.path.join(ROOT, "include")
    libdir = os.path.dirname(nsfrb.LIB_PATH)
    exe = tmp_path / "caller"
    subprocess.check_call([gcc, "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", inc, str(src), "-o", str(exe),
                           "-L", libdir, "-l:libnsfrb.so", f"-Wl,-rpath,{libdir}"])
    assert exe.exists()
    import torch
    if torch.cuda.is_available():   # on the GPU box also run it: create, two rejected calls, destroy -> exit code 0
        assert subprocess.run([str(exe)]).returncode == 0
