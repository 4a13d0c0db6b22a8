"""-m "not gpu": the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/fasttracks_b200.h declares; struct layouts of the binding match the header.  No compute."""
import ctypes as C
import os
import re

from paper_2411_18370_b200 import binding as B
from paper_2411_18370_b200 import build as bld

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "fasttracks_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ft_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    so = bld.build()
    lib = C.CDLL(so)
    names = _declared()
    assert set(names) == set(B.SYMBOLS), names
    for n in names:
        assert hasattr(lib, n), n


def test_struct_layouts():
    assert C.sizeof(B.FtCand) == 32 and B.CAND_DTYPE.itemsize == 32 and B.CAND_BOX_DTYPE.itemsize == 48
    assert C.sizeof(B.FtBankBox) == 104 and C.sizeof(B.FtPeaks) == 40
    assert C.sizeof(B.FtCounters) == 56
    assert B.FtGrid.n_f0.offset == 16 and B.FtGrid.t_ref.offset == 48
    assert C.sizeof(B.FtGrid) == 120


def test_no_device_is_a_loud_error():
    """Without a GPU ft_create fails with FT_ERR_CUDA: there is no CPU fallback."""
    import torch
    if torch.cuda.is_available():
        return
    lib = B.load_library()
    h = C.c_void_p()
    import numpy as np
    t = np.zeros(4); v = np.zeros((4, 3)); w = np.ones(4, np.float32)
    fake = C.c_void_p(256)  # never dereferenced on the host
    rc = lib.ft_create(C.byref(h), fake, 4, 8, 8, t.ctypes.data_as(C.c_void_p), v.ctypes.data_as(C.c_void_p),
                       w.ctypes.data_as(C.c_void_p), 1, 100.0, 1.0 / 1800, None)
    assert rc == -3 and b"no CPU fallback" in lib.ft_last_error(h)
    lib.ft_destroy(h)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2411_18370_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                for line in open(os.path.join(dp, f)):
                    s = line.strip()
                    if s.startswith(("import ", "from ", "#include")) or "CDLL" in s or "dlopen" in s:
                        assert "oracle" not in s, (f, s)


def test_header_is_plain_c():
    """The boundary is a C ABI: the header compiles as C99 with no C++ or torch types."""
    import subprocess
    hdr = os.path.join(ROOT, "include", "fasttracks_b200.h")
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-fsyntax-only", "-x", "c", hdr],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    assert "torch" not in open(hdr).read().lower().replace("pytorch allocates", "")
