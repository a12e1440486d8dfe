"""Host-side checks that need no GPU: libctqr.so builds for sm_100a, loads, and exports every
symbol include/ctqr.h declares; the ctypes mirrors of the two ABI structs have the C layout;
argument errors are reported LAPACK-style without touching a device."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2412_07631_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build.build()
    return binding.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "ctqr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ct_qr_\w+)\s*\(", src)))


def test_every_declared_symbol_is_exported_and_bound(L):
    syms = declared_symbols()
    assert {"ct_qr_factor", "ct_qr_solve", "ct_qr_apply_qt", "ct_qr_trsm", "ct_qr_get_R", "ct_qr_get_V",
            "ct_qr_get_T", "ct_qr_get_tau", "ct_qr_get_stats", "ct_qr_destroy"} <= set(syms)
    raw = ctypes.CDLL(binding.LIB_PATH)
    for s in syms:
        assert hasattr(raw, s), f"{s} declared in ctqr.h but not exported"
        assert s in binding.EXPORTS, f"{s} has no ctypes prototype in binding.py"
    assert set(binding.EXPORTS) <= set(syms)


def test_struct_layouts_match_the_header(tmp_path):
    """The ctypes mirrors against the C compiler's view of include/ctqr.h: a small C program prints sizeof and
    every offsetof; names, order, offsets and sizes must agree."""
    import subprocess
    pairs = (("ctqr_options_t", binding.Options), ("ctqr_stats_t", binding.Stats))
    pairs += (("ctqr_csr_t", binding.Csr), ("ctqr_refine_info_t", binding.RefineInfo))
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "ctqr.h"', 'int main(void) {']
    for cname, cls in pairs:
        lines.append(f'printf("%zu\\n", sizeof({cname}));')
        for fld, _ in cls._fields_:
            lines.append(f'printf("%zu\\n", offsetof({cname}, {fld}));')
    lines += ['return 0; }']
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    got = [int(x) for x in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    want = []
    for _, cls in pairs:
        want.append(ctypes.sizeof(cls))
        want += [getattr(cls, fld).offset for fld, _ in cls._fields_]
    assert got == want
    # every member the header declares has a mirror (count the declarators of each struct body)
    hdr = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "ctqr.h")).read(), flags=re.S)
    for cname, cls in pairs:
        body = re.search(r"typedef struct \{([^}]*)\} " + cname, hdr, flags=re.S).group(1)
        n_decl = sum(len(d.split(",")) for d in body.split(";") if d.strip())
        assert n_decl == len(cls._fields_), (cname, n_decl, len(cls._fields_))


def test_version_and_error_strings(L):
    assert L.ct_qr_version() >= 100
    assert b"success" in L.ct_qr_strerror(0)
    assert b"argument" in L.ct_qr_strerror(-3)
    assert b"zero" in L.ct_qr_strerror(4)


def test_argument_errors_need_no_device(L):
    h = ctypes.c_void_p()
    A = np.zeros((4, 2), order="F")
    P = A.ctypes.data
    assert L.ct_qr_factor(None, 4, 2, 4, 1, None, ctypes.byref(h)) == -1
    assert L.ct_qr_factor(P, 0, 2, 4, 1, None, ctypes.byref(h)) == -2
    assert L.ct_qr_factor(P, 4, 5, 4, 1, None, ctypes.byref(h)) == -3
    assert L.ct_qr_factor(P, 4, 2, 3, 1, None, ctypes.byref(h)) == -4
    assert L.ct_qr_factor(P, 4, 2, 4, 7, None, ctypes.byref(h)) == -5
    assert L.ct_qr_factor(P, 4, 2, 4, 1, None, None) == -7
    assert L.ct_qr_solve(None, P, 4, 1, P, 2) == -1
    assert L.ct_qr_get_stats(None, None) == -1
    assert b"" != L.ct_qr_last_error()


def test_persistence_argument_and_file_errors_need_no_device(L, tmp_path):
    h = ctypes.c_void_p()
    assert L.ct_qr_save(None, b"/tmp/x") == -1
    assert L.ct_qr_load(None, None, ctypes.byref(h)) == -1
    assert L.ct_qr_load(b"/tmp/x", None, None) == -3
    assert L.ct_qr_dtype(None) == -1
    # missing file, empty file, wrong magic, right magic with a corrupt header: all CTQR_ERR_IO (3), no device touched
    assert L.ct_qr_load(os.fsencode(tmp_path / "missing.ctqr"), None, ctypes.byref(h)) == 3
    (tmp_path / "empty.ctqr").write_bytes(b"")
    assert L.ct_qr_load(os.fsencode(tmp_path / "empty.ctqr"), None, ctypes.byref(h)) == 3
    (tmp_path / "junk.ctqr").write_bytes(b"NOTAFACT" + bytes(8192))
    assert L.ct_qr_load(os.fsencode(tmp_path / "junk.ctqr"), None, ctypes.byref(h)) == 3
    (tmp_path / "hdr.ctqr").write_bytes(b"CTQRFAC1" + bytes(8192))
    assert L.ct_qr_load(os.fsencode(tmp_path / "hdr.ctqr"), None, ctypes.byref(h)) == 3
    assert b"not a ctqr factor file" in L.ct_qr_last_error()
    assert h.value is None


def test_no_cpu_fallback(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    h = ctypes.c_void_p()
    A = np.eye(4, 2).copy(order="F")
    rc = L.ct_qr_factor(A.ctypes.data, 4, 2, 4, 1, None, ctypes.byref(h))
    assert rc == 1 and b"no CPU fallback" in L.ct_qr_last_error()
