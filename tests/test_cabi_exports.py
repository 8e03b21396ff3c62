"""The C-ABI library loads without a GPU and exports every symbol include/tpc_tracker.h declares; the
host-side argument checks answer without touching a device (no compute calls here)."""
import ctypes as C
import os
import re

import numpy as np

import paper_2009_07515_b200 as tpc
from tpc_synth import default_params, generate_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "tpc_tracker.h")


def _declared():
    src = open(HEADER).read()
    return sorted(set(re.findall(r"TPC_API\s+[\w\s\*]+?\b(tpc_\w+)\s*\(", src)))


def test_header_symbols_are_exported():
    names = _declared()
    assert len(names) >= 11 and {"tpc_tracker_create", "tpc_track_timeframe", "tpc_tracker_destroy"} <= set(names)
    lib = tpc.load_library()
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(tpc.EXPORTS) == names        # the binding wraps exactly what the header declares


def test_nothing_else_leaks_from_the_library():
    """-fvisibility=hidden: only the tpc_* entry points are dynamic symbols of our own."""
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", tpc.library_path()], capture_output=True, text=True, check=True).stdout
    ours = [ln.split()[-1] for ln in out.splitlines() if " T " in ln]
    assert sorted(ours) == _declared(), ours


def test_error_strings_and_host_side_argument_checks():
    lib = tpc.load_library()
    lib.tpc_error_string.restype = C.c_char_p
    assert lib.tpc_error_string(0) == b"ok"
    assert lib.tpc_error_string(-1) and lib.tpc_error_string(-12345) == b"unknown error"
    # null handle / null params are rejected on the host
    assert lib.tpc_tracker_destroy(None) != 0
    lib.tpc_tracker_workspace_bytes.restype = C.c_size_t
    assert lib.tpc_tracker_workspace_bytes(None, C.c_int64(10), C.c_int64(10), C.c_int64(10), C.c_int64(10), C.c_int64(10), 0) == 0


def test_workspace_bytes_is_host_only_and_monotone():
    tf = generate_config("cfg1")
    P = default_params(tf)
    lib = tpc.load_library()
    lib.tpc_tracker_workspace_bytes.restype = C.c_size_t
    pp, keep = tpc.pack_params(P)

    def ws(n, nb, ns, nt, ntc, host):
        return lib.tpc_tracker_workspace_bytes(C.byref(pp), C.c_int64(n), C.c_int64(nb), C.c_int64(ns), C.c_int64(nt),
                                               C.c_int64(ntc), C.c_int32(host))
    a = ws(10_000, 20_000, 1000, 1000, 10_000, 0)
    b = ws(20_000, 20_000, 1000, 1000, 10_000, 0)
    c = ws(10_000, 20_000, 1000, 1000, 10_000, 1)
    assert 0 < a < b and a < c
    assert a >= 10_000 * (16 + 4 + 8 + 2 + 4 * 4 + 4 + 8)   # rec, perm, yz, srow, four link arrays, seed bits, owner
    assert ws(0, 20_000, 1000, 1000, 10_000, 0) == 0         # capacities must be >= 1
    # bad geometry is rejected: non-increasing row_x
    Q = dict(P)
    Q["row_x"] = np.array(P["row_x"][::-1], dtype=np.float32)
    qq, keep2 = tpc.pack_params(Q)
    assert lib.tpc_tracker_workspace_bytes(C.byref(qq), C.c_int64(10), C.c_int64(10), C.c_int64(10), C.c_int64(10),
                                           C.c_int64(10), C.c_int32(0)) == 0


def test_header_is_plain_c(tmp_path):
    """include/tpc_tracker.h compiles as C99 (no C++ or torch types cross the boundary)."""
    import subprocess
    src = tmp_path / "t.c"
    src.write_text('#include "tpc_tracker.h"\nint main(void) { tpc_params_t p; tpc_tracks_t t; tpc_fit_t f; (void)p; (void)t; (void)f; return TPC_OK; }\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-fsyntax-only", "-I", os.path.join(ROOT, "include"), str(src)],
                   check=True)
