"""CPU-only checks of the C-ABI boundary: the library builds for sm_100a, loads, exports every symbol
that include/hlc2.h declares, and its host-side logic (size queries, argument checks, error strings)
behaves.  No compute call is made here (no GPU)."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def P():
    from paper_2301_07331_b200 import build
    build.build()
    import paper_2301_07331_b200 as P
    return P


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "hlc2.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hlc2_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(P):
    names = declared_symbols()
    assert {"hlc2_build_index", "hlc2_crossmatch", "hlc2_stream_crossmatch", "hlc2_index_sizes"} <= set(names)
    lib = ctypes.CDLL(P.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/hlc2.h but not exported by libhlc2.so"


def test_library_holds_sm100a_code(P):
    out = subprocess.run(["cuobjdump", "-lelf", P.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_size_queries_and_argument_checks(P):
    ib, tb = P.hlc2_index_sizes(0)
    assert ib > 0 and tb > 0
    ib1, tb1 = P.hlc2_index_sizes(1_000_000, P.make_opts(1.0))
    ib2, tb2 = P.hlc2_index_sizes(2_000_000, P.make_opts(1.0))
    assert ib2 > ib1 > 40 * 1_000_000 and tb2 > tb1          # >= 32 B/source of SoA + keys + cell table
    assert ib1 % 256 == 0 and tb1 % 256 == 0
    for bad in (P.make_opts(0.0), P.make_opts(-1.0), P.make_opts(float("nan")), P.make_opts(1e9),
                P.make_opts(1.0, target_occupancy=-1.0), P.make_opts(1.0, cell_arcsec=-5.0)):
        with pytest.raises(P.Hlc2Error) as e:
            P.hlc2_index_sizes(10, bad)
        assert e.value.status == P.HLC2_ERR_INVALID_ARG
    with pytest.raises(P.Hlc2Error) as e:
        P.hlc2_index_sizes(-1)
    assert e.value.status == P.HLC2_ERR_INVALID_ARG
    with pytest.raises(P.Hlc2Error) as e:
        P.hlc2_index_sizes(2 ** 32)
    assert e.value.status == P.HLC2_ERR_TOO_MANY


def test_null_handles_are_rejected(P):
    L = P.lib()
    assert L.hlc2_index_status(None, None) == P.HLC2_ERR_INVALID_ARG
    assert L.hlc2_grid_describe(None, None, None) == P.HLC2_ERR_INVALID_ARG
    assert L.hlc2_crossmatch(None, None, 1.0, 0, None, None, None, 0, None, None, 0, None) == P.HLC2_ERR_INVALID_ARG
    assert L.hlc2_crossmatch_static(None, None, 1.0, 0, None, None, None, 0, None, None) == P.HLC2_ERR_INVALID_ARG
    out = ctypes.c_void_p()
    assert L.hlc2_build_index(None, None, None, 5, None, None, 0, None, 0, None, ctypes.byref(out)) == P.HLC2_ERR_INVALID_ARG
    L.hlc2_index_destroy(None)


def test_error_strings(P):
    L = P.lib()
    seen = set()
    for code in range(0, -9, -1):
        s = L.hlc2_strerror(code).decode()
        assert s and s != "unknown status"
        seen.add(s)
    assert len(seen) == 9
    assert "8 MiB" in L.hlc2_strerror(P.HLC2_ERR_STATIC_LIMIT).decode()          # the limit is named in the message
    assert L.hlc2_strerror(-99).decode() == "unknown status"
    assert "sm_100a" in P.version()


def test_product_has_no_cpu_fallback(P):
    """The binding must fail loudly without a device rather than route anywhere else."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        P.hlc2_build_index(torch.zeros(4, dtype=torch.float64), torch.zeros(4, dtype=torch.float64))
    pkg = os.path.join(ROOT, "paper_2301_07331_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "hlc2_oracle" not in txt


def test_size_queries_grow_with_n(P):
    """hlc2_stream_crossmatch sizes its arena for the largest band and builds smaller ones inside it: the size queries
    must never shrink when n grows (also across the automatic-occupancy brackets)."""
    import numpy as np
    o = P.make_opts(1.0)
    ns = sorted({int(x) for x in np.concatenate([np.arange(1, 2000), np.logspace(3.3, 8.9, 1500)])})
    prev = (0, 0)
    for n in ns:
        cur = P.hlc2_index_sizes(n, o)
        assert cur[0] >= prev[0] and cur[1] >= prev[1], (n, cur, prev)
        prev = cur
