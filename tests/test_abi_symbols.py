"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads without a GPU
driver, exports every function include/tpcclus.h declares, and fails loudly (no CPU fallback)
when there is no device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "tpcclus.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tpcclus_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for n in ("tpcclus_create", "tpcclus_run", "tpcclus_result", "tpcclus_destroy"):
        assert n in names


def test_library_builds_loads_and_exports_every_symbol():
    import paper_2412_13755_b200 as T

    L = T.lib()
    for name in declared_functions():
        assert hasattr(L, name), name
    assert set(T.EXPORTS) == set(declared_functions())
    assert T.tpcclus_strerror(0) == "ok" and "capacity" in T.tpcclus_strerror(T.TPCCLUS_ERR_CAPACITY)


def test_record_layouts_match_header():
    import paper_2412_13755_b200 as T

    assert ctypes.sizeof(T.tpcclus_geometry) == 56
    assert ctypes.sizeof(T.tpcclus_run_stats) == 32
    assert ctypes.sizeof(T.tpcclus_fragment) == 40
    assert T.CLUSTER_DTYPE.fields["time"][1] == 4 and T.CLUSTER_DTYPE.fields["qtot"][1] == 12


def test_no_cpu_fallback():
    """Without a CUDA device create() must fail with ERR_CUDA; geometry errors come first."""
    import torch
    import paper_2412_13755_b200 as T

    with pytest.raises(T.TpcclusError) as ei:
        T.tpcclus_create([0], n_sectors=1, tf_time_bins=10, max_digits=1)
    assert ei.value.code == T.TPCCLUS_ERR_GEOMETRY
    if not torch.cuda.is_available():
        with pytest.raises(T.TpcclusError) as ei:
            T.tpcclus_create([10], n_sectors=1, tf_time_bins=10, max_digits=1)
        assert ei.value.code == T.TPCCLUS_ERR_CUDA


def test_product_does_not_import_oracle():
    """The product path may not route through oracle/ (and the oracle not through the product)."""
    pkg = os.path.join(ROOT, "paper_2412_13755_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "tpc_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2412_13755_b200" not in txt and "from paper_2412_13755_b200" not in txt
            assert "#include \"../include" not in txt and "#include \"tpcclus" not in txt


def test_product_reads_no_environment_variables():
    """behaviour is selected by the geometry struct only — no env vars, no global state."""
    pkg = os.path.join(ROOT, "paper_2412_13755_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".cu", ".cuh", ".h")):
                assert "getenv" not in open(os.path.join(dirpath, f)).read(), f


def test_binding_constants_match_the_header():
    """Every integer `#define TPCCLUS_*` of include/tpcclus.h has the same value in the ctypes binding (error codes,
    flag and option bits, limits), and every error code has a message of its own."""
    import paper_2412_13755_b200 as T

    src = open(os.path.join(ROOT, "include", "tpcclus.h")).read()
    defs = dict(re.findall(r"^#define\s+(TPCCLUS_[A-Z0-9_]+)\s+(-?(?:0x[0-9a-fA-F]+|\d+))(?:u|ull)?\b", src, flags=re.M))
    assert {"TPCCLUS_OK", "TPCCLUS_ERR_CAPACITY", "TPCCLUS_ERR_TOO_LARGE", "TPCCLUS_OPT_BIN_DIRECT",
            "TPCCLUS_SELECT_STATIC_MAX_RECORDS", "TPCCLUS_FLAG_SPLIT"} <= set(defs)
    missing = [n for n in defs if not hasattr(T, n) and not n.endswith("_H")]
    # limits that only the C side needs may be absent from the binding; codes, flags and options may not
    assert not [n for n in missing if n.startswith(("TPCCLUS_ERR_", "TPCCLUS_FLAG_", "TPCCLUS_OPT_"))], missing
    for name, text in defs.items():
        if hasattr(T, name):
            assert getattr(T, name) == int(text, 0), name
    msgs = {T.tpcclus_strerror(int(v, 0)) for n, v in defs.items() if n.startswith("TPCCLUS_ERR_")}
    assert len(msgs) == len([n for n in defs if n.startswith("TPCCLUS_ERR_")]) and "unknown status" not in msgs
