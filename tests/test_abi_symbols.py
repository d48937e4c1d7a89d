"""The C-ABI library loads without a GPU and exports every symbol include/lqcd.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1209_5942_b200 import build
    return build.build()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "lqcd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lqcd_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(lib_path):
    lib = ctypes.CDLL(lib_path)
    names = _declared_symbols()
    assert "lqcd_init" in names and "lqcd_dslash_eo" in names and "lqcd_mtm" in names and "lqcd_cg_mdagm" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/lqcd.h but not exported"


def test_binding_covers_every_symbol(lib_path):
    import paper_1209_5942_b200.binding as B
    assert sorted(B.SYMBOLS) == _declared_symbols()
    for n in B.SYMBOLS:
        assert callable(getattr(B, n))


def test_host_logic_without_gpu(lib_path):
    """Argument validation and size queries need no device."""
    import paper_1209_5942_b200.binding as B
    B.lqcd_init((8, 8, 8, 16), [1, 1, 1, -1])
    assert B.lqcd_spinor_bytes() == 4096 * 192          # 192 B per spinor
    assert B.lqcd_gauge_bytes() == 8192 * 576           # 576 B per site
    B.lqcd_set_format(B.LQCD_DOUBLE, 12)
    assert B.lqcd_gauge_bytes() == 8192 * 384           # REC12
    B.lqcd_set_format(B.LQCD_SINGLE, 18)
    assert B.lqcd_gauge_bytes() == 8192 * 288 and B.lqcd_spinor_bytes() == 4096 * 96
    for bad in ((8, 8, 7, 16), (8, 0, 8, 16), (8, 8, 8, -2)):
        with pytest.raises(B.LqcdError) as e:
            B.lqcd_init(bad, [1, 1, 1, -1])
        assert e.value.status == B.LQCD_BAD_DIMS
    with pytest.raises(B.LqcdError) as e:
        B.lqcd_init((8, 8, 8, 16), [1, 1, 1, 0.5])
    assert e.value.status == B.LQCD_BAD_DIMS
    B.lqcd_init((4, 4, 4, 4), [1, 1, 1, -1])
    with pytest.raises(B.LqcdError) as e:
        B.lqcd_set_block_size(48)
    assert e.value.status == B.LQCD_BAD_ARG
    assert B.lqcd_last_error() != ""


def test_plaquette_static_argument_checks_without_gpu(lib_path):
    """lqcd_plaquette_static (the no-allocation entry point) rejects null pointers and lattices whose partial sums do not
    fit its static scratch array before it touches the device."""
    import ctypes
    import paper_1209_5942_b200.binding as B
    B.lqcd_init((4, 4, 4, 4), [1, 1, 1, -1])
    assert B._lib.lqcd_plaquette_static(None, None) == B.LQCD_BAD_ARG
    B.lqcd_init((64, 32, 32, 34), [1, 1, 1, -1])     # 8 * ceil(V / 256) = 69632 partial sums > 65536
    dummy = ctypes.c_void_p(256)                     # never dereferenced: the size check comes first
    assert B._lib.lqcd_plaquette_static(dummy, dummy) == B.LQCD_BAD_ARG
    assert "static scratch array holds 65536" in B.lqcd_last_error()
    B.lqcd_init((4, 4, 4, 4), [1, 1, 1, -1])


def test_paper_sizes_fixture():
    vals = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "paper_table2_table3_sizes.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            vals[k] = int(v)
    # Table 2's 2880 B = 8 links + 8 neighbour spinors + 1 store
    assert vals["dslash_rw_bytes_per_site"] == 8 * vals["su3_bytes"] + 8 * vals["spinor_bytes"] + vals["spinor_bytes"]
    assert vals["gauge_bytes_per_site"] == 4 * vals["su3_bytes"]
    assert vals["gauge_rec12_bytes_per_site"] == 4 * 12 * 8
    assert vals["spinor_eo_bytes_per_site_of_V"] * 2 == vals["spinor_bytes"]
