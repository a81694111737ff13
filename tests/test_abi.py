"""CPU-only checks of the boundary: libmosaic.so builds, loads and exports every symbol that
include/mosaic.h declares; host-side argument validation answers without touching a GPU."""
import ctypes
import re

import pytest

from conftest import ROOT
from paper_2606_03014_b200 import build as mbuild


@pytest.fixture(scope="module")
def lib():
    mbuild.build_library()
    from paper_2606_03014_b200 import mosaic
    return mosaic.load()


def _declared_symbols():
    text = (ROOT / "include" / "mosaic.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mosaic_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    from paper_2606_03014_b200 import mosaic
    names = _declared_symbols()
    assert {"mosaic_gate", "mosaic_compact", "mosaic_agg_prefill_attn"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
        assert n in mosaic.SIGNATURES, f"binding lacks {n}"
    assert set(mosaic.SIGNATURES) == set(names)


def test_version_and_status_strings(lib):
    assert lib.mosaic_version() >= 100
    assert lib.mosaic_status_string(0) == b"MOSAIC_OK"
    assert lib.mosaic_status_string(2) == b"MOSAIC_ERR_UNSUPPORTED"


def test_workspace_helpers(lib):
    assert lib.mosaic_compact_workspace_bytes(0) >= 16
    assert lib.mosaic_compact_workspace_bytes(1 << 20) >= 16 * ((1 << 20) // 256)
    a = lib.mosaic_agg_prefill_attn_workspace_bytes(78, 179057, 28, 4, 128)
    assert 8 * (179057 // 128 + 78) <= a < (1 << 20)
    assert lib.mosaic_stage_host_arena_bytes(256, 3, 1000, 28, 4, 128) > 1000 * 28 * 128 * 4


def test_host_side_validation_needs_no_gpu(lib):
    nan = float("nan")
    fake = ctypes.c_void_p(0x1000)  # never dereferenced: validation fails first
    assert lib.mosaic_gate(fake, None, 8, 0, 0.5, 0, None, None, None, None, fake, None) == 1
    assert lib.mosaic_gate(fake, None, 8, 33, 0.5, 0, None, None, None, None, fake, None) == 1
    assert lib.mosaic_gate(fake, None, 8, 3, nan, 0, None, None, None, None, fake, None) == 1
    assert lib.mosaic_gate(fake, None, 8, 3, 0.5, 1, None, None, None, None, fake, None) == 1
    assert lib.mosaic_gate(fake, None, -1, 3, 0.5, 0, None, None, None, None, fake, None) == 1
    assert lib.mosaic_gate(fake, None, 0, 3, 0.5, 0, None, None, None, None, None, None) == 0
    # attention: Hq % Hkv, unsupported head dim, empty batch
    args = lambda Hq, Hkv, D, n, T: (fake, fake, fake, fake, n, T, 128, Hq, Hkv, D, 0.1, fake, fake,
                                     fake, 1 << 20, None)
    assert lib.mosaic_agg_prefill_attn(*args(7, 2, 128, 1, 128)) == 1
    assert lib.mosaic_agg_prefill_attn(*args(8, 2, 96, 1, 128)) == 2
    assert lib.mosaic_agg_prefill_attn(*args(8, 2, 128, 0, 0)) == 0
    assert lib.mosaic_agg_prefill_attn(*args(8, 2, 128, 1, 1 << 31)) == 1
    # the SURVEY 8(f) entries validate before they touch the device too
    kv = lambda Hq, Hkv, D, n, Tq, Tk: (fake, fake, fake, fake, fake, n, Tq, Tk, 128, Hq, Hkv, D, 0.1,
                                        1, fake, fake, fake, 1 << 20, None)
    assert lib.mosaic_agg_prefill_attn_kv(*kv(7, 2, 128, 1, 128, 256)) == 1
    assert lib.mosaic_agg_prefill_attn_kv(*kv(8, 2, 96, 1, 128, 256)) == 2
    assert lib.mosaic_agg_prefill_attn_kv(*kv(8, 2, 128, 1, 128, 1 << 31)) == 1
    assert lib.mosaic_agg_prefill_attn_kv(*kv(8, 2, 128, 0, 0, 0)) == 0
    asm = lambda n, E: (fake, fake, n, 100, fake, fake, fake, fake, E, fake, fake, None, None)
    assert lib.mosaic_assemble_context(*asm(4, 0)) == 1
    assert lib.mosaic_assemble_context(*asm(4, 33)) == 1
    assert lib.mosaic_assemble_context(*asm(-1, 3)) == 1
    assert lib.mosaic_rope_packed(fake, fake, fake, 16, 4, 2, 96, 1e6, None) == 2
    assert lib.mosaic_rope_packed(fake, fake, fake, 16, 4, 2, 128, 0.0, None) == 1
    assert lib.mosaic_rope_packed(fake, fake, fake, 0, 4, 2, 128, 1e6, None) == 0
    assert lib.mosaic_lse_merge(fake, fake, fake, fake, 16, 4, 100, fake, fake, None) == 1
    assert lib.mosaic_lse_merge(fake, fake, fake, fake, 0, 4, 128, fake, fake, None) == 0
    dec = lambda Hq, Hkv, D, n: (fake, fake, fake, fake, n, 1000, Hq, Hkv, D, 0.1, fake, fake, fake,
                                 1 << 20, None)
    assert lib.mosaic_agg_decode_attn(*dec(7, 2, 128, 4)) == 1
    assert lib.mosaic_agg_decode_attn(*dec(8, 2, 96, 4)) == 2
    assert lib.mosaic_agg_decode_attn(*dec(8, 2, 128, 0)) == 0
    assert lib.mosaic_agg_decode_attn_workspace_bytes(4, 1000, 8, 2, 128) > 0
    assert lib.mosaic_agg_decode_attn_workspace_bytes(4, 1000, 7, 2, 128) == 0


def test_product_path_does_not_import_oracle():
    """The oracle is test infrastructure: nothing under the package may import or include it."""
    pkg = ROOT / "paper_2606_03014_b200"
    pat = re.compile(r"^\s*(import\s+oracle|from\s+oracle|#\s*include\s*[<\"].*oracle)", re.M)
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")):
        assert not pat.search(f.read_text()), f
