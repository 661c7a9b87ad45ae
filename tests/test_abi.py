"""CPU-side checks of the boundary: liblqcd.so loads, exports every symbol include/lqcd.h
declares, and the host logic that needs no GPU (parameter validation, size queries)."""
import ctypes
import os
import re

import pytest

import paper_1112_5280_b200 as L

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "lqcd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lqcd_[a-zA-Z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_1112_5280_b200 import _build
    _build.build()
    lib = ctypes.CDLL(_build.LIB)
    names = _declared()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(L.EXPORTS) == names


def test_create_validation_and_sizes():
    c = L.Context((32, 32, 32, 64), 32, 12)
    Vh = 32 * 32 * 32 * 64 // 2
    assert c.Vh == Vh
    assert c.spinor_bytes(True) == Vh * 24 * 4
    assert c.spinor_bytes(False) == Vh * 48 * 4
    assert c.gauge_bytes() == 2 * 8 * 12 * Vh * 4  # gathered by output site: every link stored twice
    assert c.workspace_bytes() == Vh * 24 * 4
    c = L.Context((4, 4, 4, 4), 64, 18)
    assert c.gauge_bytes() == 2 * 8 * 18 * 128 * 8
    c6 = L.Context((6, 6, 6, 6), 32, 12)  # Vh = 648 is padded to 21 tiles of 32 sites
    assert c6.spinor_bytes(True) == 21 * 32 * 24 * 4 and c6.gauge_bytes() == 2 * 21 * 32 * 8 * 12 * 4
    assert c.host_workspace_bytes() >= c.gauge_bytes() + 4 * 256 * 18 * 8 + 4 * c.spinor_bytes(True)
    c8 = L.Context((8, 8, 8, 16), 64, 8)
    assert c8.gauge_bytes() == 2 * 8 * 4096 * 8 * 8
    c16 = L.Context((8, 8, 8, 16), 16, 12)
    assert c16.spinor_bytes(True) == 4096 * 52 and c16.gauge_bytes() == 2 * 8 * 4096 * 24
    with pytest.raises(L.LqcdError) as e:
        L.Context((8, 8, 8, 16), 16, 18)
    assert e.value.status == L.LQCD_EUNSUPPORTED
    for bad in [dict(dims=(4, 4, 3, 4)), dict(dims=(2, 4, 4, 4)), dict(precision=8), dict(recon=10),
                dict(bc=(1, 1, 1, 0.5))]:
        kw = dict(dims=(4, 4, 4, 4), precision=64, recon=18, bc=(1, 1, 1, -1))
        kw.update(bad)
        with pytest.raises(L.LqcdError) as e:
            L.Context(**kw)
        assert e.value.status == L.LQCD_EINVAL


def test_null_pointers_rejected_without_gpu():
    c = L.Context((4, 4, 4, 4), 64, 18)
    lib = L._lib()
    assert lib.lqcd_dslash_eo(c._h, None, None, None, 0, None) == L.LQCD_EINVAL
    assert lib.lqcd_dslash_full(None, None, None, None, None) == L.LQCD_EINVAL
    assert lib.lqcd_apply_M(c._h, None, None, None, 0.1, 2, None, None) == L.LQCD_EINVAL
    assert lib.lqcd_spinor_bytes(None, 1) == 0
    assert lib.lqcd_status_string(L.LQCD_EALIAS).decode() == "output overlaps an input"


def test_alignment_contract_checked_before_any_launch():
    """Native fields are accessed with 256-bit words: every native pointer must be 32-byte aligned, canonical buffers
    16-byte aligned.  The check precedes any CUDA call, so fake addresses exercise it without a GPU."""
    lib = L._lib()
    base = 1 << 20
    for precision, recon in ((64, 12), (64, 18), (32, 12), (32, 18), (16, 12)):
        c = L.Context((4, 4, 4, 4), precision, recon)
        far = base + (1 << 16)
        for off in (8, 16, 24):
            assert lib.lqcd_dslash_eo(c._h, base + off, base + (1 << 18), far, 0, None) == L.LQCD_EALIGN
            assert lib.lqcd_dslash_eo(c._h, base, base + (1 << 18) + off, far, 0, None) == L.LQCD_EALIGN
            assert lib.lqcd_dslash_eo(c._h, base, base + (1 << 18), far + off, 0, None) == L.LQCD_EALIGN
            assert lib.lqcd_dslash_full(c._h, base + off, base + (1 << 18), far + (1 << 16), None) == L.LQCD_EALIGN
            assert lib.lqcd_apply_M(c._h, base, base + (1 << 18), far, 0.1, 1, base + (1 << 17) + off, None) == L.LQCD_EALIGN
            assert lib.lqcd_apply_M(c._h, base + off, base + (1 << 18), far, 0.1, 0, None, None) == L.LQCD_EALIGN
            assert lib.lqcd_pack_spinor(c._h, base + off, far, 0, None) == L.LQCD_EALIGN      # native side: 32
            assert lib.lqcd_unpack_spinor(c._h, far, base + off, 0, None) == L.LQCD_EALIGN
            assert lib.lqcd_pack_gauge(c._h, base + off, far, None) == L.LQCD_EALIGN
        assert lib.lqcd_pack_spinor(c._h, base, far + 8, 0, None) == L.LQCD_EALIGN            # canonical side: 16
        assert lib.lqcd_unpack_spinor(c._h, far + 8, base, 0, None) == L.LQCD_EALIGN
    assert b"32" in lib.lqcd_status_string(L.LQCD_EALIGN)


def test_division_free_index_map_equals_integer_division():
    """decode_site divides checkerboard indices (< 2^30) by the run-time extents with a multiply-shift (geometry.cuh);
    the library's own routine, on the host, against n // d: every extent up to 600, large and awkward ones, indices at
    both ends of the range, around multiples of d, and random."""
    import numpy as np
    lib = L._lib()
    rng = np.random.default_rng(0)
    for d in list(range(1, 601)) + [1023, 1024, 1025, 4097, 65535, 65536, 65537, 100003, (1 << 20) - 1, (1 << 24) + 5, (1 << 29) + 1]:
        ns = set(int(x) for x in rng.integers(0, 1 << 30, 40))
        ns |= {0, 1, d - 1, d, d + 1, (1 << 30) - 1, (1 << 30) - d, ((1 << 30) // d) * d - 1, ((1 << 30) // d) * d}
        for k in (3, 1000, 123457):
            ns |= {k * d - 1, k * d, k * d + 1}
        for n in ns:
            if 0 <= n < (1 << 30):
                assert lib.lqcd_selftest_fastdiv(d, n) == n // d, (d, n)
