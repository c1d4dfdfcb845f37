"""Host-side checks of the C-ABI library (no GPU): it loads, exports every symbol include/qcd.h
declares, and validates arguments before touching CUDA."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def qcd():
    from paper_1212_0785_b200 import build
    build.build()
    from paper_1212_0785_b200 import binding
    return binding


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "qcd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qcd_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound(qcd):
    names = declared_symbols()
    assert len(names) >= 24 and "qcd_gauge_force" in names and "qcd_sum_multi" in names
    raw = C.CDLL(qcd.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), f"{n} declared in include/qcd.h but not exported"
        assert n in qcd.SIGNATURES, f"{n} has no binding"
    for n in ("qcd_gauge_force", "qcd_mom_update", "qcd_link_update", "qcd_reunit", "qcd_mom_refresh",
              "qcd_plaquette", "qcd_sum", "qcd_sum_multi"):  # the eight north_star names
        assert n in names
        assert callable(getattr(qcd, n))


def test_lattice_object_and_sizes(qcd):
    lat = qcd.Lattice((4, 6, 8, 10))
    assert lat.V == 4 * 6 * 8 * 10
    assert lat.field_bytes(qcd.F64) == lat.V * 72 * 8
    assert lat.field_bytes(qcd.F32) == lat.V * 72 * 4
    assert lat.field_bytes(qcd.F32, 3) == lat.V * 3 * 4
    assert lat.workspace_bytes() >= 4096 * 256 * 8
    assert lat.md_host_work_bytes(qcd.F64) == 4 * lat.field_bytes(qcd.F64)
    big = qcd.Lattice((48, 48, 48, 96))
    assert big.V == 10616832 and big.field_bytes(qcd.F64) == 6115295232
    # fields are whole chunks of 32 sites: V = 16 occupies one chunk, V = 480 fifteen
    assert qcd.Lattice((2, 2, 2, 2)).field_bytes(qcd.F64) == 32 * 72 * 8
    assert qcd.Lattice((4, 10, 6, 2)).field_bytes(qcd.F32, 24) == 480 * 24 * 4
    assert qcd.Lattice((2, 2, 2, 6)).field_bytes(qcd.F64) == 64 * 72 * 8  # V = 48 -> two chunks
    assert qcd.lib.qcd_version().decode().startswith("qcdmd")
    assert qcd.Lattice((128, 128, 128, 56)).V == 117440512  # largest class of lattices: 36 V < 2^32


@pytest.mark.parametrize("dims", [(3, 4, 4, 4), (4, 4, 4, 1), (0, 2, 2, 2), (2048, 2048, 2048, 2),
                                  (128, 128, 128, 58)])  # the last: V = 121.6 M, 36 V >= 2^32
def test_bad_extents(qcd, dims):
    with pytest.raises(qcd.QcdError) as e:
        qcd.Lattice(dims)
    assert e.value.code == qcd.EDIMS


def test_argument_validation_happens_before_any_cuda_call(qcd):
    lat = qcd.Lattice((4, 4, 4, 4))
    h = lat.handle
    L = qcd.lib
    fb = lat.field_bytes(qcd.F64)
    a, b = 0x10000000, 0x10000000 + 2 * fb  # fake, never dereferenced: every call must fail first
    assert L.qcd_gauge_force(h, qcd.F64, qcd.ALL, 5.0, None, b, None) == qcd.EINVAL
    assert L.qcd_gauge_force(None, qcd.F64, qcd.ALL, 5.0, a, b, None) == qcd.EINVAL
    assert L.qcd_gauge_force(h, 7, qcd.ALL, 5.0, a, b, None) == qcd.EINVAL
    assert L.qcd_gauge_force(h, qcd.F64, 3, 5.0, a, b, None) == qcd.EINVAL
    assert L.qcd_gauge_force(h, qcd.F64, qcd.ALL, 5.0, a + 8, b, None) == qcd.EALIGN
    assert L.qcd_gauge_force(h, qcd.F64, qcd.ALL, 5.0, a, a + fb // 2, None) == qcd.EALIAS
    assert b"overlap" in L.qcd_last_error()
    assert L.qcd_mom_update(h, qcd.F64, qcd.ALL, 0.1, a, a, None) == qcd.EALIAS
    assert L.qcd_force_mom_update(h, qcd.F64, qcd.ALL, 5.0, 0.1, a, a + 16, None) == qcd.EALIAS
    assert L.qcd_link_update(h, qcd.F32, qcd.EVEN, 0.1, a, a, 1, None) == qcd.EALIAS
    assert L.qcd_reunit(h, qcd.F64, qcd.ALL, None, None) == qcd.EINVAL
    assert L.qcd_mom_refresh(h, qcd.F64, 5, 1, 0, a, None) == qcd.EINVAL
    assert L.qcd_plaquette(h, qcd.F64, a, None, None, b, None) == qcd.EINVAL
    assert L.qcd_sum(h, qcd.F64, qcd.ALL, 9, 72, a, b, b, None) == qcd.EINVAL
    assert L.qcd_sum(h, qcd.F64, qcd.ALL, qcd.SUM_NORM2, 70, a, b, b, None) == qcd.EINVAL
    assert L.qcd_sum(h, qcd.F64, qcd.ALL, qcd.SUM_SCALAR, 65, a, b, b, None) == qcd.EINVAL
    assert L.qcd_sum_multi(h, qcd.F64, qcd.SUM_SCALAR, 1, a, None, 5, b, b, None) == qcd.EINVAL  # nsub != Lt
    assert L.qcd_sum_multi(h, qcd.F64, qcd.SUM_SCALAR, 1, a, b, 0, b, b, None) == qcd.EINVAL
    assert L.qcd_sum_multi(h, qcd.F64, qcd.SUM_SCALAR, 1, a, b, 5000, b, b, None) == qcd.EINVAL
    assert L.qcd_leapfrog(h, qcd.F64, 5.0, 0.1, 0, a, b, None) == qcd.EINVAL
    assert L.qcd_get_map(h, 12, a, None) == qcd.EINVAL
    assert L.qcd_pack(h, qcd.F64, 72, qcd.LAYOUT_PAIRS, a, a, None) == qcd.EALIAS
    assert L.qcd_md_host(h, qcd.F64, 5.0, 0.1, 1, None, a, b, None) == qcd.EINVAL


def test_multi_step_integrators_refuse_slab_lattices_and_views(qcd):
    """several link updates in one call cannot refresh halos in between: QCD_EINVAL before anything is enqueued"""
    L = qcd.lib
    full = qcd.Lattice((4, 4, 4, 8))
    slab = qcd.Lattice((4, 4, 4, 8), slab=(2, 4))
    view = full.view_t(2, 6)
    fb = full.field_bytes(qcd.F64)
    a, b, c, o = 0x10000000, 0x10000000 + 2 * fb, 0x10000000 + 4 * fb, 0x10000000 + 6 * fb
    two = (C.c_double * 2)(5.0, 1.0)
    for lat in (slab, view):
        h = lat.handle
        assert L.qcd_leapfrog(h, qcd.F64, 5.0, 0.1, 2, a, b, None) == qcd.EINVAL
        assert b"whole lattice" in L.qcd_last_error()
        assert L.qcd_leapfrog(h, qcd.F64, 5.0, 0.1, 1, a, b, None) == qcd.EINVAL
        assert L.qcd_leapfrog_energy(h, qcd.F64, 5.0, 0.1, 2, a, b, o, o, None) == qcd.EINVAL
        assert L.qcd_leapfrog_single_pass(h, qcd.F64, 5.0, 0.1, 2, a, b, c, None) == qcd.EINVAL
        assert L.qcd_trajectory(h, qcd.F64, 5.0, 0.1, 2, a, b, c, o, None, o, 1 << 30, None) == qcd.EINVAL
        assert L.qcd_nested_leapfrog(h, qcd.F64, C.byref(two), C.byref(two), 1.0, 2, 2, a, b, None) == qcd.EINVAL
        assert L.qcd_md_host(h, qcd.F64, 5.0, 0.1, 1, a, b, c, None) == qcd.EINVAL
    # a view that spans every timeslice is the whole lattice again: the call gets past this check (and fails the next)
    assert L.qcd_leapfrog(full.view_t(0, 8).handle, qcd.F64, 5.0, 0.1, 2, a, a, None) == qcd.EALIAS


def test_product_path_does_not_import_the_oracle():
    """the CUDA package must not reference oracle/ (and the oracle must not reference the package)"""
    pkg = os.path.join(ROOT, "paper_1212_0785_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower().replace("no cpu fallback", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1212_0785_b200" not in text and "from paper_1212_0785_b200" not in text
            assert "csrc/" not in text or "shares no code" in text


def test_tuning_database_roundtrip_and_validation():
    """qcd_tune_set / qcd_tune_get / qcd_tune_clear are host-only (the N_t database)"""
    from paper_1212_0785_b200 import binding as qcd
    qcd.qcd_tune_clear()
    lat, other = qcd.Lattice((8, 8, 8, 16)), qcd.Lattice((8, 8, 8, 4))
    assert qcd.qcd_tune_get(lat, qcd.F64, qcd.ALL, qcd.KERNEL_FORCE) is None
    qcd.qcd_tune_set(lat, qcd.F64, qcd.ALL, qcd.KERNEL_FORCE, qcd.FORCE_VARIANTS.index("plane"), (8, 4, 2, 2))
    qcd.qcd_tune_set(lat, qcd.F64, qcd.EVEN, qcd.KERNEL_LINK_UPDATE, threads=64)
    assert qcd.qcd_tune_get(lat, qcd.F64, qcd.ALL, qcd.KERNEL_FORCE) == (1, (8, 4, 2, 2), 0)
    assert qcd.qcd_tune_get(lat, qcd.F64, qcd.ODD, qcd.KERNEL_LINK_UPDATE) == (0, (0, 0, 0, 0), 64)  # EVEN/ODD share
    assert qcd.qcd_tune_get(lat, qcd.F32, qcd.ALL, qcd.KERNEL_FORCE) is None  # keyed on precision
    assert qcd.qcd_tune_get(other, qcd.F64, qcd.ALL, qcd.KERNEL_FORCE) is None  # and on the extents
    qcd.qcd_tune_set(lat, qcd.F64, qcd.ALL, qcd.KERNEL_FORCE, 0, None)  # overwrite: library's own tile
    assert qcd.qcd_tune_get(lat, qcd.F64, qcd.ALL, qcd.KERNEL_FORCE) == (0, (0, 0, 0, 0), 0)
    for bad in [dict(kernel=qcd.KERNEL_FORCE, variant=9), dict(kernel=qcd.KERNEL_FORCE, variant=0, tile=(3, 2, 2, 2)),
                dict(kernel=qcd.KERNEL_FORCE, variant=0, tile=(8, 8, 8, 2)),  # 1024 sites > 128-thread block
                dict(kernel=qcd.KERNEL_FORCE, variant=0, tile=(8, 4, 4, 4)),  # 512 sites = 256 per parity > 128
                dict(kernel=qcd.KERNEL_FORCE, variant=0, tile=(5, 2, 2, 2)), dict(kernel=qcd.KERNEL_MOM_UPDATE, threads=48),
                dict(kernel=qcd.KERNEL_LINK_UPDATE, threads=512), dict(kernel=7, threads=64)]:
        with pytest.raises(qcd.QcdError) as e:
            qcd.qcd_tune_set(lat, qcd.F64, qcd.ALL, **bad)
        assert e.value.code == qcd.EINVAL
    qcd.qcd_tune_clear()
    assert qcd.qcd_tune_get(lat, qcd.F64, qcd.EVEN, qcd.KERNEL_LINK_UPDATE) is None
