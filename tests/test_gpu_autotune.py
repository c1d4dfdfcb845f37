"""the auto-tuner.  Launch parameters taken from the database must not
change results beyond rounding; the tuner must measure, pick, persist and reload."""
import json

import numpy as np
import pytest

from tests import inputs
from tests.test_gpu_parity import dev, host, rel

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qcd():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1212_0785_b200 import binding
    return binding


def test_database_entries_drive_the_launch_and_keep_parity(qcd, orc_omp):
    dims = (8, 8, 8, 16)
    lat = qcd.Lattice(dims)
    beta, eps = 5.8, 0.05
    U = orc_omp.hot_start(dims, inputs.config_seed(2), 0.5)
    P = orc_omp.mom_refresh(dims, inputs.config_seed(2))
    P1 = orc_omp.mom_update(dims, eps, orc_omp.gauge_force(dims, beta, U), P)
    U1 = orc_omp.link_update(dims, eps, P1, U, reunit=True)
    try:
        for variant, tile, nt in [("staple", (8, 4, 2, 2), 32), ("staple", None, 96), ("plane", (4, 4, 4, 2), 256),
                                  ("plane", (8, 2, 2, 2), 160), ("plane", None, 64), ("plane", (8, 8, 2, 1), 224)]:
            qcd.qcd_tune_set(lat, qcd.F64, qcd.ALL, qcd.KERNEL_FORCE, qcd.FORCE_VARIANTS.index(variant), tile)
            qcd.qcd_tune_set(lat, qcd.F64, qcd.ALL, qcd.KERNEL_LINK_UPDATE, threads=nt)
            qcd.qcd_tune_set(lat, qcd.F64, qcd.ALL, qcd.KERNEL_MOM_UPDATE, threads=nt)
            dU, dP = dev(qcd, lat, U, "f64"), dev(qcd, lat, P, "f64")
            qcd.qcd_md_step(lat, dU, dP, beta, eps, eps)
            assert rel(host(qcd, lat, dP), P1) < 1e-12, variant
            assert rel(host(qcd, lat, dU), U1) < 1e-12, variant
            F = lat.new_matrix_field()
            qcd.qcd_gauge_force(lat, dev(qcd, lat, U, "f64"), F, beta)
            dP = dev(qcd, lat, P, "f64")
            qcd.qcd_mom_update(lat, F, dP, eps)
            assert rel(host(qcd, lat, dP), P1) < 1e-12, variant
    finally:
        qcd.qcd_tune_clear()


def test_autotune_measures_picks_persists_and_reloads(qcd, tmp_path):
    import torch
    from paper_1212_0785_b200 import autotune
    dims = (8, 8, 8, 8)
    try:
        entries = autotune.tune(dims, torch.float64, reps=3, verbose=False)
        assert [e["kernel"] for e in entries] == ["force", "link_update", "mom_update"]
        for e in entries:
            assert len(e["candidates"]) >= 4 and all(c["ms"] > 0 for c in e["candidates"])
            assert e["best"]["ms"] == min(c["ms"] for c in e["candidates"])
        lat = qcd.Lattice(dims)
        b = entries[0]["best"]
        want = (qcd.FORCE_VARIANTS.index(b["variant"]), tuple(b["tile"]), 0)
        assert qcd.qcd_tune_get(lat, qcd.F64, qcd.ALL, qcd.KERNEL_FORCE) == want
        path = str(tmp_path / "tune.json")
        autotune.save(entries, path)
        autotune.write_csv(entries, str(tmp_path / "tune.csv"))
        assert "B200" in json.load(open(path))["device"] or json.load(open(path))["device"]
        qcd.qcd_tune_clear()
        assert qcd.qcd_tune_get(lat, qcd.F64, qcd.ALL, qcd.KERNEL_FORCE) is None
        assert autotune.load(path) == 3
        assert qcd.qcd_tune_get(lat, qcd.F64, qcd.ALL, qcd.KERNEL_FORCE) == want
        assert qcd.qcd_tune_get(lat, qcd.F64, qcd.ALL, qcd.KERNEL_LINK_UPDATE)[2] == entries[1]["best"]["threads"]
    finally:
        qcd.qcd_tune_clear()
