"""GPU parity for SURVEY.md 8(f)-1: anisotropic Wilson force, space-space / space-time plaquette and the
two-level leapfrog, through the C ABI against the oracle (O13, O14).  Tolerances as in test_gpu_parity.py."""
import numpy as np
import pytest

from tests import inputs
from tests.test_gpu_parity import TOL, dev, host, rel, round_to, tdtype

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qcd():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1212_0785_b200 import binding
    return binding


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (6, 4, 2, 8), (12, 6, 10, 4), (16, 16, 16, 32)])
def test_aniso_force_all_subsets_and_fused(qcd, orc_omp, prec, dims):
    lat = qcd.Lattice(dims)
    U = round_to(prec, orc_omp.hot_start(dims, 51, 0.5))
    P = round_to(prec, orc_omp.mom_refresh(dims, 52))
    dU = dev(qcd, lat, U, prec)
    for bs, bt in [(2.5, 8.0), (6.0, 0.0), (0.0, 4.5)]:  # generic, space-space only, space-time only
        Fr = orc_omp.gauge_force_aniso(dims, bs, bt, U)
        for subset in (qcd.ALL, qcd.EVEN, qcd.ODD):
            F = lat.new_matrix_field(tdtype(prec))
            F.zero_()
            qcd.qcd_gauge_force_aniso(lat, dU, F, bs, bt, subset=subset)
            ref = Fr if subset == qcd.ALL else orc_omp.gauge_force_aniso(dims, bs, bt, U, subset=subset)
            assert rel(host(qcd, lat, F), ref) < TOL[prec] or np.abs(ref).max() == 0
            assert np.abs(host(qcd, lat, F) - ref).max() <= TOL[prec] * max(np.abs(Fr).max(), 1e-300)
        dP = dev(qcd, lat, P, prec)
        qcd.qcd_force_mom_update_aniso(lat, dU, dP, bs, bt, 0.07)
        assert rel(host(qcd, lat, dP), P + 0.07 * Fr) < TOL[prec]
    # the isotropic limit is the isotropic kernel's answer
    F1, F2 = lat.new_matrix_field(tdtype(prec)), lat.new_matrix_field(tdtype(prec))
    qcd.qcd_gauge_force_aniso(lat, dU, F1, 5.7, 5.7)
    qcd.qcd_gauge_force(lat, dU, F2, 5.7)
    assert rel(host(qcd, lat, F1), host(qcd, lat, F2)) < TOL[prec]


def test_aniso_force_generic_matrices(qcd, orc):
    dims = (4, 6, 2, 4)
    lat = qcd.Lattice(dims)
    U = inputs.random_matrix_field(61, lat.V)  # not unitary: the formula, not the group, is checked
    F = lat.new_matrix_field()
    qcd.qcd_gauge_force_aniso(lat, dev(qcd, lat, U, "f64"), F, 1.7, 3.3)
    assert rel(host(qcd, lat, F), orc.gauge_force_aniso(dims, 1.7, 3.3, U)) < 1e-12


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (6, 4, 2, 8), (16, 16, 16, 32)])
def test_plaquette_st(qcd, orc_omp, prec, dims):
    import torch
    lat = qcd.Lattice(dims)
    U = round_to(prec, orc_omp.hot_start(dims, 71, 0.5))
    dU = dev(qcd, lat, U, prec)
    ws = lat.new_workspace()
    avg = torch.zeros(2, dtype=torch.float64, device="cuda")
    per_t = torch.zeros((dims[3], 2), dtype=torch.float64, device="cuda")
    qcd.qcd_plaquette_st(lat, dU, avg, per_t, ws)
    ravg, rper_t = orc_omp.plaquette_st(dims, U)
    assert rel(avg.cpu().numpy(), ravg) < TOL[prec] and rel(per_t.cpu().numpy(), rper_t) < TOL[prec]
    qcd.qcd_plaquette_st(lat, dU, avg, None, ws)  # per-timeslice output is optional
    assert rel(avg.cpu().numpy(), ravg) < TOL[prec]
    iso = torch.zeros(1, dtype=torch.float64, device="cuda")
    qcd.qcd_plaquette(lat, dU, iso, None, ws)
    assert abs(avg.mean().item() - iso.item()) < (1e-13 if prec == "f64" else 1e-6)


@pytest.mark.parametrize("prec,n_outer,n_inner", [("f64", 1, 1), ("f64", 3, 2), ("f64", 2, 5), ("f32", 2, 3)])
def test_nested_leapfrog_matches_oracle_and_reverses(qcd, orc_omp, prec, n_outer, n_inner):
    dims = (8, 8, 8, 16)
    lat = qcd.Lattice(dims)
    bs, bt = (0.0, 2.9), (8.7, 0.0)  # inner level: space-time planes; outer level: space-space planes
    tau = 0.25
    U = round_to(prec, orc_omp.hot_start(dims, inputs.config_seed(2), 0.5))
    P = round_to(prec, orc_omp.mom_refresh(dims, inputs.config_seed(2)))
    dU, dP = dev(qcd, lat, U, prec), dev(qcd, lat, P, prec)
    qcd.qcd_nested_leapfrog(lat, dU, dP, bs, bt, tau, n_outer, n_inner)
    U1, P1 = orc_omp.nested_leapfrog(dims, bs, bt, tau, n_outer, n_inner, U, P)
    assert rel(host(qcd, lat, dU), U1) < TOL[prec] and rel(host(qcd, lat, dP), P1) < TOL[prec]
    if prec == "f64":
        dP.mul_(-1.0)
        qcd.qcd_nested_leapfrog(lat, dU, dP, bs, bt, tau, n_outer, n_inner)
        dP.mul_(-1.0)
        assert rel(host(qcd, lat, dU), U) < 1e-12 and rel(host(qcd, lat, dP), P) < 1e-12


def test_nested_leapfrog_general_split_and_energy(qcd, orc_omp):
    """both levels carry both plane classes; dH from the GPU's own observables matches the oracle's"""
    import torch
    dims = (4, 4, 4, 8)
    lat = qcd.Lattice(dims)
    bs, bt = (1.0, 2.0), (5.0, 1.5)
    U = orc_omp.hot_start(dims, 81, 0.4)
    P = orc_omp.mom_refresh(dims, 82)
    dU, dP = dev(qcd, lat, U, "f64"), dev(qcd, lat, P, "f64")
    ws = lat.new_workspace()

    def H():
        o = torch.zeros(3, dtype=torch.float64, device="cuda")
        qcd.qcd_sum(lat, qcd.SUM_NORM2, 72, dP, o[0:1], ws)
        qcd.qcd_plaquette_st(lat, dU, o[1:3], None, ws)
        K, ps, pt = o.cpu().numpy()
        return K + 3 * lat.V * (sum(bs) * (1 - ps) + sum(bt) * (1 - pt))

    H0 = H()
    qcd.qcd_nested_leapfrog(lat, dU, dP, bs, bt, 0.2, 4, 3)
    H1 = H()
    U1, P1 = orc_omp.nested_leapfrog(dims, bs, bt, 0.2, 4, 3, U, P)
    assert rel(host(qcd, lat, dU), U1) < 1e-12 and rel(host(qcd, lat, dP), P1) < 1e-12
    r0 = float(np.sum(np.abs(P) ** 2)) + orc_omp.action_aniso(dims, sum(bs), sum(bt), U)
    r1 = float(np.sum(np.abs(P1) ** 2)) + orc_omp.action_aniso(dims, sum(bs), sum(bt), U1)
    assert abs((H1 - H0) - (r1 - r0)) <= 1e-12 * abs(r0)
    with pytest.raises(qcd.QcdError):
        qcd.qcd_nested_leapfrog(lat, dU, dP, bs, bt, 0.2, 0, 3)
