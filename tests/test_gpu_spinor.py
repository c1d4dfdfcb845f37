"""GPU parity for SURVEY.md 8(f)-4: Gaussian spin-colour fill (O15) and inner products (O16) through the C
ABI against the oracle.  The generator output is compared at fp64 round-off (the integer words are pinned
bit-exact in test_gpu_parity.py); reductions within the north_star tolerances."""
import numpy as np
import pytest

from oracle import oracle as O
from tests.test_gpu_parity import TOL, round_to, tdtype

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qcd():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1212_0785_b200 import binding
    return binding


def spinor_to_device(qcd, lat, a, prec):
    import torch
    t = torch.view_as_real(torch.from_numpy(np.ascontiguousarray(a))).reshape(-1).to(tdtype(prec)).cuda()
    out = lat.new_pair_field(a.shape[1], tdtype(prec))
    qcd.qcd_pack(lat, 2 * a.shape[1], qcd.LAYOUT_PAIRS, t, out)
    return out


def spinor_to_host(qcd, lat, d):
    import torch
    nc = d.shape[1]
    t = torch.empty(lat.V * nc * 2, dtype=d.dtype, device="cuda")
    qcd.qcd_unpack(lat, 2 * nc, qcd.LAYOUT_PAIRS, d, t)
    return t.to(torch.float64).cpu().numpy().view("complex128").reshape(lat.V, nc)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (6, 4, 2, 8), (4, 10, 6, 2), (16, 16, 16, 8)])
def test_spinor_gaussian(qcd, orc_omp, prec, dims):
    lat = qcd.Lattice(dims)
    seed = 0x1212078500000007
    ref = orc_omp.spinor_gaussian(dims, seed, stream_id=3)
    eta = lat.new_spinor_field(tdtype(prec))
    qcd.qcd_spinor_gaussian(lat, eta, seed, stream_id=3)
    got = spinor_to_host(qcd, lat, eta)
    tol = 1e-14 if prec == "f64" else 1e-7
    assert np.abs(got - ref).max() < tol * np.abs(ref).max()
    # subsets write only their sites
    par = orc_omp.map(dims, O.MAP_PARITY)
    for subset, p in ((qcd.EVEN, 0), (qcd.ODD, 1)):
        eta.fill_(7.0)
        qcd.qcd_spinor_gaussian(lat, eta, seed, stream_id=3, subset=subset)
        g = spinor_to_host(qcd, lat, eta)
        assert np.abs(g[par == p] - ref[par == p]).max() < tol * np.abs(ref).max()
        assert np.all(g[par != p] == 7.0 + 7.0j)
    # layout: component k of checkerboard site cb at [cb >> 5][k][cb & 31]
    cb = orc_omp.map(dims, O.MAP_CB_OF_LEX)
    qcd.qcd_spinor_gaussian(lat, eta, seed, stream_id=3)
    raw = lat.by_component(eta).to("cpu").numpy().astype(np.float64)
    assert np.abs(raw[5, cb, 0] - ref[:, 5].real).max() < tol * 5 and np.abs(raw[11, cb, 1] - ref[:, 11].imag).max() < tol * 5


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (6, 4, 2, 8), (16, 16, 16, 32)])
def test_inner_product_and_norm(qcd, orc_omp, prec, dims):
    import torch
    lat = qcd.Lattice(dims)
    V = lat.V
    rng = np.random.default_rng(11)
    a = round_to(prec, rng.standard_normal((V, 12)) + 1j * rng.standard_normal((V, 12)))
    b = round_to(prec, rng.standard_normal((V, 12)) + 1j * rng.standard_normal((V, 12)))
    da, db = spinor_to_device(qcd, lat, a, prec), spinor_to_device(qcd, lat, b, prec)
    ws = lat.new_workspace()
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    scale = np.sqrt(np.vdot(a, a).real * np.vdot(b, b).real)  # |<a,b>| <= |a||b|: the natural size for the tolerance
    for subset in (qcd.ALL, qcd.EVEN, qcd.ODD):
        qcd.qcd_inner_product(lat, 12, da, db, out, ws, subset=subset)
        got = complex(*out.cpu().numpy())
        assert abs(got - orc_omp.inner_product(dims, a, b, subset=subset)) < TOL[prec] * scale
    per_t = torch.zeros((dims[3], 2), dtype=torch.float64, device="cuda")
    qcd.qcd_inner_product_multi(lat, 12, da, db, per_t, ws)
    g = per_t.cpu().numpy()
    assert np.abs((g[:, 0] + 1j * g[:, 1]) - orc_omp.inner_product_multi(dims, a, b)).max() < TOL[prec] * scale
    # <a,a> is the norm: real, equal to qcd_sum(NORM2) on the 24-real field, deterministic
    qcd.qcd_inner_product(lat, 12, da, da, out, ws)
    n2 = torch.zeros(1, dtype=torch.float64, device="cuda")
    qcd.qcd_sum(lat, qcd.SUM_NORM2, 24, da, n2, ws)
    ref = orc_omp.sum(dims, O.SUM_NORM2, a.view(np.float64).reshape(V, 24))
    assert out[1].item() == 0.0 and abs(out[0].item() - ref) < TOL[prec] * ref and abs(n2.item() - ref) < TOL[prec] * ref
    again = torch.zeros(2, dtype=torch.float64, device="cuda")
    qcd.qcd_inner_product(lat, 12, da, db, out, ws)
    qcd.qcd_inner_product(lat, 12, da, db, again, ws)
    assert torch.equal(out, again)


def test_inner_product_on_matrix_fields_and_arguments(qcd, orc_omp):
    """nc = 36: <P, F> of two momentum-like fields, as used for energy-conservation diagnostics"""
    import torch
    from tests.test_gpu_parity import dev
    dims = (4, 4, 4, 8)
    lat = qcd.Lattice(dims)
    A, B = orc_omp.mom_refresh(dims, 1), orc_omp.mom_refresh(dims, 2)
    dA, dB = dev(qcd, lat, A, "f64"), dev(qcd, lat, B, "f64")
    ws = lat.new_workspace()
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    qcd.qcd_inner_product(lat, 36, dA, dB, out, ws)
    ref = np.vdot(A, B)
    assert abs(complex(*out.cpu().numpy()) - ref) < 1e-12 * np.sqrt(np.vdot(A, A).real * np.vdot(B, B).real)
    with pytest.raises(qcd.QcdError):
        qcd.qcd_inner_product(lat, 0, dA, dB, out, ws)
    with pytest.raises(qcd.QcdError):
        qcd.qcd_sum(lat, qcd.SUM_NORM2, 20, dA, out, ws)  # not a complex-pair field size
