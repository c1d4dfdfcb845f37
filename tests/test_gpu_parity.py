"""GPU parity: the CUDA path (through the C ABI of include/qcd.h) against the CPU oracle, element by
element on the same seeded inputs.

Tolerances (BASELINE.json north_star; norm per DESIGN.md R15): fields max|gpu-ref| / max|ref| <= 1e-12 in
fp64 and 2e-5 in fp32; scalars |d|/|ref|; integer maps and RNG words bit-exact.  fp32 runs feed the
fp64 oracle the fp32-rounded inputs (R14).
"""
import numpy as np
import pytest

from oracle import oracle as O
from tests import inputs

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}


@pytest.fixture(scope="module")
def qcd():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1212_0785_b200 import binding
    return binding


def tdtype(prec):
    import torch
    return torch.float64 if prec == "f64" else torch.float32


def rel(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def round_to(prec, a):
    """inputs as the GPU sees them: fp32-rounded for the fp32 path"""
    if prec == "f64":
        return a
    return a.astype(np.complex64).astype(np.complex128) if np.iscomplexobj(a) else a.astype(np.float32).astype(np.float64)


def dev(qcd, lat, a, prec):
    return qcd.field_to_device(lat, a, tdtype(prec))


def host(qcd, lat, t):
    return qcd.field_to_host(lat, t)


def sync():
    import torch
    torch.cuda.synchronize()


DIMS_SMALL = [(2, 2, 2, 2), (4, 4, 4, 4), (6, 4, 2, 8), (4, 10, 6, 2), (8, 8, 8, 16)]


# ------------------------------------------------------------------ integer work: bit-exact

@pytest.mark.parametrize("dims", DIMS_SMALL + [(16, 16, 16, 32), (12, 6, 10, 4)])
def test_maps_bit_exact(qcd, orc, dims):
    import torch
    lat = qcd.Lattice(dims)
    out = torch.empty(lat.V, dtype=torch.int32, device="cuda")
    for which in range(12):
        out.fill_(-1)
        qcd.qcd_get_map(lat, which, out)
        assert np.array_equal(out.cpu().numpy(), orc.map(dims, which)), which


def test_rng_words_and_uniforms_bit_exact(qcd, orc):
    import torch
    n = 4096
    rng = np.random.default_rng(7)
    site = rng.integers(0, 2 ** 31 - 1, n, dtype=np.int64).astype(np.uint32)
    site[:4] = [0, 1, 0xFFFFFFFF, 10616831]
    mu_j = rng.integers(0, 64, n).astype(np.uint32)
    seed, stream_id, purpose = 0x1212078500000003, 5, 1
    d_site = torch.from_numpy(site.view(np.int32)).cuda()
    d_muj = torch.from_numpy(mu_j.view(np.int32)).cuda()
    words = torch.empty(4 * n, dtype=torch.int32, device="cuda")
    uni = torch.empty(2 * n, dtype=torch.float64, device="cuda")
    gau = torch.empty(2 * n, dtype=torch.float64, device="cuda")
    qcd.qcd_rng_blocks(seed, stream_id, purpose, d_site, d_muj, words, uni, gau)
    w = words.cpu().numpy().view(np.uint32).reshape(n, 4)
    u = uni.cpu().numpy().reshape(n, 2)
    g = gau.cpu().numpy().reshape(n, 2)
    for i in range(n):
        rw, ru, rg = orc.rng_block(seed, int(site[i]), int(mu_j[i]) // 16, int(mu_j[i]) % 16, stream_id, purpose)
        assert list(w[i]) == rw
        assert u[i, 0] == ru[0] and u[i, 1] == ru[1]  # exact dyadic uniforms
        assert np.abs(g[i] - rg).max() < 1e-14 * max(1.0, np.abs(rg).max())
    # empty request is a no-op
    e = torch.empty(0, dtype=torch.int32, device="cuda")
    qcd.qcd_rng_blocks(seed, 0, 0, e, e)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(4, 6, 2, 4), (2, 2, 2, 2), (4, 10, 6, 2), (16, 8, 8, 6)])
def test_pack_unpack_layout(qcd, orc, prec, dims):
    """bit-exact; V = 192, 16, 480, 6144: whole 64-site chunks of the transposing kernel and ragged tails"""
    import torch
    lat = qcd.Lattice(dims)
    V = lat.V
    A = round_to(prec, inputs.random_matrix_field(3, V))
    d = dev(qcd, lat, A, prec)
    assert np.array_equal(host(qcd, lat, d), A)  # round trip is exact
    # documented layout: pair k = mu*9+e of site cb at [cb >> 5][k][cb & 31] (chunks of 32 checkerboard sites)
    assert tuple(d.shape) == ((V + 31) // 32, 36, 32, 2) and d.numel() * d.element_size() == lat.field_bytes(
        qcd.F64 if prec == "f64" else qcd.F32)
    raw4 = d.cpu().numpy().astype(np.float64)
    cb = orc.map(dims, O.MAP_CB_OF_LEX)
    k_probe, s_probe = 17, V - 1  # one element by the index formula itself
    assert raw4[cb[s_probe] >> 5, k_probe, cb[s_probe] & 31, 0] == A.reshape(V, 36)[s_probe, k_probe].real
    raw = lat.by_component(d).cpu().numpy().astype(np.float64)  # [36][V][2] by checkerboard index
    ref = np.empty((36, V, 2))
    flat = A.reshape(V, 36)
    ref[:, cb, 0] = flat.real.T
    ref[:, cb, 1] = flat.imag.T
    assert np.array_equal(raw, ref)
    # real-field layout [comp][cb]
    R = round_to(prec, inputs.random_real_field(4, V, 3))
    src = torch.from_numpy(R).to(tdtype(prec)).cuda().reshape(-1)
    dst = lat.new_real_field(3, tdtype(prec))
    qcd.qcd_pack(lat, 3, qcd.LAYOUT_REAL, src, dst)
    got = lat.by_component(dst).cpu().numpy().astype(np.float64)
    assert np.array_equal(got[:, cb], R.T)
    back = torch.empty_like(src)
    qcd.qcd_unpack(lat, 3, qcd.LAYOUT_REAL, dst, back)
    assert torch.equal(back, src)
    # many components per site: the direct (non-transposing) kernel
    R = round_to(prec, inputs.random_real_field(5, V, 100))
    src = torch.from_numpy(R).to(tdtype(prec)).cuda().reshape(-1)
    dst = lat.new_real_field(100, tdtype(prec))
    qcd.qcd_pack(lat, 100, qcd.LAYOUT_REAL, src, dst)
    assert np.array_equal(lat.by_component(dst).cpu().numpy().astype(np.float64)[:, cb], R.T)
    back = torch.empty_like(src)
    qcd.qcd_unpack(lat, 100, qcd.LAYOUT_REAL, dst, back)
    assert torch.equal(back, src)


# ------------------------------------------------------------------ generators

@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 8), (16, 16, 16, 8), (16, 16, 16, 32)])
def test_mom_refresh_and_hot_start(qcd, orc_omp, prec, dims):
    lat = qcd.Lattice(dims)
    seed = inputs.config_seed(3)
    tol = TOL[prec] if prec == "f64" else 2e-7  # fp32: fp64 Gaussians rounded once
    P = lat.new_matrix_field(tdtype(prec))
    qcd.qcd_mom_refresh(lat, P, seed, stream_id=2)
    ref = orc_omp.mom_refresh(dims, seed, stream_id=2)
    assert rel(host(qcd, lat, P), ref) < tol
    par = orc_omp.map(dims, O.MAP_PARITY)
    for subset, keep in ((qcd.EVEN, 1), (qcd.ODD, 0)):
        P.fill_(7.0)
        qcd.qcd_mom_refresh(lat, P, seed, stream_id=2, subset=subset)
        got = host(qcd, lat, P)
        assert np.all(got[par == keep] == 7.0 + 7.0j)  # other parity untouched, bit-identical
        assert rel(got[par != keep], ref[par != keep]) < tol
    U = lat.new_matrix_field(tdtype(prec))
    for sigma in (0.2, 0.5, 3.0):
        qcd.qcd_hot_start(lat, U, seed, sigma)
        assert rel(host(qcd, lat, U), orc_omp.hot_start(dims, seed, sigma)) < tol


# ------------------------------------------------------------------ plaquette, sums

@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", DIMS_SMALL + [(16, 16, 16, 32)])
def test_plaquette(qcd, orc_omp, prec, dims):
    import torch
    lat = qcd.Lattice(dims)
    U = round_to(prec, orc_omp.hot_start(dims, inputs.config_seed(3), 0.5))
    dU = dev(qcd, lat, U, prec)
    ws = lat.new_workspace()
    avg = torch.zeros(1, dtype=torch.float64, device="cuda")
    per_t = torch.zeros(dims[3], dtype=torch.float64, device="cuda")
    qcd.qcd_plaquette(lat, dU, avg, per_t, ws)
    ravg, rper_t = orc_omp.plaquette(dims, U)
    tol = TOL[prec]
    assert abs(avg.item() - ravg) / abs(ravg) < tol
    assert rel(per_t.cpu().numpy(), rper_t) < tol
    assert abs(per_t.mean().item() - avg.item()) < 1e-14
    # deterministic: bit-identical on a second run, and without the per-timeslice output
    avg2 = torch.zeros(1, dtype=torch.float64, device="cuda")
    qcd.qcd_plaquette(lat, dU, avg2, None, ws)
    assert avg2.item() == avg.item()
    # generic (non-unitary) matrices exercise every entry of the products
    G = round_to(prec, inputs.random_matrix_field(5, lat.V) * 0.7)
    qcd.qcd_plaquette(lat, dev(qcd, lat, G, prec), avg, per_t, ws)
    gavg, gper_t = orc_omp.plaquette(dims, G)
    scale = np.abs(gper_t).max()
    assert np.abs(per_t.cpu().numpy() - gper_t).max() / scale < tol
    assert abs(avg.item() - gavg) / scale < tol


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 6, 2, 8), (16, 16, 16, 32)])
def test_sum_and_sum_multi(qcd, orc, prec, dims):
    import torch
    lat = qcd.Lattice(dims)
    V, Lt = lat.V, dims[3]
    ws = lat.new_workspace()
    tol = 1e-12 if prec == "f64" else 1e-6  # inputs identical (rounded), accumulation always fp64
    cb = orc.map(dims, O.MAP_CB_OF_LEX)
    # matrix kinds on a momentum-like field
    M = round_to(prec, inputs.random_matrix_field(11, V))
    dM = dev(qcd, lat, M, prec)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    for kind, okind in ((qcd.SUM_NORM2, O.SUM_NORM2), (qcd.SUM_RETR, O.SUM_RETR)):
        scale = np.sum(np.abs(M) ** 2) if kind == qcd.SUM_NORM2 else np.abs(np.trace(M, axis1=-2, axis2=-1).real).sum()
        for subset in (qcd.ALL, qcd.EVEN, qcd.ODD):
            qcd.qcd_sum(lat, kind, 72, dM, out, ws, subset=subset)
            assert abs(out.item() - orc.sum(dims, okind, M, subset=subset)[0]) / scale < tol, (kind, subset)
        outt = torch.zeros(Lt, dtype=torch.float64, device="cuda")
        qcd.qcd_sum_multi(lat, kind, 72, dM, None, Lt, outt, ws)
        assert np.abs(outt.cpu().numpy() - orc.sum_multi(dims, okind, M)).max() / scale < tol
        nsub = 7
        ids = inputs.random_subset_ids(5, V, nsub)
        ids[::11] = -1  # sites in no subset
        ids_cb = np.empty_like(ids)
        ids_cb[cb] = ids
        outs = torch.zeros(nsub, dtype=torch.float64, device="cuda")
        qcd.qcd_sum_multi(lat, kind, 72, dM, torch.from_numpy(ids_cb).cuda(), nsub, outs, ws)
        assert np.abs(outs.cpu().numpy() - orc.sum_multi(dims, okind, M, subset_id=ids, nsub=nsub)).max() / scale < tol
    # scalar kind, 3 components, closed forms included
    R = inputs.random_real_field(13, V, 3)
    R[:, 1] = orc.map(dims, O.MAP_TSLICE)
    R[:, 2] = 1 - 2 * orc.map(dims, O.MAP_PARITY)
    R = round_to(prec, R)
    dR = lat.new_real_field(3, tdtype(prec))
    qcd.qcd_pack(lat, 3, qcd.LAYOUT_REAL, torch.from_numpy(R).to(tdtype(prec)).cuda().reshape(-1), dR)
    out3 = torch.zeros(3, dtype=torch.float64, device="cuda")
    for subset in (qcd.ALL, qcd.EVEN, qcd.ODD):
        qcd.qcd_sum(lat, qcd.SUM_SCALAR, 3, dR, out3, ws, subset=subset)
        ref = orc.sum(dims, O.SUM_SCALAR, R, subset=subset)
        got = out3.cpu().numpy()
        assert abs(got[0] - ref[0]) < tol * np.abs(R[:, 0]).sum()
        assert got[1] == ref[1] and got[2] == ref[2]  # integer-valued sums are exact
    assert out3[2].item() == -V / 2
    outm = torch.zeros(Lt * 3, dtype=torch.float64, device="cuda")
    qcd.qcd_sum_multi(lat, qcd.SUM_SCALAR, 3, dR, None, Lt, outm, ws)
    refm = orc.sum_multi(dims, O.SUM_SCALAR, R)
    got = outm.cpu().numpy().reshape(Lt, 3)
    assert np.abs(got[:, 0] - refm[:, 0]).max() < tol * np.abs(R[:, 0]).sum()
    assert np.array_equal(got[:, 1:], refm[:, 1:])


# ------------------------------------------------------------------ force, momentum update

@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", DIMS_SMALL + [(16, 16, 16, 32), (12, 6, 10, 4)])
def test_gauge_force_all_subsets(qcd, orc_omp, prec, dims):
    lat = qcd.Lattice(dims)
    beta = 5.8
    U = round_to(prec, orc_omp.hot_start(dims, inputs.config_seed(3), 0.5))
    dU = dev(qcd, lat, U, prec)
    ref = orc_omp.gauge_force(dims, beta, U)
    par = orc_omp.map(dims, O.MAP_PARITY)
    F = lat.new_matrix_field(tdtype(prec))
    qcd.qcd_gauge_force(lat, dU, F, beta)
    got = host(qcd, lat, F)
    assert rel(got, ref) < TOL[prec]
    assert np.abs(got - np.conj(np.swapaxes(got, -1, -2))).max() == 0  # exactly Hermitian by construction
    for subset, keep in ((qcd.EVEN, 1), (qcd.ODD, 0)):
        F.fill_(3.0)
        qcd.qcd_gauge_force(lat, dU, F, beta, subset=subset)
        got = host(qcd, lat, F)
        assert np.all(got[par == keep] == 3.0 + 3.0j)
        assert rel(got[par != keep], ref[par != keep]) < TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_gauge_force_generic_matrices(qcd, orc, prec):
    """O7 is a formula on arbitrary 3x3 matrices; non-unitary input catches any dagger/order slip"""
    dims = (4, 6, 4, 2)
    lat = qcd.Lattice(dims)
    U = round_to(prec, inputs.random_matrix_field(17, lat.V) * 0.6)
    F = lat.new_matrix_field(tdtype(prec))
    qcd.qcd_gauge_force(lat, dev(qcd, lat, U, prec), F, 6.1)
    assert rel(host(qcd, lat, F), orc.gauge_force(dims, 6.1, U)) < TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("variant,tile", [("plane", None), ("plane", (4, 2, 2, 2)), ("plane", (8, 4, 2, 2)),
                                          ("plane", (4, 4, 4, 2)), ("plane", (2, 2, 2, 2)), ("staple", None),
                                          ("staple", (4, 2, 2, 2)), ("staple", (8, 2, 2, 4)),
                                          # blocks of 1, 2 and 4 threads: fewer threads than the hop table has rows
                                          ("plane", (2, 1, 1, 1)), ("plane", (2, 2, 1, 1)), ("staple", (2, 1, 1, 1))])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 4, 6, 4), (16, 8, 8, 16)])
def test_force_kernel_variants(qcd, orc_omp, prec, variant, tile, dims):
    """both force kernels (the tuner's database is the knob: variant and 4-D block tile) against the oracle,
    fused and unfused, over several tiles, with tiles that span a whole extent (periodic wrap inside the
    tile), with blocks that are not a whole number of warps, and with blocks of one, two and four threads"""
    if tile and any(d % t for d, t in zip(dims, tile)):
        pytest.skip("tile does not divide the lattice")
    lat = qcd.Lattice(dims)
    beta, eps = 6.0, 0.07
    U = round_to(prec, orc_omp.hot_start(dims, inputs.config_seed(2), 0.5))
    P = round_to(prec, orc_omp.mom_refresh(dims, inputs.config_seed(2)))
    Fr = orc_omp.gauge_force(dims, beta, U)
    dU = dev(qcd, lat, U, prec)
    F = lat.new_matrix_field(tdtype(prec))
    p = qcd.F64 if prec == "f64" else qcd.F32
    try:
        for subset in (qcd.ALL, qcd.EVEN):
            qcd.qcd_tune_set(lat, p, subset, qcd.KERNEL_FORCE, qcd.FORCE_VARIANTS.index(variant), tile)
        qcd.qcd_gauge_force(lat, dU, F, beta)
        assert rel(host(qcd, lat, F), Fr) < TOL[prec]
        dP = dev(qcd, lat, P, prec)
        qcd.qcd_force_mom_update(lat, dU, dP, beta, eps)
        assert rel(host(qcd, lat, dP), P + eps * Fr) < TOL[prec]
        par = orc_omp.map(dims, O.MAP_PARITY)
        dP = dev(qcd, lat, P, prec)
        qcd.qcd_force_mom_update(lat, dU, dP, beta, eps, subset=qcd.ODD)
        want = P.copy()
        want[par == 1] += eps * Fr[par == 1]
        assert rel(host(qcd, lat, dP), want) < TOL[prec]
    finally:
        qcd.qcd_tune_clear()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 8), (16, 16, 16, 32)])
def test_mom_update_and_fused_force_mom_update(qcd, orc_omp, prec, dims):
    lat = qcd.Lattice(dims)
    beta, eps = 5.8, 0.05
    U = round_to(prec, orc_omp.hot_start(dims, inputs.config_seed(3), 0.5))
    P = round_to(prec, orc_omp.mom_refresh(dims, inputs.config_seed(3)))
    Fr = orc_omp.gauge_force(dims, beta, U)
    par = orc_omp.map(dims, O.MAP_PARITY)
    dU = dev(qcd, lat, U, prec)
    for subset, osub in ((qcd.ALL, O.ALL), (qcd.EVEN, O.EVEN), (qcd.ODD, O.ODD)):
        # unfused: F from the oracle (rounded), P += eps F
        Fin = round_to(prec, Fr)
        dP = dev(qcd, lat, P, prec)
        qcd.qcd_mom_update(lat, dev(qcd, lat, Fin, prec), dP, eps, subset=subset)
        ref = orc_omp.mom_update(dims, eps, Fin, P, subset=osub)
        got = host(qcd, lat, dP)
        assert rel(got, ref) < (1e-15 if prec == "f64" else 2e-7)  # one rounding (FMA vs mul+add)
        # fused
        dP = dev(qcd, lat, P, prec)
        qcd.qcd_force_mom_update(lat, dU, dP, beta, eps, subset=subset)
        ref = orc_omp.mom_update(dims, eps, Fr, P, subset=osub)
        got = host(qcd, lat, dP)
        assert rel(got, ref) < TOL[prec]
        if subset != qcd.ALL:
            keep = 1 if subset == qcd.EVEN else 0
            assert np.array_equal(got[par == keep], P[par == keep])


# ------------------------------------------------------------------ link update, reunitarisation

@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (6, 4, 2, 8), (16, 16, 16, 32)])
def test_link_update_and_reunit(qcd, orc_omp, prec, dims):
    lat = qcd.Lattice(dims)
    eps = 0.05
    seed = inputs.config_seed(3)
    U = round_to(prec, orc_omp.hot_start(dims, seed, 0.5))
    P = round_to(prec, orc_omp.mom_refresh(dims, seed))
    par = orc_omp.map(dims, O.MAP_PARITY)
    dP = dev(qcd, lat, P, prec)
    for reunit in (False, True):
        for subset, osub in ((qcd.ALL, O.ALL), (qcd.EVEN, O.EVEN), (qcd.ODD, O.ODD)):
            dU = dev(qcd, lat, U, prec)
            qcd.qcd_link_update(lat, dP, dU, eps, reunit=reunit, subset=subset)
            got = host(qcd, lat, dU)
            ref = orc_omp.link_update(dims, eps, P, U, reunit=reunit, subset=osub)
            assert rel(got, ref) < TOL[prec], (reunit, subset)
            if subset != qcd.ALL:
                keep = 1 if subset == qcd.EVEN else 0
                assert np.array_equal(got[par == keep], U[par == keep])
    # large steps: exp(i eps P) for norms far beyond the series radius (scaling and squaring path)
    for big in (1.0, 7.0, 40.0):
        dU = dev(qcd, lat, U, prec)
        qcd.qcd_link_update(lat, dP, dU, big, reunit=False)
        ref = orc_omp.link_update(dims, big, P, U)
        assert rel(host(qcd, lat, dU), ref) < TOL[prec] * max(1.0, big / 20), big  # DESIGN.md R15: 2^n squarings amplify rounding by ~|eps P|
    # reunitarisation of links pushed off SU(3) by sigma = 1e-3 noise (config 3), GPU noise vs oracle noise
    dU = dev(qcd, lat, U, prec)
    qcd.qcd_perturb(lat, dU, seed + 1, 1e-3)
    Up = round_to(prec, orc_omp.perturb(dims, seed + 1, 1e-3, U))
    assert rel(host(qcd, lat, dU), Up) < (1e-14 if prec == "f64" else 2e-7)
    for subset, osub in ((qcd.ALL, O.ALL), (qcd.EVEN, O.EVEN), (qcd.ODD, O.ODD)):
        dU = dev(qcd, lat, Up, prec)
        qcd.qcd_reunit(lat, dU, subset=subset)
        got = host(qcd, lat, dU)
        assert rel(got, orc_omp.reunit(dims, Up, subset=osub)) < TOL[prec]
        if subset != qcd.ALL:
            keep = 1 if subset == qcd.EVEN else 0
            assert np.array_equal(got[par == keep], Up[par == keep])
    if prec == "f64":
        got = host(qcd, lat, dU)[par == 1]
        assert np.abs(got @ np.conj(np.swapaxes(got, -1, -2)) - np.eye(3)).max() < 1e-14


def test_expi_degenerate_and_zero_momenta(qcd, orc):
    """exp of Q = 0 and of Q with degenerate eigenvalues (T8 direction), through qcd_link_update"""
    dims = (2, 2, 2, 2)
    lat = qcd.Lattice(dims)
    V = lat.V
    U = orc.hot_start(dims, 3, 0.5)
    P = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    P[1::2, :] = np.diag([1.0, 1.0, -2.0]) / np.sqrt(12.0)
    P[2, 1] = np.diag([0.3, -0.3, 0.0])
    for eps in (0.1, 3.0):
        dU = dev(qcd, lat, U, "f64")
        qcd.qcd_link_update(lat, dev(qcd, lat, P, "f64"), dU, eps)
        got = host(qcd, lat, dU)
        assert rel(got, orc.link_update(dims, eps, P, U)) < 1e-12
        assert np.array_equal(got[0], U[0])  # P = 0 -> exp = 1 exactly -> U unchanged


# ------------------------------------------------------------------ configs 1 and 2: trajectories

def gpu_H(qcd, lat, dU, dP, beta, ws):
    import torch
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    qcd.qcd_sum(lat, qcd.SUM_NORM2, 72, dP, out[0:1], ws)
    qcd.qcd_plaquette(lat, dU, out[1:2], None, ws)
    K, plaq = out.cpu().numpy()
    return K, beta * 6 * lat.V * (1 - plaq), plaq


def test_config1_one_leapfrog_step(qcd, orc):
    c = inputs.CONFIGS[1]
    dims, beta, eps = c["dims"], c["beta"], c["eps"]
    seed = inputs.config_seed(1)
    lat = qcd.Lattice(dims)
    ws = lat.new_workspace()
    U0 = orc.hot_start(dims, seed, c["sigma"])
    P0 = orc.mom_refresh(dims, seed)
    # the GPU generates its own start from the same (seed, counter) definition
    dU = lat.new_matrix_field()
    dP = lat.new_matrix_field()
    qcd.qcd_hot_start(lat, dU, seed, c["sigma"])
    qcd.qcd_mom_refresh(lat, dP, seed)
    assert rel(host(qcd, lat, dU), U0) < 1e-12 and rel(host(qcd, lat, dP), P0) < 1e-12
    K0, S0, plaq0 = gpu_H(qcd, lat, dU, dP, beta, ws)
    rK0, rS0 = orc.hamiltonian(dims, beta, U0, P0)
    assert abs(K0 - rK0) / rK0 < 1e-12 and abs(S0 - rS0) / rS0 < 1e-12
    assert abs(plaq0 - orc.plaquette(dims, U0)[0]) < 1e-12
    qcd.qcd_leapfrog(lat, dU, dP, beta, eps, 1)
    U1, P1 = orc.leapfrog(dims, beta, eps, 1, U0, P0)
    assert rel(host(qcd, lat, dU), U1) < 1e-12 and rel(host(qcd, lat, dP), P1) < 1e-12
    K1, S1, plaq1 = gpu_H(qcd, lat, dU, dP, beta, ws)
    rK1, rS1 = orc.hamiltonian(dims, beta, U1, P1)
    dH, rdH = (K1 + S1) - (K0 + S0), (rK1 + rS1) - (rK0 + rS0)
    assert abs(dH - rdH) <= 1e-12 * abs(rK0 + rS0)  # DESIGN.md R15: dH against |H|
    assert abs(plaq1 - orc.plaquette(dims, U1)[0]) < 1e-12 and abs(K1 - rK1) / rK1 < 1e-12


def test_config2_trajectory_parity_each_step_and_reversibility(qcd, orc_omp):
    c = inputs.CONFIGS[2]
    dims, beta, eps, n = c["dims"], c["beta"], c["eps"], c["nsteps"]
    seed = inputs.config_seed(2)
    lat = qcd.Lattice(dims)
    ws = lat.new_workspace()
    U = orc_omp.hot_start(dims, seed, c["sigma"])
    P = orc_omp.mom_refresh(dims, seed)
    U0, P0 = U.copy(), P.copy()
    dU, dP = dev(qcd, lat, U, "f64"), dev(qcd, lat, P, "f64")
    K0, S0, _ = gpu_H(qcd, lat, dU, dP, beta, ws)
    # leapfrog as its steps (O11): P += eps/2 F; n x { U update+reunit; P += eps F (eps/2 last) }
    qcd.qcd_force_mom_update(lat, dU, dP, beta, eps / 2)
    P = orc_omp.mom_update(dims, eps / 2, orc_omp.gauge_force(dims, beta, U), P)
    for k in range(n):
        e = eps / 2 if k == n - 1 else eps
        qcd.qcd_link_update(lat, dP, dU, eps, reunit=True)
        qcd.qcd_force_mom_update(lat, dU, dP, beta, e)
        U = orc_omp.link_update(dims, eps, P, U, reunit=True)
        P = orc_omp.mom_update(dims, e, orc_omp.gauge_force(dims, beta, U), P)
        assert rel(host(qcd, lat, dU), U) < 1e-12, k
        assert rel(host(qcd, lat, dP), P) < 1e-12, k
    K1, S1, plaq1 = gpu_H(qcd, lat, dU, dP, beta, ws)
    rK0, rS0 = orc_omp.hamiltonian(dims, beta, U0, P0)
    rK1, rS1 = orc_omp.hamiltonian(dims, beta, U, P)
    assert abs(((K1 + S1) - (K0 + S0)) - ((rK1 + rS1) - (rK0 + rS0))) <= 1e-12 * abs(rK0 + rS0)
    assert abs(plaq1 - orc_omp.plaquette(dims, U)[0]) < 1e-12
    # reversed trajectory through the single-call driver returns to the start
    dP.mul_(-1.0)
    qcd.qcd_leapfrog(lat, dU, dP, beta, eps, n)
    dP.mul_(-1.0)
    assert rel(host(qcd, lat, dU), U0) < 1e-12
    assert rel(host(qcd, lat, dP), P0) < 1e-12


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (6, 4, 2, 8), (12, 6, 10, 4), (16, 16, 16, 32)])
def test_md_step_single_pass(qcd, orc_omp, prec, dims):
    """the one-kernel MD step (force + momentum + exp + reunit, ping-pong U) against the oracle's three steps"""
    beta, eps_p, eps_u = 5.7, 0.03, 0.07
    lat = qcd.Lattice(dims)
    U = round_to(prec, orc_omp.hot_start(dims, 41, 0.5))
    P = round_to(prec, orc_omp.mom_refresh(dims, 42))
    dU, dP = dev(qcd, lat, U, prec), dev(qcd, lat, P, prec)
    dV = lat.new_matrix_field(tdtype(prec))
    dV.fill_(float("nan"))
    keep = dU.clone()
    qcd.qcd_md_step_single_pass(lat, dU, dP, dV, beta, eps_p, eps_u)
    P1 = orc_omp.mom_update(dims, eps_p, orc_omp.gauge_force(dims, beta, U), P)
    U1 = orc_omp.link_update(dims, eps_u, P1, U, reunit=True)
    assert rel(host(qcd, lat, dP), P1) < TOL[prec]
    assert rel(host(qcd, lat, dV), U1) < TOL[prec]
    import torch
    assert torch.equal(dU, keep)  # the input links are only read
    # aliasing is refused
    with pytest.raises(qcd.QcdError) as e:
        qcd.qcd_md_step_single_pass(lat, dU, dP, dU, beta, eps_p, eps_u)
    assert e.value.code == qcd.EALIAS


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(8, 8, 8, 16), (12, 6, 10, 4), (32, 32, 48, 8)])
def test_kernels_write_nothing_outside_their_fields(qcd, dims, prec):
    """every output of the step kernels sits inside a larger buffer filled with a sentinel: momenta, second gauge
    field, workspace, observables, and the neighbours' fields of the calls that push halos.  After the calls the
    guard bands are untouched (whole warps, partial warps, the z-blocked launch order)"""
    import torch
    dt = tdtype(prec)
    G, SENT = 4096, -7.25

    def guarded(n, dtype):
        base = torch.full((n + 2 * G,), SENT, dtype=dtype, device="cuda")
        return base, base[G: G + n]

    def intact(base, n):
        return bool((base[:G] == SENT).all()) and bool((base[G + n:] == SENT).all())

    lat = qcd.Lattice(dims)
    n = lat.nchunks * 36 * 32 * 2
    bases, f = zip(*(guarded(n, dt) for _ in range(3)))
    U, P, W = (x.view(lat.nchunks, 36, 32, 2) for x in f)
    qcd.qcd_hot_start(lat, U, 11, 0.4)
    qcd.qcd_mom_refresh(lat, P, 12)
    nws = lat.workspace_bytes() // 8
    wsb, ws = guarded(nws, torch.float64)
    obb, obs = guarded(2 * 3, torch.float64)
    ptb, per_t = guarded(3 * dims[3], torch.float64)
    qcd.qcd_md_step_single_pass(lat, U, P, W, 5.8, 0.03, 0.03)
    qcd.qcd_force_mom_update(lat, W, P, 5.8, 0.03)
    qcd.qcd_link_update(lat, P, W, 0.03, reunit=True)
    qcd.qcd_trajectory(lat, U, P, W, 5.8, 0.03, 2, obs.view(3, 2), per_t.view(3, dims[3]), ws)
    qcd.qcd_plaquette(lat, U, obs[0:1], per_t[: dims[3]], ws)
    torch.cuda.synchronize()
    assert all(intact(b, n) for b in bases) and intact(wsb, nws) and intact(obb, 6) and intact(ptb, 3 * dims[3])
    assert bool(torch.isfinite(U).all()) and bool(torch.isfinite(P).all())
    if dims[3] % 4 == 0 and dims[3] >= 8:  # two slabs, halos pushed by the kernels
        half = dims[3] // 2
        a, b = qcd.Lattice(dims, slab=(0, half)), qcd.Lattice(dims, slab=(half, half))
        m = a.nchunks * 36 * 32 * 2
        sb, sf = zip(*(guarded(m, dt) for _ in range(6)))
        Ua, Pa, Wa, Ub, Pb, Wb = (x.view(a.nchunks, 36, 32, 2) for x in sf)
        for L, Uf, Pf in ((a, Ua, Pa), (b, Ub, Pb)):
            qcd.qcd_hot_start(L, Uf, 11, 0.4)
            qcd.qcd_mom_refresh(L, Pf, 12)
        qcd.qcd_md_step_single_pass_push(a, Ua, Pa, Wa, 5.8, 0.03, 0.03, b, Wb, b, Wb)
        qcd.qcd_md_step_single_pass_push(b, Ub, Pb, Wb, 5.8, 0.03, 0.03, a, Wa, a, Wa)
        qcd.qcd_link_update_push(a, Pa, Wa, 0.03, True, b, Wb, b, Wb)
        qcd.qcd_link_update_push(b, Pb, Wb, 0.03, True, a, Wa, a, Wa)
        torch.cuda.synchronize()
        assert all(intact(x, m) for x in sb)


def test_z_blocked_launch_order_whole_field(qcd, orc_omp):
    """32x32x48x8 fp64: three timeslices of U are 85 MB, above the threshold at which the plane kernel launches its
    blocks z-block by z-block (force.cu: canonical_block, two z-blocks of 24 planes here).  Whole-field comparison of
    the single-pass step and of the by-product sums (global, per timeslice, K) of one trajectory step: every tile is
    visited exactly once and its partial sums land in their timeslice's slot"""
    import torch
    dims, beta, eps = (32, 32, 48, 8), 5.9, 0.04
    lat = qcd.Lattice(dims)
    U = orc_omp.hot_start(dims, 91, 0.4)
    P = orc_omp.mom_refresh(dims, 92)
    dU, dP, dV = dev(qcd, lat, U, "f64"), dev(qcd, lat, P, "f64"), lat.new_matrix_field(torch.float64)
    dV.fill_(float("nan"))
    qcd.qcd_md_step_single_pass(lat, dU, dP, dV, beta, eps, eps)
    P1 = orc_omp.mom_update(dims, eps, orc_omp.gauge_force(dims, beta, U), P)
    U1 = orc_omp.link_update(dims, eps, P1, U, reunit=True)
    assert rel(host(qcd, lat, dP), P1) < TOL["f64"] and rel(host(qcd, lat, dV), U1) < TOL["f64"]
    # one trajectory step with observables from the same kernel
    dU2, dP2 = dev(qcd, lat, U, "f64"), dev(qcd, lat, P, "f64")
    ws = lat.new_workspace()
    obs = torch.zeros((2, 2), dtype=torch.float64, device="cuda")
    per_t = torch.zeros((2, dims[3]), dtype=torch.float64, device="cuda")
    qcd.qcd_trajectory(lat, dU2, dP2, dV, beta, eps, 1, obs, per_t, ws)
    rplaq, rper_t = orc_omp.plaquette(dims, U)
    o = obs.cpu().numpy()
    assert abs(o[0, 0] - rplaq) < TOL["f64"] and np.abs(per_t[0].cpu().numpy() - rper_t).max() < TOL["f64"]
    rK = orc_omp.sum(dims, O.SUM_NORM2, P.view(np.float64).reshape(lat.V, 72))[0]
    assert abs(o[0, 1] - rK) < TOL["f64"] * rK


@pytest.mark.parametrize("prec,nsteps", [("f64", 1), ("f64", 4), ("f64", 5), ("f32", 3)])
def test_leapfrog_single_pass_matches_oracle_trajectory(qcd, orc_omp, prec, nsteps):
    c = inputs.CONFIGS[2]
    dims, beta, eps = c["dims"], c["beta"], c["eps"]
    seed = inputs.config_seed(2)
    lat = qcd.Lattice(dims)
    U = round_to(prec, orc_omp.hot_start(dims, seed, c["sigma"]))
    P = round_to(prec, orc_omp.mom_refresh(dims, seed))
    dU, dP = dev(qcd, lat, U, prec), dev(qcd, lat, P, prec)
    dW = lat.new_matrix_field(tdtype(prec))
    qcd.qcd_leapfrog_single_pass(lat, dU, dP, dW, beta, eps, nsteps)
    U1, P1 = orc_omp.leapfrog(dims, beta, eps, nsteps, U, P)
    assert rel(host(qcd, lat, dU), U1) < TOL[prec] and rel(host(qcd, lat, dP), P1) < TOL[prec]
    if prec == "f64":  # reversibility through the same driver
        dP.mul_(-1.0)
        qcd.qcd_leapfrog_single_pass(lat, dU, dP, dW, beta, eps, nsteps)
        dP.mul_(-1.0)
        assert rel(host(qcd, lat, dU), U) < 1e-12 and rel(host(qcd, lat, dP), P) < 1e-12


def test_fp32_trajectory_tracks_fp64_oracle(qcd, orc_omp):
    c = inputs.CONFIGS[2]
    dims, beta, eps = c["dims"], c["beta"], c["eps"]
    seed = inputs.config_seed(2)
    lat = qcd.Lattice(dims)
    U = round_to("f32", orc_omp.hot_start(dims, seed, c["sigma"]))
    P = round_to("f32", orc_omp.mom_refresh(dims, seed))
    dU, dP = dev(qcd, lat, U, "f32"), dev(qcd, lat, P, "f32")
    qcd.qcd_leapfrog(lat, dU, dP, beta, eps, 10)
    U1, P1 = orc_omp.leapfrog(dims, beta, eps, 10, U, P)
    assert rel(host(qcd, lat, dU), U1) < 2e-5 and rel(host(qcd, lat, dP), P1) < 2e-5


# ------------------------------------------------------------------ full sizes, in bench.py's launch configuration

def sample_sites(dims, n, seed):
    """lexicographic sites: corners and faces of the lattice (periodic wrap) plus random interior ones"""
    Lx, Ly, Lz, Lt = dims
    rng = np.random.default_rng(seed)
    pts = []
    for x in (0, 1, Lx - 1):
        for y in (0, Ly - 1):
            for z in (0, Lz - 1):
                for t in (0, 1, Lt - 1):
                    pts.append(x + Lx * (y + Ly * (z + Lz * t)))
    pts += list(rng.integers(0, Lx * Ly * Lz * Lt, n - len(pts)))
    return np.unique(np.array(pts, dtype=np.int32))


_full_start = {}


def full_start(orc_omp, cfg):
    """hot-start links and Gaussian momenta of a BASELINE config, whole lattice, from the oracle (cached: the
    48^3x96 fields are 6 GB each)"""
    if cfg not in _full_start:
        _full_start.clear()  # one config at a time
        c = inputs.CONFIGS[cfg]
        seed = inputs.config_seed(cfg)
        _full_start[cfg] = (orc_omp.hot_start(c["dims"], seed, c["sigma"]), orc_omp.mom_refresh(c["dims"], seed))
    return _full_start[cfg]


@pytest.mark.parametrize("cfg,prec,single", [(4, "f64", False), (4, "f64", True), (5, "f64", False), (5, "f64", True),
                                             (5, "f32", False), (5, "f32", True)])
def test_full_size_md_step_sampled_parity(qcd, orc_omp, cfg, prec, single):
    """BASELINE configs 4 (32^3x64 fp64, the headline) and 5 (48^3x96, both precisions): the fused MD step
    exactly as bench.py launches it (two kernels in place, or the single-pass kernel), checked at sampled sites
    the oracle computes one by one, the reductions of configs[3] ("sumMulti of plaquette per timeslice and
    global kinetic-energy sum") on the WHOLE field against the oracle, plus properties that hold at any size."""
    import torch
    c = inputs.CONFIGS[cfg]
    dims, beta, eps = c["dims"], c["beta"], c["eps"]
    seed = inputs.config_seed(cfg)
    lat = qcd.Lattice(dims)
    dt = tdtype(prec)
    dU, dP = lat.new_matrix_field(dt), lat.new_matrix_field(dt)
    qcd.qcd_hot_start(lat, dU, seed, c["sigma"])
    qcd.qcd_mom_refresh(lat, dP, seed)
    # the oracle builds the same start from the (seed, counter) definition, never from the GPU
    U0, P0 = full_start(orc_omp, cfg)
    sites = sample_sites(dims, 600, 1)
    cbmap = orc_omp.map(dims, O.MAP_CB_OF_LEX)
    cbs = torch.from_numpy(cbmap[sites].astype(np.int64)).cuda()

    def gather(field):  # device field [chunk][36][32][2] -> complex [n,4,3,3] at the sampled sites
        g = field[cbs >> 5, :, cbs & 31, :].permute(1, 0, 2).to(torch.float64).cpu().numpy()
        return (g[..., 0] + 1j * g[..., 1]).T.reshape(len(sites), 4, 3, 3)

    tolgen = 1e-12 if prec == "f64" else 2e-7
    assert rel(gather(dU), U0[sites]) < tolgen
    if prec == "f32":  # the fp32 path starts from rounded fields: give the oracle the same
        U0, P0 = round_to(prec, U0), round_to(prec, P0)
    # momenta at a few sampled sites once more from the oracle's generator blocks (the RNG is keyed on the site)
    for s_ in sites[:8]:
        for mu in range(4):
            q = np.concatenate([orc_omp.rng_block(seed, int(s_), mu, j, 0, 1)[2] for j in range(4)])
            assert np.abs(round_to(prec, orc_omp.herm_from_coeffs(q)) - P0[s_, mu]).max() == 0
    Psites = P0[sites]
    assert rel(gather(dP), Psites) < tolgen
    ws = lat.new_workspace()
    plaq = torch.zeros(1, dtype=torch.float64, device="cuda")
    per_t = torch.zeros(dims[3], dtype=torch.float64, device="cuda")
    qcd.qcd_plaquette(lat, dU, plaq, per_t, ws)
    rplaq, rper_t = orc_omp.plaquette(dims, U0)
    assert abs(plaq.item() - rplaq) / rplaq < TOL[prec]
    assert rel(per_t.cpu().numpy(), rper_t) < TOL[prec]
    # one fused MD step (two kernels in place, or the single-pass kernel writing a second gauge field)
    if single:
        dV = lat.new_matrix_field(dt)
        qcd.qcd_md_step_single_pass(lat, dU, dP, dV, beta, eps, eps)
        dU = dV
    else:
        qcd.qcd_md_step(lat, dU, dP, beta, eps, eps)
    Fs = orc_omp.gauge_force_sites(dims, beta, U0, sites)
    P1 = Psites + eps * Fs
    assert rel(gather(dP), P1) < TOL[prec]
    # link update is site-local: run the oracle on the sampled sites laid out as a small lattice
    n = len(sites) // 16 * 16
    sub = (2, 2, 2, n // 8)
    U1 = orc_omp.link_update(sub, eps, np.ascontiguousarray(P1[:n]), np.ascontiguousarray(U0[sites][:n]), reunit=True)
    gU = gather(dU)
    assert rel(gU[:n], U1) < TOL[prec]
    # any-size properties: links stay in SU(3), momenta stay Hermitian traceless
    utol = 1e-14 if prec == "f64" else 1e-6
    assert np.abs(gU @ np.conj(np.swapaxes(gU, -1, -2)) - np.eye(3)).max() < utol
    assert np.abs(np.linalg.det(gU) - 1).max() < utol
    gP = gather(dP)
    assert np.abs(gP - np.conj(np.swapaxes(gP, -1, -2))).max() < utol * 10
    assert np.abs(np.trace(gP, axis1=-2, axis2=-1)).max() < utol * 10
    # the reductions on the whole field: kinetic energy (sum) and per timeslice (sumMulti) of the UPDATED momenta
    # against the oracle's own force on the whole lattice, and the per-timeslice plaquette of the updated links
    P1full = P0 + eps * orc_omp.gauge_force(dims, beta, U0)
    K = torch.zeros(1, dtype=torch.float64, device="cuda")
    Kt = torch.zeros(dims[3], dtype=torch.float64, device="cuda")
    qcd.qcd_sum(lat, qcd.SUM_NORM2, 72, dP, K, ws)
    qcd.qcd_sum_multi(lat, qcd.SUM_NORM2, 72, dP, None, dims[3], Kt, ws)
    flat = P1full.view(np.float64).reshape(lat.V, 72)
    rK, rKt = orc_omp.sum(dims, O.SUM_NORM2, flat)[0], orc_omp.sum_multi(dims, O.SUM_NORM2, flat)
    assert abs(K.item() - rK) < TOL[prec] * rK
    assert rel(Kt.cpu().numpy(), rKt) < TOL[prec]
    assert abs(K.item() / (16 * lat.V) - 1) < 0.01


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (6, 4, 2, 8), (12, 6, 10, 4), (16, 16, 16, 32)])
def test_force_mom_update_with_fused_sums(qcd, orc_omp, prec, dims):
    """plaquette and kinetic energy as by-products of the force kernel (sum rule: sum Re tr W = 4 sum Re tr P)"""
    import torch
    lat = qcd.Lattice(dims)
    beta, eps = 5.9, 0.04
    U = round_to(prec, orc_omp.hot_start(dims, 91, 0.5))
    P = round_to(prec, orc_omp.mom_refresh(dims, 92))
    dU, dP = dev(qcd, lat, U, prec), dev(qcd, lat, P, prec)
    ws = lat.new_workspace()
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    qcd.qcd_force_mom_update_sums(lat, dU, dP, beta, eps, out, ws)
    P1 = orc_omp.mom_update(dims, eps, orc_omp.gauge_force(dims, beta, U), P)
    assert rel(host(qcd, lat, dP), P1) < TOL[prec]
    plaq, K = out.cpu().numpy()
    rplaq = orc_omp.plaquette(dims, U)[0]
    rK = orc_omp.sum(dims, O.SUM_NORM2, P1.view(np.float64).reshape(lat.V, 72))
    assert abs(plaq - rplaq) < TOL[prec] * abs(rplaq) and abs(K - rK) < TOL[prec] * rK
    # deterministic, and the same numbers as the stand-alone reductions up to rounding order
    dP2 = dev(qcd, lat, P, prec)
    out2 = torch.zeros(2, dtype=torch.float64, device="cuda")
    qcd.qcd_force_mom_update_sums(lat, dU, dP2, beta, eps, out2, ws)
    assert torch.equal(out, out2) and torch.equal(dP, dP2)


def test_leapfrog_energy_gives_the_final_hamiltonian(qcd, orc_omp):
    import torch
    c = inputs.CONFIGS[2]
    dims, beta, eps = c["dims"], c["beta"], c["eps"]
    lat = qcd.Lattice(dims)
    U = orc_omp.hot_start(dims, inputs.config_seed(2), c["sigma"])
    P = orc_omp.mom_refresh(dims, inputs.config_seed(2))
    dU, dP = dev(qcd, lat, U, "f64"), dev(qcd, lat, P, "f64")
    ws = lat.new_workspace()
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    qcd.qcd_leapfrog_energy(lat, dU, dP, beta, eps, 4, out, ws)
    U1, P1 = orc_omp.leapfrog(dims, beta, eps, 4, U, P)
    assert rel(host(qcd, lat, dU), U1) < 1e-12 and rel(host(qcd, lat, dP), P1) < 1e-12
    rK, rS = orc_omp.hamiltonian(dims, beta, U1, P1)
    plaq, K = out.cpu().numpy()
    H = K + beta * 6 * lat.V * (1 - plaq)
    assert abs(H - (rK + rS)) < 1e-12 * abs(rK + rS)


@pytest.mark.parametrize("n", [1, 2])
def test_config_observables_against_stored_oracle_values(qcd, n):
    """BASELINE configs 1 and 2: plaquette, kinetic energy and dH of the GPU trajectory (start generated on the
    device, qcd_leapfrog_energy) against tests/golden/config_values.json, written by the oracle alone"""
    import json
    import os
    import torch
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "config_values.json")))[str(n)]
    dims, beta = tuple(g["dims"]), g["beta"]
    seed = int(g["seed"], 16)
    lat = qcd.Lattice(dims)
    ws = lat.new_workspace()
    dU, dP = lat.new_matrix_field(), lat.new_matrix_field()
    qcd.qcd_hot_start(lat, dU, seed, g["sigma"])
    qcd.qcd_mom_refresh(lat, dP, seed)
    K0, S0, plaq0 = gpu_H(qcd, lat, dU, dP, beta, ws)
    assert abs(plaq0 - g["plaq0"]) < 1e-12 and abs(K0 - g["K0"]) < 1e-12 * g["K0"] and abs(S0 - g["S0"]) < 1e-12 * g["S0"]
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    qcd.qcd_leapfrog_energy(lat, dU, dP, beta, g["eps"], g["nsteps"], out, ws)
    plaq1, K1 = out.cpu().numpy()
    S1 = beta * 6 * lat.V * (1 - plaq1)
    assert abs(plaq1 - g["plaq1"]) < 1e-12 and abs(K1 - g["K1"]) < 1e-12 * g["K1"]
    assert abs(((K1 + S1) - (K0 + S0)) - g["dH"]) <= 1e-12 * abs(g["K0"] + g["S0"])  # R15: dH against |H|


def test_trajectory_driver_reports_the_stored_dH(qcd):
    """paper_1212_0785_b200.trajectory (one qcd_trajectory call, observables from the force kernel) on config 2"""
    import json
    import os
    from paper_1212_0785_b200 import trajectory
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "config_values.json")))["2"]
    r = trajectory.run(2)
    scale = abs(g["K0"] + g["S0"])
    assert abs(r["dH"] - g["dH"]) <= 1e-12 * scale and abs(r["H_end_from_fused_sums"] - r["H_end"]) <= 1e-12 * scale
    assert abs(r["plaq_end"] - g["plaq1"]) < 1e-12 and len(r["per_step_plaq_K"]) == g["nsteps"] + 1
    assert abs(r["per_step_plaq_K"][-1][0] - r["plaq_end"]) < 1e-13
    assert abs(np.mean(r["plaq_per_timeslice_end"]) - r["plaq_end"]) < 1e-13
    r2 = trajectory.run(2, observables=False)
    assert abs(r2["H_end"] - r["H_end"]) <= 1e-12 * scale


def oracle_trajectory_observed(orc, dims, beta, eps, n, U, P):
    """O11 step by step on the oracle with the observables qcd_trajectory reports (include/qcd.h): row k =
    (plaquette of U_k, K of the momenta after the kick that follows link update k; row 0: K of the initial momenta),
    and the per-timeslice plaquette of U_k"""
    V = O.Oracle.volume(dims)
    obs, per_t = np.empty((n + 1, 2)), np.empty((n + 1, dims[3]))

    def K(P):
        return orc.sum(dims, O.SUM_NORM2, P.view(np.float64).reshape(V, 72))[0]

    obs[0, 0], per_t[0] = orc.plaquette(dims, U)
    obs[0, 1] = K(P)
    P = orc.mom_update(dims, eps / 2, orc.gauge_force(dims, beta, U), P)
    for k in range(1, n + 1):
        U = orc.link_update(dims, eps, P, U, reunit=True)
        obs[k, 0], per_t[k] = orc.plaquette(dims, U)
        P = orc.mom_update(dims, eps / 2 if k == n else eps, orc.gauge_force(dims, beta, U), P)
        obs[k, 1] = K(P)
    return U, P, obs, per_t


@pytest.mark.parametrize("dims,prec,n,tile", [((4, 4, 4, 4), "f64", 1, None), ((8, 8, 8, 16), "f64", 4, None),
                                               ((8, 8, 8, 16), "f64", 5, None), ((6, 4, 2, 8), "f64", 3, None),
                                               ((8, 8, 8, 16), "f64", 3, (8, 2, 2, 2)), ((8, 8, 8, 16), "f32", 3, None),
                                               ((8, 8, 8, 16), "f64", 4, (8, 4, 4, 1)), ((8, 8, 8, 16), "f32", 2, (8, 4, 4, 1)),
                                               ((8, 8, 8, 16), "f64", 3, (8, 4, 2, 1)), ((8, 8, 8, 16), "f64", 2, "staple"),
                                               ((8, 8, 8, 16), "f64", 3, (4, 2, 2, 4)), ((8, 8, 8, 16), "f32", 2, (8, 2, 2, 2)),
                                               ((4, 6, 2, 8), "f64", 2, (4, 3, 2, 2))])
def test_trajectory_observables_every_step(qcd, orc_omp, dims, prec, n, tile):
    """qcd_trajectory: final fields and the per-step (plaquette, per-timeslice plaquette, K) series against the
    oracle's leapfrog step by step; odd and even step counts (the ping-pong starts differently), a block that
    is not a whole number of warps, tiles inside one timeslice and tiles that span two or four timeslices
    (per-timeslice values are by-products of the force kernel: one partial per block and timeslice of its tile) and
    the staple variant (they then come from the stand-alone plaquette kernel)"""
    import torch
    beta, eps = 5.8, 0.05
    lat = qcd.Lattice(dims)
    U = round_to(prec, orc_omp.hot_start(dims, 77, 0.4))
    P = round_to(prec, orc_omp.mom_refresh(dims, 78))
    dU, dP, dW = dev(qcd, lat, U, prec), dev(qcd, lat, P, prec), lat.new_matrix_field(tdtype(prec))
    ws = lat.new_workspace()
    obs = torch.zeros((n + 1, 2), dtype=torch.float64, device="cuda")
    per_t = torch.zeros((n + 1, dims[3]), dtype=torch.float64, device="cuda")
    p = qcd.F64 if prec == "f64" else qcd.F32
    try:
        if tile == "staple":
            qcd.qcd_tune_set(lat, p, qcd.ALL, qcd.KERNEL_FORCE, qcd.FORCE_VARIANTS.index("staple"), None)
        elif tile:
            qcd.qcd_tune_set(lat, p, qcd.ALL, qcd.KERNEL_FORCE, qcd.FORCE_VARIANTS.index("plane"), tile)
        qcd.qcd_trajectory(lat, dU, dP, dW, beta, eps, n, obs, per_t, ws)
        obs2, per_t2 = torch.zeros_like(obs), torch.zeros_like(per_t)
        dU2, dP2 = dev(qcd, lat, U, prec), dev(qcd, lat, P, prec)
        qcd.qcd_trajectory(lat, dU2, dP2, dW, beta, eps, n, obs2, per_t2, ws)
        # without the per-timeslice output
        dU3, dP3, obs3 = dev(qcd, lat, U, prec), dev(qcd, lat, P, prec), torch.zeros_like(obs)
        qcd.qcd_trajectory(lat, dU3, dP3, dW, beta, eps, n, obs3, None, ws)
    finally:
        qcd.qcd_tune_clear()
    rU, rP, robs, rper_t = oracle_trajectory_observed(orc_omp, dims, beta, eps, n, U, P)
    assert rel(host(qcd, lat, dU), rU) < TOL[prec] and rel(host(qcd, lat, dP), rP) < TOL[prec]
    o = obs.cpu().numpy()
    assert np.abs(o[:, 0] - robs[:, 0]).max() < TOL[prec] and rel(o[:, 1], robs[:, 1]) < TOL[prec]
    assert np.abs(per_t.cpu().numpy() - rper_t).max() < TOL[prec]
    H = o[:, 1] + beta * 6 * lat.V * (1 - o[:, 0])
    rH = robs[:, 1] + beta * 6 * lat.V * (1 - robs[:, 0])
    assert abs((H[n] - H[0]) - (rH[n] - rH[0])) <= TOL[prec] * abs(rH[0])  # R15: dH against |H|
    # deterministic run to run, per-timeslice values average to the global one
    assert torch.equal(obs, obs2) and torch.equal(per_t, per_t2) and torch.equal(dU, dU2) and torch.equal(dP, dP2)
    assert np.abs(per_t.cpu().numpy().mean(axis=1) - o[:, 0]).max() < (1e-13 if prec == "f64" else 1e-7)
    # argument checks come before anything is enqueued
    assert np.abs(obs3.cpu().numpy() - o).max() < 1e-12 * np.abs(o).max() and torch.equal(dU3, dU)
    small = torch.empty(8, dtype=torch.float64, device="cuda")
    with pytest.raises(qcd.QcdError) as e:
        qcd.qcd_trajectory(lat, dU3, dP3, dW, beta, eps, n, obs3, None, small)
    assert e.value.code == qcd.EWORKSPACE and torch.equal(dU3, dU)
    with pytest.raises(qcd.QcdError) as e:
        qcd.qcd_trajectory(lat, dU3, dP3, dU3, beta, eps, n, obs3, None, ws)
    assert e.value.code == qcd.EALIAS


@pytest.mark.parametrize("cfg,prec,n", [(4, "f64", 4), (5, "f64", 20), (5, "f32", 2)])
def test_config_trajectory_full_size_against_oracle(qcd, orc_omp, cfg, prec, n):
    """BASELINE configs 4 and 5 at full size ("sustained 20-step leapfrog trajectory with per-step
    reunitarization and reductions ... reports dH"): qcd_trajectory against the OpenMP build of the oracle,
    step by step — plaquette, per-timeslice plaquette and K of every step, dH (R15: against |H|), final links and
    momenta at sampled sites, and at EVERY site for config 4.  Config 5 fp64 runs all 20 steps; the other two rows are shortened to 4 and 2 steps
    to keep the suite's time down (the oracle needs about 9 s per 48^3x96 step on 16 host cores)."""
    import torch
    c = inputs.CONFIGS[cfg]
    dims, beta, eps = c["dims"], c["beta"], c["eps"]
    seed = inputs.config_seed(cfg)
    lat = qcd.Lattice(dims)
    dt = tdtype(prec)
    dU, dP, dW = lat.new_matrix_field(dt), lat.new_matrix_field(dt), lat.new_matrix_field(dt)
    qcd.qcd_hot_start(lat, dU, seed, c["sigma"])
    qcd.qcd_mom_refresh(lat, dP, seed)
    ws = lat.new_workspace()
    obs = torch.zeros((n + 1, 2), dtype=torch.float64, device="cuda")
    per_t = torch.zeros((n + 1, dims[3]), dtype=torch.float64, device="cuda")
    qcd.qcd_trajectory(lat, dU, dP, dW, beta, eps, n, obs, per_t, ws)
    U0, P0 = full_start(orc_omp, cfg)
    rU, rP, robs, rper_t = oracle_trajectory_observed(orc_omp, dims, beta, eps, n, round_to(prec, U0), round_to(prec, P0))
    _full_start.clear()
    o = obs.cpu().numpy()
    assert np.abs(o[:, 0] - robs[:, 0]).max() < TOL[prec] and rel(o[:, 1], robs[:, 1]) < TOL[prec]
    assert np.abs(per_t.cpu().numpy() - rper_t).max() < TOL[prec]
    H = o[:, 1] + beta * 6 * lat.V * (1 - o[:, 0])
    rH = robs[:, 1] + beta * 6 * lat.V * (1 - robs[:, 0])
    assert abs((H[n] - H[0]) - (rH[n] - rH[0])) <= TOL[prec] * abs(rH[0])
    sites = sample_sites(dims, 2000, 3)
    cbs = torch.from_numpy(orc_omp.map(dims, O.MAP_CB_OF_LEX)[sites].astype(np.int64)).cuda()

    def gather(field):
        g = field[cbs >> 5, :, cbs & 31, :].permute(1, 0, 2).to(torch.float64).cpu().numpy()
        return (g[..., 0] + 1j * g[..., 1]).T.reshape(len(sites), 4, 3, 3)

    assert rel(gather(dU), rU[sites]) < TOL[prec] and rel(gather(dP), rP[sites]) < TOL[prec]
    if cfg == 4:  # every link of every site as well (a 1.2 GB unpack per field; config 5 would need 6 GB per copy)
        assert rel(host(qcd, lat, dU), rU) < TOL[prec]
        assert rel(host(qcd, lat, dP), rP) < TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,nsteps", [((8, 8, 8, 16), 1), ((8, 8, 8, 16), 3), ((8, 8, 8, 32), 2), ((6, 4, 2, 8), 1),
                                         ((8, 8, 8, 16), 0), ((4, 4, 4, 4), 2)])
def test_md_host_pipeline_matches_the_oracle(qcd, orc_omp, prec, dims, nsteps):
    """qcd_md_host (the end-to-end call of bench.py) on pinned host buffers: slabs of 1 and 2 timeslices on three
    streams, one / several / zero steps, and the single-stream path of small lattices, against nsteps oracle MD steps;
    back-to-back calls on one stream stay ordered"""
    import torch
    beta, eps = 5.9, 0.04
    lat = qcd.Lattice(dims)
    dt = tdtype(prec)
    U = round_to(prec, orc_omp.hot_start(dims, 21, 0.5))
    P = round_to(prec, orc_omp.mom_refresh(dims, 22))

    def to_host(a):
        return torch.from_numpy(np.ascontiguousarray(a).view(np.float64).reshape(-1)).to(dt).pin_memory()

    hU, hP = to_host(U), to_host(P)
    p = qcd.F64 if prec == "f64" else qcd.F32
    work = torch.empty(lat.md_host_work_bytes(p) // hU.element_size(), dtype=dt, device="cuda")
    qcd.qcd_md_host(lat, hU, hP, beta, eps, nsteps, work)
    torch.cuda.synchronize()
    rU, rP = U, P
    for _ in range(nsteps):
        rU, rP = orc_omp.md_step(dims, beta, eps, eps, rU, rP)

    def from_host(h):
        return h.to(torch.float64).numpy().view(np.complex128).reshape(-1, 4, 3, 3)

    if nsteps == 0:
        assert np.array_equal(from_host(hU), U) and np.array_equal(from_host(hP), P)
    else:
        assert rel(from_host(hU), rU) < TOL[prec] and rel(from_host(hP), rP) < TOL[prec]
    # a second call continues from the first one's output without a host synchronisation in between
    hU2, hP2 = to_host(U), to_host(P)
    qcd.qcd_md_host(lat, hU2, hP2, beta, eps, 1, work)
    qcd.qcd_md_host(lat, hU2, hP2, beta, eps, 1, work)
    torch.cuda.synchronize()
    rU, rP = orc_omp.md_step(dims, beta, eps, eps, *orc_omp.md_step(dims, beta, eps, eps, U, P))
    assert rel(from_host(hU2), rU) < TOL[prec] and rel(from_host(hP2), rP) < TOL[prec]
