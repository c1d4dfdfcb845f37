"""domain decomposition in t with a one-site halo, tested on ONE GPU: the lattice is split
into 2 and 4 slabs in one process, halos travel through qcd_copy_timeslices (what peer stores over NVLink would
do), and the gathered result must equal the undecomposed lattice — bit for bit for the generator, and for the
trajectory because every site runs the same arithmetic in the same order whatever tile it falls in — and the
oracle within the usual tolerance.  PAPER.md:24 (multi-GPU support), PAPER.md:121 (overlap, work in progress)."""
import numpy as np
import pytest

from oracle import oracle as O
from tests.test_gpu_parity import TOL, host, rel, tdtype

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qcd():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1212_0785_b200 import binding
    return binding


def slab_rows(a, dims, t_begin, t_count):
    """timeslices t_begin-1 .. t_begin+t_count (periodic) of a canonical global array: what the slab stores"""
    Vs = dims[0] * dims[1] * dims[2]
    t = (np.arange(t_begin - 1, t_begin + t_count + 1)) % dims[3]
    return a.reshape(dims[3], Vs, 4, 3, 3)[t].reshape(-1, 4, 3, 3)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,nslabs", [((8, 8, 8, 16), 2), ((8, 8, 8, 16), 4), ((4, 6, 2, 8), 2), ((4, 4, 4, 4), 1)])
def test_generator_is_decomposition_independent(qcd, orc_omp, dims, nslabs, prec):
    """hot start, momentum refresh and perturbation on slab lattices give, halos included, exactly the fields of
    the whole lattice; EVEN / ODD mean the global parity on every slab"""
    from paper_1212_0785_b200 import slabs
    seed = 0x1212078500000002
    full = qcd.Lattice(dims)
    dt = tdtype(prec)
    fU, fP = full.new_matrix_field(dt), full.new_matrix_field(dt)
    qcd.qcd_hot_start(full, fU, seed, 0.5)
    qcd.qcd_mom_refresh(full, fP, seed, stream_id=3)
    gU, gP = host(qcd, full, fU), host(qcd, full, fP)
    assert rel(gU, orc_omp.hot_start(dims, seed, 0.5)) < (1e-12 if prec == "f64" else 2e-7)
    gpar = orc_omp.map(dims, O.MAP_PARITY)
    for tb, tc in slabs.partition(dims[3], nslabs):
        lat = qcd.Lattice(dims, slab=(tb, tc))
        assert lat.dims == dims[:3] + (tc + 2,) and lat.interior_t == (1, tc + 1)
        U, P = lat.new_matrix_field(dt), lat.new_matrix_field(dt)
        qcd.qcd_hot_start(lat, U, seed, 0.5)
        qcd.qcd_mom_refresh(lat, P, seed, stream_id=3)
        assert np.array_equal(host(qcd, lat, U), slab_rows(gU, dims, tb, tc))
        assert np.array_equal(host(qcd, lat, P), slab_rows(gP, dims, tb, tc))
        # subset call: only globally even sites are written
        P.fill_(7.0)
        qcd.qcd_mom_refresh(lat, P, seed, stream_id=3, subset=qcd.EVEN)
        got = host(qcd, lat, P)
        par = slab_rows(np.repeat(gpar, 36).reshape(-1, 4, 3, 3).astype(np.complex128), dims, tb, tc).real[:, 0, 0, 0]
        assert np.array_equal(got[par == 0], slab_rows(gP, dims, tb, tc)[par == 0]) and np.all(got[par == 1] == 7.0 + 7.0j)
        # perturbation noise as well
        qcd.qcd_perturb(lat, U, seed + 1, 1e-3)
        fU2 = fU.clone()
        qcd.qcd_perturb(full, fU2, seed + 1, 1e-3)
        assert np.array_equal(host(qcd, lat, U), slab_rows(host(qcd, full, fU2), dims, tb, tc))


@pytest.mark.parametrize("fused", [False, True])
@pytest.mark.parametrize("dims,nslabs,prec,overlap", [((8, 8, 8, 16), 2, "f64", False), ((8, 8, 8, 16), 4, "f64", True),
                                                      ((16, 16, 16, 32), 4, "f64", True), ((16, 16, 16, 32), 2, "f32", True),
                                                      ((8, 8, 8, 16), 1, "f64", False), ((4, 6, 2, 8), 2, "f64", True),
                                                      ((8, 8, 8, 16), 3, "f64", True)])
def test_slab_trajectory_equals_the_whole_lattice(qcd, orc_omp, dims, nslabs, prec, overlap, fused):
    """fused = True: the halo transport is done by the link update itself (qcd_link_update_push: the thread that has a
    boundary link in registers stores it into the neighbour's halo) instead of qcd_copy_timeslices"""
    import torch
    from paper_1212_0785_b200 import slabs
    beta, eps, n, seed = 5.8, 0.05, 3, 0x1212078500000002
    dt = tdtype(prec)
    full = qcd.Lattice(dims)
    fU, fP = full.new_matrix_field(dt), full.new_matrix_field(dt)
    qcd.qcd_hot_start(full, fU, seed, 0.5)
    qcd.qcd_mom_refresh(full, fP, seed)
    U0, P0 = host(qcd, full, fU), host(qcd, full, fP)
    qcd.qcd_leapfrog(full, fU, fP, beta, eps, n)
    ss = slabs.SlabSet(qcd, dims, nslabs, dt)
    ss.start(seed, 0.5)
    ss.leapfrog(beta, eps, n, overlap=overlap, fused=fused)
    torch.cuda.synchronize()
    gU, gP = ss.gather("U"), ss.gather("P")
    # the same arithmetic per site whatever the decomposition: bit-identical to the undecomposed run
    assert np.array_equal(gU, host(qcd, full, fU)) and np.array_equal(gP, host(qcd, full, fP))
    rU, rP = orc_omp.leapfrog(dims, beta, eps, n, U0, P0)
    assert rel(gU, rU) < TOL[prec] and rel(gP, rP) < TOL[prec]
    # reductions: per-timeslice values of the slabs in rank order = the whole lattice's; K summed in rank order
    plaq, K, plaq_t = ss.global_observables()
    rplaq, rper_t = orc_omp.plaquette(dims, rU)
    rK = orc_omp.sum(dims, O.SUM_NORM2, rP.view(np.float64).reshape(full.V, 72))[0]
    assert abs(plaq - rplaq) < TOL[prec] and np.abs(plaq_t.cpu().numpy() - rper_t).max() < TOL[prec]
    assert abs(K - rK) < TOL[prec] * rK
    plaq2, K2, _ = ss.global_observables()
    assert plaq2 == plaq and K2 == K  # fixed order: the same bits on every call
    # the by-product sums of a slab average over its interior only
    s = ss.slabs[0]
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    ss.exchange()
    qcd.qcd_force_mom_update_sums(s.lat, s.U, s.P, beta, 0.0, out, s.ws)
    assert abs(out[0].item() - rper_t[s.t_begin: s.t_begin + s.n].mean()) < TOL[prec]


@pytest.mark.parametrize("dims,nslabs,prec,overlap", [((8, 8, 8, 16), 2, "f64", False), ((8, 8, 8, 16), 4, "f64", True),
                                                      ((16, 16, 16, 32), 4, "f64", True), ((16, 16, 16, 32), 2, "f32", True),
                                                      ((8, 8, 8, 16), 1, "f64", False), ((4, 6, 2, 8), 2, "f64", True),
                                                      ((8, 8, 8, 16), 3, "f64", True), ((32, 8, 8, 16), 2, "f64", True)])
@pytest.mark.parametrize("nsteps", [1, 4])
def test_slab_single_pass_trajectory_with_in_kernel_halo_push(qcd, orc_omp, dims, nslabs, prec, overlap, nsteps):
    """the single-pass step on slabs, halos written by the step kernel of the neighbouring slab
    (qcd_md_step_single_pass_push): bit-identical to qcd_leapfrog_single_pass on the undecomposed lattice and within
    tolerance of the oracle; odd and even step counts (the ping-pong ends in either buffer)"""
    import torch
    from paper_1212_0785_b200 import slabs
    beta, eps, seed = 5.8, 0.05, 0x1212078500000002
    dt = tdtype(prec)
    full = qcd.Lattice(dims)
    fU, fP, fW = full.new_matrix_field(dt), full.new_matrix_field(dt), full.new_matrix_field(dt)
    qcd.qcd_hot_start(full, fU, seed, 0.5)
    qcd.qcd_mom_refresh(full, fP, seed)
    U0, P0 = host(qcd, full, fU), host(qcd, full, fP)
    qcd.qcd_leapfrog_single_pass(full, fU, fP, fW, beta, eps, nsteps)
    ss = slabs.SlabSet(qcd, dims, nslabs, dt)
    ss.start(seed, 0.5)
    ss.leapfrog_single_pass(beta, eps, nsteps, overlap=overlap)
    torch.cuda.synchronize()
    gU, gP = ss.gather("U"), ss.gather("P")
    assert np.array_equal(gU, host(qcd, full, fU)) and np.array_equal(gP, host(qcd, full, fP))
    rU, rP = orc_omp.leapfrog(dims, beta, eps, nsteps, U0, P0)
    assert rel(gU, rU) < TOL[prec] and rel(gP, rP) < TOL[prec]


def test_link_update_push_arguments_and_halo_only_stores(qcd):
    """argument checks before anything is enqueued; the push writes the neighbours' halos and nothing else of them,
    and leaves the slab's own halos alone"""
    import torch
    a, b = qcd.Lattice((8, 8, 8, 16), slab=(0, 8)), qcd.Lattice((8, 8, 8, 16), slab=(8, 8))
    c, full = qcd.Lattice((8, 8, 4, 16), slab=(0, 8)), qcd.Lattice((8, 8, 8, 16))
    Ua, Pa, Ub = a.new_matrix_field(), a.new_matrix_field(), b.new_matrix_field()
    Uc, Uf, Pf = c.new_matrix_field(), full.new_matrix_field(), full.new_matrix_field()
    for args, code in (((a, Pa, Ua, 0.1, True, c, Uc, b, Ub), qcd.EDIMS), ((a, Pa, Ua, 0.1, True, b, None, b, Ub), qcd.EINVAL),
                       ((full, Pf, Uf, 0.1, True, None, None, None, None), qcd.EINVAL),
                       ((a, Pa, Pa, 0.1, True, None, None, None, None), qcd.EALIAS)):
        with pytest.raises(qcd.QcdError) as e:
            qcd.qcd_link_update_push(*args)
        assert e.value.code == code
    qcd.qcd_hot_start(a, Ua, 5, 0.5)
    qcd.qcd_mom_refresh(a, Pa, 5)
    Ub.fill_(7.0)
    ref = Ua.clone()
    qcd.qcd_link_update(a, Pa, ref, 0.1, reunit=True)
    before = qcd.field_to_host(a, Ua).reshape(10, 512, 4, 3, 3)
    qcd.qcd_link_update_push(a, Pa, Ua, 0.1, True, b, Ub, b, Ub)
    got, want = qcd.field_to_host(a, Ua).reshape(10, 512, 4, 3, 3), qcd.field_to_host(a, ref).reshape(10, 512, 4, 3, 3)
    assert np.array_equal(got[1:9], want[1:9]) and np.array_equal(got[0], before[0]) and np.array_equal(got[9], before[9])
    nb = qcd.field_to_host(b, Ub).reshape(10, 512, 4, 3, 3)
    assert np.array_equal(nb[0], want[8])                      # my last interior timeslice -> its lower halo, all links
    assert np.array_equal(nb[9][:, :3], want[1][:, :3])        # my first -> its upper halo, spatial links
    assert np.all(nb[1:9] == 7.0 + 7.0j) and np.all(nb[9][:, 3] == 7.0 + 7.0j)


def test_copy_timeslices_arguments(qcd):
    import torch
    a, b = qcd.Lattice((8, 8, 8, 16), slab=(0, 8)), qcd.Lattice((8, 8, 4, 16), slab=(0, 8))
    Ua, Ub = a.new_matrix_field(), b.new_matrix_field()
    for args, code in (((a, Ua, 0, b, Ub, 0, 1), qcd.EDIMS), ((a, Ua, 9, a, Ua.clone(), 0, 2), qcd.EINVAL),
                       ((a, Ua, 0, a, Ua, 0, 1), qcd.EALIAS)):
        with pytest.raises(qcd.QcdError) as e:
            qcd.qcd_copy_timeslices(*args)
        assert e.value.code == code
    with pytest.raises(qcd.QcdError) as e:
        qcd.Lattice((8, 8, 8, 16), slab=(0, 3))  # odd slab length
    assert e.value.code == qcd.EDIMS
    # mu_mask copies only the selected links
    qcd.qcd_hot_start(a, Ua, 5, 0.5)
    Uc = torch.zeros_like(Ua)
    qcd.qcd_copy_timeslices(a, Ua, 2, a, Uc, 5, 1, 72, 0x5)
    got, src = qcd.field_to_host(a, Uc).reshape(10, 512, 4, 3, 3), qcd.field_to_host(a, Ua).reshape(10, 512, 4, 3, 3)
    assert np.array_equal(got[5, :, 0], src[2, :, 0]) and np.array_equal(got[5, :, 2], src[2, :, 2])
    assert np.all(got[5, :, 1] == 0) and np.all(got[5, :, 3] == 0) and np.all(got[4] == 0)
