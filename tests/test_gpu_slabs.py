"""domain decomposition in t with a one-site halo, tested on ONE GPU: the lattice is split
into 2 and 4 slabs in one process, halos travel through qcd_copy_timeslices (what peer stores over NVLink would
do), and the gathered result must equal the undecomposed lattice — bit for bit for the generator, and for the
trajectory because every site runs the same arithmetic in the same order whatever tile it falls in — and the
oracle within the usual tolerance.  PAPER.md:24 (multi-GPU support), PAPER.md:121 (overlap, work in progress)."""
import json
import os
import socket
import subprocess
import sys
import time

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


# ---- DistSlab: one slab per PROCESS, faces through torch.distributed (the class a multi-GPU job runs) ----------

def _full_lattice_leapfrog(qcd, dims, prec, beta, eps, n, seed):
    full = qcd.Lattice(dims)
    dt = tdtype(prec)
    fU, fP = full.new_matrix_field(dt), full.new_matrix_field(dt)
    qcd.qcd_hot_start(full, fU, seed, 0.5)
    qcd.qcd_mom_refresh(full, fP, seed)
    qcd.qcd_leapfrog(full, fU, fP, beta, eps, n)
    return host(qcd, full, fU), host(qcd, full, fP)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(8, 8, 8, 16), (4, 6, 2, 8), (2, 2, 2, 4)])
def test_dist_slab_alone_equals_the_whole_lattice(qcd, dims, prec):
    """world = 1: the slab's halos are its own boundary timeslices, sent to itself as compact face messages (only the
    chunks of one timeslice, three links for the face that goes down); bit-identical to qcd_leapfrog"""
    import torch
    from paper_1212_0785_b200 import slabs
    beta, eps, n, seed = 5.8, 0.05, 3, 0x1212078500000002
    wU, wP = _full_lattice_leapfrog(qcd, dims, prec, beta, eps, n, seed)
    ds = slabs.DistSlab(qcd, dims, slabs.SlabComm(0, 1), tdtype(prec))
    ds.start(seed, 0.5)
    ds.leapfrog(beta, eps, n)
    torch.cuda.synchronize()
    assert np.array_equal(ds.gather("U"), wU) and np.array_equal(ds.gather("P"), wP)
    # a face message holds one timeslice, not the two-timeslice staging field
    Vs = dims[0] * dims[1] * dims[2]
    up, down = ds.face(ds.n, slabs.MASK_ALL), ds.face(1, slabs.MASK_SPATIAL)
    assert up.shape[1:] == (36, 32, 2) and down.shape[1:] == (27, 32, 2)
    assert up.shape[0] <= (Vs // 2 + 31) // 32 * 2 + 1 and up.is_contiguous() and down.is_contiguous()
    # and the observables are the whole lattice's
    full = qcd.Lattice(dims)
    ws = full.new_workspace()
    avg = torch.zeros(1, dtype=torch.float64, device="cuda")
    per_t = torch.zeros(dims[3], dtype=torch.float64, device="cuda")
    qcd.qcd_plaquette(full, qcd.field_to_device(full, wU, tdtype(prec)), avg, per_t, ws)
    plaq, K, plaq_t = ds.global_observables(beta)
    # (the two parities of a timeslice are summed in the slab's local order: equal up to rounding, not bit for bit)
    assert np.abs(plaq_t.cpu().numpy() - per_t.cpu().numpy()).max() < TOL[prec] and abs(plaq - avg.item()) < TOL[prec]


def _dist_slab_worker(rank, world, port, out, dims, prec, beta, eps, n, seed):
    """one rank of a DistSlab job: every rank uses cuda:0 (the box has one GPU); faces and reductions travel over gloo
    through host memory.  The ranks' kernels never wait on one another: each rank's host blocks in the exchange."""
    import datetime

    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world, timeout=datetime.timedelta(seconds=90))
    torch.cuda.set_device(0)
    from paper_1212_0785_b200 import binding as qcd
    from paper_1212_0785_b200 import slabs
    ds = slabs.DistSlab(qcd, dims, slabs.SlabComm(rank, world, dist), tdtype(prec))
    ds.start(seed, 0.5)
    ds.leapfrog(beta, eps, n)
    plaq, K, plaq_t = ds.global_observables(beta)
    torch.cuda.synchronize()
    np.savez(f"{out}.{rank}.npz", U=ds.gather("U"), P=ds.gather("P"), plaq=plaq, K=K, plaq_t=plaq_t.cpu().numpy(),
             t_begin=ds.t_begin, t_count=ds.n)
    dist.destroy_process_group()


@pytest.mark.parametrize("dims,world,prec", [((8, 8, 8, 16), 2, "f64"), ((4, 6, 2, 12), 3, "f64"), ((8, 8, 8, 16), 2, "f32")])
def test_dist_slab_processes_equal_the_whole_lattice(qcd, orc_omp, tmp_path, dims, world, prec):
    """the decomposition as a multi-GPU job runs it — one process per slab, halo faces exchanged between processes
     — here with all processes on the one GPU and gloo as the transport: the gathered trajectory is
    bit-identical to the undecomposed run and within tolerance of the oracle, and every rank holds the same global
    observables"""
    import torch
    import torch.multiprocessing as mp
    beta, eps, n, seed = 5.8, 0.05, 3, 0x1212078500000002
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    out = str(tmp_path / "ds")
    ctx = mp.start_processes(_dist_slab_worker, args=(world, port, out, dims, prec, beta, eps, n, seed), nprocs=world,
                             join=False, start_method="spawn")
    deadline = time.time() + 240.0
    try:
        while not ctx.join(timeout=5.0):
            assert time.time() < deadline, "DistSlab ranks did not finish"
    finally:
        for p in ctx.processes:  # only the processes this test started
            if p.is_alive():
                p.kill()
    res = [np.load(f"{out}.{r}.npz") for r in range(world)]
    assert [int(x["t_begin"]) for x in res] == sorted(int(x["t_begin"]) for x in res)
    gU, gP = np.concatenate([x["U"] for x in res]), np.concatenate([x["P"] for x in res])
    wU, wP = _full_lattice_leapfrog(qcd, dims, prec, beta, eps, n, seed)
    assert np.array_equal(gU, wU) and np.array_equal(gP, wP)
    full = qcd.Lattice(dims)
    dt = tdtype(prec)
    fU, fP = full.new_matrix_field(dt), full.new_matrix_field(dt)
    qcd.qcd_hot_start(full, fU, seed, 0.5)
    qcd.qcd_mom_refresh(full, fP, seed)
    rU, rP = orc_omp.leapfrog(dims, beta, eps, n, host(qcd, full, fU), host(qcd, full, fP))
    assert rel(gU, rU) < TOL[prec] and rel(gP, rP) < TOL[prec]
    rplaq, rper_t = orc_omp.plaquette(dims, rU)
    rK = orc_omp.sum(dims, O.SUM_NORM2, rP.view(np.float64).reshape(full.V, 72))[0]
    for x in res:
        assert float(x["plaq"]) == float(res[0]["plaq"]) and float(x["K"]) == float(res[0]["K"])
        assert np.array_equal(x["plaq_t"], res[0]["plaq_t"]) and x["plaq_t"].shape == (dims[3],)
        assert abs(float(x["plaq"]) - rplaq) < TOL[prec] and abs(float(x["K"]) - rK) < TOL[prec] * rK
        assert np.abs(x["plaq_t"] - rper_t).max() < TOL[prec]


@pytest.mark.parametrize("world", [1, 2])
def test_bench_decompose_mode_runs(world):
    """bench.py --decompose (one lattice cut into one slab per rank, DistSlab) prints one strong-scaling JSON object;
    world = 2: two ranks share the one GPU over gloo — a check of the N > 1 code path, not a measurement"""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    tail = [os.path.join(root, "bench.py"), "--gpus", str(world), "--decompose", "--config", "3", "--steps", "2"]
    cmd = [sys.executable] + tail if world == 1 else \
        [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world), "--master-addr",
         "127.0.0.1", "--master-port", str(port)] + tail + ["--backend", "gloo"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=root)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1  # rank 0 only
    d = json.loads(lines[0])
    assert d["scaling"] == "strong" and d["n_gpus"] == world and d["config"]["mode"] == "decompose"
    assert d["value"] > 0 and 0.0 < d["plaquette"] < 1.0 and d["kinetic_energy"] > 0
    assert d["config"]["sent_bytes_per_rank_per_step"] == 16 ** 3 * (72 + 54) * 8  # one timeslice up, three links down
