"""qcd_plaquette_noalloc: the plaquette for callers that cannot allocate device memory.

Who that is: a routine running inside an application whose memory manager has reserved the whole GPU for its own
pool (the arrangement of PAPER.md:71,83 — the caller has no handle to that pool, and a cudaMalloc of its own
fails or fights it), and measurement code inside a running trajectory, where cudaMalloc / cudaFree would stall
every stream of the device.  Such a caller cannot build the `workspace` that qcd_plaquette wants, so this entry
point keeps the first-pass partial sums in a 256 KiB array that is part of libqcdmd.so (32768 doubles; larger
lattices are refused).

What is checked: its results against qcd_plaquette's on the same field, within the tolerances of the parity tests
(and bit for bit, since both run the same kernels in the same order), on two calls in a row — the second on a
smaller lattice and another field, so that it runs on top of what the first call left in the shared array.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It needs neither the oracle nor any state of the other tests: it passes alone in a fresh process.
"""
import pytest

TOL = {"f64": 1e-12, "f32": 2e-5}  # tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def qcd():
    from paper_1212_0785_b200 import binding
    return binding


def test_lattices_beyond_the_built_in_scratch_are_refused_before_any_cuda_call(qcd):
    """32768 partial sums are all the array holds: 64^3 x 130 needs 2*130*128 = 33280 -> QCD_EWORKSPACE, nothing
    enqueued (the pointers are fake and never dereferenced)"""
    big = qcd.Lattice((64, 64, 64, 130))
    a, out = 0x10000000, 0x20000000
    assert qcd.lib.qcd_plaquette_noalloc(big.handle, qcd.F64, a, out, None, None) == qcd.EWORKSPACE
    text = qcd.lib.qcd_last_error().decode()
    assert "33280" in text and "32768" in text and "qcd_plaquette" in text
    small = qcd.Lattice((4, 4, 4, 4))
    assert qcd.lib.qcd_plaquette_noalloc(small.handle, qcd.F64, a, None, None, None) == qcd.EINVAL
    assert qcd.lib.qcd_plaquette_noalloc(small.handle, qcd.F64, a + 8, out, None, None) == qcd.EALIGN
    assert qcd.lib.qcd_plaquette_noalloc(None, qcd.F64, a, out, None, None) == qcd.EINVAL


def _both_paths(qcd, torch, dims, dtype, seed, sigma):
    """(avg, per_t) of a seeded hot-start field from qcd_plaquette_noalloc and from qcd_plaquette"""
    lat = qcd.Lattice(dims)
    U = lat.new_matrix_field(dtype)
    qcd.qcd_hot_start(lat, U, seed, sigma)
    avg = torch.full((2, 1), float("nan"), dtype=torch.float64, device="cuda")
    per_t = torch.full((2, dims[3]), float("nan"), dtype=torch.float64, device="cuda")
    qcd.qcd_plaquette_noalloc(lat, U, avg[0], per_t[0])
    qcd.qcd_plaquette(lat, U, avg[1], per_t[1], lat.new_workspace())
    torch.cuda.synchronize()
    return avg.cpu().numpy(), per_t.cpu().numpy()


@pytest.mark.gpu
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_two_calls_in_a_row_match_the_workspace_path(qcd, prec):
    import numpy as np
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    dtype = torch.float64 if prec == "f64" else torch.float32
    tol = TOL[prec]
    # call 1 fills 2*32*2 = 128 slots of the array; call 2 (16 slots, other field) runs over their remains
    for dims, seed, sigma in (((16, 16, 16, 32), 0x1212078500000003, 0.5), ((4, 6, 2, 8), 77, 0.2)):
        avg, per_t = _both_paths(qcd, torch, dims, dtype, seed, sigma)
        assert np.isfinite(avg).all() and np.isfinite(per_t).all()
        assert 0.0 < avg[1, 0] < 1.0  # a hot start is neither ordered nor garbage
        assert abs(avg[0, 0] - avg[1, 0]) / abs(avg[1, 0]) < tol
        assert np.abs(per_t[0] - per_t[1]).max() / np.abs(per_t[1]).max() < tol
        # same kernels, same order: not merely close
        assert avg[0, 0] == avg[1, 0] and np.array_equal(per_t[0], per_t[1])
    # without the per-timeslice output, twice on one stream with no host synchronisation in between
    lat = qcd.Lattice((8, 8, 8, 16))
    U1, U2 = lat.new_matrix_field(dtype), lat.new_matrix_field(dtype)
    qcd.qcd_hot_start(lat, U1, 5, 0.3)
    qcd.qcd_hot_start(lat, U2, 6, 0.6)
    got = torch.zeros(2, dtype=torch.float64, device="cuda")
    want = torch.zeros(2, dtype=torch.float64, device="cuda")
    qcd.qcd_plaquette_noalloc(lat, U1, got[0:1], None)
    qcd.qcd_plaquette_noalloc(lat, U2, got[1:2], None)
    ws = lat.new_workspace()
    qcd.qcd_plaquette(lat, U1, want[0:1], None, ws)
    qcd.qcd_plaquette(lat, U2, want[1:2], None, ws)
    torch.cuda.synchronize()
    g, w = got.cpu().numpy(), want.cpu().numpy()
    assert g[0] != g[1]
    assert np.abs(g - w).max() / np.abs(w).max() < tol and np.array_equal(g, w)
