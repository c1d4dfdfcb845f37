"""Pins for the oracle's pseudofermion-side site operations (O15 Gaussian spin-colour fill, O16 inner
product; "a pseudofermion refresh", PAPER.md:26 reductions; R21): generator-block
layout retyped from the definition, Gaussian moments, numpy's vdot, sesquilinearity.  All CPU."""
import numpy as np

from oracle import oracle as O
from tests import inputs


def test_spinor_gaussian_block_layout_and_subsets(orc):
    dims = (4, 2, 2, 4)
    seed = inputs.config_seed(3)
    eta = orc.spinor_gaussian(dims, seed, stream_id=5)
    for s in (0, 7, 63):
        for k in (0, 5, 11):
            g = orc.rng_block(seed, s, 4, k, 5, 4)[2]  # counter (s, 64 + k, stream 5, purpose 4)
            assert abs(eta[s, k] - complex(g[0], g[1]) / np.sqrt(2.0)) <= 4e-16 * abs(eta[s, k])
    assert not np.array_equal(eta, orc.spinor_gaussian(dims, seed, stream_id=6))  # streams are independent
    par = orc.map(dims, O.MAP_PARITY)
    e = orc.spinor_gaussian(dims, seed, stream_id=5, subset=O.EVEN)
    assert np.array_equal(e[par == 0], eta[par == 0]) and np.all(e[par == 1] == 0)
    # never the momentum / hot-start numbers: other purpose and counter range
    P = orc.mom_refresh(dims, seed, stream_id=5)
    assert abs(np.corrcoef(eta[:, 0].real, P[:, 0, 0, 1].real)[0, 1]) < 0.2


def test_spinor_gaussian_moments(orc_omp):
    dims = (8, 8, 8, 16)
    eta = orc_omp.spinor_gaussian(dims, 12345)
    n = eta.size
    x = np.concatenate([eta.real.ravel(), eta.imag.ravel()])
    sig = 4 / np.sqrt(2 * n)
    assert abs(x.mean()) < sig
    assert abs(x.var() - 0.5) < sig  # re and im ~ N(0, 1/2): <|eta_k|^2> = 1, weight exp(-eta^dag eta)
    assert abs(np.mean(x ** 4) / x.var() ** 2 - 3) < 6 * sig * 4
    assert abs(np.mean(eta.real * eta.imag)) < sig
    norm2 = orc_omp.sum(dims, O.SUM_NORM2, eta.view(np.float64).reshape(eta.shape[0], 24))
    assert abs(norm2 / n - 1) < 4 / np.sqrt(n)
    # components and neighbouring sites are uncorrelated
    assert abs(np.mean(eta[:, 0] * np.conj(eta[:, 1]))) < 4 / np.sqrt(eta.shape[0])
    assert abs(np.mean(eta[:-1, 3] * np.conj(eta[1:, 3]))) < 4 / np.sqrt(eta.shape[0])


def test_inner_product_against_numpy_and_sesquilinearity(orc):
    dims = (4, 6, 2, 4)
    V = int(np.prod(dims))
    rng = np.random.default_rng(5)
    a = rng.standard_normal((V, 12)) + 1j * rng.standard_normal((V, 12))
    b = rng.standard_normal((V, 12)) + 1j * rng.standard_normal((V, 12))
    ip = orc.inner_product(dims, a, b)
    assert np.isclose(ip, np.vdot(a, b), rtol=1e-13)  # vdot conjugates its first argument
    assert np.isclose(orc.inner_product(dims, b, a), np.conj(ip), rtol=1e-13)
    z = 0.3 - 1.7j
    assert np.isclose(orc.inner_product(dims, a, z * b), z * ip, rtol=1e-13)
    assert np.isclose(orc.inner_product(dims, z * a, b), np.conj(z) * ip, rtol=1e-13)
    aa = orc.inner_product(dims, a, a)
    assert aa.imag == 0 and np.isclose(aa.real, orc.sum(dims, O.SUM_NORM2, a.view(np.float64).reshape(V, 24)), rtol=1e-14)
    par = orc.map(dims, O.MAP_PARITY)
    assert np.isclose(orc.inner_product(dims, a, b, subset=O.ODD), np.vdot(a[par == 1], b[par == 1]), rtol=1e-13)
    per_t = orc.inner_product_multi(dims, a, b)
    Vs = V // dims[3]
    ref = np.array([np.vdot(a[t * Vs:(t + 1) * Vs], b[t * Vs:(t + 1) * Vs]) for t in range(dims[3])])
    assert np.allclose(per_t, ref, rtol=1e-13) and np.isclose(per_t.sum(), ip, rtol=1e-13)
    # other component counts (e.g. a colour vector, 3 components)
    a3, b3 = np.ascontiguousarray(a[:, :3]), np.ascontiguousarray(b[:, :3])
    assert np.isclose(orc.inner_product(dims, a3, b3), np.vdot(a3, b3), rtol=1e-13)
