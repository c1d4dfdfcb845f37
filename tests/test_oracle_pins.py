"""Pins for the CPU oracle (oracle/), against what the mathematics fixes — never against itself.

Every test cites the definition in SURVEY.md section 8(c) (O1..O12) / DESIGN.md it pins; the paper
passage that names the operation is PAPER.md:17 (section 1) and PAPER.md:26 for the reductions.
All CPU, no GPU marker.
"""
import os

import numpy as np
import pytest
import scipy.linalg

from oracle import oracle as O
from tests import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")

# Gell-Mann matrices retyped here from the textbook table (independent of the oracle's O2 code)
_s3 = np.sqrt(3.0)
LAMBDA = np.array([
    [[0, 1, 0], [1, 0, 0], [0, 0, 0]],
    [[0, -1j, 0], [1j, 0, 0], [0, 0, 0]],
    [[1, 0, 0], [0, -1, 0], [0, 0, 0]],
    [[0, 0, 1], [0, 0, 0], [1, 0, 0]],
    [[0, 0, -1j], [0, 0, 0], [1j, 0, 0]],
    [[0, 0, 0], [0, 0, 1], [0, 1, 0]],
    [[0, 0, 0], [0, 0, -1j], [0, 1j, 0]],
    [[1 / _s3, 0, 0], [0, 1 / _s3, 0], [0, 0, -2 / _s3]],
], dtype=np.complex128)
T = LAMBDA / 2


def dag(m):
    return np.conj(np.swapaxes(m, -1, -2))


def unit_gauge(V):
    U = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1
    return U


# ------------------------------------------------------------------ O1 maps

@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 4), (4, 4, 4, 4), (6, 4, 2, 8)])
def test_maps_bruteforce(orc, dims):
    Lx, Ly, Lz, Lt = dims
    V = Lx * Ly * Lz * Lt
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    x, y, z, t = (a.reshape(-1) for a in (x, y, z, t))
    s = x + Lx * (y + Ly * (z + Lz * t))
    assert np.array_equal(s, np.arange(V))
    par = (x + y + z + t) & 1
    assert np.array_equal(orc.map(dims, O.MAP_PARITY), par)
    assert np.array_equal(orc.map(dims, O.MAP_TSLICE), t)
    cb = orc.map(dims, O.MAP_CB_OF_LEX)
    assert np.array_equal(cb, par * (V // 2) + (s >> 1))
    # bijection, V/2 per parity, even sites first
    assert np.array_equal(np.sort(cb), np.arange(V))
    assert np.all(cb[par == 0] < V // 2) and np.all(cb[par == 1] >= V // 2)
    lex = orc.map(dims, O.MAP_LEX_OF_CB)
    assert np.array_equal(lex[cb], s)
    c = [x, y, z, t]
    for mu in range(4):
        cf = [a.copy() for a in c]
        cf[mu] = (cf[mu] + 1) % dims[mu]
        sf = cf[0] + Lx * (cf[1] + Ly * (cf[2] + Lz * cf[3]))
        fwd = orc.map(dims, O.MAP_NBR_FWD0 + mu)
        bwd = orc.map(dims, O.MAP_NBR_BWD0 + mu)
        assert np.array_equal(fwd, sf)
        assert np.array_equal(bwd[fwd], s) and np.array_equal(fwd[bwd], s)
        assert np.all(par[fwd] != par)  # each hop flips parity
        h = s.copy()
        for _ in range(dims[mu]):
            h = fwd[h]
        assert np.array_equal(h, s)  # L_mu hops = identity


def test_map_rejects_odd_or_small_extents(orc):
    for dims in [(3, 4, 4, 4), (4, 4, 4, 1), (0, 2, 2, 2)]:
        with pytest.raises(ValueError):
            orc.map(dims, O.MAP_PARITY)


# ------------------------------------------------------------------ O3 RNG

def test_philox_known_answers(orc):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(h, 16) for h in r]
        assert orc.philox(v[0:4], v[4:6]) == v[6:10]


def test_rng_block_counter_layout_and_uniforms(orc):
    seed = 0x0123456789ABCDEF
    s, mu, j, stream, purpose = 1234, 3, 2, 7, 1
    w, u, g = orc.rng_block(seed, s, mu, j, stream, purpose)
    # counter = (s, mu*16+j, stream_id, purpose), key = (seed low, seed high)
    assert w == orc.philox([s, mu * 16 + j, stream, purpose], [seed & 0xFFFFFFFF, seed >> 32])
    # u = (2k+1) 2^-53 with k the top 26 bits of each word pair: exact dyadic strictly inside (0,1)
    for (wa, wb), uu in (((w[0], w[1]), u[0]), ((w[2], w[3]), u[1])):
        k = ((wa >> 6) << 26) | (wb >> 6)
        assert uu == (2 * k + 1) / 2.0 ** 53
        assert 0.0 < uu < 1.0
        m = uu * 2.0 ** 53
        assert m == int(m) and int(m) % 2 == 1
    # Box-Muller pair
    r = np.sqrt(-2 * np.log(u[0]))
    assert np.allclose(g, [r * np.cos(2 * np.pi * u[1]), r * np.sin(2 * np.pi * u[1])], rtol=1e-14, atol=1e-15)


def test_uniform_extremes_stay_inside_unit_interval(orc):
    # all-zero and all-one words are the extreme k; the map must stay strictly inside (0,1)
    k_max = (1 << 52) - 1
    assert (2 * 0 + 1) / 2.0 ** 53 > 0.0
    assert (2 * k_max + 1) / 2.0 ** 53 < 1.0
    assert float(2 * k_max + 1) == 2 * k_max + 1  # exactly representable


def test_gaussian_moments_and_kinetic_energy(orc_omp):
    dims = (16, 16, 16, 8)  # 32768 sites * 4 links * 8 = 1,048,576 Gaussians
    V = int(np.prod(dims))
    P = orc_omp.mom_refresh(dims, seed=inputs.config_seed(3))
    # p_a = 2 tr(T_a P) with the test's own Gell-Mann table
    p = 2 * np.einsum("aij,xmji->xma", T, P).real.reshape(-1)
    n = p.size
    assert n == 1 << 20
    assert abs(p.mean()) < 4 / np.sqrt(n)
    assert abs(p.var() - 1) < 4 * np.sqrt(2 / n)
    kurt = np.mean((p - p.mean()) ** 4) / p.var() ** 2
    assert abs(kurt - 3) < 4 * np.sqrt(24 / n)
    # no correlation between the two Box-Muller outputs or between neighbouring links
    pa = p.reshape(V, 4, 8)
    assert abs(np.mean(pa[:, :, 0] * pa[:, :, 1])) < 5 / np.sqrt(V * 4)
    assert abs(np.mean(pa[:, 0, :] * pa[:, 1, :])) < 5 / np.sqrt(V * 8)
    # P Hermitian traceless; K = sum tr P^2 = 1/2 sum p_a^2 ; <K> = 16 V
    assert np.abs(P - dag(P)).max() == 0
    assert np.abs(np.trace(P, axis1=-2, axis2=-1)).max() < 1e-15
    K = orc_omp.sum(dims, O.SUM_NORM2, P)[0]
    assert np.isclose(K, 0.5 * np.sum(p ** 2), rtol=1e-12)
    assert abs(K / (16 * V) - 1) < 4 * np.sqrt(2.0 / (32 * V))


def test_rng_is_independent_of_subset_and_stream(orc):
    dims = (4, 4, 4, 4)
    seed = 99
    P = orc.mom_refresh(dims, seed)
    Pe = orc.mom_refresh(dims, seed, subset=O.EVEN)
    Po = orc.mom_refresh(dims, seed, subset=O.ODD)
    par = orc.map(dims, O.MAP_PARITY)
    assert np.array_equal(Pe[par == 0], P[par == 0]) and np.all(Pe[par == 1] == 0)
    assert np.array_equal(Po[par == 1], P[par == 1]) and np.all(Po[par == 0] == 0)
    P2 = orc.mom_refresh(dims, seed, stream_id=1)
    assert not np.any(P2 == P)


# ------------------------------------------------------------------ O2 generators

def test_generators(orc):
    Ts = np.array([orc.herm_from_coeffs(np.eye(8)[a]) for a in range(8)])
    assert np.allclose(Ts, T, atol=1e-16)
    gram = np.einsum("aij,bji->ab", Ts, Ts)
    assert np.allclose(gram, np.eye(8) / 2, atol=1e-15)
    assert np.allclose(Ts, dag(Ts)) and np.allclose(np.trace(Ts, axis1=1, axis2=2), 0)
    q = np.random.default_rng(5).standard_normal(8)
    Q = orc.herm_from_coeffs(q)
    assert np.isclose(np.trace(Q @ Q).real, 0.5 * np.sum(q ** 2))


# ------------------------------------------------------------------ O8 exp

@pytest.mark.parametrize("scale", [1e-8, 0.05, 0.5, 1.4, 5.6, 40.0])
def test_expi_against_library_and_group_properties(orc, scale):
    for Q in inputs.random_hermitian_traceless(11, 20, scale):
        E = orc.expi(Q)
        ref = scipy.linalg.expm(1j * Q)
        assert np.abs(E - ref).max() < 5e-14 * max(1.0, scale)
        assert np.abs(E @ dag(E) - np.eye(3)).max() < 1e-14 * max(1.0, scale)
        assert abs(np.linalg.det(E) - 1) < 1e-14 * max(1.0, scale)
        assert np.abs(E @ orc.expi(-Q) - np.eye(3)).max() < 1e-14 * max(1.0, scale)


def test_expi_closed_forms(orc):
    assert np.array_equal(orc.expi(np.zeros((3, 3))), np.eye(3))
    for a, b in [(0.3, -1.1), (2.0, 0.7), (-4.0, 3.0)]:
        Q = a * T[2] + b * T[7]  # diagonal: span of T3, T8
        th = np.diag(Q).real
        assert np.abs(orc.expi(Q) - np.diag(np.exp(1j * th))).max() < 2e-15 * max(1, np.abs(th).max())
    # degenerate eigenvalues (T8 direction) and a rotation generator with known closed form
    th = 0.9
    E = orc.expi(2 * th * T[1])  # exp(i th lambda_2) = rotation by th in the 1-2 block
    ref = np.array([[np.cos(th), np.sin(th), 0], [-np.sin(th), np.cos(th), 0], [0, 0, 1]])
    assert np.abs(E - ref).max() < 1e-15


# ------------------------------------------------------------------ O6 plaquette

def numpy_plaquette(dims, U):
    """independent brute force with np.roll on a [t,z,y,x,mu,3,3] view"""
    Lx, Ly, Lz, Lt = dims
    A = U.reshape(Lt, Lz, Ly, Lx, 4, 3, 3)
    axis = {0: 3, 1: 2, 2: 1, 3: 0}
    per_site = np.zeros((Lt, Lz, Ly, Lx))
    for mu in range(4):
        for nu in range(mu + 1, 4):
            Umu, Unu = A[..., mu, :, :], A[..., nu, :, :]
            Unu_xpmu = np.roll(Unu, -1, axis=axis[mu])
            Umu_xpnu = np.roll(Umu, -1, axis=axis[nu])
            Pl = Umu @ Unu_xpmu @ dag(Umu_xpnu) @ dag(Unu)
            per_site += np.trace(Pl, axis1=-2, axis2=-1).real / 3
    return per_site.mean() / 6, per_site.mean(axis=(1, 2, 3)) / 6


def test_plaquette_unit_and_pure_gauge(orc):
    dims = (4, 2, 4, 6)
    V = int(np.prod(dims))
    U = unit_gauge(V)
    avg, per_t = orc.plaquette(dims, U)
    assert avg == 1.0 and np.all(per_t == 1.0)
    G, Upure = orc.gauge_transform(dims, 3, 1.0, U)  # U_mu(x) = G(x) G(x+mu)^dagger
    assert np.abs(G @ dag(G) - np.eye(3)).max() < 1e-14
    avg, per_t = orc.plaquette(dims, Upure)
    assert abs(avg - 1) < 1e-14 and np.abs(per_t - 1).max() < 1e-14


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 6, 2, 4)])
def test_plaquette_bruteforce_generic_matrices(orc, dims):
    # generic non-unitary matrices: any index / dagger / ordering slip shows up
    V = int(np.prod(dims))
    U = inputs.random_matrix_field(21, V)
    avg, per_t = orc.plaquette(dims, U)
    ravg, rper_t = numpy_plaquette(dims, U)
    assert np.isclose(avg, ravg, rtol=1e-13)
    assert np.allclose(per_t, rper_t, rtol=1e-13)
    assert np.isclose(per_t.mean(), avg, rtol=1e-13)
    beta = 5.5
    assert np.isclose(orc.action(dims, beta, U), beta * 6 * V * (1 - avg), rtol=1e-12)


def test_plaquette_gauge_invariance_and_hot_start_expectation(orc_omp):
    dims = (8, 8, 8, 8)
    seed = inputs.config_seed(2)
    for sigma, expect in [(0.2, 0.898), (0.3, 0.784), (0.5, 0.503)]:
        U = orc_omp.hot_start(dims, seed, sigma)
        assert np.abs(U @ dag(U) - np.eye(3)).max() < 1e-14
        assert np.abs(np.linalg.det(U) - 1).max() < 1e-14
        avg, per_t = orc_omp.plaquette(dims, U)
        # <plaq> = chi(sigma)^4, chi = <1/3 tr exp(i sigma Q)>: each plaquette is a product of four
        # independent links (SURVEY.md section 8(c) pin table); measure chi from the links themselves
        chi = np.trace(U, axis1=-2, axis2=-1).real.mean() / 3
        assert abs(avg - chi ** 4) < 0.01
        assert abs(avg - expect) < 0.02
        G, Ug = orc_omp.gauge_transform(dims, seed + 17, 1.0, U)
        avg_g, per_t_g = orc_omp.plaquette(dims, Ug)
        assert abs(avg_g - avg) < 1e-13 and np.abs(per_t_g - per_t).max() < 1e-13


# ------------------------------------------------------------------ O7 force

def test_force_equals_finite_difference_of_action(orc):
    """f_a = 2 tr(T_a F) = - dS/d omega_a for U_mu(x) -> exp(i omega T_a) U_mu(x), on 2^4 (north_star)"""
    dims = (2, 2, 2, 2)
    beta = 5.6
    U = orc.hot_start(dims, inputs.config_seed(1), 0.5)
    F = orc.gauge_force(dims, beta, U)
    h = 1e-5
    rng = np.random.default_rng(0)
    worst = 0.0
    for _ in range(6):
        s, mu = int(rng.integers(0, 16)), int(rng.integers(0, 4))
        for a in range(8):
            Up, Um = U.copy(), U.copy()
            Up[s, mu] = scipy.linalg.expm(1j * h * T[a]) @ U[s, mu]
            Um[s, mu] = scipy.linalg.expm(-1j * h * T[a]) @ U[s, mu]
            dS = (orc.action(dims, beta, Up) - orc.action(dims, beta, Um)) / (2 * h)
            fa = 2 * np.trace(T[a] @ F[s, mu]).real
            worst = max(worst, abs(fa + dS))
    assert worst < 5e-8, worst
    assert np.abs(F).max() > 0.1  # the check is not vacuous


def test_force_structure_and_covariance(orc):
    dims = (4, 4, 2, 4)
    V = int(np.prod(dims))
    beta = 6.0
    U = orc.hot_start(dims, 7, 0.5)
    F = orc.gauge_force(dims, beta, U)
    assert np.abs(F - dag(F)).max() < 1e-14  # Hermitian
    assert np.abs(np.trace(F, axis1=-2, axis2=-1)).max() < 1e-14  # traceless
    # unit and pure gauge: zero force
    U1 = unit_gauge(V)
    assert np.abs(orc.gauge_force(dims, beta, U1)).max() == 0
    G, Upure = orc.gauge_transform(dims, 5, 1.0, U1)
    assert np.abs(orc.gauge_force(dims, beta, Upure)).max() < 1e-13
    # covariance F'(x) = G(x) F(x) G(x)^dagger
    G, Ug = orc.gauge_transform(dims, 6, 1.0, U)
    Fg = orc.gauge_force(dims, beta, Ug)
    ref = G[:, None] @ F @ dag(G)[:, None]
    assert np.abs(Fg - ref).max() < 1e-13
    # sum rule: sum_{x,mu} Re tr W_mu(x) = 4 sum_{x,mu<nu} Re tr P_mu_nu(x)
    avg, _ = orc.plaquette(dims, U)
    assert np.isclose(orc.sum_retr_w(dims, U), 4 * 3 * 6 * V * avg, rtol=1e-12)
    # linear in beta
    assert np.allclose(orc.gauge_force(dims, 2 * beta, U), 2 * F, rtol=1e-15)


def test_force_generic_matrices_against_numpy_staples(orc):
    """the formula of O7 on arbitrary (non-unitary) input, via np.roll staples"""
    dims = (4, 2, 2, 4)
    Lx, Ly, Lz, Lt = dims
    V = int(np.prod(dims))
    beta = 5.0
    U = inputs.random_matrix_field(33, V) * 0.5
    A = U.reshape(Lt, Lz, Ly, Lx, 4, 3, 3)
    ax = {0: 3, 1: 2, 2: 1, 3: 0}
    ref = np.zeros_like(A)
    for mu in range(4):
        St = np.zeros(A.shape[:4] + (3, 3), dtype=np.complex128)
        Umu = A[..., mu, :, :]
        for nu in range(4):
            if nu == mu:
                continue
            Unu = A[..., nu, :, :]
            up = np.roll(Unu, -1, ax[mu]) @ dag(np.roll(Umu, -1, ax[nu])) @ dag(Unu)
            Unu_d = np.roll(Unu, +1, ax[nu])  # U_nu(x-nu)
            Umu_d = np.roll(Umu, +1, ax[nu])  # U_mu(x-nu)
            dn = dag(np.roll(Unu_d, -1, ax[mu])) @ dag(Umu_d) @ Unu_d
            St += up + dn
        W = Umu @ St
        X = W - dag(W)
        X = X - np.trace(X, axis1=-2, axis2=-1)[..., None, None] * np.eye(3) / 3
        ref[..., mu, :, :] = 1j * beta / 12 * X
    F = orc.gauge_force(dims, beta, U)
    assert np.abs(F - ref.reshape(V, 4, 3, 3)).max() < 1e-12 * np.abs(ref).max()


def test_force_subsets(orc):
    dims = (4, 4, 4, 2)
    U = orc.hot_start(dims, 8, 0.5)
    F = orc.gauge_force(dims, 5.7, U)
    par = orc.map(dims, O.MAP_PARITY)
    sentinel = np.full_like(F, 7.0)
    Fe = orc.gauge_force(dims, 5.7, U, subset=O.EVEN, out=sentinel.copy())
    assert np.array_equal(Fe[par == 0], F[par == 0]) and np.all(Fe[par == 1] == 7.0)
    Fo = orc.gauge_force(dims, 5.7, U, subset=O.ODD, out=sentinel.copy())
    assert np.array_equal(Fo[par == 1], F[par == 1]) and np.all(Fo[par == 0] == 7.0)


# ------------------------------------------------------------------ O3/O5: perturbation noise (config 3)

def test_perturb_noise_layout_and_moments(orc_omp, orc):
    """"Perturbation noise: 18 Gaussians from blocks 0..8 in storage order [row][col][re,im]",
    purpose 2, counter keyed on the lexicographic site, stride-16 block index mu*16 + j; O5: U + sigma N.
    Rebuilt here by hand from the generator blocks (rng_block itself is pinned by the Philox known answers and
    the uniform / Gaussian tests above), then the moments of the 18 reals over 1.3 x 10^5 links: a wrong block
    index, purpose, storage order, sign or a variance-of-2 slip fails."""
    dims, seed, sigma = (16, 16, 16, 8), 0x1212078500000003, 1e-3
    V = O.Oracle.volume(dims)
    U = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    N = orc_omp.perturb(dims, seed, sigma, U) / sigma  # the noise itself
    # elements by hand: entry e = 3*row + col of link (s, mu) is g[0] + i g[1] of block (s, mu, j = e, stream 0, purpose 2)
    for s_, mu, row, col in [(0, 0, 0, 0), (V - 1, 3, 2, 2), (4711, 2, 1, 2), (17, 1, 2, 0), (V // 2 + 5, 0, 0, 1)]:
        g = orc.rng_block(seed, s_, mu, 3 * row + col, 0, 2)[2]
        assert abs(N[s_, mu, row, col] - (g[0] + 1j * g[1])) < 1e-12
    # other purposes / streams / a neighbouring block give different numbers
    g1 = orc.rng_block(seed, 0, 0, 0, 0, 1)[2]
    g2 = orc.rng_block(seed, 0, 0, 1, 0, 2)[2]
    assert abs(N[0, 0, 0, 0] - (g1[0] + 1j * g1[1])) > 1e-6 and abs(N[0, 0, 0, 0] - (g2[0] + 1j * g2[1])) > 1e-6
    # perturbation is additive and linear in sigma
    U0 = orc_omp.hot_start(dims, 5, 0.5)
    assert np.abs(orc_omp.perturb(dims, seed, sigma, U0) - (U0 + sigma * N)).max() < 1e-15
    # moments: 18 iid N(0,1) reals per link
    x = N.reshape(-1, 9).view(np.float64).reshape(-1, 18)
    n = x.shape[0]
    assert n >= 100000
    assert np.abs(x.mean(axis=0)).max() < 5 / np.sqrt(n)
    assert np.abs(x.var(axis=0) - 1).max() < 5 * np.sqrt(2.0 / n)
    assert abs((x ** 4).mean() - 3) < 5 * np.sqrt(96.0 / x.size)
    c = np.corrcoef(x.T)
    assert np.abs(c - np.eye(18)).max() < 5 / np.sqrt(n)  # re/im and entries uncorrelated
    # and across links of a site / neighbouring sites
    flat = x.reshape(V, 4 * 18)
    assert abs(np.corrcoef(flat[:, 0], flat[:, 18])[0, 1]) < 5 / np.sqrt(V)
    assert abs(np.corrcoef(flat[:-1, 0], flat[1:, 0])[0, 1]) < 5 / np.sqrt(V)


# ------------------------------------------------------------------ O9, O10

def test_reunit_pins(orc):
    dims = (4, 4, 2, 2)
    U = orc.hot_start(dims, 12, 0.5)
    Up = orc.perturb(dims, 13, 1e-3, U)
    assert 1e-4 < np.abs(Up - U).max() < 1e-2
    R = orc.reunit(dims, Up)
    assert np.abs(R @ dag(R) - np.eye(3)).max() < 2e-15
    assert np.abs(np.linalg.det(R) - 1).max() < 2e-15
    assert np.abs(orc.reunit(dims, R) - R).max() < 2e-15  # idempotent
    assert np.abs(orc.reunit(dims, U) - U).max() < 2e-15  # identity on SU(3)
    assert np.abs(R - U).max() < 1e-2  # moves a sigma=1e-3 perturbed link by O(sigma)
    # row Gram-Schmidt specifically: first row keeps its direction, second stays in span(r0, r1)
    M = inputs.random_complex_matrices(4, 1)[0]
    Rm = orc.reunit_mat(M)
    assert np.allclose(Rm[0], M[0] / np.linalg.norm(M[0]))
    r1 = M[1] - np.vdot(Rm[0], M[1]) * Rm[0]
    assert np.allclose(Rm[1], r1 / np.linalg.norm(r1))
    assert np.allclose(Rm[2], np.conj(np.cross(Rm[0], Rm[1])))
    # subsets leave the other parity bit-identical
    par = orc.map(dims, O.MAP_PARITY)
    Re = orc.reunit(dims, Up, subset=O.EVEN)
    assert np.array_equal(Re[par == 1], Up[par == 1]) and np.array_equal(Re[par == 0], R[par == 0])


def test_mom_and_link_update(orc):
    dims = (2, 4, 2, 4)
    V = int(np.prod(dims))
    F = inputs.random_matrix_field(1, V)
    P = inputs.random_matrix_field(2, V)
    eps = 0.37
    Pn = orc.mom_update(dims, eps, F, P)
    assert np.array_equal(Pn, P + eps * F)
    par = orc.map(dims, O.MAP_PARITY)
    Po = orc.mom_update(dims, eps, F, P, subset=O.ODD)
    assert np.array_equal(Po[par == 0], P[par == 0]) and np.array_equal(Po[par == 1], Pn[par == 1])
    # U <- exp(i eps P) U against the library exponential
    Ph = orc.mom_refresh(dims, 5)
    U = orc.hot_start(dims, 6, 0.5)
    Un = orc.link_update(dims, eps, Ph, U)
    ref = np.array([scipy.linalg.expm(1j * eps * p) @ u for p, u in zip(Ph.reshape(-1, 3, 3), U.reshape(-1, 3, 3))])
    assert np.abs(Un.reshape(-1, 3, 3) - ref).max() < 5e-15
    Ur = orc.link_update(dims, eps, Ph, U, reunit=True)
    assert np.abs(Ur - orc.reunit(dims, Un)).max() == 0
    Ue = orc.link_update(dims, eps, Ph, U, subset=O.EVEN)
    assert np.array_equal(Ue[par == 1], U[par == 1]) and np.array_equal(Ue[par == 0], Un[par == 0])


# ------------------------------------------------------------------ O11 leapfrog

def test_leapfrog_reversibility(orc_omp):
    c = inputs.CONFIGS[2]
    dims = (4, 4, 4, 8)
    U0 = orc_omp.hot_start(dims, inputs.config_seed(2), c["sigma"])
    P0 = orc_omp.mom_refresh(dims, inputs.config_seed(2))
    U1, P1 = orc_omp.leapfrog(dims, c["beta"], c["eps"], 10, U0, P0)
    assert np.abs(U1 - U0).max() > 0.1
    U2, P2 = orc_omp.leapfrog(dims, c["beta"], c["eps"], 10, U1, -P1)
    assert np.abs(U2 - U0).max() < 1e-13
    assert np.abs(-P2 - P0).max() < 1e-13


def test_leapfrog_dH_scales_as_eps_squared(orc_omp):
    dims = (4, 4, 4, 4)
    beta = 5.6
    U0 = orc_omp.hot_start(dims, inputs.config_seed(1), 0.5)
    P0 = orc_omp.mom_refresh(dims, inputs.config_seed(1))
    K0, S0 = orc_omp.hamiltonian(dims, beta, U0, P0)
    tau = 0.2
    dH = []
    for n in (4, 8, 16, 32):
        U1, P1 = orc_omp.leapfrog(dims, beta, tau / n, n, U0, P0)
        K1, S1 = orc_omp.hamiltonian(dims, beta, U1, P1)
        dH.append(K1 + S1 - K0 - S0)
    ratios = [dH[i] / dH[i + 1] for i in range(3)]
    assert abs(ratios[1] - 4) < 0.2 and abs(ratios[2] - 4) < 0.06, (dH, ratios)
    # one leapfrog step = fused md_step with half steps: P += eps/2 F; U; P += eps/2 F
    eps = 0.1
    Ua, Pa = orc_omp.leapfrog(dims, beta, eps, 1, U0, P0)
    Ub, Pb = orc_omp.md_step(dims, beta, eps / 2, eps, U0, P0)
    Pb = orc_omp.mom_update(dims, eps / 2, orc_omp.gauge_force(dims, beta, Ub), Pb)
    assert np.array_equal(Ua, Ub) and np.array_equal(Pa, Pb)


# ------------------------------------------------------------------ O12 sums

def test_sums_closed_forms(orc):
    dims = (4, 2, 4, 6)
    Lx, Ly, Lz, Lt = dims
    V = int(np.prod(dims))
    par = orc.map(dims, O.MAP_PARITY).astype(np.float64)
    tsl = orc.map(dims, O.MAP_TSLICE).astype(np.float64)
    const = np.full((V, 1), 2.5)
    assert orc.sum(dims, O.SUM_SCALAR, const)[0] == 2.5 * V
    assert orc.sum(dims, O.SUM_SCALAR, const, subset=O.EVEN)[0] == 2.5 * V / 2
    f = np.stack([tsl, 1 - 2 * par], axis=1)
    out = orc.sum(dims, O.SUM_SCALAR, f)
    assert out[0] == (V // Lt) * Lt * (Lt - 1) / 2 and out[1] == 0
    assert orc.sum(dims, O.SUM_SCALAR, f, subset=O.EVEN)[1] == V / 2
    assert orc.sum(dims, O.SUM_SCALAR, f, subset=O.ODD)[1] == -V / 2
    m = orc.sum_multi(dims, O.SUM_SCALAR, f)
    assert np.array_equal(m[:, 0], np.arange(Lt) * (V // Lt)) and np.all(m[:, 1] == 0)
    # matrix kinds against numpy
    M = inputs.random_matrix_field(9, V)
    assert np.isclose(orc.sum(dims, O.SUM_NORM2, M)[0], np.sum(np.abs(M) ** 2), rtol=1e-13)
    assert np.isclose(orc.sum(dims, O.SUM_RETR, M)[0], np.trace(M, axis1=-2, axis2=-1).real.sum(), rtol=1e-12)
    ids = inputs.random_subset_ids(3, V, 5)
    mm = orc.sum_multi(dims, O.SUM_NORM2, M, subset_id=ids, nsub=5)
    ref = np.array([np.sum(np.abs(M[ids == k]) ** 2) for k in range(5)])
    assert np.allclose(mm, ref, rtol=1e-13)
    assert np.isclose(mm.sum(), orc.sum(dims, O.SUM_NORM2, M)[0], rtol=1e-13)
    # long-double accumulation: a sum that plain fp64 left-to-right gets wrong
    big = np.zeros((V, 1))
    big[0, 0] = 1e16
    big[1:, 0] = 1.0
    assert orc.sum(dims, O.SUM_SCALAR, big)[0] == 1e16 + (V - 1)


def test_hamiltonian_pieces(orc):
    dims = (2, 2, 4, 4)
    V = int(np.prod(dims))
    U = orc.hot_start(dims, 4, 0.3)
    P = orc.mom_refresh(dims, 4)
    K, S = orc.hamiltonian(dims, 5.9, U, P)
    assert np.isclose(K, np.einsum("xmij,xmji->", P, P).real, rtol=1e-13)  # K = sum tr P^2
    avg, _ = orc.plaquette(dims, U)
    assert np.isclose(S, 5.9 * 6 * V * (1 - avg), rtol=1e-13)


def test_serial_and_openmp_builds_agree_bitwise(orc, orc_omp):
    dims = (4, 4, 4, 4)
    U = orc.hot_start(dims, 1, 0.5)
    assert np.array_equal(U, orc_omp.hot_start(dims, 1, 0.5))
    P = orc.mom_refresh(dims, 1)
    Ua, Pa = orc.leapfrog(dims, 5.6, 0.1, 2, U, P)
    Ub, Pb = orc_omp.leapfrog(dims, 5.6, 0.1, 2, U, P)
    assert np.array_equal(Ua, Ub) and np.array_equal(Pa, Pb)
    assert orc.plaquette(dims, Ua)[0] == orc_omp.plaquette(dims, Ub)[0]
    assert orc.num_threads() == 1


def test_force_at_listed_sites_is_the_full_force(orc):
    dims = (4, 4, 2, 4)
    U = orc.hot_start(dims, 3, 0.5)
    F = orc.gauge_force(dims, 5.5, U)
    sites = np.array([0, 5, 127, 17, 5], dtype=np.int32)
    assert np.array_equal(orc.gauge_force_sites(dims, 5.5, U, sites), F[sites])


def test_oracle_reproduces_stored_config_values(orc):
    """tests/golden/config_values.json (written by tests/golden/make_config_values.py from the oracle alone):
    the oracle still gives the same config-1 observables; hot-start plaquette near its expectation chi(sigma)^4"""
    import json
    g = json.load(open(os.path.join(GOLDEN, "config_values.json")))["1"]
    dims, beta = tuple(g["dims"]), g["beta"]
    seed = int(g["seed"], 16)
    U0, P0 = orc.hot_start(dims, seed, g["sigma"]), orc.mom_refresh(dims, seed)
    K0, S0 = orc.hamiltonian(dims, beta, U0, P0)
    U1, P1 = orc.leapfrog(dims, beta, g["eps"], g["nsteps"], U0, P0)
    K1, S1 = orc.hamiltonian(dims, beta, U1, P1)
    assert np.isclose(orc.plaquette(dims, U0)[0], g["plaq0"], rtol=1e-13) and np.isclose(K0, g["K0"], rtol=1e-13)
    assert np.isclose(orc.plaquette(dims, U1)[0], g["plaq1"], rtol=1e-13) and np.isclose(K1, g["K1"], rtol=1e-13)
    assert abs(((K1 + S1) - (K0 + S0)) - g["dH"]) < 1e-9 * abs(K0 + S0)
    assert abs(g["K0"] / (16 * np.prod(dims)) - 1) < 4 / np.sqrt(16 * np.prod(dims))  # <K> = 16 V
    assert abs(g["plaq0"] - 0.503) < 0.03  # chi(0.5)^4 (SURVEY.md 8(c) pin table), 4^4 statistics
