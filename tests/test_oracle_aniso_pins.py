"""Pins for the oracle's anisotropic Wilson action (O13, R19; PAPER.md:101 names the action) and
two-level leapfrog (O14, R20; "Multi-timescale integrators"), against what the
mathematics fixes: an independent numpy brute force, finite differences of the action, the isotropic
limit, linearity in the coefficients, degenerate nestings that reduce to the plain leapfrog,
reversibility and the eps^2 scaling of dH.  All CPU."""
import numpy as np
import pytest
import scipy.linalg

from tests import inputs
from tests.test_oracle_pins import T, dag, unit_gauge


def numpy_plaquette_st(dims, U):
    """independent brute force with np.roll: mean (1/3) Re tr P over space-space / space-time planes"""
    Lx, Ly, Lz, Lt = dims
    A = U.reshape(Lt, Lz, Ly, Lx, 4, 3, 3)
    axis = {0: 3, 1: 2, 2: 1, 3: 0}
    per_site = np.zeros((2, Lt, Lz, Ly, Lx))
    for mu in range(4):
        for nu in range(mu + 1, 4):
            Umu, Unu = A[..., mu, :, :], A[..., nu, :, :]
            Pl = Umu @ np.roll(Unu, -1, axis=axis[mu]) @ dag(np.roll(Umu, -1, axis=axis[nu])) @ dag(Unu)
            per_site[1 if nu == 3 else 0] += np.trace(Pl, axis1=-2, axis2=-1).real / 3
    return per_site.mean(axis=(1, 2, 3, 4)) / 3, per_site.mean(axis=(2, 3, 4)).T / 3


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 6, 2, 4)])
def test_plaquette_st_bruteforce_and_consistency(orc, dims):
    V = int(np.prod(dims))
    U = inputs.random_matrix_field(31, V)  # generic matrices: a wrong plane class or index shows up
    avg, per_t = orc.plaquette_st(dims, U)
    ravg, rper_t = numpy_plaquette_st(dims, U)
    assert np.allclose(avg, ravg, rtol=1e-13) and np.allclose(per_t, rper_t, rtol=1e-13)
    # the two classes average to the isotropic plaquette; per-timeslice means give the global ones
    iso, iso_t = orc.plaquette(dims, U)
    assert np.isclose(avg.mean(), iso, rtol=1e-13) and np.allclose(per_t.mean(axis=1), iso_t, rtol=1e-13)
    assert np.allclose(per_t.mean(axis=0), avg, rtol=1e-13)
    bs, bt = 2.3, 7.1
    assert np.isclose(orc.action_aniso(dims, bs, bt, U), 3 * V * (bs * (1 - avg[0]) + bt * (1 - avg[1])), rtol=1e-12)
    assert np.isclose(orc.action_aniso(dims, 5.5, 5.5, U), orc.action(dims, 5.5, U), rtol=1e-13)
    a1, p1 = orc.plaquette_st(dims, unit_gauge(V))
    assert np.all(a1 == 1.0) and np.all(p1 == 1.0)


def test_aniso_force_equals_finite_difference_of_aniso_action(orc):
    """f_a = 2 tr(T_a F) = -dS/d omega_a with beta_s != beta_t: a wrong coefficient on any plane fails;
    2^4 and a lattice with distinct extents; spatial and temporal links"""
    h = 1e-5
    worst = 0.0
    for dims, bs, bt in [((2, 2, 2, 2), 2.0, 9.0), ((4, 2, 2, 4), 7.5, 1.5)]:
        U = orc.hot_start(dims, inputs.config_seed(1), 0.5)
        F = orc.gauge_force_aniso(dims, bs, bt, U)
        rng = np.random.default_rng(1)
        V = int(np.prod(dims))
        for mu in (0, 1, 2, 3, 3):
            s = int(rng.integers(0, V))
            for a in range(8):
                Up, Um = U.copy(), U.copy()
                Up[s, mu] = scipy.linalg.expm(1j * h * T[a]) @ U[s, mu]
                Um[s, mu] = scipy.linalg.expm(-1j * h * T[a]) @ U[s, mu]
                dS = (orc.action_aniso(dims, bs, bt, Up) - orc.action_aniso(dims, bs, bt, Um)) / (2 * h)
                worst = max(worst, abs(2 * np.trace(T[a] @ F[s, mu]).real + dS))
        assert np.abs(F).max() > 0.1
    assert worst < 1e-7, worst


def test_aniso_force_isotropic_limit_linearity_and_structure(orc):
    dims = (4, 4, 2, 4)
    U = orc.hot_start(dims, 7, 0.5)
    beta = 5.9
    assert np.abs(orc.gauge_force_aniso(dims, beta, beta, U) - orc.gauge_force(dims, beta, U)).max() < 1e-14
    bs, bt = 3.1, 8.2
    F = orc.gauge_force_aniso(dims, bs, bt, U)
    Fs, Ft = orc.gauge_force_aniso(dims, bs, 0.0, U), orc.gauge_force_aniso(dims, 0.0, bt, U)
    assert np.abs(F - (Fs + Ft)).max() < 1e-14
    assert np.abs(Fs[:, 3]).max() == 0  # no space-space plane contains a time link
    assert np.abs(F - dag(F)).max() < 1e-14 and np.abs(np.trace(F, axis1=-2, axis2=-1)).max() < 1e-14
    # subsets write only their sites
    Fe = orc.gauge_force_aniso(dims, bs, bt, U, subset=1)
    Fo = orc.gauge_force_aniso(dims, bs, bt, U, subset=2)
    assert np.array_equal(Fe + Fo, F) and np.abs(Fe).sum(axis=(1, 2, 3)).astype(bool).sum() == U.shape[0] // 2


def H_aniso(orc, dims, bs, bt, U, P):
    return float(np.sum(np.abs(P) ** 2)) + orc.action_aniso(dims, bs, bt, U)


def test_nested_leapfrog_degenerate_cases_reduce_to_plain_leapfrog(orc_omp):
    dims = (4, 4, 4, 4)
    beta, tau = 5.6, 0.3
    U0 = orc_omp.hot_start(dims, inputs.config_seed(1), 0.5)
    P0 = orc_omp.mom_refresh(dims, inputs.config_seed(1))
    # outer level empty: n_outer x n_inner plain steps of the inner action
    Ua, Pa = orc_omp.nested_leapfrog(dims, (beta, 0.0), (beta, 0.0), tau, 2, 3, U0, P0)
    Ub, Pb = orc_omp.leapfrog(dims, beta, tau / 6, 6, U0, P0)
    assert np.abs(Ua - Ub).max() < 1e-13 and np.abs(Pa - Pb).max() < 1e-13
    # inner level empty, one inner step: plain leapfrog of the outer action
    Ua, Pa = orc_omp.nested_leapfrog(dims, (0.0, beta), (0.0, beta), tau, 5, 1, U0, P0)
    Ub, Pb = orc_omp.leapfrog(dims, beta, tau / 5, 5, U0, P0)
    assert np.abs(Ua - Ub).max() < 1e-13 and np.abs(Pa - Pb).max() < 1e-13
    # inner level empty, several inner steps: exp(i e0 P)^n = exp(i e1 P) for constant P
    Ua, Pa = orc_omp.nested_leapfrog(dims, (0.0, beta), (0.0, beta), tau, 5, 4, U0, P0)
    assert np.abs(Ua - Ub).max() < 1e-13 and np.abs(Pa - Pb).max() < 1e-13
    # one outer, one inner step with the action split in halves: one plain step
    Ua, Pa = orc_omp.nested_leapfrog(dims, (beta / 2, beta / 2), (beta / 2, beta / 2), 0.1, 1, 1, U0, P0)
    Ub, Pb = orc_omp.leapfrog(dims, beta, 0.1, 1, U0, P0)
    assert np.abs(Ua - Ub).max() < 1e-13 and np.abs(Pa - Pb).max() < 1e-13


def test_nested_leapfrog_reversibility_and_dH_scaling(orc_omp):
    """space-space planes on the outer level, space-time planes (the stiff part, beta_t > beta_s) inside"""
    dims = (4, 4, 4, 4)
    bs, bt = (0.0, 3.0), (9.0, 0.0)  # level 0 (inner): (bs=0, bt=9); level 1 (outer): (bs=3, bt=0)
    U0 = orc_omp.hot_start(dims, inputs.config_seed(1), 0.5)
    P0 = orc_omp.mom_refresh(dims, inputs.config_seed(1))
    tau = 0.2
    U1, P1 = orc_omp.nested_leapfrog(dims, bs, bt, tau, 4, 3, U0, P0)
    assert np.abs(U1 - U0).max() > 0.05
    U2, P2 = orc_omp.nested_leapfrog(dims, bs, bt, tau, 4, 3, U1, -P1)
    assert np.abs(U2 - U0).max() < 1e-13 and np.abs(-P2 - P0).max() < 1e-13
    H0 = H_aniso(orc_omp, dims, 3.0, 9.0, U0, P0)
    dH = []
    for n in (4, 8, 16, 32):
        U1, P1 = orc_omp.nested_leapfrog(dims, bs, bt, tau, n, 2, U0, P0)
        dH.append(H_aniso(orc_omp, dims, 3.0, 9.0, U1, P1) - H0)
    ratios = [dH[i] / dH[i + 1] for i in range(3)]
    assert abs(ratios[1] - 4) < 0.3 and abs(ratios[2] - 4) < 0.1, (dH, ratios)
    # the finer inner level buys accuracy: same outer step, more inner steps -> smaller |dH|
    Ua, Pa = orc_omp.nested_leapfrog(dims, bs, bt, tau, 4, 1, U0, P0)
    Ub, Pb = orc_omp.nested_leapfrog(dims, bs, bt, tau, 4, 4, U0, P0)
    assert abs(H_aniso(orc_omp, dims, 3.0, 9.0, Ub, Pb) - H0) < abs(H_aniso(orc_omp, dims, 3.0, 9.0, Ua, Pa) - H0)
