"""Seeded synthetic inputs shared by the oracle tests and the GPU parity tests.

This module holds NONE of the method's arithmetic: it only draws generic random numbers
(numpy PCG64) and shapes them.  Inputs that ARE outputs of the method (hot-start links,
Gaussian momenta) are produced by the side under test from the (seed, counter) definition
in DESIGN.md, never here.
"""
import numpy as np

CONFIG_SEED_BASE = 0x1212078500000000  # seed = base + config number

# the five BASELINE.json configs: dims, hot-start sigma, beta, eps, steps
CONFIGS = {
    1: dict(dims=(4, 4, 4, 4), sigma=0.5, beta=5.6, eps=0.1, nsteps=1),
    2: dict(dims=(8, 8, 8, 16), sigma=0.5, beta=5.8, eps=0.05, nsteps=10),
    3: dict(dims=(16, 16, 16, 32), sigma=0.5, beta=5.8, eps=0.05, nsteps=1),
    4: dict(dims=(32, 32, 32, 64), sigma=0.2, beta=6.0, eps=0.02, nsteps=20),
    5: dict(dims=(48, 48, 48, 96), sigma=0.3, beta=6.2, eps=0.01, nsteps=20),
}


def config_seed(n):
    return CONFIG_SEED_BASE + n


def random_complex_matrices(seed, n):
    """n generic (non-unitary) 3x3 complex matrices, entries O(1)."""
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n, 3, 3)) + 1j * rng.standard_normal((n, 3, 3))


def random_hermitian_traceless(seed, n, scale=1.0):
    m = random_complex_matrices(seed, n)
    h = 0.5 * (m + np.conj(np.swapaxes(m, -1, -2)))
    h -= np.trace(h, axis1=-2, axis2=-1)[:, None, None] * np.eye(3) / 3.0
    return scale * h


def random_matrix_field(seed, V):
    """generic complex matrix field [V,4,3,3] (not unitary): exercises formulas on arbitrary input"""
    return np.ascontiguousarray(random_complex_matrices(seed, 4 * V).reshape(V, 4, 3, 3))


def random_real_field(seed, V, ncomp):
    return np.random.default_rng(seed).standard_normal((V, ncomp))


def random_subset_ids(seed, V, nsub):
    return np.random.default_rng(seed).integers(0, nsub, size=V, dtype=np.int32)
