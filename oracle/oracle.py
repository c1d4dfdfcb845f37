"""ctypes/numpy face of the CPU oracle.  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It never imports paper_1212_0785_b200 and shares no code with it.

Fields are numpy arrays in the canonical lexicographic layout of oracle/qcd_oracle.h:
    matrix field  complex128[V, 4, 3, 3]      real field  float64[V, ncomp]
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

ALL, EVEN, ODD = 0, 1, 2
SUM_SCALAR, SUM_NORM2, SUM_RETR = 0, 1, 2
MAP_CB_OF_LEX, MAP_LEX_OF_CB, MAP_NBR_FWD0, MAP_NBR_BWD0, MAP_PARITY, MAP_TSLICE = 0, 1, 2, 6, 10, 11

_c_int4 = C.c_int * 4
_dp = C.POINTER(C.c_double)


def _ptr(a):
    return a.ctypes.data_as(_dp)


def _mat(a, V):
    assert a.dtype == np.complex128 and a.flags.c_contiguous and a.shape == (V, 4, 3, 3), (a.dtype, a.shape)
    return _ptr(a)


class Oracle:
    """One loaded oracle library (serial by default; omp=True loads the OpenMP build)."""

    def __init__(self, omp=False):
        serial, par = _build.build()
        self.lib = C.CDLL(par if omp else serial)
        self.omp = omp
        L = self.lib
        L.orc_rng_block.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32,
                                    C.POINTER(C.c_uint32), _dp, _dp]
        L.orc_rng_block.restype = None
        L.orc_mom_refresh.argtypes = [_c_int4, C.c_int, C.c_uint64, C.c_uint32, _dp]
        L.orc_hot_start.argtypes = [_c_int4, C.c_uint64, C.c_double, _dp]
        L.orc_perturb.argtypes = [_c_int4, C.c_uint64, C.c_double, _dp]
        L.orc_gauge_transform.argtypes = [_c_int4, C.c_uint64, C.c_double, _dp, _dp, _dp]
        L.orc_plaquette.argtypes = [_c_int4, _dp, _dp, _dp]
        L.orc_action.argtypes = [_c_int4, C.c_double, _dp, _dp]
        L.orc_gauge_force.argtypes = [_c_int4, C.c_int, C.c_double, _dp, _dp]
        L.orc_gauge_force_sites.argtypes = [_c_int4, C.c_double, _dp, C.c_int, C.POINTER(C.c_int32), _dp]
        L.orc_sum_retr_w.argtypes = [_c_int4, _dp, _dp]
        L.orc_mom_update.argtypes = [_c_int4, C.c_int, C.c_double, _dp, _dp]
        L.orc_link_update.argtypes = [_c_int4, C.c_int, C.c_double, _dp, _dp, C.c_int]
        L.orc_reunit.argtypes = [_c_int4, C.c_int, _dp]
        L.orc_sum.argtypes = [_c_int4, C.c_int, C.c_int, C.c_int, _dp, _dp]
        L.orc_sum_multi.argtypes = [_c_int4, C.c_int, C.c_int, _dp, C.POINTER(C.c_int32), C.c_int, _dp]
        L.orc_hamiltonian.argtypes = [_c_int4, C.c_double, _dp, _dp, _dp, _dp]
        L.orc_leapfrog.argtypes = [_c_int4, C.c_double, C.c_double, C.c_int, _dp, _dp]
        L.orc_md_step.argtypes = [_c_int4, C.c_double, C.c_double, C.c_double, _dp, _dp]
        L.orc_spinor_gaussian.argtypes = [_c_int4, C.c_int, C.c_uint64, C.c_uint32, _dp]
        L.orc_inner_product.argtypes = [_c_int4, C.c_int, C.c_int, _dp, _dp, _dp]
        L.orc_inner_product_multi.argtypes = [_c_int4, C.c_int, _dp, _dp, _dp]
        L.orc_plaquette_st.argtypes = [_c_int4, _dp, _dp, _dp]
        L.orc_action_aniso.argtypes = [_c_int4, C.c_double, C.c_double, _dp, _dp]
        L.orc_gauge_force_aniso.argtypes = [_c_int4, C.c_int, C.c_double, C.c_double, _dp, _dp]
        L.orc_nested_leapfrog.argtypes = [_c_int4, _dp, _dp, C.c_double, C.c_int, C.c_int, _dp, _dp]
        L.orc_map.argtypes = [_c_int4, C.c_int, C.POINTER(C.c_int32)]
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.orc_philox4x32_10.restype = None
        for f in ("orc_herm_from_coeffs", "orc_expi"):
            getattr(L, f).argtypes = [_dp, _dp]
            getattr(L, f).restype = None
        L.orc_reunit_mat.argtypes = [_dp]
        L.orc_reunit_mat.restype = None

    # ---- helpers
    @staticmethod
    def volume(dims):
        return int(np.prod(dims))

    def num_threads(self):
        return int(self.lib.orc_num_threads())

    @staticmethod
    def _ok(rc, what):
        if rc != 0:
            raise ValueError(f"oracle {what} failed with code {rc}")

    # ---- O1
    def map(self, dims, which):
        out = np.empty(self.volume(dims), dtype=np.int32)
        self._ok(self.lib.orc_map(_c_int4(*dims), which, out.ctypes.data_as(C.POINTER(C.c_int32))), "map")
        return out

    # ---- O3
    def philox(self, ctr, key):
        c = (C.c_uint32 * 4)(*ctr)
        k = (C.c_uint32 * 2)(*key)
        o = (C.c_uint32 * 4)()
        self.lib.orc_philox4x32_10(c, k, o)
        return [int(x) for x in o]

    def rng_block(self, seed, s, mu, j, stream_id, purpose):
        w = (C.c_uint32 * 4)()
        u = np.empty(2)
        g = np.empty(2)
        self.lib.orc_rng_block(seed, s, mu, j, stream_id, purpose, w, _ptr(u), _ptr(g))
        return [int(x) for x in w], u, g

    # ---- O2, O8, O9 single-matrix
    def herm_from_coeffs(self, q):
        q = np.ascontiguousarray(q, dtype=np.float64)
        Q = np.empty((3, 3), dtype=np.complex128)
        self.lib.orc_herm_from_coeffs(_ptr(q), _ptr(Q))
        return Q

    def expi(self, Q):
        Q = np.ascontiguousarray(Q, dtype=np.complex128)
        E = np.empty((3, 3), dtype=np.complex128)
        self.lib.orc_expi(_ptr(Q), _ptr(E))
        return E

    def reunit_mat(self, M):
        M = np.array(M, dtype=np.complex128, order="C")
        self.lib.orc_reunit_mat(_ptr(M))
        return M

    # ---- O4, O5
    def mom_refresh(self, dims, seed, stream_id=0, subset=ALL, out=None):
        V = self.volume(dims)
        P = np.zeros((V, 4, 3, 3), dtype=np.complex128) if out is None else out
        self._ok(self.lib.orc_mom_refresh(_c_int4(*dims), subset, seed, stream_id, _mat(P, V)), "mom_refresh")
        return P

    def hot_start(self, dims, seed, sigma):
        V = self.volume(dims)
        U = np.empty((V, 4, 3, 3), dtype=np.complex128)
        self._ok(self.lib.orc_hot_start(_c_int4(*dims), seed, sigma, _mat(U, V)), "hot_start")
        return U

    def perturb(self, dims, seed, sigma, U):
        V = self.volume(dims)
        U = U.copy()
        self._ok(self.lib.orc_perturb(_c_int4(*dims), seed, sigma, _mat(U, V)), "perturb")
        return U

    def gauge_transform(self, dims, seed, sigma, U):
        V = self.volume(dims)
        G = np.empty((V, 3, 3), dtype=np.complex128)
        Uo = np.empty_like(U)
        self._ok(self.lib.orc_gauge_transform(_c_int4(*dims), seed, sigma, _mat(U, V), _ptr(G), _mat(Uo, V)),
                 "gauge_transform")
        return G, Uo

    # ---- O6
    def plaquette(self, dims, U):
        V = self.volume(dims)
        avg = np.empty(1)
        per_t = np.empty(dims[3])
        self._ok(self.lib.orc_plaquette(_c_int4(*dims), _mat(U, V), _ptr(avg), _ptr(per_t)), "plaquette")
        return float(avg[0]), per_t

    def action(self, dims, beta, U):
        S = np.empty(1)
        self._ok(self.lib.orc_action(_c_int4(*dims), beta, _mat(U, self.volume(dims)), _ptr(S)), "action")
        return float(S[0])

    def hamiltonian(self, dims, beta, U, P):
        V = self.volume(dims)
        K, S = np.empty(1), np.empty(1)
        self._ok(self.lib.orc_hamiltonian(_c_int4(*dims), beta, _mat(U, V), _mat(P, V), _ptr(K), _ptr(S)), "H")
        return float(K[0]), float(S[0])

    # ---- O7
    def gauge_force(self, dims, beta, U, subset=ALL, out=None):
        V = self.volume(dims)
        F = np.zeros_like(U) if out is None else out
        self._ok(self.lib.orc_gauge_force(_c_int4(*dims), subset, beta, _mat(U, V), _mat(F, V)), "gauge_force")
        return F

    def gauge_force_sites(self, dims, beta, U, sites):
        sites = np.ascontiguousarray(sites, dtype=np.int32)
        F = np.empty((len(sites), 4, 3, 3), dtype=np.complex128)
        self._ok(self.lib.orc_gauge_force_sites(_c_int4(*dims), beta, _mat(U, self.volume(dims)), len(sites),
                                                sites.ctypes.data_as(C.POINTER(C.c_int32)), _ptr(F)),
                 "gauge_force_sites")
        return F

    def sum_retr_w(self, dims, U):
        out = np.empty(1)
        self._ok(self.lib.orc_sum_retr_w(_c_int4(*dims), _mat(U, self.volume(dims)), _ptr(out)), "sum_retr_w")
        return float(out[0])

    # ---- O10 (in place on copies: inputs are never modified)
    def mom_update(self, dims, eps, F, P, subset=ALL):
        V = self.volume(dims)
        P = P.copy()
        self._ok(self.lib.orc_mom_update(_c_int4(*dims), subset, eps, _mat(F, V), _mat(P, V)), "mom_update")
        return P

    def link_update(self, dims, eps, P, U, reunit=False, subset=ALL):
        V = self.volume(dims)
        U = U.copy()
        self._ok(self.lib.orc_link_update(_c_int4(*dims), subset, eps, _mat(P, V), _mat(U, V), int(reunit)),
                 "link_update")
        return U

    def reunit(self, dims, U, subset=ALL):
        V = self.volume(dims)
        U = U.copy()
        self._ok(self.lib.orc_reunit(_c_int4(*dims), subset, _mat(U, V)), "reunit")
        return U

    # ---- O12
    def sum(self, dims, kind, field, subset=ALL):
        V = self.volume(dims)
        f = np.ascontiguousarray(field)
        if f.dtype == np.complex128:
            f = f.view(np.float64)
        assert f.dtype == np.float64
        f = f.reshape(V, -1)
        ncomp = f.shape[1]
        out = np.empty(ncomp if kind == SUM_SCALAR else 1)
        self._ok(self.lib.orc_sum(_c_int4(*dims), subset, kind, ncomp, _ptr(f), _ptr(out)), "sum")
        return out

    def sum_multi(self, dims, kind, field, subset_id=None, nsub=None):
        V = self.volume(dims)
        f = np.ascontiguousarray(field)
        if f.dtype == np.complex128:
            f = f.view(np.float64)
        f = f.reshape(V, -1)
        ncomp = f.shape[1]
        if subset_id is None:
            nsub = dims[3]
            idp = None
        else:
            subset_id = np.ascontiguousarray(subset_id, dtype=np.int32)
            idp = subset_id.ctypes.data_as(C.POINTER(C.c_int32))
        out = np.empty((nsub, ncomp) if kind == SUM_SCALAR else (nsub,))
        self._ok(self.lib.orc_sum_multi(_c_int4(*dims), kind, ncomp, _ptr(f), idp, nsub, _ptr(out)), "sum_multi")
        return out

    # ---- O13 anisotropic Wilson action, O14 two-level leapfrog
    def plaquette_st(self, dims, U):
        """(avg[2], per_t[Lt,2]): space-space and space-time plaquette averages"""
        avg, per_t = np.empty(2), np.empty((dims[3], 2))
        self._ok(self.lib.orc_plaquette_st(_c_int4(*dims), _mat(U, self.volume(dims)), _ptr(avg), _ptr(per_t)), "plaq_st")
        return avg, per_t

    def action_aniso(self, dims, beta_s, beta_t, U):
        S = np.empty(1)
        self._ok(self.lib.orc_action_aniso(_c_int4(*dims), beta_s, beta_t, _mat(U, self.volume(dims)), _ptr(S)),
                 "action_aniso")
        return float(S[0])

    def gauge_force_aniso(self, dims, beta_s, beta_t, U, subset=ALL, out=None):
        V = self.volume(dims)
        F = np.zeros_like(U) if out is None else out
        self._ok(self.lib.orc_gauge_force_aniso(_c_int4(*dims), subset, beta_s, beta_t, _mat(U, V), _mat(F, V)),
                 "gauge_force_aniso")
        return F

    def nested_leapfrog(self, dims, bs, bt, tau, n_outer, n_inner, U, P):
        """bs, bt: (level 0 = inner, level 1 = outer) coefficients"""
        V = self.volume(dims)
        U, P = U.copy(), P.copy()
        bs, bt = np.asarray(bs, dtype=np.float64), np.asarray(bt, dtype=np.float64)
        self._ok(self.lib.orc_nested_leapfrog(_c_int4(*dims), _ptr(bs), _ptr(bt), tau, n_outer, n_inner, _mat(U, V),
                                              _mat(P, V)), "nested_leapfrog")
        return U, P

    # ---- O15 / O16 spin-colour vectors: complex128[V, 12]
    def spinor_gaussian(self, dims, seed, stream_id=0, subset=ALL, out=None):
        eta = np.zeros((self.volume(dims), 12), dtype=np.complex128) if out is None else out
        self._ok(self.lib.orc_spinor_gaussian(_c_int4(*dims), subset, seed, stream_id, _ptr(eta)), "spinor_gaussian")
        return eta

    def inner_product(self, dims, a, b, subset=ALL):
        assert a.dtype == b.dtype == np.complex128 and a.shape == b.shape and a.flags.c_contiguous and b.flags.c_contiguous
        out = np.empty(2)
        self._ok(self.lib.orc_inner_product(_c_int4(*dims), subset, a.shape[1], _ptr(a), _ptr(b), _ptr(out)), "inner")
        return complex(out[0], out[1])

    def inner_product_multi(self, dims, a, b):
        assert a.dtype == b.dtype == np.complex128 and a.shape == b.shape and a.flags.c_contiguous and b.flags.c_contiguous
        out = np.empty((dims[3], 2))
        self._ok(self.lib.orc_inner_product_multi(_c_int4(*dims), a.shape[1], _ptr(a), _ptr(b), _ptr(out)), "inner_multi")
        return out[:, 0] + 1j * out[:, 1]

    # ---- O11
    def leapfrog(self, dims, beta, eps, nsteps, U, P):
        V = self.volume(dims)
        U, P = U.copy(), P.copy()
        self._ok(self.lib.orc_leapfrog(_c_int4(*dims), beta, eps, nsteps, _mat(U, V), _mat(P, V)), "leapfrog")
        return U, P

    def md_step(self, dims, beta, eps_p, eps_u, U, P, inplace=False):
        V = self.volume(dims)
        if not inplace:
            U, P = U.copy(), P.copy()
        self._ok(self.lib.orc_md_step(_c_int4(*dims), beta, eps_p, eps_u, _mat(U, V), _mat(P, V)), "md_step")
        return U, P
