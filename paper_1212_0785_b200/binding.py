"""Thin Python binding of the C ABI in include/qcd.h (same names, argument marshalling only).

Every step of the path runs in the CUDA kernels of libqcdmd.so; PyTorch is used for device memory
(tensors), streams and nothing else.  There is no CPU fallback: if the library is missing the import
fails loudly.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqcdmd.so")

F32, F64 = 0, 1
ALL, EVEN, ODD = 0, 1, 2
SUM_SCALAR, SUM_NORM2, SUM_RETR = 0, 1, 2
LAYOUT_REAL, LAYOUT_PAIRS = 0, 1
PROBE_FMA, PROBE_L1, PROBE_LDS, PROBE_L2 = 0, 1, 2, 3
OK, EINVAL, EDIMS, EALIGN, EALIAS, EWORKSPACE, ECUDA = range(7)
KERNEL_FORCE, KERNEL_LINK_UPDATE, KERNEL_MOM_UPDATE = 0, 1, 2
FORCE_VARIANTS = ("staple", "plane")  # index = QCD_FORCE_* value
MAP_CB_OF_LEX, MAP_LEX_OF_CB, MAP_NBR_FWD0, MAP_NBR_BWD0, MAP_PARITY, MAP_TSLICE = 0, 1, 2, 6, 10, 11

# every symbol include/qcd.h declares, with its ctypes signature (restype, argtypes)
_vp, _i, _d, _u64, _u32, _sz = C.c_void_p, C.c_int, C.c_double, C.c_uint64, C.c_uint32, C.c_size_t
SIGNATURES = {
    "qcd_lattice_create": (_i, [C.POINTER(C.c_int * 4), C.POINTER(_vp)]),
    "qcd_lattice_create_slab": (_i, [C.POINTER(C.c_int * 4), _i, _i, C.POINTER(_vp)]),
    "qcd_lattice_view_t": (_i, [_vp, _i, _i, C.POINTER(_vp)]),
    "qcd_lattice_dims": (_i, [_vp, C.POINTER(C.c_int * 4), C.POINTER(C.c_int * 2)]),
    "qcd_copy_timeslices": (_i, [_vp, _vp, _i, _vp, _vp, _i, _i, _i, _i, C.c_uint, _vp]),
    "qcd_link_update_push": (_i, [_vp, _i, _d, _vp, _vp, _i, _vp, _vp, _vp, _vp, _vp]),
    "qcd_md_step_single_pass_push": (_i, [_vp, _i, _d, _d, _d, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "qcd_lattice_destroy": (_i, [_vp]),
    "qcd_lattice_volume": (C.c_int64, [_vp]),
    "qcd_field_bytes": (_sz, [_vp, _i, _i]),
    "qcd_workspace_bytes": (_sz, [_vp]),
    "qcd_md_host_work_bytes": (_sz, [_vp, _i]),
    "qcd_last_error": (C.c_char_p, []),
    "qcd_version": (C.c_char_p, []),
    "qcd_gauge_force": (_i, [_vp, _i, _i, _d, _vp, _vp, _vp]),
    "qcd_mom_update": (_i, [_vp, _i, _i, _d, _vp, _vp, _vp]),
    "qcd_force_mom_update": (_i, [_vp, _i, _i, _d, _d, _vp, _vp, _vp]),
    "qcd_link_update": (_i, [_vp, _i, _i, _d, _vp, _vp, _i, _vp]),
    "qcd_reunit": (_i, [_vp, _i, _i, _vp, _vp]),
    "qcd_mom_refresh": (_i, [_vp, _i, _i, _u64, _u32, _vp, _vp]),
    "qcd_plaquette": (_i, [_vp, _i, _vp, _vp, _vp, _vp, _vp]),
    "qcd_plaquette_noalloc": (_i, [_vp, _i, _vp, _vp, _vp, _vp]),
    "qcd_sum": (_i, [_vp, _i, _i, _i, _i, _vp, _vp, _vp, _vp]),
    "qcd_sum_multi": (_i, [_vp, _i, _i, _i, _vp, _vp, _i, _vp, _vp, _vp]),
    "qcd_md_step": (_i, [_vp, _i, _d, _d, _d, _vp, _vp, _vp]),
    "qcd_leapfrog": (_i, [_vp, _i, _d, _d, _i, _vp, _vp, _vp]),
    "qcd_force_mom_update_sums": (_i, [_vp, _i, _d, _d, _vp, _vp, _vp, _vp, _vp]),
    "qcd_leapfrog_energy": (_i, [_vp, _i, _d, _d, _i, _vp, _vp, _vp, _vp, _vp]),
    "qcd_md_step_single_pass": (_i, [_vp, _i, _d, _d, _d, _vp, _vp, _vp, _vp]),
    "qcd_leapfrog_single_pass": (_i, [_vp, _i, _d, _d, _i, _vp, _vp, _vp, _vp]),
    "qcd_trajectory": (_i, [_vp, _i, _d, _d, _i, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    "qcd_gauge_force_aniso": (_i, [_vp, _i, _i, _d, _d, _vp, _vp, _vp]),
    "qcd_force_mom_update_aniso": (_i, [_vp, _i, _i, _d, _d, _d, _vp, _vp, _vp]),
    "qcd_plaquette_st": (_i, [_vp, _i, _vp, _vp, _vp, _vp, _vp]),
    "qcd_nested_leapfrog": (_i, [_vp, _i, C.POINTER(C.c_double * 2), C.POINTER(C.c_double * 2), _d, _i, _i, _vp, _vp,
                                 _vp]),
    "qcd_spinor_gaussian": (_i, [_vp, _i, _i, _u64, _u32, _vp, _vp]),
    "qcd_inner_product": (_i, [_vp, _i, _i, _i, _vp, _vp, _vp, _vp, _vp]),
    "qcd_inner_product_multi": (_i, [_vp, _i, _i, _vp, _vp, _vp, _vp, _vp]),
    "qcd_tune_set": (_i, [_vp, _i, _i, _i, _i, C.POINTER(C.c_int * 4), _i]),
    "qcd_tune_get": (_i, [_vp, _i, _i, _i, C.POINTER(_i), C.POINTER(C.c_int * 4), C.POINTER(_i)]),
    "qcd_tune_clear": (_i, []),
    "qcd_pack": (_i, [_vp, _i, _i, _i, _vp, _vp, _vp]),
    "qcd_unpack": (_i, [_vp, _i, _i, _i, _vp, _vp, _vp]),
    "qcd_get_map": (_i, [_vp, _i, _vp, _vp]),
    "qcd_hot_start": (_i, [_vp, _i, _u64, _d, _vp, _vp]),
    "qcd_perturb": (_i, [_vp, _i, _u64, _d, _vp, _vp]),
    "qcd_rng_blocks": (_i, [_u64, _u32, _u32, _i, _vp, _vp, _vp, _vp, _vp, _vp]),
    "qcd_probe_scratch_bytes": (_sz, [_i]),
    "qcd_probe_work": (_d, [_i, _i, _i]),
    "qcd_probe_launch": (_i, [_i, _i, _i, _vp, _sz, _vp]),
    "qcd_md_host": (_i, [_vp, _i, _d, _d, _i, _vp, _vp, _vp, _vp]),
}


def load_library(path=LIB_PATH):
    if not os.path.exists(path):
        raise ImportError(
            f"{path} is missing: build it with `python paper_1212_0785_b200/build.py` "
            "(there is no CPU fallback for the CUDA path)")
    lib = C.CDLL(path)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)  # AttributeError if the library does not export a declared symbol
        fn.restype = res
        fn.argtypes = args
    return lib


lib = load_library()


class QcdError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"qcd error {code}: {text}")
        self.code = code


def _check(rc):
    if rc != OK:
        raise QcdError(rc, lib.qcd_last_error().decode())


def _prec(t):
    if t.dtype == torch.float64:
        return F64
    if t.dtype == torch.float32:
        return F32
    raise TypeError(f"field dtype must be float32 or float64, got {t.dtype}")


def _ptr(t):
    return None if t is None else t.data_ptr()


def _stream(stream):
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


class Lattice:
    """qcd_lattice handle (host side)."""

    def __init__(self, dims, slab=None):
        """dims: extents of the (global) lattice; slab = (t_begin, t_count): the slab lattice of
        qcd_lattice_create_slab (stored extents (Lx, Ly, Lz, t_count + 2), interior timeslices 1 .. t_count)"""
        gdims = tuple(int(d) for d in dims)
        h = _vp()
        arr = (C.c_int * 4)(*gdims) if len(gdims) == 4 else None
        if arr is None:
            raise QcdError(EINVAL, "dims must have 4 entries")
        if slab is None:
            _check(lib.qcd_lattice_create(C.byref(arr), C.byref(h)))
        else:
            _check(lib.qcd_lattice_create_slab(C.byref(arr), int(slab[0]), int(slab[1]), C.byref(h)))
        self.handle = h
        self.V = int(lib.qcd_lattice_volume(h))
        d, it = (C.c_int * 4)(), (C.c_int * 2)()
        _check(lib.qcd_lattice_dims(h, C.byref(d), C.byref(it)))
        self.dims = tuple(d)          # stored (local) extents
        self.interior_t = tuple(it)   # timeslices the stencil kernels update
        self.global_dims, self.slab = gdims, slab

    def view_t(self, t0, t1):
        """the same stored lattice with the stencil calls restricted to the timeslices [t0, t1) (qcd_lattice_view_t)"""
        v = object.__new__(Lattice)
        h = _vp()
        _check(lib.qcd_lattice_view_t(self.handle, int(t0), int(t1), C.byref(h)))
        v.handle, v.V, v.dims, v.interior_t = h, self.V, self.dims, (int(t0), int(t1))
        v.global_dims, v.slab = self.global_dims, self.slab
        return v

    def __del__(self):
        h = getattr(self, "handle", None)
        if h and lib is not None:  # `lib` is already None when the interpreter is shutting down
            lib.qcd_lattice_destroy(h)
            self.handle = None

    def field_bytes(self, prec, ncomp=72):
        return int(lib.qcd_field_bytes(self.handle, prec, ncomp))

    def workspace_bytes(self):
        return int(lib.qcd_workspace_bytes(self.handle))

    def md_host_work_bytes(self, prec):
        return int(lib.qcd_md_host_work_bytes(self.handle, prec))

    # ---- device memory (PyTorch owns it).  Layout of include/qcd.h: chunks of 32 checkerboard sites,
    # [chunk = cb >> 5][unit][lane = cb & 31]; zero-filled so that the padding of the last chunk is defined
    @property
    def nchunks(self):
        return (self.V + 31) // 32

    def new_matrix_field(self, dtype=torch.float64, device="cuda"):
        """[chunk][36][32][2]: entry k = mu*9+e of site cb at [cb >> 5, k, cb & 31, re/im]"""
        return torch.zeros((self.nchunks, 36, 32, 2), dtype=dtype, device=device)

    def new_spinor_field(self, dtype=torch.float64, device="cuda"):
        """[chunk][12][32][2]: spin-colour component k = 3*spin + colour"""
        return torch.zeros((self.nchunks, 12, 32, 2), dtype=dtype, device=device)

    def new_pair_field(self, nc, dtype=torch.float64, device="cuda"):
        """[chunk][nc][32][2]: nc complex units per site (QCD_LAYOUT_PAIRS)"""
        return torch.zeros((self.nchunks, nc, 32, 2), dtype=dtype, device=device)

    def new_real_field(self, ncomp, dtype=torch.float64, device="cuda"):
        """[chunk][ncomp][32]"""
        return torch.zeros((self.nchunks, ncomp, 32), dtype=dtype, device=device)

    def by_component(self, field):
        """view-free copy of a device field as [unit][cb] (+ [2] for pair fields): what the layout holds, site by site"""
        if field.dim() == 4:
            return field.permute(1, 0, 2, 3).reshape(field.shape[1], -1, 2)[:, :self.V]
        return field.permute(1, 0, 2).reshape(field.shape[1], -1)[:, :self.V]

    def new_workspace(self, device="cuda"):
        return torch.empty(self.workspace_bytes() // 8, dtype=torch.float64, device=device)


# ---- the calls, named as in include/qcd.h ---------------------------------------------------

def qcd_gauge_force(lat, U, F, beta, subset=ALL, stream=None):
    _check(lib.qcd_gauge_force(lat.handle, _prec(U), subset, beta, _ptr(U), _ptr(F), _stream(stream)))


def qcd_mom_update(lat, F, P, eps, subset=ALL, stream=None):
    _check(lib.qcd_mom_update(lat.handle, _prec(P), subset, eps, _ptr(F), _ptr(P), _stream(stream)))


def qcd_force_mom_update(lat, U, P, beta, eps, subset=ALL, stream=None):
    _check(lib.qcd_force_mom_update(lat.handle, _prec(U), subset, beta, eps, _ptr(U), _ptr(P), _stream(stream)))


def qcd_link_update(lat, P, U, eps, reunit=False, subset=ALL, stream=None):
    _check(lib.qcd_link_update(lat.handle, _prec(U), subset, eps, _ptr(P), _ptr(U), int(reunit), _stream(stream)))


def qcd_reunit(lat, U, subset=ALL, stream=None):
    _check(lib.qcd_reunit(lat.handle, _prec(U), subset, _ptr(U), _stream(stream)))


def qcd_mom_refresh(lat, P, seed, stream_id=0, subset=ALL, stream=None):
    _check(lib.qcd_mom_refresh(lat.handle, _prec(P), subset, seed, stream_id, _ptr(P), _stream(stream)))


def qcd_plaquette(lat, U, out_avg, out_per_t, workspace, stream=None):
    _check(lib.qcd_plaquette(lat.handle, _prec(U), _ptr(U), _ptr(out_avg), _ptr(out_per_t), _ptr(workspace),
                             _stream(stream)))


def qcd_plaquette_noalloc(lat, U, out_avg, out_per_t, stream=None):
    """qcd_plaquette for a caller that cannot get device memory for a workspace (a routine inside an application
    whose memory manager owns the whole device, or one that must not stall a running trajectory with cudaMalloc):
    the partial sums use the 256 KiB array built into the library.  Lattices that need more than 32768 partial
    sums raise QcdError(EWORKSPACE); calls that overlap on one GPU race on that array (include/qcd.h)."""
    _check(lib.qcd_plaquette_noalloc(lat.handle, _prec(U), _ptr(U), _ptr(out_avg), _ptr(out_per_t), _stream(stream)))


def qcd_sum(lat, kind, ncomp, field, out, workspace, subset=ALL, stream=None):
    _check(lib.qcd_sum(lat.handle, _prec(field), subset, kind, ncomp, _ptr(field), _ptr(out), _ptr(workspace),
                       _stream(stream)))


def qcd_sum_multi(lat, kind, ncomp, field, subset_id, nsub, out, workspace, stream=None):
    _check(lib.qcd_sum_multi(lat.handle, _prec(field), kind, ncomp, _ptr(field), _ptr(subset_id), nsub, _ptr(out),
                             _ptr(workspace), _stream(stream)))


def qcd_md_step(lat, U, P, beta, eps_p, eps_u, stream=None):
    _check(lib.qcd_md_step(lat.handle, _prec(U), beta, eps_p, eps_u, _ptr(U), _ptr(P), _stream(stream)))


def qcd_leapfrog(lat, U, P, beta, eps, nsteps, stream=None):
    _check(lib.qcd_leapfrog(lat.handle, _prec(U), beta, eps, nsteps, _ptr(U), _ptr(P), _stream(stream)))


def qcd_force_mom_update_sums(lat, U, P, beta, eps, out, workspace, stream=None):
    _check(lib.qcd_force_mom_update_sums(lat.handle, _prec(U), beta, eps, _ptr(U), _ptr(P), _ptr(out), _ptr(workspace),
                                         _stream(stream)))


def qcd_leapfrog_energy(lat, U, P, beta, eps, nsteps, out, workspace, stream=None):
    _check(lib.qcd_leapfrog_energy(lat.handle, _prec(U), beta, eps, nsteps, _ptr(U), _ptr(P), _ptr(out), _ptr(workspace),
                                   _stream(stream)))


def qcd_md_step_single_pass(lat, U_in, P, U_out, beta, eps_p, eps_u, stream=None):
    _check(lib.qcd_md_step_single_pass(lat.handle, _prec(U_in), beta, eps_p, eps_u, _ptr(U_in), _ptr(P), _ptr(U_out),
                                       _stream(stream)))


def qcd_leapfrog_single_pass(lat, U, P, U_work, beta, eps, nsteps, stream=None):
    _check(lib.qcd_leapfrog_single_pass(lat.handle, _prec(U), beta, eps, nsteps, _ptr(U), _ptr(P), _ptr(U_work),
                                        _stream(stream)))


def qcd_trajectory(lat, U, P, U_work, beta, eps, nsteps, obs, per_t, workspace, stream=None):
    _check(lib.qcd_trajectory(lat.handle, _prec(U), beta, eps, nsteps, _ptr(U), _ptr(P), _ptr(U_work), _ptr(obs),
                              _ptr(per_t), _ptr(workspace), workspace.numel() * workspace.element_size(),
                              _stream(stream)))


def qcd_gauge_force_aniso(lat, U, F, beta_s, beta_t, subset=ALL, stream=None):
    _check(lib.qcd_gauge_force_aniso(lat.handle, _prec(U), subset, beta_s, beta_t, _ptr(U), _ptr(F), _stream(stream)))


def qcd_force_mom_update_aniso(lat, U, P, beta_s, beta_t, eps, subset=ALL, stream=None):
    _check(lib.qcd_force_mom_update_aniso(lat.handle, _prec(U), subset, beta_s, beta_t, eps, _ptr(U), _ptr(P),
                                          _stream(stream)))


def qcd_plaquette_st(lat, U, out_avg, out_per_t, workspace, stream=None):
    _check(lib.qcd_plaquette_st(lat.handle, _prec(U), _ptr(U), _ptr(out_avg), _ptr(out_per_t), _ptr(workspace),
                                _stream(stream)))


def qcd_nested_leapfrog(lat, U, P, beta_s, beta_t, tau, n_outer, n_inner, stream=None):
    """beta_s, beta_t: (level 0 = inner, level 1 = outer)"""
    bs, bt = (C.c_double * 2)(*beta_s), (C.c_double * 2)(*beta_t)
    _check(lib.qcd_nested_leapfrog(lat.handle, _prec(U), C.byref(bs), C.byref(bt), tau, n_outer, n_inner, _ptr(U),
                                   _ptr(P), _stream(stream)))


def qcd_spinor_gaussian(lat, eta, seed, stream_id=0, subset=ALL, stream=None):
    _check(lib.qcd_spinor_gaussian(lat.handle, _prec(eta), subset, seed, stream_id, _ptr(eta), _stream(stream)))


def qcd_inner_product(lat, nc, a, b, out, workspace, subset=ALL, stream=None):
    _check(lib.qcd_inner_product(lat.handle, _prec(a), subset, nc, _ptr(a), _ptr(b), _ptr(out), _ptr(workspace),
                                 _stream(stream)))


def qcd_inner_product_multi(lat, nc, a, b, out, workspace, stream=None):
    _check(lib.qcd_inner_product_multi(lat.handle, _prec(a), nc, _ptr(a), _ptr(b), _ptr(out), _ptr(workspace),
                                       _stream(stream)))


def qcd_tune_set(lat, prec, subset, kernel, variant=0, tile=None, threads=0):
    arr = (C.c_int * 4)(*tile) if tile else None
    _check(lib.qcd_tune_set(lat.handle, prec, subset, kernel, variant, C.byref(arr) if tile else None, threads))


def qcd_tune_get(lat, prec, subset, kernel):
    """(variant, tile, threads) or None when the database has no entry"""
    v, t, arr = _i(), _i(), (C.c_int * 4)()
    rc = lib.qcd_tune_get(lat.handle, prec, subset, kernel, C.byref(v), C.byref(arr), C.byref(t))
    return None if rc != OK else (v.value, tuple(arr), t.value)


def qcd_tune_clear():
    _check(lib.qcd_tune_clear())


def qcd_pack(lat, ncomp, layout, lex_aos, dev_soa, stream=None):
    _check(lib.qcd_pack(lat.handle, _prec(dev_soa), ncomp, layout, _ptr(lex_aos), _ptr(dev_soa), _stream(stream)))


def qcd_unpack(lat, ncomp, layout, dev_soa, lex_aos, stream=None):
    _check(lib.qcd_unpack(lat.handle, _prec(dev_soa), ncomp, layout, _ptr(dev_soa), _ptr(lex_aos), _stream(stream)))


def qcd_get_map(lat, which, out, stream=None):
    _check(lib.qcd_get_map(lat.handle, which, _ptr(out), _stream(stream)))


def qcd_hot_start(lat, U, seed, sigma, stream=None):
    _check(lib.qcd_hot_start(lat.handle, _prec(U), seed, sigma, _ptr(U), _stream(stream)))


def qcd_perturb(lat, U, seed, sigma, stream=None):
    _check(lib.qcd_perturb(lat.handle, _prec(U), seed, sigma, _ptr(U), _stream(stream)))


def qcd_rng_blocks(seed, stream_id, purpose, site, mu_j, words=None, uniforms=None, gauss=None, stream=None):
    _check(lib.qcd_rng_blocks(seed, stream_id, purpose, site.numel(), _ptr(site), _ptr(mu_j), _ptr(words),
                              _ptr(uniforms), _ptr(gauss), _stream(stream)))


def qcd_md_host(lat, U_host, P_host, beta, eps, nsteps, device_work, stream=None):
    """U_host, P_host: host tensors (pinned for asynchronous copies) in the canonical layout [V,4,3,3,2]."""
    _check(lib.qcd_md_host(lat.handle, _prec(U_host), beta, eps, nsteps, _ptr(U_host), _ptr(P_host),
                           _ptr(device_work), _stream(stream)))


def qcd_copy_timeslices(src_lat, src, src_t, dst_lat, dst, dst_t, nt, ncomp=72, mu_mask=0xF, stream=None):
    _check(lib.qcd_copy_timeslices(src_lat.handle, _ptr(src), src_t, dst_lat.handle, _ptr(dst), dst_t, nt, _prec(src),
                                   ncomp, mu_mask, _stream(stream)))


def qcd_md_step_single_pass_push(lat, U_in, P, U_out, beta, eps_p, eps_u, lo_lat, lo_U_out, hi_lat, hi_U_out,
                                 stream=None):
    _check(lib.qcd_md_step_single_pass_push(lat.handle, _prec(U_in), beta, eps_p, eps_u, _ptr(U_in), _ptr(P),
                                            _ptr(U_out), None if lo_lat is None else lo_lat.handle, _ptr(lo_U_out),
                                            None if hi_lat is None else hi_lat.handle, _ptr(hi_U_out), _stream(stream)))


def qcd_link_update_push(lat, P, U, eps, reunit, lo_lat, lo_U, hi_lat, hi_U, stream=None):
    _check(lib.qcd_link_update_push(lat.handle, _prec(U), eps, _ptr(P), _ptr(U), int(reunit),
                                    None if lo_lat is None else lo_lat.handle, _ptr(lo_U),
                                    None if hi_lat is None else hi_lat.handle, _ptr(hi_U), _stream(stream)))


def qcd_probe_launch(what, prec, reps, scratch, stream=None):
    _check(lib.qcd_probe_launch(what, prec, reps, _ptr(scratch), scratch.numel() * scratch.element_size(),
                                _stream(stream)))


def probe_rate(what, prec=F64, reps=None):
    """work per second of one probe launch (FMA/s or bytes/s), CUDA events, best of 3 after a warm-up"""
    reps = reps or {PROBE_FMA: 4000, PROBE_L1: 2000, PROBE_LDS: 4000, PROBE_L2: 20}[what]
    scratch = torch.zeros(lib.qcd_probe_scratch_bytes(what) // 8 + 1, dtype=torch.float64, device="cuda")
    qcd_probe_launch(what, prec, max(1, reps // 50), scratch)
    best = float("inf")
    for _ in range(3):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        qcd_probe_launch(what, prec, reps, scratch)
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    return lib.qcd_probe_work(what, prec, reps) / (best * 1e-3)


# ---- convenience used by tests and bench: canonical host arrays <-> device fields (via qcd_pack) ----

def field_to_device(lat, host_array, dtype=torch.float64):
    """numpy complex128 [V,4,3,3] (canonical layout) -> device matrix field of `dtype`"""
    t = torch.view_as_real(torch.from_numpy(host_array)).reshape(-1).to(dtype).cuda()
    out = lat.new_matrix_field(dtype)
    qcd_pack(lat, 72, LAYOUT_PAIRS, t, out)
    torch.cuda.current_stream().synchronize()
    return out


def field_to_host(lat, dev_field):
    """device matrix field -> numpy complex128 [V,4,3,3]"""
    t = torch.empty(lat.V * 72, dtype=dev_field.dtype, device=dev_field.device)  # canonical: no padding
    qcd_unpack(lat, 72, LAYOUT_PAIRS, dev_field, t)
    return t.to(torch.float64).cpu().numpy().view("complex128").reshape(lat.V, 4, 3, 3)
