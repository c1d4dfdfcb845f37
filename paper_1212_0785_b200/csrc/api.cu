// api.cu — the C ABI of include/qcd.h: argument checks, error text, dispatch to the kernel launchers.
#include <cstdarg>
#include <cstdio>
#include <new>

#include "qcd_internal.h"
#include "site.cuh"

namespace qcd {

static thread_local char g_err[256] = "";

void set_error(const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

int check_launch(const char *what) {
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        set_error("%s: %s", what, cudaGetErrorString(e));
        return QCD_ECUDA;
    }
    return QCD_OK;
}

static size_t real_bytes(int prec) { return prec == QCD_F64 ? 8 : 4; }

static int bad(int code, const char *fmt, const char *a = "") {
    set_error(fmt, a);
    return code;
}

static int check_common(const qcd_lattice *lat, int prec, const char *fn) {
    if (!lat) return bad(QCD_EINVAL, "%s: lattice is NULL", fn);
    if (prec != QCD_F32 && prec != QCD_F64) return bad(QCD_EINVAL, "%s: unknown prec", fn);
    return QCD_OK;
}
static int check_subset(int subset, const char *fn) {
    if (subset != QCD_ALL && subset != QCD_EVEN && subset != QCD_ODD) return bad(QCD_EINVAL, "%s: unknown subset", fn);
    return QCD_OK;
}
// EVEN / ODD always mean the GLOBAL parity; a slab lattice whose first stored timeslice is globally odd flips them
static int local_subset(const qcd_lattice *lat, int subset) {
    if (subset == QCD_ALL || !lat->par_flip) return subset;
    return subset == QCD_EVEN ? QCD_ODD : QCD_EVEN;
}
static int check_ptr(const void *p, const char *fn) {
    if (!p) return bad(QCD_EINVAL, "%s: NULL field pointer", fn);
    if (((uintptr_t)p) & 15) return bad(QCD_EALIGN, "%s: field pointer not 16-byte aligned", fn);
    return QCD_OK;
}
static int check_alias2(const void *a, size_t bytes_a, const void *b, size_t bytes_b, const char *fn) {
    const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
    if (x < y + bytes_b && y < x + bytes_a) return bad(QCD_EALIAS, "%s: input and output fields overlap", fn);
    return QCD_OK;
}
static int check_alias(const void *a, const void *b, size_t bytes, const char *fn) {
    return check_alias2(a, bytes, b, bytes, fn);
}
// The multi-step integrators run several link updates in a row and have no way to refresh halo timeslices in
// between (and their link update on QCD_ALL would advance the halos with stale momenta), so on a slab lattice or
// a t-view they would return wrong fields without saying so: whole lattices only.
static int check_whole(const qcd_lattice *lat, const char *fn) {
    if (lat->p.t0 != 0 || lat->p.t1 != lat->p.L[3] || lat->p.gV != lat->p.V)
        return bad(QCD_EINVAL, "%s: needs the whole lattice, not a slab lattice or a t-view (halos cannot be refreshed inside the call)", fn);
    return QCD_OK;
}
// the kernels index the units of a field with 32 bits: nc units per site need nc (V + 32) < 2^32
static int check_units(const qcd_lattice *lat, long long nc, const char *fn) {
    if (nc * ((long long)lat->p.V + 32) >= (1ll << 32)) return bad(QCD_EDIMS, "%s: units per site x V must be < 2^32", fn);
    return QCD_OK;
}

}  // namespace qcd

using namespace qcd;

#define QCD_TRY(expr)            \
    do {                         \
        const int rc_ = (expr);  \
        if (rc_ != QCD_OK) return rc_; \
    } while (0)

extern "C" {

// the descriptor of a lattice with extents dims whose stencil kernels update the timeslices [t0, t1)
static int make_lattice(const int dims[4], int t0, int t1, long long site_off, long long gV, int par_flip,
                        qcd_lattice **out, const char *fn) {
    long long V = 1;
    for (int d = 0; d < 4; d++) {
        if (dims[d] < 2 || (dims[d] & 1)) return bad(QCD_EDIMS, "%s: extents must be even and >= 2", fn);
        V *= dims[d];
        // 36 V < 2^32: the kernels index the 36 V complex pairs of a matrix field with 32 bits
        if (36 * (V + 32) >= (1ll << 32)) return bad(QCD_EDIMS, "%s: V must be < 2^32 / 36", fn);
    }
    qcd_lattice *lat = new (std::nothrow) qcd_lattice;
    if (!lat) return bad(QCD_EINVAL, "%s: out of host memory", fn);
    int stride = 1;
    for (int d = 0; d < 4; d++) {
        lat->p.L[d] = dims[d];
        lat->p.stride[d] = stride;
        stride *= dims[d];
    }
    lat->p.V = (int)V;
    lat->p.Vh = (int)(V / 2);
    lat->p.t0 = t0;
    lat->p.t1 = t1;
    lat->p.site_off = (int)site_off;
    lat->p.gV = (int)(gV ? gV : V);
    lat->par_flip = par_flip;
    const int Vsh = lat->p.Vh / dims[3];
    lat->red_chunks_per_seg = (Vsh + RED_CHUNK - 1) / RED_CHUNK;
    lat->red_nseg = 2 * dims[3];
    const size_t a = (size_t)MAX_SUM_NCOMP * lat->red_nseg * lat->red_chunks_per_seg;
    const size_t b = (size_t)MAX_NSUB * RED_GENERIC_CHUNKS;
    const size_t c = 2 * ((size_t)V / 32 + 1);  // per-block partial pairs of the kernels that reduce as a by-product
    lat->workspace_doubles = (a > b ? (a > c ? a : c) : (b > c ? b : c)) + 64;
    default_force_tile(lat->p, 2, lat->tile_all);
    default_force_tile(lat->p, 1, lat->tile_par);
    *out = lat;
    return QCD_OK;
}

int qcd_lattice_create(const int dims[4], qcd_lattice **out) {
    if (!dims || !out) return bad(QCD_EINVAL, "%s: NULL argument", "qcd_lattice_create");
    return make_lattice(dims, 0, dims[3], 0, 0, 0, out, "qcd_lattice_create");
}

int qcd_lattice_create_slab(const int global_dims[4], int t_begin, int t_count, qcd_lattice **out) {
    const char *fn = "qcd_lattice_create_slab";
    if (!global_dims || !out) return bad(QCD_EINVAL, "%s: NULL argument", fn);
    long long gV = 1;
    for (int d = 0; d < 4; d++) {
        if (global_dims[d] < 2 || (global_dims[d] & 1)) return bad(QCD_EDIMS, "%s: extents must be even and >= 2", fn);
        gV *= global_dims[d];
    }
    const int Lt = global_dims[3];
    if (t_count < 2 || (t_count & 1) || t_count > Lt || t_begin < 0 || t_begin >= Lt)
        return bad(QCD_EDIMS, "%s: t_count must be even, 2..Lt, and 0 <= t_begin < Lt", fn);
    const int dims[4] = {global_dims[0], global_dims[1], global_dims[2], t_count + 2};
    const long long Vs = gV / Lt;
    // slab timeslice te is global timeslice (t_begin + te - 1) mod Lt
    return make_lattice(dims, 1, t_count + 1, Vs * ((t_begin - 1 + Lt) % Lt), gV, (t_begin - 1 + Lt) & 1, out, fn);
}

int qcd_lattice_view_t(const qcd_lattice *lat, int t0, int t1, qcd_lattice **out) {
    const char *fn = "qcd_lattice_view_t";
    if (!lat || !out) return bad(QCD_EINVAL, "%s: NULL argument", fn);
    if (t0 < 0 || t1 > lat->p.L[3] || t1 <= t0) return bad(QCD_EDIMS, "%s: need 0 <= t0 < t1 <= Lt", fn);
    qcd_lattice *v = new (std::nothrow) qcd_lattice(*lat);
    if (!v) return bad(QCD_EINVAL, "%s: out of host memory", fn);
    v->p.t0 = t0;
    v->p.t1 = t1;
    default_force_tile(v->p, 2, v->tile_all);
    default_force_tile(v->p, 1, v->tile_par);
    *out = v;
    return QCD_OK;
}

int qcd_lattice_dims(const qcd_lattice *lat, int dims[4], int interior_t[2]) {
    if (!lat || !dims) return bad(QCD_EINVAL, "%s: NULL argument", "qcd_lattice_dims");
    for (int d = 0; d < 4; d++) dims[d] = lat->p.L[d];
    if (interior_t) {
        interior_t[0] = lat->p.t0;
        interior_t[1] = lat->p.t1;
    }
    return QCD_OK;
}

int qcd_lattice_destroy(qcd_lattice *lat) {
    delete lat;
    return QCD_OK;
}

int64_t qcd_lattice_volume(const qcd_lattice *lat) { return lat ? lat->p.V : 0; }

size_t qcd_field_bytes(const qcd_lattice *lat, int prec, int ncomp) {
    if (!lat || ncomp < 1 || (prec != QCD_F32 && prec != QCD_F64)) return 0;
    const size_t padded = ((size_t)lat->p.V + 31) / 32 * 32;  // whole chunks of 32 sites
    return padded * ncomp * real_bytes(prec);
}

size_t qcd_workspace_bytes(const qcd_lattice *lat) { return lat ? lat->workspace_doubles * sizeof(double) : 0; }

size_t qcd_md_host_work_bytes(const qcd_lattice *lat, int prec) { return 4 * qcd_field_bytes(lat, prec, 72); }

const char *qcd_last_error(void) { return g_err; }

const char *qcd_version(void) { return "qcdmd 0.1 sm_100a"; }

int qcd_gauge_force(const qcd_lattice *lat, int prec, int subset, double beta, const void *U, void *F, void *stream) {
    const char *fn = "qcd_gauge_force";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(F, fn));
    QCD_TRY(check_alias(U, F, qcd_field_bytes(lat, prec, 72), fn));
    return launch_gauge_force(lat, prec, local_subset(lat, subset), beta, 0.0, U, F, false, (cudaStream_t)stream);
}

int qcd_mom_update(const qcd_lattice *lat, int prec, int subset, double eps, const void *F, void *P, void *stream) {
    const char *fn = "qcd_mom_update";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    QCD_TRY(check_ptr(F, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_alias(F, P, qcd_field_bytes(lat, prec, 72), fn));
    return launch_mom_update(lat, prec, local_subset(lat, subset), eps, F, P, (cudaStream_t)stream);
}

int qcd_force_mom_update(const qcd_lattice *lat, int prec, int subset, double beta, double eps, const void *U,
                         void *P, void *stream) {
    const char *fn = "qcd_force_mom_update";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_alias(U, P, qcd_field_bytes(lat, prec, 72), fn));
    return launch_gauge_force(lat, prec, local_subset(lat, subset), beta, eps, U, P, true, (cudaStream_t)stream);
}

int qcd_link_update(const qcd_lattice *lat, int prec, int subset, double eps, const void *P, void *U, int reunit,
                    void *stream) {
    const char *fn = "qcd_link_update";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_alias(P, U, qcd_field_bytes(lat, prec, 72), fn));
    return launch_link_update(lat, prec, local_subset(lat, subset), eps, P, U, reunit ? 1 : 0, (cudaStream_t)stream);
}

int qcd_reunit(const qcd_lattice *lat, int prec, int subset, void *U, void *stream) {
    const char *fn = "qcd_reunit";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    QCD_TRY(check_ptr(U, fn));
    return launch_link_update(lat, prec, local_subset(lat, subset), 0.0, U, U, 2, (cudaStream_t)stream);
}

int qcd_mom_refresh(const qcd_lattice *lat, int prec, int subset, uint64_t seed, uint32_t stream_id, void *P,
                    void *stream) {
    const char *fn = "qcd_mom_refresh";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    QCD_TRY(check_ptr(P, fn));
    return launch_mom_refresh(lat, prec, local_subset(lat, subset), seed, stream_id, P, (cudaStream_t)stream);
}

int qcd_plaquette(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                  void *workspace, void *stream) {
    const char *fn = "qcd_plaquette";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(U, fn));
    if (!out_avg || !workspace) return bad(QCD_EINVAL, "%s: NULL output or workspace", fn);
    return launch_plaquette(lat, prec, U, out_avg, out_per_t, (double *)workspace, (cudaStream_t)stream);
}

// qcd_plaquette for callers that have no device memory to offer as workspace (include/qcd.h): the partial sums
// go to the array built into the library (reduce.cu).  No allocation here or below; the size is checked before
// any CUDA call.
int qcd_plaquette_noalloc(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                          void *stream) {
    const char *fn = "qcd_plaquette_noalloc";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(U, fn));
    if (!out_avg) return bad(QCD_EINVAL, "%s: NULL output", fn);
    const long long need = (long long)lat->red_nseg * lat->red_chunks_per_seg;
    if (need > NOALLOC_MAX_PARTIALS) {
        set_error("%s: this lattice needs %lld partial sums, the built-in scratch holds %d (2 Lt ceil(Lx Ly Lz / 2048) "
                  "must not exceed it); use qcd_plaquette with a workspace of your own",
                  fn, need, NOALLOC_MAX_PARTIALS);
        return QCD_EWORKSPACE;
    }
    return launch_plaquette_noalloc(lat, prec, U, out_avg, out_per_t, (cudaStream_t)stream);
}

static int check_sum_args(int kind, int ncomp, const char *fn) {
    if (kind != QCD_SUM_SCALAR && kind != QCD_SUM_NORM2 && kind != QCD_SUM_RETR) return bad(QCD_EINVAL, "%s: unknown kind", fn);
    if (ncomp < 1) return bad(QCD_EINVAL, "%s: ncomp < 1", fn);
    if (kind == QCD_SUM_SCALAR && ncomp > MAX_SUM_NCOMP) return bad(QCD_EINVAL, "%s: ncomp > 64 for SCALAR", fn);
    if (kind == QCD_SUM_RETR && ncomp % 18) return bad(QCD_EINVAL, "%s: RETR needs ncomp %% 18 == 0", fn);
    if (kind == QCD_SUM_NORM2 && ncomp % 18 && ncomp % 24)
        return bad(QCD_EINVAL, "%s: NORM2 needs a complex-pair field (ncomp %% 18 == 0 or ncomp %% 24 == 0)", fn);
    return QCD_OK;
}

int qcd_sum(const qcd_lattice *lat, int prec, int subset, int kind, int ncomp, const void *field, double *out,
            void *workspace, void *stream) {
    const char *fn = "qcd_sum";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    QCD_TRY(check_sum_args(kind, ncomp, fn));
    QCD_TRY(check_units(lat, kind == QCD_SUM_SCALAR ? ncomp : ncomp / 2, fn));
    QCD_TRY(check_ptr(field, fn));
    if (!out || !workspace) return bad(QCD_EINVAL, "%s: NULL output or workspace", fn);
    return launch_sum(lat, prec, local_subset(lat, subset), kind, ncomp, field, out, (double *)workspace, (cudaStream_t)stream);
}

int qcd_sum_multi(const qcd_lattice *lat, int prec, int kind, int ncomp, const void *field, const int32_t *subset_id,
                  int nsub, double *out, void *workspace, void *stream) {
    const char *fn = "qcd_sum_multi";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_sum_args(kind, ncomp, fn));
    QCD_TRY(check_units(lat, kind == QCD_SUM_SCALAR ? ncomp : ncomp / 2, fn));
    QCD_TRY(check_ptr(field, fn));
    if (!out || !workspace) return bad(QCD_EINVAL, "%s: NULL output or workspace", fn);
    if (nsub < 1 || nsub > MAX_NSUB) return bad(QCD_EINVAL, "%s: nsub out of range [1,4096]", fn);
    if (!subset_id && nsub != lat->p.L[3]) return bad(QCD_EINVAL, "%s: timeslice set needs nsub == Lt", fn);
    if (subset_id && (size_t)nsub * (kind == QCD_SUM_SCALAR ? ncomp : 1) > (size_t)MAX_NSUB)
        return bad(QCD_EINVAL, "%s: nsub*ncomp > 4096 on the subset_id path", fn);
    return launch_sum_multi(lat, prec, kind, ncomp, field, subset_id, nsub, out, (double *)workspace,
                            (cudaStream_t)stream);
}

int qcd_md_step(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u, void *U, void *P,
                void *stream) {
    const char *fn = "qcd_md_step";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_alias(U, P, qcd_field_bytes(lat, prec, 72), fn));
    QCD_TRY(launch_gauge_force(lat, prec, QCD_ALL, beta, eps_p, U, P, true, (cudaStream_t)stream));
    return launch_link_update(lat, prec, QCD_ALL, eps_u, P, U, 1, (cudaStream_t)stream);
}

int qcd_leapfrog(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U, void *P,
                 void *stream) {
    const char *fn = "qcd_leapfrog";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_whole(lat, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_alias(U, P, qcd_field_bytes(lat, prec, 72), fn));
    if (nsteps < 1) return bad(QCD_EINVAL, "%s: nsteps < 1", fn);
    cudaStream_t st = (cudaStream_t)stream;
    QCD_TRY(launch_gauge_force(lat, prec, QCD_ALL, beta, 0.5 * eps, U, P, true, st));
    for (int k = 0; k < nsteps; k++) {
        QCD_TRY(launch_link_update(lat, prec, QCD_ALL, eps, P, U, 1, st));
        QCD_TRY(launch_gauge_force(lat, prec, QCD_ALL, beta, k == nsteps - 1 ? 0.5 * eps : eps, U, P, true, st));
    }
    return QCD_OK;
}

int qcd_force_mom_update_sums(const qcd_lattice *lat, int prec, double beta, double eps, const void *U, void *P,
                              double *out, void *workspace, void *stream) {
    const char *fn = "qcd_force_mom_update_sums";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_alias(U, P, qcd_field_bytes(lat, prec, 72), fn));
    if (!out || !workspace) return bad(QCD_EINVAL, "%s: NULL output or workspace", fn);
    return launch_force_sums(lat, prec, beta, eps, 0.0, U, P, nullptr, out, out + 1, nullptr, (double *)workspace,
                             (cudaStream_t)stream);
}

int qcd_leapfrog_energy(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U, void *P,
                        double *out, void *workspace, void *stream) {
    const char *fn = "qcd_leapfrog_energy";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_whole(lat, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_alias(U, P, qcd_field_bytes(lat, prec, 72), fn));
    if (nsteps < 1) return bad(QCD_EINVAL, "%s: nsteps < 1", fn);
    if (!out || !workspace) return bad(QCD_EINVAL, "%s: NULL output or workspace", fn);
    cudaStream_t st = (cudaStream_t)stream;
    QCD_TRY(launch_gauge_force(lat, prec, QCD_ALL, beta, 0.5 * eps, U, P, true, st));
    for (int k = 0; k < nsteps; k++) {
        QCD_TRY(launch_link_update(lat, prec, QCD_ALL, eps, P, U, 1, st));
        if (k < nsteps - 1) QCD_TRY(launch_gauge_force(lat, prec, QCD_ALL, beta, eps, U, P, true, st));
    }
    return launch_force_sums(lat, prec, beta, 0.5 * eps, 0.0, U, P, nullptr, out, out + 1, nullptr, (double *)workspace, st);
}

int qcd_md_step_single_pass(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u,
                            const void *U_in, void *P, void *U_out, void *stream) {
    const char *fn = "qcd_md_step_single_pass";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(U_in, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_ptr(U_out, fn));
    const size_t fb = qcd_field_bytes(lat, prec, 72);
    QCD_TRY(check_alias(U_in, P, fb, fn));
    QCD_TRY(check_alias(U_in, U_out, fb, fn));
    QCD_TRY(check_alias(P, U_out, fb, fn));
    return launch_md_single(lat, prec, beta, eps_p, eps_u, U_in, P, U_out, (cudaStream_t)stream);
}

int qcd_leapfrog_single_pass(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U,
                             void *P, void *U_work, void *stream) {
    const char *fn = "qcd_leapfrog_single_pass";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_whole(lat, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_ptr(U_work, fn));
    const size_t fb = qcd_field_bytes(lat, prec, 72);
    QCD_TRY(check_alias(U, P, fb, fn));
    QCD_TRY(check_alias(U, U_work, fb, fn));
    QCD_TRY(check_alias(P, U_work, fb, fn));
    if (nsteps < 1) return bad(QCD_EINVAL, "%s: nsteps < 1", fn);
    cudaStream_t st = (cudaStream_t)stream;
    // O11 regrouped: n x { P += a_k F(U); U <- reunit(exp(i eps P) U) } with a_0 = eps/2, then P += (eps/2) F(U)
    void *cur = U, *other = U_work;
    int k = 0;
    if (nsteps & 1) {  // keep the number of ping-pong steps even so the result lands in U
        QCD_TRY(launch_gauge_force(lat, prec, QCD_ALL, beta, 0.5 * eps, U, P, true, st));
        QCD_TRY(launch_link_update(lat, prec, QCD_ALL, eps, P, U, 1, st));
        k = 1;
    }
    for (; k < nsteps; k++) {
        QCD_TRY(launch_md_single(lat, prec, beta, k == 0 ? 0.5 * eps : eps, eps, cur, P, other, st));
        void *t = cur;
        cur = other;
        other = t;
    }
    return launch_gauge_force(lat, prec, QCD_ALL, beta, 0.5 * eps, cur, P, true, st);
}

int qcd_trajectory(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U, void *P, void *U_work,
                   double *obs, double *per_t, void *workspace, size_t workspace_bytes, void *stream) {
    const char *fn = "qcd_trajectory";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_whole(lat, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_ptr(U_work, fn));
    const size_t fb = qcd_field_bytes(lat, prec, 72);
    QCD_TRY(check_alias(U, P, fb, fn));
    QCD_TRY(check_alias(U, U_work, fb, fn));
    QCD_TRY(check_alias(P, U_work, fb, fn));
    if (nsteps < 1) return bad(QCD_EINVAL, "%s: nsteps < 1", fn);
    if (!obs || !workspace) return bad(QCD_EINVAL, "%s: NULL output or workspace", fn);
    if (workspace_bytes < qcd_workspace_bytes(lat)) return bad(QCD_EWORKSPACE, "%s: workspace smaller than qcd_workspace_bytes", fn);
    QCD_TRY(force_sums_check(lat, prec));
    cudaStream_t st = (cudaStream_t)stream;
    double *ws = (double *)workspace;
    double *scratch = ws + lat->workspace_doubles - 8;  // K after the opening half kick has no slot in obs
    const int Lt = lat->p.L[3];
    // One kick (+ link update into `to` when to != NULL) with plaq(U), per-timeslice plaq(U) and K(P after) as
    // by-products; the per-timeslice values fall back to the stand-alone plaquette kernel when the launch
    // configuration cannot give them.
    auto kick = [&](double eps_p, void *from, void *to, double *o_plaq, double *o_K, double *o_per_t) -> int {
        int rc = launch_force_sums(lat, prec, beta, eps_p, eps, from, P, to, o_plaq, o_K, o_per_t, ws, st);
        if (rc == -1) {
            QCD_TRY(launch_plaquette(lat, prec, from, o_plaq, o_per_t, ws, st));
            rc = launch_force_sums(lat, prec, beta, eps_p, eps, from, P, to, o_plaq, o_K, nullptr, ws, st);
        }
        return rc;
    };
    // O11 regrouped as in qcd_leapfrog_single_pass; step k reports plaq(U_k) and K of the momenta after its kick
    QCD_TRY(launch_sum(lat, prec, QCD_ALL, QCD_SUM_NORM2, 72, P, obs + 1, ws, st));  // K of the initial momenta
    void *cur = U, *other = U_work;
    int k = 0;
    if (nsteps & 1) {  // keep the number of ping-pong steps even so the result lands in U
        QCD_TRY(kick(0.5 * eps, U, nullptr, obs, scratch, per_t));
        QCD_TRY(launch_link_update(lat, prec, QCD_ALL, eps, P, U, 1, st));
        k = 1;
    }
    for (; k < nsteps; k++) {
        QCD_TRY(kick(k == 0 ? 0.5 * eps : eps, cur, other, obs + 2 * k, k == 0 ? scratch : obs + 2 * k + 1,
                     per_t ? per_t + (size_t)k * Lt : nullptr));
        void *t = cur;
        cur = other;
        other = t;
    }
    return kick(0.5 * eps, cur, nullptr, obs + 2 * nsteps, obs + 2 * nsteps + 1,
                per_t ? per_t + (size_t)nsteps * Lt : nullptr);
}

int qcd_gauge_force_aniso(const qcd_lattice *lat, int prec, int subset, double beta_s, double beta_t, const void *U,
                          void *F, void *stream) {
    const char *fn = "qcd_gauge_force_aniso";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(F, fn));
    QCD_TRY(check_alias(U, F, qcd_field_bytes(lat, prec, 72), fn));
    return launch_gauge_force_aniso(lat, prec, local_subset(lat, subset), beta_s, beta_t, 0.0, U, F, false, (cudaStream_t)stream);
}

int qcd_force_mom_update_aniso(const qcd_lattice *lat, int prec, int subset, double beta_s, double beta_t,
                               double eps, const void *U, void *P, void *stream) {
    const char *fn = "qcd_force_mom_update_aniso";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_alias(U, P, qcd_field_bytes(lat, prec, 72), fn));
    return launch_gauge_force_aniso(lat, prec, local_subset(lat, subset), beta_s, beta_t, eps, U, P, true, (cudaStream_t)stream);
}

int qcd_plaquette_st(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                     void *workspace, void *stream) {
    const char *fn = "qcd_plaquette_st";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(U, fn));
    if (!out_avg || !workspace) return bad(QCD_EINVAL, "%s: NULL output or workspace", fn);
    return launch_plaquette_st(lat, prec, U, out_avg, out_per_t, (double *)workspace, (cudaStream_t)stream);
}

int qcd_nested_leapfrog(const qcd_lattice *lat, int prec, const double beta_s[2], const double beta_t[2], double tau,
                        int n_outer, int n_inner, void *U, void *P, void *stream) {
    const char *fn = "qcd_nested_leapfrog";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_whole(lat, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_alias(U, P, qcd_field_bytes(lat, prec, 72), fn));
    if (!beta_s || !beta_t) return bad(QCD_EINVAL, "%s: NULL coefficient array", fn);
    if (n_outer < 1 || n_inner < 1) return bad(QCD_EINVAL, "%s: step counts must be >= 1", fn);
    cudaStream_t st = (cudaStream_t)stream;
    const double e1 = tau / n_outer, e0 = e1 / n_inner;
    // a momentum update with step a0 of level 0 and a1 of level 1 at fixed U is one force kernel with plane
    // weights a0*beta[0] + a1*beta[1] and eps = 1
    auto kick = [&](double a0, double a1) {
        return launch_gauge_force_aniso(lat, prec, QCD_ALL, a0 * beta_s[0] + a1 * beta_s[1],
                                        a0 * beta_t[0] + a1 * beta_t[1], 1.0, U, P, true, st);
    };
    QCD_TRY(kick(0.5 * e0, 0.5 * e1));
    for (int k = 0; k < n_outer; k++)
        for (int j = 0; j < n_inner; j++) {
            QCD_TRY(launch_link_update(lat, prec, QCD_ALL, e0, P, U, 1, st));
            const bool inner_end = j == n_inner - 1, traj_end = inner_end && k == n_outer - 1;
            if (!inner_end) QCD_TRY(kick(e0, 0.0));
            else if (!traj_end) QCD_TRY(kick(e0, e1));  // (e0/2 + e1/2) closing this outer step + the same opening the next
            else QCD_TRY(kick(0.5 * e0, 0.5 * e1));
        }
    return QCD_OK;
}

int qcd_spinor_gaussian(const qcd_lattice *lat, int prec, int subset, uint64_t seed, uint32_t stream_id, void *eta,
                        void *stream) {
    const char *fn = "qcd_spinor_gaussian";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    QCD_TRY(check_ptr(eta, fn));
    return launch_spinor_gaussian(lat, prec, local_subset(lat, subset), seed, stream_id, eta, (cudaStream_t)stream);
}

static int check_inner(const qcd_lattice *lat, int prec, int nc, const void *a, const void *b, const double *out,
                       const void *workspace, const char *fn) {
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(a, fn));
    QCD_TRY(check_ptr(b, fn));
    if (nc < 1) return bad(QCD_EINVAL, "%s: nc < 1", fn);
    QCD_TRY(check_units(lat, nc, fn));
    if (!out || !workspace) return bad(QCD_EINVAL, "%s: NULL output or workspace", fn);
    return QCD_OK;
}

int qcd_inner_product(const qcd_lattice *lat, int prec, int subset, int nc, const void *a, const void *b, double *out,
                      void *workspace, void *stream) {
    const char *fn = "qcd_inner_product";
    QCD_TRY(check_inner(lat, prec, nc, a, b, out, workspace, fn));
    QCD_TRY(check_subset(subset, fn));
    return launch_inner_product(lat, prec, local_subset(lat, subset), nc, a, b, false, out, (double *)workspace, (cudaStream_t)stream);
}

int qcd_inner_product_multi(const qcd_lattice *lat, int prec, int nc, const void *a, const void *b, double *out,
                            void *workspace, void *stream) {
    const char *fn = "qcd_inner_product_multi";
    QCD_TRY(check_inner(lat, prec, nc, a, b, out, workspace, fn));
    return launch_inner_product(lat, prec, QCD_ALL, nc, a, b, true, out, (double *)workspace, (cudaStream_t)stream);
}

int qcd_tune_set(const qcd_lattice *lat, int prec, int subset, int kernel, int variant, const int tile[4],
                 int threads) {
    const char *fn = "qcd_tune_set";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    TuneCfg cfg = {0, {0, 0, 0, 0}, 0};
    if (kernel == QCD_KERNEL_FORCE) {
        if (variant != QCD_FORCE_STAPLE && variant != QCD_FORCE_PLANE) return bad(QCD_EINVAL, "%s: unknown force variant", fn);
        cfg.variant = variant;
        if (tile && tile[0]) {
            long sites = 1;
            for (int d = 0; d < 4; d++) {
                const int ext = d == 3 ? lat->p.t1 - lat->p.t0 : lat->p.L[d];
                if (tile[d] < 1 || ext % tile[d]) return bad(QCD_EINVAL, "%s: tile must divide the lattice", fn);
                sites *= tile[d];
                cfg.tile[d] = tile[d];
            }
            if (tile[0] & 1) return bad(QCD_EINVAL, "%s: tile[0] must be even", fn);
            const long threads_needed = subset == QCD_ALL ? sites : sites / 2;
            if (threads_needed > 128) return bad(QCD_EINVAL, "%s: tile has more sites than a block can hold (128)", fn);
        }
    } else if (kernel == QCD_KERNEL_LINK_UPDATE || kernel == QCD_KERNEL_MOM_UPDATE) {
        if (threads < 32 || threads > 256 || threads % 32) return bad(QCD_EINVAL, "%s: threads must be 32..256, multiple of 32", fn);
        cfg.threads = threads;
    } else {
        return bad(QCD_EINVAL, "%s: unknown kernel", fn);
    }
    tune_store(lat, prec, subset, kernel, cfg);
    return QCD_OK;
}

int qcd_tune_get(const qcd_lattice *lat, int prec, int subset, int kernel, int *variant, int tile[4], int *threads) {
    const char *fn = "qcd_tune_get";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_subset(subset, fn));
    TuneCfg cfg;
    if (!tune_lookup(lat, prec, subset, kernel, cfg)) return bad(QCD_EINVAL, "%s: no entry", fn);
    if (variant) *variant = cfg.variant;
    if (tile)
        for (int d = 0; d < 4; d++) tile[d] = cfg.tile[d];
    if (threads) *threads = cfg.threads;
    return QCD_OK;
}

int qcd_tune_clear(void) {
    tune_clear_all();
    return QCD_OK;
}

static int check_layout(const qcd_lattice *lat, int ncomp, int layout, const char *fn) {
    if (ncomp < 1) return bad(QCD_EINVAL, "%s: ncomp < 1", fn);
    if (layout != QCD_LAYOUT_REAL && layout != QCD_LAYOUT_PAIRS) return bad(QCD_EINVAL, "%s: unknown layout", fn);
    if (layout == QCD_LAYOUT_PAIRS && (ncomp & 1)) return bad(QCD_EINVAL, "%s: the pair layout needs an even ncomp", fn);
    return check_units(lat, layout == QCD_LAYOUT_PAIRS ? ncomp / 2 : ncomp, fn);
}

int qcd_pack(const qcd_lattice *lat, int prec, int ncomp, int layout, const void *lex_aos, void *dev_soa, void *stream) {
    const char *fn = "qcd_pack";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_layout(lat, ncomp, layout, fn));
    QCD_TRY(check_ptr(lex_aos, fn));
    QCD_TRY(check_ptr(dev_soa, fn));
    // the canonical array has exactly V sites, the device field whole chunks of 32
    QCD_TRY(check_alias2(lex_aos, (size_t)lat->p.V * ncomp * real_bytes(prec), dev_soa, qcd_field_bytes(lat, prec, ncomp), fn));
    return launch_pack(lat, prec, ncomp, layout == QCD_LAYOUT_PAIRS, lex_aos, dev_soa, false, (cudaStream_t)stream);
}

int qcd_unpack(const qcd_lattice *lat, int prec, int ncomp, int layout, const void *dev_soa, void *lex_aos, void *stream) {
    const char *fn = "qcd_unpack";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_layout(lat, ncomp, layout, fn));
    QCD_TRY(check_ptr(lex_aos, fn));
    QCD_TRY(check_ptr(dev_soa, fn));
    QCD_TRY(check_alias2(lex_aos, (size_t)lat->p.V * ncomp * real_bytes(prec), dev_soa, qcd_field_bytes(lat, prec, ncomp), fn));
    return launch_pack(lat, prec, ncomp, layout == QCD_LAYOUT_PAIRS, dev_soa, lex_aos, true, (cudaStream_t)stream);
}

int qcd_get_map(const qcd_lattice *lat, int which, int32_t *dev_out, void *stream) {
    const char *fn = "qcd_get_map";
    if (!lat || !dev_out) return bad(QCD_EINVAL, "%s: NULL argument", fn);
    if (which < QCD_MAP_CB_OF_LEX || which > QCD_MAP_TSLICE) return bad(QCD_EINVAL, "%s: unknown map", fn);
    return launch_get_map(lat, which, dev_out, (cudaStream_t)stream);
}

int qcd_hot_start(const qcd_lattice *lat, int prec, uint64_t seed, double sigma, void *U, void *stream) {
    const char *fn = "qcd_hot_start";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(U, fn));
    return launch_hot_start(lat, prec, seed, sigma, U, (cudaStream_t)stream);
}

int qcd_perturb(const qcd_lattice *lat, int prec, uint64_t seed, double sigma, void *U, void *stream) {
    const char *fn = "qcd_perturb";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(U, fn));
    return launch_perturb(lat, prec, seed, sigma, U, (cudaStream_t)stream);
}

int qcd_rng_blocks(uint64_t seed, uint32_t stream_id, uint32_t purpose, int n, const uint32_t *site,
                   const uint32_t *mu_j, uint32_t *words, double *uniforms, double *gauss, void *stream) {
    const char *fn = "qcd_rng_blocks";
    if (n < 0 || (n > 0 && (!site || !mu_j))) return bad(QCD_EINVAL, "%s: bad arguments", fn);
    return launch_rng_blocks(seed, stream_id, purpose, n, site, mu_j, words, uniforms, gauss, (cudaStream_t)stream);
}

int qcd_copy_timeslices(const qcd_lattice *src_lat, const void *src, int src_t, const qcd_lattice *dst_lat, void *dst,
                        int dst_t, int nt, int prec, int ncomp, unsigned mu_mask, void *stream) {
    const char *fn = "qcd_copy_timeslices";
    QCD_TRY(check_common(src_lat, prec, fn));
    QCD_TRY(check_common(dst_lat, prec, fn));
    QCD_TRY(check_ptr(src, fn));
    QCD_TRY(check_ptr(dst, fn));
    for (int d = 0; d < 3; d++)
        if (src_lat->p.L[d] != dst_lat->p.L[d]) return bad(QCD_EDIMS, "%s: the two lattices differ in a spatial extent", fn);
    if (ncomp < 2 || (ncomp & 1)) return bad(QCD_EINVAL, "%s: ncomp must be even (pair layout)", fn);
    if (nt < 1 || src_t < 0 || src_t + nt > src_lat->p.L[3] || dst_t < 0 || dst_t + nt > dst_lat->p.L[3])
        return bad(QCD_EINVAL, "%s: timeslice range outside a lattice", fn);
    if (src == dst && src_t < dst_t + nt && dst_t < src_t + nt) return bad(QCD_EALIAS, "%s: overlapping timeslices of one field", fn);
    return launch_copy_timeslices(src_lat, src, src_t, dst_lat, dst, dst_t, nt, prec, ncomp / 2, mu_mask,
                                  (cudaStream_t)stream);
}

// neighbours of a slab for the calls that store into their halos: both or neither of (lattice, field), a slab lattice
// with the same spatial extents
static int check_push_neighbours(const qcd_lattice *lat, int prec, const qcd_lattice *const nb[2], void *const nbU[2],
                                 const void *P, const char *fn) {
    if (lat->p.L[3] < 3 || lat->p.t0 < 1 || lat->p.t1 > lat->p.L[3] - 1)
        return bad(QCD_EINVAL, "%s: needs a slab lattice (halo timeslices on both sides) or a view of one", fn);
    for (int k = 0; k < 2; k++) {
        if ((nb[k] == nullptr) != (nbU[k] == nullptr)) return bad(QCD_EINVAL, "%s: a neighbour needs both its lattice and its field", fn);
        if (!nb[k]) continue;
        QCD_TRY(check_common(nb[k], prec, fn));
        QCD_TRY(check_ptr(nbU[k], fn));
        if (nb[k]->p.L[3] < 3) return bad(QCD_EINVAL, "%s: a neighbour is not a slab lattice", fn);
        for (int d = 0; d < 3; d++)
            if (nb[k]->p.L[d] != lat->p.L[d]) return bad(QCD_EDIMS, "%s: a neighbour differs in a spatial extent", fn);
        if (nbU[k] == P) return bad(QCD_EALIAS, "%s: a neighbour's gauge field is this slab's momentum field", fn);
    }
    return QCD_OK;
}

int qcd_md_step_single_pass_push(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u,
                                 const void *U_in, void *P, void *U_out, const qcd_lattice *lo_lat, void *lo_U_out,
                                 const qcd_lattice *hi_lat, void *hi_U_out, void *stream) {
    const char *fn = "qcd_md_step_single_pass_push";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(U_in, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_ptr(U_out, fn));
    const size_t fb = qcd_field_bytes(lat, prec, 72);
    QCD_TRY(check_alias(U_in, P, fb, fn));
    QCD_TRY(check_alias(U_in, U_out, fb, fn));
    QCD_TRY(check_alias(P, U_out, fb, fn));
    const qcd_lattice *nb[2] = {lo_lat, hi_lat};
    void *nbU[2] = {lo_U_out, hi_U_out};
    QCD_TRY(check_push_neighbours(lat, prec, nb, nbU, P, fn));
    for (int k = 0; k < 2; k++)
        if (nbU[k] == U_in) return bad(QCD_EALIAS, "%s: a neighbour's output field is this slab's input field", fn);
    return launch_md_single_push(lat, prec, beta, eps_p, eps_u, U_in, P, U_out, lo_lat, lo_U_out, hi_lat, hi_U_out,
                                 (cudaStream_t)stream);
}

int qcd_link_update_push(const qcd_lattice *lat, int prec, double eps, const void *P, void *U, int reunit,
                         const qcd_lattice *lo_lat, void *lo_U, const qcd_lattice *hi_lat, void *hi_U, void *stream) {
    const char *fn = "qcd_link_update_push";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_ptr(P, fn));
    QCD_TRY(check_ptr(U, fn));
    QCD_TRY(check_alias(P, U, qcd_field_bytes(lat, prec, 72), fn));
    const qcd_lattice *nb[2] = {lo_lat, hi_lat};
    void *nbU[2] = {lo_U, hi_U};
    QCD_TRY(check_push_neighbours(lat, prec, nb, nbU, P, fn));
    return launch_link_update_push(lat, prec, eps, P, U, reunit ? 1 : 0, lo_lat, lo_U, hi_lat, hi_U, (cudaStream_t)stream);
}

size_t qcd_probe_scratch_bytes(int what) {
    return what >= QCD_PROBE_FMA && what <= QCD_PROBE_L2 ? probe_scratch_bytes(what) : 0;
}

double qcd_probe_work(int what, int prec, int reps) {
    if (what < QCD_PROBE_FMA || what > QCD_PROBE_L2 || reps < 1) return 0.0;
    return probe_work(what, prec, reps);
}

int qcd_probe_launch(int what, int prec, int reps, void *scratch, size_t scratch_bytes, void *stream) {
    const char *fn = "qcd_probe_launch";
    if (what < QCD_PROBE_FMA || what > QCD_PROBE_L2) return bad(QCD_EINVAL, "%s: unknown probe", fn);
    if (prec != QCD_F32 && prec != QCD_F64) return bad(QCD_EINVAL, "%s: unknown prec", fn);
    if (reps < 1) return bad(QCD_EINVAL, "%s: reps < 1", fn);
    QCD_TRY(check_ptr(scratch, fn));
    if (scratch_bytes < probe_scratch_bytes(what)) return bad(QCD_EWORKSPACE, "%s: scratch smaller than qcd_probe_scratch_bytes", fn);
    return launch_probe(what, prec, reps, scratch, (cudaStream_t)stream);
}

int qcd_md_host(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U_host, void *P_host,
                void *device_work, void *stream) {
    const char *fn = "qcd_md_host";
    QCD_TRY(check_common(lat, prec, fn));
    QCD_TRY(check_whole(lat, fn));
    if (!U_host || !P_host) return bad(QCD_EINVAL, "%s: NULL host buffer", fn);
    QCD_TRY(check_ptr(device_work, fn));
    if (nsteps < 0) return bad(QCD_EINVAL, "%s: nsteps < 0", fn);
    cudaStream_t st = (cudaStream_t)stream;
    const size_t fb = qcd_field_bytes(lat, prec, 72);                // device field (whole chunks of 32 sites)
    const size_t hb = (size_t)lat->p.V * 72 * real_bytes(prec);      // canonical host array
    if (md_host_can_pipeline(lat))  // slabs of timeslices on three streams (host_pipeline.cu)
        return md_host_pipelined(lat, prec, beta, eps, nsteps, U_host, P_host, device_work, fb, st);
    // small lattices (fewer than 8 slabs): one stream, whole fields
    char *w = (char *)device_work;
    void *stageU = w, *stageP = w + fb, *U = w + 2 * fb, *P = w + 3 * fb;
    cudaError_t e = cudaMemcpyAsync(stageU, U_host, hb, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(stageP, P_host, hb, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) {
        set_error("%s: H2D copy: %s", fn, cudaGetErrorString(e));
        return QCD_ECUDA;
    }
    QCD_TRY(launch_pack(lat, prec, 72, true, stageU, U, false, st));
    QCD_TRY(launch_pack(lat, prec, 72, true, stageP, P, false, st));
    for (int k = 0; k < nsteps; k++) {
        QCD_TRY(launch_gauge_force(lat, prec, QCD_ALL, beta, eps, U, P, true, st));
        QCD_TRY(launch_link_update(lat, prec, QCD_ALL, eps, P, U, 1, st));
    }
    QCD_TRY(launch_pack(lat, prec, 72, true, U, stageU, true, st));
    QCD_TRY(launch_pack(lat, prec, 72, true, P, stageP, true, st));
    e = cudaMemcpyAsync(U_host, stageU, hb, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(P_host, stageP, hb, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) {
        set_error("%s: D2H copy: %s", fn, cudaGetErrorString(e));
        return QCD_ECUDA;
    }
    return QCD_OK;
}

}  // extern "C"
