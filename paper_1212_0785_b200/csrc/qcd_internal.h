// qcd_internal.h — host/device shared declarations of libqcdmd (not part of the public ABI).
//
// Device layout (include/qcd.h, su3.cuh): chunks of 32 checkerboard sites; unit k (of NC per site) of site cb at
// ((cb >> 5)*NC + k)*32 + (cb & 31); a matrix field has NC = 36 complex pairs per site, k = mu*9 + 3*row + col.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/qcd.h"

namespace qcd {

// Lattice geometry handed to kernels by value.
struct LatP {
    int L[4];       // extents
    int stride[4];  // lexicographic strides 1, Lx, Lx*Ly, Lx*Ly*Lz
    int V;          // sites
    int Vh;         // V/2 sites per parity
    // domain decomposition in t: a slab lattice stores its timeslices plus a one-site halo on
    // both sides; the stencil kernels update the interior timeslices [t0, t1) only (a full lattice: 0, Lt), and the
    // generator is keyed on the GLOBAL lexicographic site (s + site_off) mod gV (a full lattice: 0, V)
    int t0, t1;
    int site_off, gV;
};

// 4-D tile handled by one thread block of the stencil kernels (force).  The block owns the sites
// of `npar` parities of the tile; T[0] is even so every x-row has T[0]/2 sites of each parity.
struct TileP {
    int T[4];   // tile extents (divide L)
    int nt[4];  // tiles per direction
    int tsp;    // sites per parity per tile = T0/2*T1*T2*T3
    int npar;   // parities per block: 2 (subset ALL) or 1
    int par0;   // parity handled when npar == 1
    int zb;     // launch order of the plane kernel: z-blocks of zb tiles (nt[2]: plain x, y, z, t order)
};

// Reduction geometry (fixed, independent of any tuning, so results are run-to-run identical).
constexpr int RED_THREADS = 256;   // threads per reduction block
constexpr int RED_CHUNK = 1024;    // sites per first-pass block
constexpr int RED_GENERIC_CHUNKS = 256;  // first-pass blocks per subset on the subset_id path
constexpr int MAX_NSUB = 4096;
constexpr int MAX_SUM_NCOMP = 64;
// qcd_plaquette_noalloc: first-pass partial sums that fit the library's built-in scratch array (reduce.cu);
// 32768 doubles = 256 KiB of device memory per GPU, held from the moment the library is loaded there until exit
constexpr int NOALLOC_MAX_PARTIALS = 32768;

}  // namespace qcd

struct qcd_lattice {
    qcd::LatP p;
    int red_chunks_per_seg;  // first-pass blocks per (timeslice, parity) segment
    int red_nseg;            // 2*Lt segments
    size_t workspace_doubles;
    int tile_all[4];  // default 4-D block tile of the stencil kernel, subset ALL (both parities per block)
    int tile_par[4];  // the same for one parity (EVEN / ODD)
    int par_flip;     // slab lattices: 1 if local parity = global parity ^ 1 (subsets are translated at the ABI)
};

namespace qcd {

// one entry of the auto-tuner's database (tune.cu)
struct TuneCfg {
    int variant;   // QCD_FORCE_* for the stencil kernel, ignored otherwise
    int tile[4];   // 4-D block tile of the stencil kernel; tile[0] == 0: library's own choice
    int threads;   // threads per block of a site-local kernel; 0: library default
};
bool tune_lookup(const qcd_lattice *lat, int prec, int subset, int kernel, TuneCfg &out);
void tune_store(const qcd_lattice *lat, int prec, int subset, int kernel, const TuneCfg &cfg);
void tune_clear_all();

void set_error(const char *fmt, ...);
int check_launch(const char *what);

// kernel launchers, one per translation unit; prec already validated. All return QCD_OK/QCD_ECUDA.
int launch_gauge_force(const qcd_lattice *lat, int prec, int subset, double beta, double eps, const void *U,
                       void *out, bool fused_mom, cudaStream_t st);
// anisotropic Wilson force (force.cu): staples of space-space planes weighted ws, space-time planes wt
// (weights include beta; eps multiplies F in the fused momentum update)
int launch_gauge_force_aniso(const qcd_lattice *lat, int prec, int subset, double ws, double wt, double eps,
                             const void *U, void *out, bool fused_mom, cudaStream_t st);
// space-space / space-time plaquette averages (reduce.cu): out_avg[2], out_per_t[Lt][2] or NULL
int launch_plaquette_st(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                        double *ws, cudaStream_t st);
// single-pass MD step (force.cu): P += eps_p F(U); Uout = reunit(exp(i eps_u P) U); U and Uout distinct
int launch_md_single(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u, const void *U, void *P,
                     void *Uout, cudaStream_t st);
int launch_md_single_push(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u, const void *U,
                          void *P, void *Uout, const qcd_lattice *lo, void *lo_U, const qcd_lattice *hi, void *hi_U,
                          cudaStream_t st);
// default block tile of the stencil kernels (force.cu), computed once per lattice
void default_force_tile(const LatP &lat, int npar, int out[4]);
// copy `nt` timeslices starting at src_t of a pair-layout field with nc units per site into dst (same spatial
// extents) starting at dst_t; mu_mask (matrix fields, nc = 36): bit mu set = copy link mu
int launch_copy_timeslices(const qcd_lattice *src_lat, const void *src, int src_t, const qcd_lattice *dst_lat, void *dst,
                           int dst_t, int nt, int prec, int nc, unsigned mu_mask, cudaStream_t st);
// timeslices [t_begin, t_begin + nt) only: the canonical side (src when packing, dst when unpacking) holds exactly
// those sites, the device side is the whole field
int launch_pack_slab(const qcd_lattice *lat, int prec, int ncomp, bool pairs, const void *src, void *dst, bool unpack,
                     int t_begin, int nt, cudaStream_t st);
int launch_mom_update(const qcd_lattice *lat, int prec, int subset, double eps, const void *F, void *P,
                      cudaStream_t st);
int launch_link_update(const qcd_lattice *lat, int prec, int subset, double eps, const void *P, void *U,
                       int mode /*0 exp, 1 exp+reunit, 2 reunit only*/, cudaStream_t st);
// link update of the interior timeslices of a slab fused with the stores of its boundary timeslices into the
// neighbours' halos (update.cu)
int launch_link_update_push(const qcd_lattice *lat, int prec, double eps, const void *P, void *U, int reunit,
                            const qcd_lattice *lo, void *lo_U, const qcd_lattice *hi, void *hi_U, cudaStream_t st);
int launch_mom_refresh(const qcd_lattice *lat, int prec, int subset, uint64_t seed, uint32_t stream_id, void *P,
                       cudaStream_t st);
int launch_hot_start(const qcd_lattice *lat, int prec, uint64_t seed, double sigma, void *U, cudaStream_t st);
int launch_perturb(const qcd_lattice *lat, int prec, uint64_t seed, double sigma, void *U, cudaStream_t st);
int launch_rng_blocks(uint64_t seed, uint32_t stream_id, uint32_t purpose, int n, const uint32_t *site,
                      const uint32_t *mu_j, uint32_t *words, double *uniforms, double *gauss, cudaStream_t st);
int launch_plaquette(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                     double *ws, cudaStream_t st);
// qcd_plaquette_noalloc (reduce.cu): launch_plaquette with the partial sums in the library's built-in scratch array;
// the caller has checked red_nseg * red_chunks_per_seg <= NOALLOC_MAX_PARTIALS
int launch_plaquette_noalloc(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                             cudaStream_t st);
int launch_sum(const qcd_lattice *lat, int prec, int subset, int kind, int ncomp, const void *field, double *out,
               double *ws, cudaStream_t st);
int launch_sum_multi(const qcd_lattice *lat, int prec, int kind, int ncomp, const void *field,
                     const int32_t *subset_id, int nsub, double *out, double *ws, cudaStream_t st);
// force + momentum update (+ link update into Uout when Uout != NULL: the single-pass step) with plaquette and
// kinetic-energy sums as by-products (force.cu); ws: 2*blocks doubles
// out_per_t != NULL: plaquette per timeslice as well; returns -1 without enqueuing anything if the launch
// configuration cannot provide it (the caller then runs launch_plaquette)
int launch_force_sums(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u, const void *U, void *P,
                      void *Uout, double *out_plaq, double *out_K, double *out_per_t, double *ws, cudaStream_t st);
int force_sums_check(const qcd_lattice *lat, int prec);  // QCD_EWORKSPACE if the tuned tile has too many blocks
int launch_sum_partials(const double *partial, int ngroups, int count, double scale, double *out, cudaStream_t st);
int launch_spinor_gaussian(const qcd_lattice *lat, int prec, int subset, uint64_t seed, uint32_t stream_id, void *eta,
                           cudaStream_t st);
int launch_inner_product(const qcd_lattice *lat, int prec, int subset, int nc, const void *a, const void *b,
                         bool per_t, double *out, double *ws, cudaStream_t st);
int launch_pack(const qcd_lattice *lat, int prec, int ncomp, bool pairs, const void *lex, void *soa, bool unpack,
                cudaStream_t st);
// qcd_md_host as a three-stream pipeline over slabs of timeslices (host_pipeline.cu)
bool md_host_can_pipeline(const qcd_lattice *lat);
int md_host_pipelined(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U_host, void *P_host,
                      void *work, size_t fb, cudaStream_t user);
// probes of the FMA / L1 / shared-memory / L2 rates (probe.cu)
double probe_work(int what, int prec, int reps);
size_t probe_scratch_bytes(int what);
int launch_probe(int what, int prec, int reps, void *scratch, cudaStream_t st);
int launch_get_map(const qcd_lattice *lat, int which, int32_t *out, cudaStream_t st);

}  // namespace qcd
