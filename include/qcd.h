/* qcd.h — C ABI of libqcdmd: B200 (sm_100a) kernels for the site-parallel SU(3) field operations of
 * the Hybrid Monte-Carlo molecular-dynamics step outside the fermion inverter.
 *
 * The operations are the ones the paper lists as having to leave the CPU (section 1:
 * "momentum updates, force term calculation, projection of fields, reunitarization of SU(3)
 * matrices, a random number generator, exponentiating of SU(3) matrices") and its "non-linear
 * algebra" reductions (section 1: "sum, sumMulti").  Every operation is site-parallel
 * (Table 1 caption and section 3).  The paper defines none of them; the definitions
 * are the textbook ones fixed in SURVEY.md section 8(c) and DESIGN.md ("Readings"), cited per call
 * below as O1..O12.
 *
 * CONVENTIONS
 *   Lattice: extents L = (Lx,Ly,Lz,Lt), all even and >= 2, V = Lx*Ly*Lz*Lt < 2^32/36 (119 304 647: 36 V pair indices fit 32 bits), periodic.
 *   Directions mu = 0..3 <-> x,y,z,t.  Lexicographic site index s = x + Lx*(y + Ly*(z + Lz*t)).
 *   parity(s) = (x+y+z+t) & 1;  checkerboard index cb(s) = parity*V/2 + (s>>1).       [O1]
 *
 *   Precision `prec`: QCD_F64 fields are double, QCD_F32 fields are float.  All field arithmetic is
 *   done in the field's precision; every reduction accumulates and returns double.
 *
 *   DEVICE layout: checkerboarded, site-fastest arrays in CHUNKS OF 32 SITES.  A field with NC units per
 *   site (a unit is a (re,im) pair = `double2`/`float2` for matrix, spin-colour and other pair fields, one
 *   real for real fields) stores unit k of checkerboard site cb at unit index
 *       ((cb >> 5)*NC + k)*32 + (cb & 31)            i.e. [chunk = cb/32][k][lane = cb%32].
 *   Matrix fields (U, P, F; 4 links per site, 3x3 complex each = 72 reals/site): NC = 36, k = mu*9 + e,
 *   e = 3*row + col.  A warp reading one entry of 32 consecutive sites reads 512 contiguous bytes (fp64), and
 *   the 36 entries of a site sit at fixed offsets (k*32 units) from the site's base address.  Even sites
 *   are cb in [0,V/2), odd sites [V/2,V).  A field occupies whole chunks: qcd_field_bytes rounds V up to a
 *   multiple of 32 sites; the padding is never read or written.
 *   Real site fields with ncomp components: NC = ncomp, unit = one real.
 *   CANONICAL (exchange) layout, used by qcd_pack/qcd_unpack and the *_host call: lexicographic
 *   array of structures [s][mu][row][col][re,im] (matrix) or [s][comp] (real).
 *
 *   Subsets: QCD_ALL, QCD_EVEN (parity 0), QCD_ODD.  A subset call writes only sites of the subset
 *   and leaves every other site bit-identical; it may read any site.
 *
 * OWNERSHIP AND ASYNCHRONY
 *   Unless a parameter says "host", every pointer is a DEVICE pointer owned by the caller (e.g. a
 *   PyTorch tensor's data_ptr()).  The library allocates no device memory: fields, outputs and
 *   workspace are the caller's and must stay alive until the stream work has completed (the library image
 *   itself carries one fixed 256 KiB device array, the scratch of qcd_plaquette_noalloc).  `stream`
 *   is a cudaStream_t passed as void* (NULL = the legacy default stream).  Every call only enqueues
 *   work on `stream` and returns without synchronising; reduction results are written to device
 *   doubles.  qcd_lattice is host-only, immutable after creation and may be shared across threads.
 *
 * ERRORS
 *   Return code only: no exceptions, no abort, no printing.  Arguments are validated before the first
 *   launch, so on any return other than QCD_ECUDA nothing was enqueued; QCD_ECUDA (a launch the CUDA runtime
 *   refused) can leave the earlier kernels of a multi-launch call (qcd_md_step, qcd_leapfrog*, qcd_trajectory,
 *   qcd_nested_leapfrog, qcd_md_host) on the stream.  qcd_last_error() returns a thread-local text for the
 *   last nonzero return.
 *     QCD_EINVAL      NULL pointer, unknown enum value, nsub < 1, ncomp < 1 ...
 *     QCD_EDIMS       an extent is odd or < 2, or 36 V >= 2^32
 *     QCD_EALIGN      a field pointer is not 16-byte aligned
 *     QCD_EALIAS      input and output overlap where the operation forbids it
 *     QCD_EWORKSPACE  the workspace is too small (calls that take its size, and tuned tiles with too many blocks)
 *     QCD_ECUDA       the CUDA runtime reported a launch error (text in qcd_last_error)
 *   Scalars beta, eps, sigma are double and rounded to float once for QCD_F32.
 */
#ifndef QCD_H
#define QCD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qcd_lattice qcd_lattice; /* opaque, host side */

enum { QCD_F32 = 0, QCD_F64 = 1 };
enum { QCD_ALL = 0, QCD_EVEN = 1, QCD_ODD = 2 };
enum { QCD_SUM_SCALAR = 0, QCD_SUM_NORM2 = 1, QCD_SUM_RETR = 2 };
enum { QCD_LAYOUT_REAL = 0, QCD_LAYOUT_PAIRS = 1 }; /* device layout of a field: NC = ncomp reals, or ncomp/2 pairs */
enum { QCD_OK = 0, QCD_EINVAL = 1, QCD_EDIMS = 2, QCD_EALIGN = 3, QCD_EALIAS = 4, QCD_EWORKSPACE = 5,
       QCD_ECUDA = 6 };
/* qcd_get_map `which`: maps are indexed by the lexicographic index and hold lexicographic indices,
 * except CB_OF_LEX (value = checkerboard index) and LEX_OF_CB (indexed by checkerboard index). */
enum { QCD_MAP_CB_OF_LEX = 0, QCD_MAP_LEX_OF_CB = 1, QCD_MAP_NBR_FWD0 = 2, QCD_MAP_NBR_FWD1 = 3,
       QCD_MAP_NBR_FWD2 = 4, QCD_MAP_NBR_FWD3 = 5, QCD_MAP_NBR_BWD0 = 6, QCD_MAP_NBR_BWD1 = 7,
       QCD_MAP_NBR_BWD2 = 8, QCD_MAP_NBR_BWD3 = 9, QCD_MAP_PARITY = 10, QCD_MAP_TSLICE = 11 };

/* ---- lattice object, sizes, errors (host only; no CUDA call is made) ---------------------- */

/* Create the host-side lattice descriptor for extents dims = (Lx,Ly,Lz,Lt).  [O1] */
int qcd_lattice_create(const int dims[4], qcd_lattice **out);
int qcd_lattice_destroy(qcd_lattice *lat);
/* Number of sites V (0 if lat is NULL). */
int64_t qcd_lattice_volume(const qcd_lattice *lat);
/* Bytes of a device field with `ncomp_reals_per_site` reals per site (72 for U, P, F). */
size_t qcd_field_bytes(const qcd_lattice *lat, int prec, int ncomp_reals_per_site);
/* Bytes of the reduction workspace required by qcd_plaquette / qcd_sum / qcd_sum_multi /
 * qcd_force_mom_update (when sums are requested). Depends only on the lattice. */
size_t qcd_workspace_bytes(const qcd_lattice *lat);
/* Device bytes needed by qcd_md_host (staging + fields). */
size_t qcd_md_host_work_bytes(const qcd_lattice *lat, int prec);
const char *qcd_last_error(void);
/* Library version string, e.g. "qcdmd 0.1 sm_100a". */
const char *qcd_version(void);

/* ---- the hot path ----------------------------------------------------------- */

/* Wilson gauge force [O7]: for every site of `subset` and every mu
 *   A = sum_{nu!=mu} [ U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag + U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu) ]
 *   W = U_mu(x) A ;  F_mu(x) = (i beta/12) [ (W - W^dag) - (1/3) tr(W - W^dag) ]      ("force term
 *   calculation", "projection of fields").  F Hermitian traceless; with dU/dt = iPU, dP/dt = F
 *   conserves H = sum tr P^2 + beta sum_{x,mu<nu} (1 - (1/3) Re tr P_mu_nu(x)).
 * U: matrix field, read at all sites.  F: matrix field, written on the subset.  U and F must not
 * overlap (QCD_EALIAS). */
int qcd_gauge_force(const qcd_lattice *lat, int prec, int subset, double beta, const void *U, void *F,
                    void *stream);

/* Momentum update [O10]: P <- P + eps*F on the subset ("momentum updates"). F and P must not overlap. */
int qcd_mom_update(const qcd_lattice *lat, int prec, int subset, double eps, const void *F, void *P,
                   void *stream);

/* Fused force + momentum update (the loop fusion of PAPER.md:32): P <- P + eps*F(U) on the subset,
 * F never stored.  U and P must not overlap. */
int qcd_force_mom_update(const qcd_lattice *lat, int prec, int subset, double beta, double eps,
                         const void *U, void *P, void *stream);

/* Link update [O8,O10]: U_mu(x) <- exp(i eps P_mu(x)) U_mu(x) on the subset ("exponentiating of
 * SU(3) matrices"); exp is exact to rounding for Hermitian traceless P of any norm.  If reunit != 0
 * the result is reunitarised in registers as by qcd_reunit before it is stored.  P and U must not
 * overlap. */
int qcd_link_update(const qcd_lattice *lat, int prec, int subset, double eps, const void *P, void *U,
                    int reunit, void *stream);

/* Reunitarisation [O9] on the subset, in place ("reunitarization of SU(3) matrices"): rows r0,r1,r2:
 * r0 <- r0/|r0| ; r1 <- r1 - (r0^dag.r1) r0, r1 <- r1/|r1| ; r2 <- conj(r0 x r1). */
int qcd_reunit(const qcd_lattice *lat, int prec, int subset, void *U, void *stream);

/* Gaussian momentum refresh [O3,O4] on the subset ("a random number generator"): for each link the
 * eight coefficients p_a ~ N(0,1) of P = sum_a p_a T_a (T_a = Gell-Mann/2) come from the counter-based
 * generator Philox4x32-10 with key = seed and counter (lexicographic site, mu*16+j, stream_id,
 * purpose=1), j = 0..3, two Box-Muller outputs per block.  The result does not depend on the subset,
 * the layout or the launch shape. */
int qcd_mom_refresh(const qcd_lattice *lat, int prec, int subset, uint64_t seed, uint32_t stream_id,
                    void *P, void *stream);

/* Plaquette [O6] ("sum", "sumMulti"): out_avg[0] = (1/6V) sum_x sum_{mu<nu} (1/3) Re tr P_mu_nu(x),
 * P_mu_nu(x) = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag, and, if out_per_t != NULL, the same
 * average over each timeslice (a plaquette belongs to the timeslice of its base site x), Lt doubles.
 * Deterministic: fixed two-pass reduction order, bit-identical from run to run.
 * out_avg, out_per_t: device doubles.  workspace: qcd_workspace_bytes(lat) device bytes. */
int qcd_plaquette(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                  void *workspace, void *stream);

/* qcd_plaquette without a workspace argument, for callers that cannot obtain device memory.  Two kinds of caller
 * are meant: code running inside an application whose memory manager has taken the whole device for its own pool
 * (the framework's allocator serves every package and a measurement routine called from inside
 * holds no handle to it, so a cudaMalloc of its own fails or competes with the pool), and code that measures inside
 * a running trajectory, where cudaMalloc / cudaFree would make every stream of the device wait.  The caller still
 * passes U and the outputs; the first-pass partial sums, which qcd_plaquette keeps in `workspace`, go to an array
 * that is part of the library itself.  Same kernels, same reduction order and same results as qcd_plaquette [O6].
 *   LIMIT    the array holds 32768 doubles (256 KiB of device memory on every GPU the library is loaded on, from
 *            load until the process exits).  A lattice needs 2 Lt ceil(Lx Ly Lz / 2048) of them: all five BASELINE
 *            lattices fit (48^3 x 96 needs 10368), 64^3 x 128 just fits; anything larger returns QCD_EWORKSPACE with
 *            the two numbers in qcd_last_error() and enqueues nothing — use qcd_plaquette there.
 *   SET-UP   the first call on each device (with that device current) asks the CUDA runtime once for the array's
 *            device address and keeps it; make that first call outside any stream capture.  Later calls only launch.
 *   ALLOCATION  none: neither this call nor anything below it calls cudaMalloc, cudaFree or an allocating library
 *            routine.
 *   SHARING  all calls on one device use the same array, and it keeps whatever the last call left there.  Nothing
 *            has to be cleared — the first pass rewrites every slot the second pass reads — but two calls whose
 *            kernels can run at the same time on one GPU (different streams without an ordering between them,
 *            different host threads) overwrite each other's partial sums and return garbage: order them, e.g. by
 *            using one stream.  Calls on different GPUs do not interfere.
 * Other errors as qcd_plaquette (QCD_EINVAL for a NULL lattice, U or out_avg; QCD_EALIGN); QCD_ECUDA if the address
 * query or a launch fails, QCD_EINVAL on a device ordinal >= 64. */
int qcd_plaquette_noalloc(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                          void *stream);

/* Global / subset sum [O12] ("sum") of a per-site quantity of `field`:
 *   QCD_SUM_SCALAR  real field (QCD_LAYOUT_REAL) with ncomp components: out[c] = sum_x field_c(x), c < ncomp <= 64
 *   QCD_SUM_NORM2   pair-layout field (QCD_LAYOUT_PAIRS) with ncomp reals per site: out[0] = sum_x sum_i field_i(x)^2
 *                   (ncomp = 72 on P gives the kinetic energy sum tr P^2)
 *   QCD_SUM_RETR    matrix field of ncomp/18 matrices per site: out[0] = sum_x sum_m Re tr M_m(x)
 * Deterministic two-pass reduction in double.  out: device doubles. */
int qcd_sum(const qcd_lattice *lat, int prec, int subset, int kind, int ncomp, const void *field,
            double *out, void *workspace, void *stream);

/* Per-subset sums [O12] ("sumMulti"): out[k] (SCALAR: out[k*ncomp + c]) = sum over the sites with
 * subset_id == k.  subset_id: device int32[V] indexed by CHECKERBOARD index with values in [0,nsub)
 * (other values: site belongs to no subset), or NULL for the timeslice set (nsub must equal Lt).
 * nsub <= 4096.  Deterministic. */
int qcd_sum_multi(const qcd_lattice *lat, int prec, int kind, int ncomp, const void *field,
                  const int32_t *subset_id, int nsub, double *out, void *workspace, void *stream);

/* One fused MD step, the unit the headline metric counts: P <- P + eps_p*F(U), then
 * U <- reunit(exp(i eps_u P) U), two kernels on `stream`. [O11 building block] */
int qcd_md_step(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u, void *U,
                void *P, void *stream);

/* qcd_force_mom_update on the whole lattice with the two sums of the Hamiltonian as by-products (reductions
 * of PAPER.md:26 fused into the site loop): out[0] = plaquette average of U (as qcd_plaquette's
 * out_avg: sum_{x,mu} Re tr W_mu(x) = 4 sum_{x,mu<nu} Re tr P_mu_nu(x)), out[1] = K = sum |P_ij|^2 of the
 * UPDATED momenta (as qcd_sum NORM2).  Saves the two extra passes (1152 B/site) per observed step.  Device
 * doubles; workspace as qcd_workspace_bytes.  Deterministic run to run at a fixed block shape (one partial
 * per block, fixed order); per timeslice: see qcd_trajectory.  QCD_EWORKSPACE if the lattice's workspace cannot
 * hold two doubles per block. */
int qcd_force_mom_update_sums(const qcd_lattice *lat, int prec, double beta, double eps, const void *U, void *P,
                              double *out, void *workspace, void *stream);
/* qcd_leapfrog whose last momentum update is qcd_force_mom_update_sums: out[0] = plaquette average and
 * out[1] = K at the END of the trajectory, i.e. H_end = out[1] + beta*6V*(1 - out[0]) at no extra pass. */
int qcd_leapfrog_energy(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U, void *P,
                        double *out, void *workspace, void *stream);

/* The same MD step in ONE pass over the lattice (SURVEY.md 8(a) "single pass, ping-pong U"; loop fusion
 * in the sense of PAPER.md:32): P <- P + eps_p*F(U_in); U_out <- reunit(exp(i eps_u P) U_in), one kernel.
 * U_in is only read; U_out is a second gauge field of the same size that must not overlap U_in or P
 * (QCD_EALIAS) because neighbouring sites still read the old links.  Results equal qcd_md_step's up to
 * rounding order (same arithmetic per link). */
int qcd_md_step_single_pass(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u,
                            const void *U_in, void *P, void *U_out, void *stream);

/* Leapfrog trajectory [O11] built from single-pass steps: same result as qcd_leapfrog; U_work is a
 * caller-owned scratch gauge field (qcd_field_bytes(lat, prec, 72) bytes) used as the ping-pong partner.
 * The final links are always left in U (an odd nsteps starts with one two-kernel in-place step). */
int qcd_leapfrog_single_pass(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U,
                             void *P, void *U_work, void *stream);

/* Leapfrog trajectory [O11] that also returns the observables of every step (BASELINE.json configs 4, 5: "per-step
 * reunitarization and reductions ... sumMulti of plaquette per timeslice ... kinetic-energy sum"; PAPER.md:26 sum /
 * sumMulti, fused into the site loop as in PAPER.md:32).  Built from single-pass steps like
 * qcd_leapfrog_single_pass; the plaquette sums and the kinetic energy are by-products of the force kernel, so a step
 * costs no extra pass over the fields.  Same U, P as qcd_leapfrog up to rounding order.
 *   obs    device double[2*(nsteps+1)]:  obs[2k] = plaquette average of U_k (U after k link updates), k = 0..nsteps;
 *          obs[1] = K of the initial momenta, obs[2k+1] (0 < k < nsteps) = K of the momenta after the full kick that
 *          follows link update k (time (k+1/2) eps), obs[2 nsteps + 1] = K of the final momenta.  Hence
 *          H_start = obs[1] + beta 6V (1 - obs[0]),  H_end = obs[2n+1] + beta 6V (1 - obs[2n]),  dH = H_end - H_start.
 *   per_t  device double[(nsteps+1)*Lt] or NULL: plaquette average of every timeslice of U_k (R13), row k.
 *   U_work scratch gauge field, qcd_field_bytes(lat, prec, 72) bytes; the final links are always left in U.
 *   workspace, workspace_bytes: at least qcd_workspace_bytes(lat), else QCD_EWORKSPACE (also returned when a tuned
 *          tile has more blocks than the workspace has room for).  All checks are made before anything is enqueued.
 * Deterministic run to run at a fixed launch configuration (one partial per block and timeslice of its tile, summed in
 * a fixed order). */
int qcd_trajectory(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U, void *P,
                   void *U_work, double *obs, double *per_t, void *workspace, size_t workspace_bytes, void *stream);

/* ---- anisotropic Wilson action and multi-timescale integrator ------------------
 * The paper's demonstration ran an anisotropic Wilson gauge action with multi-timescale
 * integrators and gives no formulas; readings R19/R20 of DESIGN.md:
 *   S = beta_s sum_x sum_{i<j<3} (1 - (1/3) Re tr P_ij(x)) + beta_t sum_x sum_{i<3} (1 - (1/3) Re tr P_i3(x)),
 *   F_mu(x) = (i/12)[(W - W^dag) - (1/3) tr(W - W^dag)],  W = U_mu(x) sum_{nu != mu} beta_{mu nu} staples_nu,
 *   beta_{mu nu} = beta_t if mu or nu is the time direction (3), else beta_s.
 * beta_s = beta_t = beta reproduces qcd_gauge_force.  Planes with coefficient 0 cost nothing. */
int qcd_gauge_force_aniso(const qcd_lattice *lat, int prec, int subset, double beta_s, double beta_t,
                          const void *U, void *F, void *stream);
/* fused P += eps * F_aniso(U) on the subset's sites */
int qcd_force_mom_update_aniso(const qcd_lattice *lat, int prec, int subset, double beta_s, double beta_t,
                               double eps, const void *U, void *P, void *stream);
/* out_avg[0] / out_avg[1] = mean of (1/3) Re tr P over the space-space / space-time planes (device doubles);
 * out_per_t: device double[Lt][2] or NULL, a plaquette counted in the timeslice of its base site.
 * S_aniso = 3 V [beta_s (1 - out_avg[0]) + beta_t (1 - out_avg[1])].  Deterministic like qcd_plaquette. */
int qcd_plaquette_st(const qcd_lattice *lat, int prec, const void *U, double *out_avg, double *out_per_t,
                     void *workspace, void *stream);
/* Two-level leapfrog (Sexton-Weingarten nesting, R20) over trajectory length tau.  The action is
 * S_1 + S_0 with coefficients (beta_s[k], beta_t[k]); level 1 takes n_outer steps of eps_1 = tau/n_outer,
 * level 0 n_inner leapfrog steps of eps_1/n_inner inside each.  Momentum updates that act on the same links
 * (adjacent half steps, both levels) are merged into ONE force kernel with summed plane weights, so the
 * trajectory is 1 + n_outer*n_inner force launches and n_outer*n_inner link updates (exp + reunit). */
int qcd_nested_leapfrog(const qcd_lattice *lat, int prec, const double beta_s[2], const double beta_t[2],
                        double tau, int n_outer, int n_inner, void *U, void *P, void *stream);

/* ---- pseudofermion-side site operations ("a pseudofermion refresh") ----
 * Only the site-parallel pieces outside the Dirac operator (which, with the solver, is out of scope:
 * PAPER.md:83): Gaussian fill of a spin-colour vector field and its norm / inner-product reductions
 * (PAPER.md:26).  A spin-colour vector has 12 complex components per site, k = 3*spin + colour; device
 * layout: complex pairs, NC = 12 units per site, component k of site cb at unit index ((cb>>5)*12 + k)*32 + (cb&31) (24 reals per site;
 * qcd_pack / qcd_unpack with QCD_LAYOUT_PAIRS; canonical layout [s][k][re,im]).  [O15] eta_k(x) = (g0 + i g1)/sqrt(2), (g0,g1) the Box-Muller pair of generator
 * block (lexicographic site, 64 + k, stream_id, purpose 4): <|eta_k|^2> = 1, weight exp(-eta^dag eta).
 * Writes only the subset's sites.  The norm is qcd_sum(QCD_SUM_NORM2, ncomp = 24). */
int qcd_spinor_gaussian(const qcd_lattice *lat, int prec, int subset, uint64_t seed, uint32_t stream_id,
                        void *eta, void *stream);
/* [O16] out[0], out[1] (device doubles) = Re, Im of <a,b> = sum over the subset's sites and the nc complex
 * components per site of conj(a) b; a, b: pair-layout fields with nc components (12 for spin-colour
 * vectors, 36 for the matrix fields).  fp64 accumulation, deterministic two-pass reduction like qcd_sum. */
int qcd_inner_product(const qcd_lattice *lat, int prec, int subset, int nc, const void *a, const void *b,
                      double *out, void *workspace, void *stream);
/* the same per timeslice ("sumMulti"): out is device double[Lt][2] */
int qcd_inner_product_multi(const qcd_lattice *lat, int prec, int nc, const void *a, const void *b, double *out,
                            void *workspace, void *stream);

/* ---- launch-parameter database of the auto-tuner (section 4) -------
 * The paper times every kernel as a function of the threads per block N_t and stores the best value in a
 * database.  Here the measuring lives in paper_1212_0785_b200/autotune.py (it calls the public kernels);
 * these calls are the database the launchers consult.  Key: (lattice extents, prec, subset ALL or
 * EVEN/ODD, kernel).  Value: for QCD_KERNEL_FORCE a kernel variant and a 4-D block tile (tile[0] = 0 or
 * tile = NULL: the library's own choice; extents must divide the lattice, tile[0] even, at most 128 sites of
 * the subset per block); for QCD_KERNEL_LINK_UPDATE / QCD_KERNEL_MOM_UPDATE the threads per block (multiple
 * of 32, 32..256).  The database is the only knob: no environment variable is read.  Both force variants
 * compute the definition [O7] for arbitrary 3x3 matrices; results never depend on these settings beyond
 * rounding order; reductions are not tunable (fixed geometry, determinism).
 * Host-only, thread-safe, process-global.  qcd_tune_get returns QCD_EINVAL when no entry exists.
 *   QCD_FORCE_STAPLE  the definition as written: per direction 6 staples of 2 products, then U_mu(x) A
 *                     (52 products, 76 link loads per site)
 *   QCD_FORCE_PLANE   (default) every plane visited once, its closed plaquette shared by the two directions
 *                     (46 products, 64 link loads per site) */
enum { QCD_KERNEL_FORCE = 0, QCD_KERNEL_LINK_UPDATE = 1, QCD_KERNEL_MOM_UPDATE = 2 };
enum { QCD_FORCE_STAPLE = 0, QCD_FORCE_PLANE = 1 };
int qcd_tune_set(const qcd_lattice *lat, int prec, int subset, int kernel, int variant, const int tile[4],
                 int threads);
int qcd_tune_get(const qcd_lattice *lat, int prec, int subset, int kernel, int *variant, int tile[4],
                 int *threads);
int qcd_tune_clear(void);

/* Leapfrog trajectory [O11]: P += (eps/2) F; n times { U <- reunit(exp(i eps P) U); P += eps F }
 * with eps/2 on the last. */
int qcd_leapfrog(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U,
                 void *P, void *stream);

/* ---- helpers (not on the hot path) -------------------------------------------------------- */

/* canonical lexicographic AoS (device, exactly V*ncomp reals) -> device layout (qcd_field_bytes bytes), and back.
 * ncomp reals per site; `layout` says which device layout the field has: QCD_LAYOUT_PAIRS (NC = ncomp/2 (re,im)
 * units per site, ncomp even: matrix fields with ncomp = 72, spin-colour vectors with ncomp = 24, what
 * QCD_SUM_NORM2 / QCD_SUM_RETR / qcd_inner_product read) or QCD_LAYOUT_REAL (NC = ncomp reals per site, what
 * QCD_SUM_SCALAR reads).  Input and output must not overlap.  QCD_EDIMS if NC (V + 32) >= 2^32. */
int qcd_pack(const qcd_lattice *lat, int prec, int ncomp, int layout, const void *lex_aos, void *dev_soa,
             void *stream);
int qcd_unpack(const qcd_lattice *lat, int prec, int ncomp, int layout, const void *dev_soa, void *lex_aos,
               void *stream);
/* index / subset maps [O1] into dev_out (int32[V]) */
int qcd_get_map(const qcd_lattice *lat, int which, int32_t *dev_out, void *stream);
/* hot start [O5]: U_mu(x) = exp(i sigma Q), Q = sum q_a T_a, q_a ~ N(0,1) from purpose 0 */
int qcd_hot_start(const qcd_lattice *lat, int prec, uint64_t seed, double sigma, void *U, void *stream);
/* U += sigma*N, 18 iid N(0,1) reals per link from purpose 2, blocks 0..8 (config 3 reunit input) */
int qcd_perturb(const qcd_lattice *lat, int prec, uint64_t seed, double sigma, void *U, void *stream);
/* raw generator output for bit-exact tests: for i < n, block counter (site[i], mu_j[i], stream_id,
 * purpose) -> words[4*i..4*i+3] (uint32), uniforms[2*i..] (double), gauss[2*i..] (double).
 * site, mu_j: device uint32[n]; any output pointer may be NULL. */
int qcd_rng_blocks(uint64_t seed, uint32_t stream_id, uint32_t purpose, int n, const uint32_t *site,
                   const uint32_t *mu_j, uint32_t *words, double *uniforms, double *gauss, void *stream);

/* ---- domain decomposition in t with a one-site halo ("multi-GPU (parallel
 * architecture) support"; PAPER.md:121 overlapping communication and computation "is work in progress").
 * A SLAB lattice holds t_count consecutive global timeslices starting at t_begin plus one halo timeslice on either
 * side: local extents (Lx, Ly, Lz, t_count + 2); local timeslice te is the global timeslice (t_begin + te - 1) mod Lt,
 * te = 0 and te = t_count + 1 are the halos.  Fields on a slab lattice have the usual device layout for the local
 * extents.  Semantics of every call on a slab lattice:
 *   - the stencil calls (qcd_gauge_force*, qcd_force_mom_update*, qcd_md_step*, qcd_leapfrog*) update the INTERIOR
 *     timeslices only and read the halos, which the caller refreshes with qcd_copy_timeslices after every link
 *     update (or which qcd_link_update_push, the link update fused with that transport, has already written) (one exchange per force evaluation: from the lower neighbour's last interior timeslice into te = 0,
 *     all four links; from the upper neighbour's first interior timeslice into te = t_count + 1, mu_mask 0x7);
 *   - the site-local calls act on all stored timeslices (halo values are recomputed or overwritten by the next
 *     exchange); EVEN / ODD always mean the GLOBAL parity;
 *   - the generator is keyed on the GLOBAL lexicographic site: qcd_mom_refresh, qcd_hot_start, qcd_perturb and
 *     qcd_spinor_gaussian give, timeslice by timeslice, exactly the field of the undecomposed lattice (halos
 *     included, so no exchange is needed after them);
 *   - qcd_force_mom_update_sums averages the plaquette over the interior sites and sums K over them; the
 *     reductions with per-timeslice outputs (qcd_plaquette out_per_t, qcd_sum_multi, qcd_inner_product_multi)
 *     return t_count + 2 values of which the interior ones are the global lattice's; ranks are combined in fixed
 *     rank order by the caller (paper_1212_0785_b200/slabs.py).  The by-product per-timeslice sums need the whole
 *     lattice;
 *   - the calls that make several link updates in a row (qcd_leapfrog, qcd_leapfrog_energy, qcd_leapfrog_single_pass,
 *     qcd_trajectory, qcd_nested_leapfrog, qcd_md_host) return QCD_EINVAL on a slab lattice or a t-view: the halos
 *     cannot be refreshed inside the call.  Build the trajectory from the single-step calls and the transport
 *     (paper_1212_0785_b200/slabs.py does).
 * qcd_copy_timeslices is the transport: it copies nt timeslices of a pair-layout field (ncomp reals per site, 72 for
 * matrix fields; mu_mask selects the links of a matrix field, bit mu) between two lattices with the same spatial
 * extents; dst may be a peer GPU's memory (direct stores over NVLink).  QCD_EDIMS if the spatial extents differ. */
int qcd_lattice_create_slab(const int global_dims[4], int t_begin, int t_count, qcd_lattice **out);
/* A second descriptor of the same stored lattice (same extents, layout, generator offsets) whose stencil calls
 * update the timeslices [t0, t1) only: the boundary / interior split that lets the force of the inner timeslices
 * run while the halos travel.  Destroy it with qcd_lattice_destroy. */
int qcd_lattice_view_t(const qcd_lattice *lat, int t0, int t1, qcd_lattice **out);
/* local (stored) extents and the interior timeslice range [interior_t[0], interior_t[1]) (NULL: not wanted) */
int qcd_lattice_dims(const qcd_lattice *lat, int dims[4], int interior_t[2]);
int qcd_copy_timeslices(const qcd_lattice *src_lat, const void *src, int src_t, const qcd_lattice *dst_lat, void *dst,
                        int dst_t, int nt, int prec, int ncomp, unsigned mu_mask, void *stream);
/* The single-pass MD step fused with the halo transport: as qcd_md_step_single_pass on the interior timeslices of the
 * slab lattice (or view) `lat` — P <- P + eps_p F(U_in), U_out <- reunit(exp(i eps_u P) U_in) — and the new links of
 * the slab's first interior timeslice are ALSO stored into the upper halo of the lower neighbour's OUTPUT field
 * lo_U_out (links mu = 0..2), those of its last interior timeslice into the lower halo of hi_U_out (all four), by the
 * thread that computed them (peer-GPU pointers allowed; a neighbour may be NULL or this slab itself).  After all slabs
 * have made the call the output fields are complete, halos included, and become the next step's input: no separate
 * exchange.  Same checks as qcd_md_step_single_pass and qcd_link_update_push. */
int qcd_md_step_single_pass_push(const qcd_lattice *lat, int prec, double beta, double eps_p, double eps_u,
                                 const void *U_in, void *P, void *U_out, const qcd_lattice *lo_lat, void *lo_U_out,
                                 const qcd_lattice *hi_lat, void *hi_U_out, void *stream);
/* Link update fused with the halo transport (SURVEY.md 8(e) "peer stores"): on the interior timeslices
 * [t0, t1) of the slab lattice (or view) `lat`, U <- exp(i eps P) U, reunitarised if reunit != 0 [O8, O9], all four
 * links of every site; the new links of the slab's first interior timeslice (te = 1) are ALSO stored into the upper
 * halo of the lower neighbour's gauge field lo_U (links mu = 0..2) and those of its last interior timeslice into the
 * lower halo of hi_U (all four links) by the thread that computed them — one kernel instead of the link update
 * followed by two qcd_copy_timeslices.  lo_lat / hi_lat: the neighbours' slab lattices (same spatial extents,
 * QCD_EDIMS otherwise; t extents may differ); lo_U / hi_U device pointers that may be peer-GPU memory; a neighbour may
 * be NULL (lattice and field together) and may be this slab itself (one slab: its halos mirror its own boundary).
 * The slab's own halo timeslices are not written: the neighbours' calls write them, so the caller orders the calls
 * of different slabs before the next force evaluation (stream or event dependencies), nothing else. */
int qcd_link_update_push(const qcd_lattice *lat, int prec, double eps, const void *P, void *U, int reunit,
                         const qcd_lattice *lo_lat, void *lo_U, const qcd_lattice *hi_lat, void *hi_U, void *stream);

/* ---- measured denominators ("Measure DFMA/FFMA peaks with a probe") --------------------
 * One kernel launch per probe, enqueued on `stream` like every other call and timed by the caller with CUDA
 * events (bench.py --peaks): rate = qcd_probe_work(...) / elapsed.
 *   QCD_PROBE_FMA  chains of 3x3 complex products in registers (the product routine of the force kernel), no
 *                  memory traffic: work = real FMAs.  prec selects double / float.
 *   QCD_PROBE_L1   every block re-reads its own 32 kB with 128-bit loads: work = bytes (L1-resident loads)
 *   QCD_PROBE_LDS  the same from 64 kB of shared memory: work = bytes
 *   QCD_PROBE_L2   all blocks stream one 48 MB buffer: work = bytes (L2-resident as the SMs see it)
 * scratch: device memory, qcd_probe_scratch_bytes(what) bytes, zero-filled by the caller; QCD_EWORKSPACE if
 * smaller.  qcd_probe_work and qcd_probe_scratch_bytes are host-only. */
enum { QCD_PROBE_FMA = 0, QCD_PROBE_L1 = 1, QCD_PROBE_LDS = 2, QCD_PROBE_L2 = 3 };
size_t qcd_probe_scratch_bytes(int what);
double qcd_probe_work(int what, int prec, int reps);
int qcd_probe_launch(int what, int prec, int reps, void *scratch, size_t scratch_bytes, void *stream);

/* End-to-end call on HOST buffers (used for the e2e measurement): U_host and P_host are host arrays
 * in the canonical layout (pinned memory makes the copies asynchronous).  `nsteps` MD steps (eps_p = eps_u = eps)
 * between a host->device and a device->host transfer of both fields, results back in U_host and P_host.  As in
 * PAPER.md:75-79 (section 5.1, transfers overlapped with kernels on CUDA streams) the work runs as a pipeline over
 * slabs of timeslices on three internal streams — H2D copies; pack, single-pass step per slab, unpack; D2H copies —
 * so that for one step both PCIe directions are busy at once.  `stream` is joined at entry and at exit with events
 * (the work is ordered after what `stream` held and before what is enqueued on it next); the host is never
 * synchronised.  Lattices with fewer than 8 slabs run on `stream` alone.
 * device_work: qcd_md_host_work_bytes(lat, prec) device bytes.
 * State the library keeps for this call (the one exception to "owns nothing" above): per host thread and device,
 * the three internal streams and a pool of events, created by the thread's first pipelined call with that device
 * current, reused afterwards and destroyed when the thread exits.  Two threads must not run the call on the same
 * device_work at the same time. */
int qcd_md_host(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U_host,
                void *P_host, void *device_work, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* QCD_H */
