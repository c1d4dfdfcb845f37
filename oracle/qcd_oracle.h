/* qcd_oracle.h — CPU ORACLE. TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct fp64 definitions of the site-parallel SU(3) operations of
 * the HMC molecular-dynamics step that the paper lists (section 1: "momentum
 * updates, force term calculation, projection of fields, reunitarization of SU(3) matrices,
 * a random number generator, exponentiating of SU(3) matrices") and of its reductions
 * ("sum, sumMulti").  The paper names these operations and defines none of
 * them; the definitions are the textbook ones fixed in SURVEY.md section 8(c) O1..O12 and
 * restated in DESIGN.md ("Readings").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this library.  It shares no code with paper_1212_0785_b200/csrc (the CUDA path).
 *
 * Canonical field layout (all functions): lexicographic array-of-structures
 *     matrix field   double[V][4][3][3][2]   = [site s][direction mu][row][col][re,im]
 *     real field     double[V][ncomp]
 * with s = x + Lx*(y + Ly*(z + Lz*t)), L = (Lx,Ly,Lz,Lt), directions mu=0..3 <-> x,y,z,t.
 * subset: 0 = all sites, 1 = even ((x+y+z+t)%2==0), 2 = odd.
 *
 * Every function returns 0 on success, nonzero on a bad argument.  Parity: all functions are
 * pinned by tests/test_oracle_*.py (see the pin table in DESIGN.md); none is "parity unpinned".
 */
#ifndef QCD_ORACLE_H
#define QCD_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* O1 maps. which: 0 CB_OF_LEX, 1 LEX_OF_CB, 2..5 NBR_FWD mu=0..3, 6..9 NBR_BWD mu=0..3,
 * 10 PARITY, 11 TSLICE.  All maps are indexed by the lexicographic index and hold
 * lexicographic indices, except CB_OF_LEX (value = checkerboard index) and LEX_OF_CB
 * (indexed by checkerboard index). out has V entries. */
int orc_map(const int L[4], int which, int32_t *out);

/* O3 RNG */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* one RNG block: words, the two uniforms and the Box-Muller pair of counter
 * (s, mu*16+j, stream_id, purpose) under key = seed */
void orc_rng_block(uint64_t seed, uint32_t s, uint32_t mu, uint32_t j, uint32_t stream_id,
                   uint32_t purpose, uint32_t words[4], double u[2], double g[2]);

/* O2: Q = sum_a q_a T_a (Hermitian traceless), Q is double[3][3][2] */
void orc_herm_from_coeffs(const double q[8], double *Q);
/* O8: E = exp(i Q) for any 3x3 complex Q (used with Hermitian traceless Q) */
void orc_expi(const double *Q, double *E);
/* O9: row Gram-Schmidt reunitarisation of one matrix, in place */
void orc_reunit_mat(double *M);

/* O4 / O5 field generators */
int orc_mom_refresh(const int L[4], int subset, uint64_t seed, uint32_t stream_id, double *P);
int orc_hot_start(const int L[4], uint64_t seed, double sigma, double *U);
int orc_perturb(const int L[4], uint64_t seed, double sigma, double *U);
/* pin helper: G(x) = exp(i sigma Q(x)) from purpose 3; U'_mu(x) = G(x) U_mu(x) G(x+mu)^dagger.
 * G (double[V][3][3][2]) is an output; pass NULL for Uout to only generate G. */
int orc_gauge_transform(const int L[4], uint64_t seed, double sigma, const double *U,
                        double *G, double *Uout);

/* O6 */
int orc_plaquette(const int L[4], const double *U, double *avg, double *per_t /*[Lt] or NULL*/);
int orc_action(const int L[4], double beta, const double *U, double *S);
/* O7 */
int orc_gauge_force(const int L[4], int subset, double beta, const double *U, double *F);
/* O7 at the listed lexicographic sites only; F is double[nsites][4][3][3][2] */
int orc_gauge_force_sites(const int L[4], double beta, const double *U, int nsites, const int32_t *sites,
                          double *F);
/* pin helper: sum over x,mu of Re tr W_mu(x), W = U_mu(x) A_mu(x) (staple sum rule) */
int orc_sum_retr_w(const int L[4], const double *U, double *out);
/* O10 */
int orc_mom_update(const int L[4], int subset, double eps, const double *F, double *P);
int orc_link_update(const int L[4], int subset, double eps, const double *P, double *U, int reunit);
int orc_reunit(const int L[4], int subset, double *U);
/* O12. kind: 0 SCALAR (field double[V][ncomp], out[ncomp]); 1 NORM2 (matrix field with
 * ncomp reals per site, out[1] = sum of squares); 2 RETR (matrix field double[V][nmat][3][3][2],
 * ncomp = 18*nmat, out[1] = sum of Re tr) */
int orc_sum(const int L[4], int subset, int kind, int ncomp, const double *field, double *out);
/* per-subset sums; subset_id[V] by lexicographic index, or NULL = timeslice (nsub must be Lt).
 * out is [nsub][ncomp] for SCALAR, [nsub] otherwise */
int orc_sum_multi(const int L[4], int kind, int ncomp, const double *field,
                  const int32_t *subset_id, int nsub, double *out);
/* O6: H = K + S with K = sum |P_ij|^2 */
int orc_hamiltonian(const int L[4], double beta, const double *U, const double *P,
                    double *K, double *S);
/* O11 leapfrog, n steps of size eps, in place */
int orc_leapfrog(const int L[4], double beta, double eps, int nsteps, double *U, double *P);
/* one fused MD step as the product path runs it: P += eps_p F(U); U <- reunit(exp(i eps_u P) U) */
int orc_md_step(const int L[4], double beta, double eps_p, double eps_u, double *U, double *P);

/* O13 anisotropic Wilson action (R19): beta_s on the three space-space planes, beta_t on the
 * three space-time planes.  avg[0]/avg[1] = mean (1/3) Re tr P over space-space / space-time planes;
 * per_t is [Lt][2] or NULL. */
int orc_plaquette_st(const int L[4], const double *U, double avg[2], double *per_t);
int orc_action_aniso(const int L[4], double beta_s, double beta_t, const double *U, double *S);
int orc_gauge_force_aniso(const int L[4], int subset, double beta_s, double beta_t, const double *U, double *F);
/* O14 two-level leapfrog (R20): level 1 (outer, n_outer steps over tau) integrates the action with
 * coefficients (bs[1], bt[1]), level 0 (n_inner steps per outer step) the one with (bs[0], bt[0]) */
int orc_nested_leapfrog(const int L[4], const double bs[2], const double bt[2], double tau, int n_outer,
                        int n_inner, double *U, double *P);

/* O15 / O16 pseudofermion-side site operations (R21): spin-colour vector fields double[V][12][2].
 * eta_k(x) = (g0 + i g1)/sqrt(2) from generator block (s, 64 + k, stream_id, purpose 4). */
int orc_spinor_gaussian(const int L[4], int subset, uint64_t seed, uint32_t stream_id, double *eta);
/* <a, b> = sum conj(a) b over the subset and nc complex components per site; out = (Re, Im) */
int orc_inner_product(const int L[4], int subset, int nc, const double *a, const double *b, double out[2]);
int orc_inner_product_multi(const int L[4], int nc, const double *a, const double *b, double *out /*[Lt][2]*/);

int orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
