/* qcd_oracle.c — CPU ORACLE. TEST INFRASTRUCTURE, NOT THE PRODUCT (see qcd_oracle.h).
 *
 * Each function is the plain definition of the operation, written out in the order and
 * notation of SURVEY.md section 8(c) (O1..O12), which fixes the conventions the paper leaves open
 * (PAPER.md:17 names the operations; PAPER.md:26 names the reductions; PAPER.md:41,51 fix
 * "one lattice site per thread", i.e. every operation is site-parallel).
 * No blocking, fusion or reordering: one loop over sites, one small dense 3x3 routine per
 * algebraic step.  fp64 throughout; reductions accumulate in long double in lexicographic
 * site order.
 *
 * Compiled twice from this one source: serial (the definition) and with -fopenmp (site loops
 * only; reductions stay serial and ordered) for the large-lattice parity runs.
 */
#include "qcd_oracle.h"

#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

static const double PI = 3.14159265358979323846264338327950288;

/* ------------------------------------------------------------------ O1 lattice and maps */

typedef struct {
    int L[4];
    long V;
} lat_t;

static int lat_init(lat_t *lat, const int L[4]) {
    long V = 1;
    for (int d = 0; d < 4; d++) {
        if (L[d] < 2 || (L[d] & 1)) return 1;
        lat->L[d] = L[d];
        V *= L[d];
    }
    if (V >= 2147483648L) return 1;
    lat->V = V;
    return 0;
}

static void coords_of(const lat_t *lat, long s, int c[4]) {
    c[0] = (int)(s % lat->L[0]); s /= lat->L[0];
    c[1] = (int)(s % lat->L[1]); s /= lat->L[1];
    c[2] = (int)(s % lat->L[2]); s /= lat->L[2];
    c[3] = (int)s;
}

static long lex_of(const lat_t *lat, const int c[4]) {
    return c[0] + (long)lat->L[0] * (c[1] + (long)lat->L[1] * (c[2] + (long)lat->L[2] * c[3]));
}

/* site reached from s by `step` (+1 or -1) in direction mu, periodic */
static long hop(const lat_t *lat, long s, int mu, int step) {
    int c[4];
    coords_of(lat, s, c);
    c[mu] = (c[mu] + step + lat->L[mu]) % lat->L[mu];
    return lex_of(lat, c);
}

static int parity_of(const lat_t *lat, long s) {
    int c[4];
    coords_of(lat, s, c);
    return (c[0] + c[1] + c[2] + c[3]) & 1;
}

static int tslice_of(const lat_t *lat, long s) {
    int c[4];
    coords_of(lat, s, c);
    return c[3];
}

static int in_subset(const lat_t *lat, long s, int subset) {
    if (subset == 0) return 1;
    return parity_of(lat, s) == (subset == 1 ? 0 : 1);
}

int orc_map(const int L[4], int which, int32_t *out) {
    lat_t lat;
    if (lat_init(&lat, L) || !out || which < 0 || which > 11) return 1;
    for (long s = 0; s < lat.V; s++) {
        long cb = (long)parity_of(&lat, s) * (lat.V / 2) + (s >> 1);
        if (which == 0) out[s] = (int32_t)cb;
        else if (which == 1) out[cb] = (int32_t)s;
        else if (which >= 2 && which <= 5) out[s] = (int32_t)hop(&lat, s, which - 2, +1);
        else if (which >= 6 && which <= 9) out[s] = (int32_t)hop(&lat, s, which - 6, -1);
        else if (which == 10) out[s] = parity_of(&lat, s);
        else out[s] = tslice_of(&lat, s);
    }
    return 0;
}

/* ------------------------------------------------------------------ 3x3 complex algebra */

/* a matrix is cplx[9], row-major: m[3*r+c] */
#define LINK(F, s, mu) ((cplx *)((F) + ((size_t)(s) * 4 + (mu)) * 18))
#define CLINK(F, s, mu) ((const cplx *)((F) + ((size_t)(s) * 4 + (mu)) * 18))

static void m_mul(cplx *c, const cplx *a, const cplx *b) { /* c = a b */
    cplx t[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx acc = 0;
            for (int k = 0; k < 3; k++) acc += a[3 * i + k] * b[3 * k + j];
            t[3 * i + j] = acc;
        }
    memcpy(c, t, sizeof t);
}

static void m_dag(cplx *c, const cplx *a) { /* c = a^dagger */
    cplx t[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) t[3 * i + j] = conj(a[3 * j + i]);
    memcpy(c, t, sizeof t);
}

static void m_add(cplx *c, const cplx *a) { /* c += a */
    for (int i = 0; i < 9; i++) c[i] += a[i];
}

static void m_zero(cplx *c) {
    for (int i = 0; i < 9; i++) c[i] = 0;
}

static void m_unit(cplx *c) {
    m_zero(c);
    c[0] = c[4] = c[8] = 1;
}

static cplx m_trace(const cplx *a) { return a[0] + a[4] + a[8]; }

/* ------------------------------------------------------------------ O3 RNG (integer, bit-exact) */

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; round++) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* 52 random bits -> u = (2k+1) 2^-53: an exact double strictly inside (0,1)
 * (reading R-RNG: the survey's 53-bit k + 1/2 is not exact for k >= 2^52). */
static double uniform_of(uint32_t wa, uint32_t wb) {
    uint64_t k = ((uint64_t)(wa >> 6) << 26) | (uint64_t)(wb >> 6);
    return (double)(2 * k + 1) * 0x1p-53;
}

void orc_rng_block(uint64_t seed, uint32_t s, uint32_t mu, uint32_t j, uint32_t stream_id,
                   uint32_t purpose, uint32_t words[4], double u[2], double g[2]) {
    uint32_t ctr[4] = {s, mu * 16u + j, stream_id, purpose};
    uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
    uint32_t w[4];
    orc_philox4x32_10(ctr, key, w);
    double u1 = uniform_of(w[0], w[1]);
    double u2 = uniform_of(w[2], w[3]);
    double r = sqrt(-2.0 * log(u1));
    double phi = 2.0 * PI * u2;
    if (words) memcpy(words, w, sizeof w);
    if (u) { u[0] = u1; u[1] = u2; }
    if (g) { g[0] = r * cos(phi); g[1] = r * sin(phi); }
}

/* eight N(0,1) coefficients of link (s,mu): q_{2j+1}, q_{2j+2} from block j = 0..3 */
static void gauss8(uint64_t seed, long s, int mu, uint32_t stream_id, uint32_t purpose, double q[8]) {
    for (int j = 0; j < 4; j++)
        orc_rng_block(seed, (uint32_t)s, (uint32_t)mu, (uint32_t)j, stream_id, purpose, NULL, NULL,
                      q + 2 * j);
}

/* ------------------------------------------------------------------ O2 generators */

/* Q = sum_a q_a T_a, T_a = lambda_a / 2 (Gell-Mann, standard order) */
static void herm_from_coeffs(const double q[8], cplx *Q) {
    const double s3 = sqrt(3.0);
    Q[0] = q[2] / 2 + q[7] / (2 * s3);
    Q[4] = -q[2] / 2 + q[7] / (2 * s3);
    Q[8] = -q[7] / s3;
    Q[1] = (q[0] - I * q[1]) / 2;
    Q[2] = (q[3] - I * q[4]) / 2;
    Q[5] = (q[5] - I * q[6]) / 2;
    Q[3] = conj(Q[1]);
    Q[6] = conj(Q[2]);
    Q[7] = conj(Q[5]);
}

void orc_herm_from_coeffs(const double q[8], double *Q) { herm_from_coeffs(q, (cplx *)Q); }

/* ------------------------------------------------------------------ O8 exp(iQ) */

/* scale by 2^-n so that ||Q||_F < 1/4, order-18 Taylor by Horner, square n times */
static void expi(const cplx *Q, cplx *E) {
    double nrm2 = 0;
    for (int i = 0; i < 9; i++) nrm2 += creal(Q[i]) * creal(Q[i]) + cimag(Q[i]) * cimag(Q[i]);
    double nrm = sqrt(nrm2);
    int n = 0;
    double scale = 1.0;
    while (nrm * scale >= 0.25) {
        scale *= 0.5;
        n++;
    }
    cplx X[9]; /* X = i Q 2^-n */
    for (int i = 0; i < 9; i++) X[i] = I * Q[i] * scale;
    /* Horner: R = 1 + X/1 (1 + X/2 (1 + ... (1 + X/18))) */
    cplx R[9], T[9];
    m_unit(R);
    for (int k = 18; k >= 1; k--) {
        m_mul(T, X, R);
        for (int i = 0; i < 9; i++) R[i] = T[i] / (double)k;
        R[0] += 1;
        R[4] += 1;
        R[8] += 1;
    }
    for (int k = 0; k < n; k++) m_mul(R, R, R);
    memcpy(E, R, sizeof R);
}

void orc_expi(const double *Q, double *E) { expi((const cplx *)Q, (cplx *)E); }

/* ------------------------------------------------------------------ O9 reunitarise */

static void reunit_mat(cplx *M) {
    cplx *r0 = M, *r1 = M + 3, *r2 = M + 6;
    double n0 = 0;
    for (int j = 0; j < 3; j++) n0 += creal(r0[j]) * creal(r0[j]) + cimag(r0[j]) * cimag(r0[j]);
    n0 = sqrt(n0);
    for (int j = 0; j < 3; j++) r0[j] /= n0;
    cplx dot = 0; /* r0^dagger . r1 */
    for (int j = 0; j < 3; j++) dot += conj(r0[j]) * r1[j];
    for (int j = 0; j < 3; j++) r1[j] -= dot * r0[j];
    double n1 = 0;
    for (int j = 0; j < 3; j++) n1 += creal(r1[j]) * creal(r1[j]) + cimag(r1[j]) * cimag(r1[j]);
    n1 = sqrt(n1);
    for (int j = 0; j < 3; j++) r1[j] /= n1;
    r2[0] = conj(r0[1] * r1[2] - r0[2] * r1[1]);
    r2[1] = conj(r0[2] * r1[0] - r0[0] * r1[2]);
    r2[2] = conj(r0[0] * r1[1] - r0[1] * r1[0]);
}

void orc_reunit_mat(double *M) { reunit_mat((cplx *)M); }

/* ------------------------------------------------------------------ O4, O5 field generators */

int orc_mom_refresh(const int L[4], int subset, uint64_t seed, uint32_t stream_id, double *P) {
    lat_t lat;
    if (lat_init(&lat, L) || !P || subset < 0 || subset > 2) return 1;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) {
        if (!in_subset(&lat, s, subset)) continue;
        for (int mu = 0; mu < 4; mu++) {
            double q[8];
            gauss8(seed, s, mu, stream_id, 1u, q);
            herm_from_coeffs(q, LINK(P, s, mu));
        }
    }
    return 0;
}

int orc_hot_start(const int L[4], uint64_t seed, double sigma, double *U) {
    lat_t lat;
    if (lat_init(&lat, L) || !U) return 1;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++)
        for (int mu = 0; mu < 4; mu++) {
            double q[8];
            cplx Q[9];
            gauss8(seed, s, mu, 0u, 0u, q);
            for (int a = 0; a < 8; a++) q[a] *= sigma;
            herm_from_coeffs(q, Q);
            expi(Q, LINK(U, s, mu));
        }
    return 0;
}

/* U += sigma N, N = 18 iid N(0,1) reals from blocks 0..8 in storage order [row][col][re,im] */
int orc_perturb(const int L[4], uint64_t seed, double sigma, double *U) {
    lat_t lat;
    if (lat_init(&lat, L) || !U) return 1;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++)
        for (int mu = 0; mu < 4; mu++) {
            double *m = U + ((size_t)s * 4 + mu) * 18;
            for (int j = 0; j < 9; j++) {
                double g[2];
                orc_rng_block(seed, (uint32_t)s, (uint32_t)mu, (uint32_t)j, 0u, 2u, NULL, NULL, g);
                m[2 * j] += sigma * g[0];
                m[2 * j + 1] += sigma * g[1];
            }
        }
    return 0;
}

int orc_gauge_transform(const int L[4], uint64_t seed, double sigma, const double *U, double *G,
                        double *Uout) {
    lat_t lat;
    if (lat_init(&lat, L) || !G) return 1;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) {
        double q[8];
        cplx Q[9];
        gauss8(seed, s, 0, 0u, 3u, q);
        for (int a = 0; a < 8; a++) q[a] *= sigma;
        herm_from_coeffs(q, Q);
        expi(Q, (cplx *)(G + (size_t)s * 18));
    }
    if (!Uout) return 0;
    if (!U) return 1;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++)
        for (int mu = 0; mu < 4; mu++) {
            cplx T[9], Gd[9];
            const cplx *Gx = (const cplx *)(G + (size_t)s * 18);
            const cplx *Gf = (const cplx *)(G + (size_t)hop(&lat, s, mu, +1) * 18);
            m_mul(T, Gx, CLINK(U, s, mu));
            m_dag(Gd, Gf);
            m_mul(LINK(Uout, s, mu), T, Gd);
        }
    return 0;
}

/* ------------------------------------------------------------------ O6 plaquette, action */

/* P_mu_nu(x) = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dagger U_nu(x)^dagger */
static void plaq_mat(const lat_t *lat, const double *U, long s, int mu, int nu, cplx *P) {
    cplx T[9], D[9];
    m_mul(T, CLINK(U, s, mu), CLINK(U, hop(lat, s, mu, +1), nu));
    m_dag(D, CLINK(U, hop(lat, s, nu, +1), mu));
    m_mul(T, T, D);
    m_dag(D, CLINK(U, s, nu));
    m_mul(P, T, D);
}

/* sum over mu<nu of (1/3) Re tr P_mu_nu(x) at one site */
static double site_plaq(const lat_t *lat, const double *U, long s) {
    double acc = 0;
    for (int mu = 0; mu < 4; mu++)
        for (int nu = mu + 1; nu < 4; nu++) {
            cplx P[9];
            plaq_mat(lat, U, s, mu, nu, P);
            acc += creal(m_trace(P)) / 3.0;
        }
    return acc;
}

int orc_plaquette(const int L[4], const double *U, double *avg, double *per_t) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !avg) return 1;
    double *w = malloc(sizeof(double) * (size_t)lat.V);
    if (!w) return 2;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) w[s] = site_plaq(&lat, U, s);
    long double tot = 0;
    int Lt = lat.L[3];
    long Vs = lat.V / Lt;
    for (int t = 0; t < Lt; t++) {
        long double acc = 0;
        for (long s = (long)t * Vs; s < (long)(t + 1) * Vs; s++) acc += w[s];
        if (per_t) per_t[t] = (double)(acc / (6.0L * Vs));
        tot += acc;
    }
    *avg = (double)(tot / (6.0L * lat.V));
    free(w);
    return 0;
}

int orc_action(const int L[4], double beta, const double *U, double *S) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !S) return 1;
    /* S = beta sum_x sum_{mu<nu} (1 - (1/3) Re tr P_mu_nu(x)) */
    double *w = malloc(sizeof(double) * (size_t)lat.V);
    if (!w) return 2;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) w[s] = 6.0 - site_plaq(&lat, U, s);
    long double acc = 0;
    for (long s = 0; s < lat.V; s++) acc += w[s];
    *S = (double)(beta * acc);
    free(w);
    return 0;
}

/* ------------------------------------------------------------------ O7 force */

/* A_mu(x) = sum_{nu != mu} [ U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
 *                           + U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu) ] */
static void staple_sum(const lat_t *lat, const double *U, long s, int mu, cplx *A) {
    m_zero(A);
    long xpm = hop(lat, s, mu, +1);
    for (int nu = 0; nu < 4; nu++) {
        if (nu == mu) continue;
        cplx T[9], D[9];
        long xpn = hop(lat, s, nu, +1);
        long xmn = hop(lat, s, nu, -1);
        long xpmmn = hop(lat, xpm, nu, -1);
        /* up */
        m_dag(D, CLINK(U, xpn, mu));
        m_mul(T, CLINK(U, xpm, nu), D);
        m_dag(D, CLINK(U, s, nu));
        m_mul(T, T, D);
        m_add(A, T);
        /* down */
        m_dag(T, CLINK(U, xpmmn, nu));
        m_dag(D, CLINK(U, xmn, mu));
        m_mul(T, T, D);
        m_mul(T, T, CLINK(U, xmn, nu));
        m_add(A, T);
    }
}

/* F = (i beta/12) [ (W - W^dag) - (1/3) tr(W - W^dag) 1 ],  W = U_mu(x) A_mu(x) */
static void force_link(const lat_t *lat, double beta, const double *U, long s, int mu, cplx *F) {
    cplx A[9], W[9], Wd[9], X[9];
    staple_sum(lat, U, s, mu, A);
    m_mul(W, CLINK(U, s, mu), A);
    m_dag(Wd, W);
    for (int i = 0; i < 9; i++) X[i] = W[i] - Wd[i];
    cplx tr3 = m_trace(X) / 3.0;
    X[0] -= tr3;
    X[4] -= tr3;
    X[8] -= tr3;
    for (int i = 0; i < 9; i++) F[i] = I * (beta / 12.0) * X[i];
}

int orc_gauge_force(const int L[4], int subset, double beta, const double *U, double *F) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !F || subset < 0 || subset > 2) return 1;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) {
        if (!in_subset(&lat, s, subset)) continue;
        for (int mu = 0; mu < 4; mu++) force_link(&lat, beta, U, s, mu, LINK(F, s, mu));
    }
    return 0;
}

/* the same force_link at a list of sites only (sampled parity on the large lattices);
 * F is double[nsites][4][3][3][2] */
int orc_gauge_force_sites(const int L[4], double beta, const double *U, int nsites, const int32_t *sites,
                          double *F) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !F || nsites < 0 || (nsites && !sites)) return 1;
    for (int i = 0; i < nsites; i++)
        if (sites[i] < 0 || sites[i] >= lat.V) return 1;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < nsites; i++)
        for (int mu = 0; mu < 4; mu++) force_link(&lat, beta, U, sites[i], mu, LINK(F, i, mu));
    return 0;
}

int orc_sum_retr_w(const int L[4], const double *U, double *out) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !out) return 1;
    long double acc = 0;
    for (long s = 0; s < lat.V; s++)
        for (int mu = 0; mu < 4; mu++) {
            cplx A[9], W[9];
            staple_sum(&lat, U, s, mu, A);
            m_mul(W, CLINK(U, s, mu), A);
            acc += creal(m_trace(W));
        }
    *out = (double)acc;
    return 0;
}

/* ------------------------------------------------------------------ O10 updates */

int orc_mom_update(const int L[4], int subset, double eps, const double *F, double *P) {
    lat_t lat;
    if (lat_init(&lat, L) || !F || !P || subset < 0 || subset > 2) return 1;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) {
        if (!in_subset(&lat, s, subset)) continue;
        for (int i = 0; i < 72; i++) P[(size_t)s * 72 + i] += eps * F[(size_t)s * 72 + i];
    }
    return 0;
}

int orc_link_update(const int L[4], int subset, double eps, const double *P, double *U, int reunit) {
    lat_t lat;
    if (lat_init(&lat, L) || !P || !U || subset < 0 || subset > 2) return 1;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) {
        if (!in_subset(&lat, s, subset)) continue;
        for (int mu = 0; mu < 4; mu++) {
            cplx Q[9], E[9];
            const cplx *p = CLINK(P, s, mu);
            for (int i = 0; i < 9; i++) Q[i] = eps * p[i];
            expi(Q, E);
            m_mul(LINK(U, s, mu), E, CLINK(U, s, mu));
            if (reunit) reunit_mat(LINK(U, s, mu));
        }
    }
    return 0;
}

int orc_reunit(const int L[4], int subset, double *U) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || subset < 0 || subset > 2) return 1;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) {
        if (!in_subset(&lat, s, subset)) continue;
        for (int mu = 0; mu < 4; mu++) reunit_mat(LINK(U, s, mu));
    }
    return 0;
}

/* ------------------------------------------------------------------ O12 reductions */

static long double site_value(int kind, int ncomp, const double *field, long s, int comp) {
    const double *p = field + (size_t)s * ncomp;
    if (kind == 0) return p[comp];
    long double acc = 0;
    if (kind == 1) {
        for (int i = 0; i < ncomp; i++) acc += (long double)p[i] * p[i];
    } else {
        for (int m = 0; m < ncomp / 18; m++) acc += (long double)p[18 * m + 0] + p[18 * m + 8] + p[18 * m + 16];
    }
    return acc;
}

int orc_sum(const int L[4], int subset, int kind, int ncomp, const double *field, double *out) {
    lat_t lat;
    if (lat_init(&lat, L) || !field || !out || subset < 0 || subset > 2 || kind < 0 || kind > 2 ||
        ncomp < 1 || (kind == 2 && ncomp % 18))
        return 1;
    int nout = kind == 0 ? ncomp : 1;
    for (int c = 0; c < nout; c++) {
        long double acc = 0;
        for (long s = 0; s < lat.V; s++)
            if (in_subset(&lat, s, subset)) acc += site_value(kind, ncomp, field, s, c);
        out[c] = (double)acc;
    }
    return 0;
}

int orc_sum_multi(const int L[4], int kind, int ncomp, const double *field, const int32_t *subset_id,
                  int nsub, double *out) {
    lat_t lat;
    if (lat_init(&lat, L) || !field || !out || nsub < 1 || kind < 0 || kind > 2 || ncomp < 1 ||
        (kind == 2 && ncomp % 18))
        return 1;
    if (!subset_id && nsub != lat.L[3]) return 1;
    int nout = kind == 0 ? ncomp : 1;
    long double *acc = calloc((size_t)nsub * nout, sizeof(long double));
    if (!acc) return 2;
    for (long s = 0; s < lat.V; s++) {
        int k = subset_id ? subset_id[s] : tslice_of(&lat, s);
        if (k < 0 || k >= nsub) continue; /* sites outside every subset */
        for (int c = 0; c < nout; c++) acc[(size_t)k * nout + c] += site_value(kind, ncomp, field, s, c);
    }
    for (long i = 0; i < (long)nsub * nout; i++) out[i] = (double)acc[i];
    free(acc);
    return 0;
}

int orc_hamiltonian(const int L[4], double beta, const double *U, const double *P, double *K,
                    double *S) {
    int rc = orc_sum(L, 0, 1, 72, P, K);
    if (rc) return rc;
    return orc_action(L, beta, U, S);
}

/* ------------------------------------------------------------------ O11 leapfrog */

int orc_md_step(const int L[4], double beta, double eps_p, double eps_u, double *U, double *P) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !P) return 1;
    double *F = malloc(sizeof(double) * 72 * (size_t)lat.V);
    if (!F) return 2;
    orc_gauge_force(L, 0, beta, U, F);
    orc_mom_update(L, 0, eps_p, F, P);
    orc_link_update(L, 0, eps_u, P, U, 1);
    free(F);
    return 0;
}

int orc_leapfrog(const int L[4], double beta, double eps, int nsteps, double *U, double *P) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !P || nsteps < 1) return 1;
    double *F = malloc(sizeof(double) * 72 * (size_t)lat.V);
    if (!F) return 2;
    orc_gauge_force(L, 0, beta, U, F);
    orc_mom_update(L, 0, 0.5 * eps, F, P);
    for (int k = 0; k < nsteps; k++) {
        orc_link_update(L, 0, eps, P, U, 1);
        orc_gauge_force(L, 0, beta, U, F);
        orc_mom_update(L, 0, k == nsteps - 1 ? 0.5 * eps : eps, F, P);
    }
    free(F);
    return 0;
}

/* ------------------------------------------------------------------ O13 anisotropic Wilson action
 * (PAPER.md:101 names an "anisotropic Wilson" gauge action and gives no formula; R19):
 *   S = beta_s sum_x sum_{i<j<3} (1 - (1/3) Re tr P_ij(x)) + beta_t sum_x sum_{i<3} (1 - (1/3) Re tr P_i3(x))
 * i.e. one coefficient for the three space-space planes and one for the three space-time planes. */

static int plane_is_temporal(int mu, int nu) { return mu == 3 || nu == 3; }

/* (1/3) Re tr of the space-space planes (out[0]) and of the space-time planes (out[1]) at one site */
static void site_plaq_st(const lat_t *lat, const double *U, long s, double out[2]) {
    out[0] = out[1] = 0;
    for (int mu = 0; mu < 4; mu++)
        for (int nu = mu + 1; nu < 4; nu++) {
            cplx P[9];
            plaq_mat(lat, U, s, mu, nu, P);
            out[plane_is_temporal(mu, nu)] += creal(m_trace(P)) / 3.0;
        }
}

/* avg[0] = mean over sites and the 3 space-space planes of (1/3) Re tr P, avg[1] = same over the 3 space-time
 * planes; per_t (or NULL) is [Lt][2], a plaquette belonging to the timeslice of its base site (R13) */
int orc_plaquette_st(const int L[4], const double *U, double avg[2], double *per_t) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !avg) return 1;
    int Lt = lat.L[3];
    long Vs = lat.V / Lt;
    long double tot[2] = {0, 0};
    for (int t = 0; t < Lt; t++) {
        long double acc[2] = {0, 0};
        for (long s = (long)t * Vs; s < (long)(t + 1) * Vs; s++) {
            double w[2];
            site_plaq_st(&lat, U, s, w);
            acc[0] += w[0];
            acc[1] += w[1];
        }
        for (int k = 0; k < 2; k++) {
            if (per_t) per_t[2 * t + k] = (double)(acc[k] / (3.0L * Vs));
            tot[k] += acc[k];
        }
    }
    for (int k = 0; k < 2; k++) avg[k] = (double)(tot[k] / (3.0L * lat.V));
    return 0;
}

int orc_action_aniso(const int L[4], double beta_s, double beta_t, const double *U, double *S) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !S) return 1;
    long double acc = 0;
    for (long s = 0; s < lat.V; s++) {
        double w[2];
        site_plaq_st(&lat, U, s, w);
        acc += beta_s * (3.0 - w[0]) + beta_t * (3.0 - w[1]);
    }
    *S = (double)acc;
    return 0;
}

/* F_mu(x) = (i/12) [ (W - W^dag) - (1/3) tr(W - W^dag) ],  W = U_mu(x) sum_{nu != mu} beta_{mu nu} (staples in nu),
 * beta_{mu nu} = beta_t if mu or nu is the time direction, else beta_s.  Staples as in O7. */
static void force_link_aniso(const lat_t *lat, double beta_s, double beta_t, const double *U, long s, int mu,
                             cplx *F) {
    cplx A[9], W[9], Wd[9], X[9];
    m_zero(A);
    long xpm = hop(lat, s, mu, +1);
    for (int nu = 0; nu < 4; nu++) {
        if (nu == mu) continue;
        double b = plane_is_temporal(mu, nu) ? beta_t : beta_s;
        cplx T[9], D[9];
        long xpn = hop(lat, s, nu, +1);
        long xmn = hop(lat, s, nu, -1);
        long xpmmn = hop(lat, xpm, nu, -1);
        m_dag(D, CLINK(U, xpn, mu));
        m_mul(T, CLINK(U, xpm, nu), D);
        m_dag(D, CLINK(U, s, nu));
        m_mul(T, T, D);
        for (int i = 0; i < 9; i++) A[i] += b * T[i];
        m_dag(T, CLINK(U, xpmmn, nu));
        m_dag(D, CLINK(U, xmn, mu));
        m_mul(T, T, D);
        m_mul(T, T, CLINK(U, xmn, nu));
        for (int i = 0; i < 9; i++) A[i] += b * T[i];
    }
    m_mul(W, CLINK(U, s, mu), A);
    m_dag(Wd, W);
    for (int i = 0; i < 9; i++) X[i] = W[i] - Wd[i];
    cplx tr3 = m_trace(X) / 3.0;
    X[0] -= tr3;
    X[4] -= tr3;
    X[8] -= tr3;
    for (int i = 0; i < 9; i++) F[i] = I * (1.0 / 12.0) * X[i];
}

int orc_gauge_force_aniso(const int L[4], int subset, double beta_s, double beta_t, const double *U, double *F) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !F || subset < 0 || subset > 2) return 1;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) {
        if (!in_subset(&lat, s, subset)) continue;
        for (int mu = 0; mu < 4; mu++) force_link_aniso(&lat, beta_s, beta_t, U, s, mu, LINK(F, s, mu));
    }
    return 0;
}

/* ------------------------------------------------------------------ O14 two-level (multi-timescale) leapfrog
 * ("Multi-timescale integrators were utilized", no formula; R20: Sexton-Weingarten
 * nesting).  The action is split as S = S_1 + S_0, each an anisotropic Wilson action with coefficients
 * (bs[k], bt[k]); S_1 is integrated with n_outer steps of eps_1 = tau/n_outer, S_0 with n_inner leapfrog
 * steps of eps_0 = eps_1/n_inner inside every outer step:
 *   outer step:  P += (eps_1/2) F_1;  inner leapfrog [P += (eps_0/2) F_0; n_inner x {U <- reunit(exp(i eps_0 P) U);
 *                P += eps_0 F_0, eps_0/2 on the last}];  P += (eps_1/2) F_1
 * written out step by step, no merging of adjacent half steps. */
int orc_nested_leapfrog(const int L[4], const double bs[2], const double bt[2], double tau, int n_outer,
                        int n_inner, double *U, double *P) {
    lat_t lat;
    if (lat_init(&lat, L) || !U || !P || n_outer < 1 || n_inner < 1) return 1;
    double *F = malloc(sizeof(double) * 72 * (size_t)lat.V);
    if (!F) return 2;
    double e1 = tau / n_outer, e0 = e1 / n_inner;
    for (int k = 0; k < n_outer; k++) {
        orc_gauge_force_aniso(L, 0, bs[1], bt[1], U, F);
        orc_mom_update(L, 0, 0.5 * e1, F, P);
        orc_gauge_force_aniso(L, 0, bs[0], bt[0], U, F);
        orc_mom_update(L, 0, 0.5 * e0, F, P);
        for (int j = 0; j < n_inner; j++) {
            orc_link_update(L, 0, e0, P, U, 1);
            orc_gauge_force_aniso(L, 0, bs[0], bt[0], U, F);
            orc_mom_update(L, 0, j == n_inner - 1 ? 0.5 * e0 : e0, F, P);
        }
        orc_gauge_force_aniso(L, 0, bs[1], bt[1], U, F);
        orc_mom_update(L, 0, 0.5 * e1, F, P);
    }
    free(F);
    return 0;
}

/* ------------------------------------------------------------------ O15 / O16 pseudofermion-side site operations
 * ("a pseudofermion refresh"; only the site-parallel pieces outside the Dirac operator: the
 * Gaussian fill of a spin-colour vector field and the norm / inner-product reductions; R21).
 * A spin-colour vector has 4 spins x 3 colours = 12 complex components per site, canonical layout
 * double[V][12][2] with component k = 3*spin + colour.
 * O15: eta_k(x) = (g0 + i g1)/sqrt(2) with (g0, g1) the Box-Muller pair of generator block
 * (site s, 64 + k, stream_id, purpose 4), so that <|eta_k|^2> = 1 and the weight is exp(-eta^dag eta). */
int orc_spinor_gaussian(const int L[4], int subset, uint64_t seed, uint32_t stream_id, double *eta) {
    lat_t lat;
    if (lat_init(&lat, L) || !eta || subset < 0 || subset > 2) return 1;
    const double isq2 = 1.0 / sqrt(2.0);
    for (long s = 0; s < lat.V; s++) {
        if (!in_subset(&lat, s, subset)) continue;
        for (int k = 0; k < 12; k++) {
            double g[2];
            orc_rng_block(seed, (uint32_t)s, 4u, (uint32_t)k, stream_id, 4u, NULL, NULL, g);
            eta[((size_t)s * 12 + k) * 2 + 0] = g[0] * isq2;
            eta[((size_t)s * 12 + k) * 2 + 1] = g[1] * isq2;
        }
    }
    return 0;
}

/* O16: <a, b> = sum over the subset's sites and the nc complex components of conj(a) b; out = (Re, Im).
 * Fields double[V][nc][2].  Serial, long double, lexicographic order. */
int orc_inner_product(const int L[4], int subset, int nc, const double *a, const double *b, double out[2]) {
    lat_t lat;
    if (lat_init(&lat, L) || !a || !b || !out || subset < 0 || subset > 2 || nc < 1) return 1;
    long double re = 0, im = 0;
    for (long s = 0; s < lat.V; s++) {
        if (!in_subset(&lat, s, subset)) continue;
        for (int k = 0; k < nc; k++) {
            const double ar = a[((size_t)s * nc + k) * 2], ai = a[((size_t)s * nc + k) * 2 + 1];
            const double br = b[((size_t)s * nc + k) * 2], bi = b[((size_t)s * nc + k) * 2 + 1];
            re += (long double)ar * br + (long double)ai * bi;
            im += (long double)ar * bi - (long double)ai * br;
        }
    }
    out[0] = (double)re;
    out[1] = (double)im;
    return 0;
}

/* the same per timeslice ("sumMulti"): out[Lt][2] */
int orc_inner_product_multi(const int L[4], int nc, const double *a, const double *b, double *out) {
    lat_t lat;
    if (lat_init(&lat, L) || !a || !b || !out || nc < 1) return 1;
    int Lt = lat.L[3];
    long Vs = lat.V / Lt;
    for (int t = 0; t < Lt; t++) {
        long double re = 0, im = 0;
        for (long s = (long)t * Vs; s < (long)(t + 1) * Vs; s++)
            for (int k = 0; k < nc; k++) {
                const double ar = a[((size_t)s * nc + k) * 2], ai = a[((size_t)s * nc + k) * 2 + 1];
                const double br = b[((size_t)s * nc + k) * 2], bi = b[((size_t)s * nc + k) * 2 + 1];
                re += (long double)ar * br + (long double)ai * bi;
                im += (long double)ar * bi - (long double)ai * br;
            }
        out[2 * t] = (double)re;
        out[2 * t + 1] = (double)im;
    }
    return 0;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
