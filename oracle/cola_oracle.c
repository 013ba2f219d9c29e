/*
 * cola_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU statement of what the COLA hot path computes: the
 * Wilson-clover fermion matrix M = A - kappa*D, its even-odd Schur complement and the CGNR
 * (CGLS-form) solver it drives.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code with the CUDA library
 * (paper_2302_00850_b200/csrc) and neither includes the other.
 *
 * Authority.  The paper (/root/reference/PAPER.md; "P:n" = line n) contains no equations: it
 * names "the fermion matrix", a "conjugate gradient inverter", one thread
 * per site and a mixed-precision solver, 32-bit inner / 64-bit outer.  The
 * operator itself is fixed by BASELINE.json north_star ("BJ:ns": "M = 1 - kappa*D_hop + clover
 * on a 4D periodic/antiperiodic lattice", "12x12 clover block (two packed 6x6 Hermitian chiral
 * blocks)", "even-odd-preconditioned CGNR") and written out in SURVEY.md section 8(c), items
 * O1..O8, whose numbering the comments below cite.  Every convention is a DESIGN.md "reading".
 *
 * Style.  Full 4x4 gamma matrices (no spin-projection trick), full 3x3 links (no compression),
 * generic dense 12x12 clover blocks (no 6x6 packing), parity masks on full-lattice vectors for
 * the even-odd operators.  No blocking, fusion or reordering beyond the definitions.
 *
 * Pins (tests/test_oracle_*.py): free-field plane-wave closed form; gamma5-hermiticity; gauge
 * covariance; pure-gauge = transformed free field; uniform Abelian field F_12 = sin(B) T;
 * clover sign via zero-mode shift; dense brute force on 2^4 (built independently in numpy) and
 * its explicit inverse vs the CGNR solution; Schur identity; monotone CGLS residual.
 * oracle_cgnr_mixed: its fp64 true residual, its agreement with oracle_cgnr, and its reliable-update
 * schedule (the iterations at which updates fire = the rule of SURVEY O8 applied to oracle_cgnr's
 * fp64 residual history, tests/schedule.py).  oracle_bicgstab: the dense inverse on 2^4, oracle_cgnr's
 * solution, scipy's iterates.  Nothing here is "parity unpinned".
 *
 * Canonical arrays (C order, complex double = two doubles):
 *   psi[i][s][c]        i = x + Lx*(y + Ly*(z + Lz*t)), s = spin 0..3, c = colour 0..2   (O1)
 *   U[i][mu][a][b]      (U psi)_a = sum_b U_ab psi_b, mu = 0..3 = x,y,z,t                 (O1)
 *   A[i][12][12]        row/column index = 3*s + c                                       (O4)
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double _Complex cplx;

/* ------------------------------------------------------------------------------------------
 * O2: gamma matrices, chiral basis.  gamma_mu = [[0, A_mu],[A_mu^dagger, 0]],
 * A_k = -i sigma_k (k = x,y,z), A_t = 1.  gamma_5 = gamma_x gamma_y gamma_z gamma_t.
 * sigma_{mu nu} = (i/2)[gamma_mu, gamma_nu].  Everything is built from the Pauli matrices by
 * matrix products here; the closed forms SURVEY lists are only checked in the tests.
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    cplx g[5][4][4];        /* g[0..3] = gamma_x..gamma_t, g[4] = gamma_5 */
    cplx sig[4][4][4][4];   /* sig[mu][nu] */
} dirac_t;

static void mat4_mul(cplx c[4][4], const cplx a[4][4], const cplx b[4][4])
{
    cplx t[4][4];
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            cplx s = 0;
            for (int k = 0; k < 4; k++) s += a[i][k] * b[k][j];
            t[i][j] = s;
        }
    memcpy(c, t, sizeof(t));
}

static void dirac_init(dirac_t *d)
{
    const cplx pauli[3][2][2] = {
        {{0, 1}, {1, 0}},
        {{0, -I}, {I, 0}},
        {{1, 0}, {0, -1}},
    };
    memset(d, 0, sizeof(*d));
    for (int mu = 0; mu < 4; mu++) {
        cplx a[2][2];
        for (int i = 0; i < 2; i++)
            for (int j = 0; j < 2; j++)
                a[i][j] = (mu < 3) ? -I * pauli[mu][i][j] : (i == j ? 1.0 : 0.0);
        for (int i = 0; i < 2; i++)
            for (int j = 0; j < 2; j++) {
                d->g[mu][i][2 + j] = a[i][j];            /* upper right: A      */
                d->g[mu][2 + i][j] = conj(a[j][i]);      /* lower left: A^dagger */
            }
    }
    mat4_mul(d->g[4], d->g[0], d->g[1]);
    mat4_mul(d->g[4], d->g[4], d->g[2]);
    mat4_mul(d->g[4], d->g[4], d->g[3]);
    for (int mu = 0; mu < 4; mu++)
        for (int nu = 0; nu < 4; nu++) {
            cplx ab[4][4], ba[4][4];
            mat4_mul(ab, d->g[mu], d->g[nu]);
            mat4_mul(ba, d->g[nu], d->g[mu]);
            for (int i = 0; i < 4; i++)
                for (int j = 0; j < 4; j++)
                    d->sig[mu][nu][i][j] = 0.5 * I * (ab[i][j] - ba[i][j]);
        }
}

/* out[5][4][4] complex: gamma_x, gamma_y, gamma_z, gamma_t, gamma_5 */
void oracle_gamma(double *out)
{
    dirac_t d;
    dirac_init(&d);
    memcpy(out, d.g, sizeof(d.g));
}

/* out[4][4][4][4] complex: sigma_{mu nu} */
void oracle_sigma(double *out)
{
    dirac_t d;
    dirac_init(&d);
    memcpy(out, d.sig, sizeof(d.sig));
}

/* ------------------------------------------------------------------------------------------
 * O1: site indexing, periodic wrap, parity.
 * ---------------------------------------------------------------------------------------- */
static long vol(const int L[4]) { return (long)L[0] * L[1] * L[2] * L[3]; }

static long site_index(const int L[4], const int x[4])
{
    return x[0] + (long)L[0] * (x[1] + (long)L[1] * (x[2] + (long)L[2] * x[3]));
}

static void site_coords(const int L[4], long i, int x[4])
{
    x[0] = (int)(i % L[0]); i /= L[0];
    x[1] = (int)(i % L[1]); i /= L[1];
    x[2] = (int)(i % L[2]); i /= L[2];
    x[3] = (int)i;
}

static int site_parity(const int L[4], long i)
{
    int x[4];
    site_coords(L, i, x);
    return (x[0] + x[1] + x[2] + x[3]) & 1;
}

/* index of x + d0*mu^ + d1*nu^ with periodic wrap */
static long site_shift2(const int L[4], const int x[4], int mu, int d0, int nu, int d1)
{
    int y[4] = {x[0], x[1], x[2], x[3]};
    y[mu] = ((y[mu] + d0) % L[mu] + L[mu]) % L[mu];
    if (nu >= 0) y[nu] = ((y[nu] + d1) % L[nu] + L[nu]) % L[nu];
    return site_index(L, y);
}

static long site_shift(const int L[4], const int x[4], int mu, int d)
{
    return site_shift2(L, x, mu, d, -1, 0);
}

/* ------------------------------------------------------------------------------------------
 * 3x3 complex helpers.
 * ---------------------------------------------------------------------------------------- */
static void m3_mul(cplx c[9], const cplx a[9], const cplx b[9])
{
    cplx t[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx s = 0;
            for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j];
            t[3 * i + j] = s;
        }
    memcpy(c, t, sizeof(t));
}

static void m3_dag(cplx c[9], const cplx a[9])
{
    cplx t[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) t[3 * i + j] = conj(a[3 * j + i]);
    memcpy(c, t, sizeof(t));
}

static const cplx *link(const cplx *U, long i, int mu) { return U + (i * 4 + mu) * 9; }

/* ------------------------------------------------------------------------------------------
 * O3: hopping term at one site.
 *   (D psi)(x) = sum_mu [ eta+_mu(x) (1 - gamma_mu) U_mu(x) psi(x+mu)
 *                       + eta-_mu(x) (1 + gamma_mu) U_mu(x-mu)^dagger psi(x-mu) ]
 * eta+ = bc_mu if x_mu = L_mu-1 else 1; eta- = bc_mu if x_mu = 0 else 1.  When L_mu = 2 the two
 * neighbours coincide and both hops are accumulated.
 * The spinor field is read through a callback so that the same statement serves full arrays,
 * parity-masked arrays and the sampled-site evaluation of composite operators (O-L).
 * ---------------------------------------------------------------------------------------- */
typedef void (*spinor_at_fn)(void *ctx, long site, cplx out[12]);

static void hop_site(const dirac_t *d, const int L[4], const int bc[4], const cplx *U,
                     spinor_at_fn get, void *ctx, long i, cplx out[12])
{
    int x[4];
    site_coords(L, i, x);
    for (int k = 0; k < 12; k++) out[k] = 0;
    for (int mu = 0; mu < 4; mu++) {
        for (int dir = 0; dir < 2; dir++) {
            cplx nb[12], w[12], u[9];
            double eta, gsign;
            if (dir == 0) {                       /* forward: U_mu(x) psi(x+mu), (1 - gamma_mu) */
                long j = site_shift(L, x, mu, +1);
                get(ctx, j, nb);
                memcpy(u, link(U, i, mu), sizeof(u));
                eta = (x[mu] == L[mu] - 1) ? (double)bc[mu] : 1.0;
                gsign = -1.0;
            } else {                              /* backward: U_mu(x-mu)^dagger psi(x-mu), (1 + gamma_mu) */
                long j = site_shift(L, x, mu, -1);
                get(ctx, j, nb);
                m3_dag(u, link(U, j, mu));
                eta = (x[mu] == 0) ? (double)bc[mu] : 1.0;
                gsign = +1.0;
            }
            for (int s = 0; s < 4; s++)
                for (int a = 0; a < 3; a++) {
                    cplx acc = 0;
                    for (int b = 0; b < 3; b++) acc += u[3 * a + b] * nb[3 * s + b];
                    w[3 * s + a] = acc;
                }
            for (int s = 0; s < 4; s++)
                for (int sp = 0; sp < 4; sp++) {
                    cplx p = (s == sp ? 1.0 : 0.0) + gsign * d->g[mu][s][sp];
                    for (int a = 0; a < 3; a++) out[3 * s + a] += eta * p * w[3 * sp + a];
                }
        }
    }
}

typedef struct { const cplx *psi; } full_field_t;

static void full_field_at(void *ctx, long site, cplx out[12])
{
    memcpy(out, ((full_field_t *)ctx)->psi + site * 12, 12 * sizeof(cplx));
}

typedef struct { const cplx *psi; const int *L; int parity; } masked_field_t;

static void masked_field_at(void *ctx, long site, cplx out[12])
{
    masked_field_t *m = (masked_field_t *)ctx;
    if (site_parity(m->L, site) == m->parity)
        memcpy(out, m->psi + site * 12, 12 * sizeof(cplx));
    else
        for (int k = 0; k < 12; k++) out[k] = 0;
}

/* out = D psi on the whole lattice */
void oracle_hop(const int *L, const int *bc, const double *U_, const double *psi_, double *out_)
{
    const cplx *U = (const cplx *)U_;
    cplx *out = (cplx *)out_;
    dirac_t d;
    dirac_init(&d);
    full_field_t f = {(const cplx *)psi_};
    long V = vol(L);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) hop_site(&d, L, bc, U, full_field_at, &f, i, out + i * 12);
}

/* ------------------------------------------------------------------------------------------
 * O4: field strength from the four-leaf clover, and the clover term.
 *   Q_mn(x) = U_m(x) U_n(x+m) U_m(x+n)^+ U_n(x)^+
 *           + U_n(x) U_m(x-m+n)^+ U_n(x-m)^+ U_m(x-m)
 *           + U_m(x-m)^+ U_n(x-m-n)^+ U_m(x-m-n) U_n(x-n)
 *           + U_n(x-n)^+ U_m(x-n) U_n(x+m-n) U_m(x)^+
 *   F_mn = -i { (Q - Q^+)/8 - (1/3) tr[(Q - Q^+)/8] }          (trace removal: flag, default on)
 *   A(x) = 1 - kappa*csw * sum_{m<n} sigma_mn (x) F_mn(x)      (spin slow, colour fast)
 * Raw periodic links, no boundary phase (it cancels in closed loops).
 * ---------------------------------------------------------------------------------------- */
static void field_strength_site(const int L[4], const cplx *U, long i, int mu, int nu, int trace_sub,
                                cplx F[9])
{
    int x[4];
    site_coords(L, i, x);
    cplx Q[9], leaf[9], t[9];
    long xpm = site_shift(L, x, mu, +1), xpn = site_shift(L, x, nu, +1);
    long xmm = site_shift(L, x, mu, -1), xmn = site_shift(L, x, nu, -1);
    long xmmpn = site_shift2(L, x, mu, -1, nu, +1);
    long xmmmn = site_shift2(L, x, mu, -1, nu, -1);
    long xpmmn = site_shift2(L, x, mu, +1, nu, -1);

    /* leaf 1: U_m(x) U_n(x+m) U_m(x+n)^+ U_n(x)^+ */
    m3_mul(leaf, link(U, i, mu), link(U, xpm, nu));
    m3_dag(t, link(U, xpn, mu)); m3_mul(leaf, leaf, t);
    m3_dag(t, link(U, i, nu));   m3_mul(leaf, leaf, t);
    memcpy(Q, leaf, sizeof(Q));
    /* leaf 2: U_n(x) U_m(x-m+n)^+ U_n(x-m)^+ U_m(x-m) */
    m3_dag(t, link(U, xmmpn, mu)); m3_mul(leaf, link(U, i, nu), t);
    m3_dag(t, link(U, xmm, nu));   m3_mul(leaf, leaf, t);
    m3_mul(leaf, leaf, link(U, xmm, mu));
    for (int k = 0; k < 9; k++) Q[k] += leaf[k];
    /* leaf 3: U_m(x-m)^+ U_n(x-m-n)^+ U_m(x-m-n) U_n(x-n) */
    m3_dag(leaf, link(U, xmm, mu));
    m3_dag(t, link(U, xmmmn, nu)); m3_mul(leaf, leaf, t);
    m3_mul(leaf, leaf, link(U, xmmmn, mu));
    m3_mul(leaf, leaf, link(U, xmn, nu));
    for (int k = 0; k < 9; k++) Q[k] += leaf[k];
    /* leaf 4: U_n(x-n)^+ U_m(x-n) U_n(x+m-n) U_m(x)^+ */
    m3_dag(leaf, link(U, xmn, nu));
    m3_mul(leaf, leaf, link(U, xmn, mu));
    m3_mul(leaf, leaf, link(U, xpmmn, nu));
    m3_dag(t, link(U, i, mu)); m3_mul(leaf, leaf, t);
    for (int k = 0; k < 9; k++) Q[k] += leaf[k];

    cplx Qd[9], G[9];
    m3_dag(Qd, Q);
    for (int k = 0; k < 9; k++) G[k] = (Q[k] - Qd[k]) / 8.0;
    if (trace_sub) {
        cplx tr = (G[0] + G[4] + G[8]) / 3.0;
        G[0] -= tr; G[4] -= tr; G[8] -= tr;
    }
    for (int k = 0; k < 9; k++) F[k] = -I * G[k];
}

/* F[V][6][3][3], planes ordered (mu,nu) = (0,1),(0,2),(0,3),(1,2),(1,3),(2,3) */
void oracle_field_strength(const int *L, const double *U_, int trace_sub, double *F_)
{
    const cplx *U = (const cplx *)U_;
    cplx *F = (cplx *)F_;
    long V = vol(L);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) {
        int p = 0;
        for (int mu = 0; mu < 4; mu++)
            for (int nu = mu + 1; nu < 4; nu++, p++)
                field_strength_site(L, U, i, mu, nu, trace_sub, F + (i * 6 + p) * 9);
    }
}

static void clover_site(const dirac_t *d, const int L[4], const cplx *U, long i, double kappa,
                        double csw, int trace_sub, cplx A[144])
{
    for (int k = 0; k < 144; k++) A[k] = 0;
    for (int k = 0; k < 12; k++) A[13 * k] = 1.0;
    for (int mu = 0; mu < 4; mu++)
        for (int nu = mu + 1; nu < 4; nu++) {
            cplx F[9];
            field_strength_site(L, U, i, mu, nu, trace_sub, F);
            for (int s = 0; s < 4; s++)
                for (int sp = 0; sp < 4; sp++)
                    for (int a = 0; a < 3; a++)
                        for (int b = 0; b < 3; b++)
                            A[(3 * s + a) * 12 + 3 * sp + b] -=
                                kappa * csw * d->sig[mu][nu][s][sp] * F[3 * a + b];
        }
}

/* A[V][12][12] */
void oracle_clover(const int *L, const double *U_, double kappa, double csw, int trace_sub, double *A_)
{
    const cplx *U = (const cplx *)U_;
    cplx *A = (cplx *)A_;
    dirac_t d;
    dirac_init(&d);
    long V = vol(L);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) clover_site(&d, L, U, i, kappa, csw, trace_sub, A + i * 144);
}

/* Generic dense n x n complex inverse, Gauss-Jordan with partial pivoting.  Returns 0 on success.
 * min_pivot (optional) receives the smallest |pivot| met. */
static int dense_inverse(int n, const cplx *a_in, cplx *inv, double *min_pivot)
{
    cplx *a = (cplx *)malloc(sizeof(cplx) * n * n);
    memcpy(a, a_in, sizeof(cplx) * n * n);
    for (int i = 0; i < n; i++)
        for (int j = 0; j < n; j++) inv[i * n + j] = (i == j) ? 1.0 : 0.0;
    double minp = INFINITY;
    for (int c = 0; c < n; c++) {
        int p = c;
        for (int r = c + 1; r < n; r++)
            if (cabs(a[r * n + c]) > cabs(a[p * n + c])) p = r;
        double piv = cabs(a[p * n + c]);
        if (piv < minp) minp = piv;
        if (piv == 0.0) { free(a); return 1; }
        if (p != c)
            for (int j = 0; j < n; j++) {
                cplx t = a[c * n + j]; a[c * n + j] = a[p * n + j]; a[p * n + j] = t;
                t = inv[c * n + j]; inv[c * n + j] = inv[p * n + j]; inv[p * n + j] = t;
            }
        cplx s = 1.0 / a[c * n + c];
        for (int j = 0; j < n; j++) { a[c * n + j] *= s; inv[c * n + j] *= s; }
        for (int r = 0; r < n; r++) {
            if (r == c) continue;
            cplx f = a[r * n + c];
            if (f == 0) continue;
            for (int j = 0; j < n; j++) {
                a[r * n + j] -= f * a[c * n + j];
                inv[r * n + j] -= f * inv[c * n + j];
            }
        }
    }
    if (min_pivot) *min_pivot = minp;
    free(a);
    return 0;
}

/* Ainv[V][12][12] = per-site dense inverse of A.  Returns the number of singular sites. */
int oracle_clover_inverse(long V, const double *A_, double *Ainv_)
{
    const cplx *A = (const cplx *)A_;
    cplx *Ainv = (cplx *)Ainv_;
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
    for (long i = 0; i < V; i++) bad += dense_inverse(12, A + i * 144, Ainv + i * 144, NULL);
    return bad;
}

/* generic dense inverse exposed for the tests (n x n complex) */
int oracle_dense_inverse(int n, const double *a, double *inv)
{
    return dense_inverse(n, (const cplx *)a, (cplx *)inv, NULL);
}

static void block12_apply(const cplx A[144], const cplx v[12], cplx out[12])
{
    for (int r = 0; r < 12; r++) {
        cplx s = 0;
        for (int c = 0; c < 12; c++) s += A[12 * r + c] * v[c];
        out[r] = s;
    }
}

/* out(x) = B(x) psi(x) for a site-diagonal field of 12x12 blocks */
void oracle_block_apply(long V, const double *B_, const double *psi_, double *out_)
{
    const cplx *B = (const cplx *)B_, *psi = (const cplx *)psi_;
    cplx *out = (cplx *)out_;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) {
        cplx t[12];
        block12_apply(B + i * 144, psi + i * 12, t);
        memcpy(out + i * 12, t, sizeof(t));
    }
}

/* ------------------------------------------------------------------------------------------
 * O5: full matrix.  (M psi)(x) = A(x) psi(x) - kappa (D psi)(x);  M^dagger = gamma_5 M gamma_5.
 * ---------------------------------------------------------------------------------------- */
static void gamma5_field(const dirac_t *d, long V, const cplx *in, cplx *out)
{
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) {
        cplx t[12];
        for (int s = 0; s < 4; s++)
            for (int a = 0; a < 3; a++) {
                cplx acc = 0;
                for (int sp = 0; sp < 4; sp++) acc += d->g[4][s][sp] * in[i * 12 + 3 * sp + a];
                t[3 * s + a] = acc;
            }
        memcpy(out + i * 12, t, sizeof(t));
    }
}

static void M_plain(const dirac_t *d, const int *L, const int *bc, const cplx *U, const cplx *A,
                    double kappa, const cplx *psi, cplx *out)
{
    long V = vol(L);
    full_field_t f = {psi};
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) {
        cplx h[12], c[12];
        hop_site(d, L, bc, U, full_field_at, &f, i, h);
        block12_apply(A + i * 144, psi + i * 12, c);
        for (int k = 0; k < 12; k++) out[i * 12 + k] = c[k] - kappa * h[k];
    }
}

void oracle_M(const int *L, const int *bc, const double *U_, const double *A_, double kappa,
              int dagger, const double *psi_, double *out_)
{
    dirac_t d;
    dirac_init(&d);
    long V = vol(L);
    const cplx *psi = (const cplx *)psi_;
    cplx *out = (cplx *)out_;
    if (!dagger) {
        M_plain(&d, L, bc, (const cplx *)U_, (const cplx *)A_, kappa, psi, out);
        return;
    }
    cplx *t = (cplx *)malloc(sizeof(cplx) * 12 * V);
    gamma5_field(&d, V, psi, t);
    M_plain(&d, L, bc, (const cplx *)U_, (const cplx *)A_, kappa, t, out);
    gamma5_field(&d, V, out, out);
    free(t);
}

/* ------------------------------------------------------------------------------------------
 * O6: even-odd form.  With sites ordered (even, odd):
 *   M = [[A_ee, -kappa D_eo], [-kappa D_oe, A_oo]]
 *   S = A_ee - kappa^2 D_eo A_oo^{-1} D_oe           (acts on even sites)
 *   bhat_e = b_e + kappa D_eo A_oo^{-1} b_o
 *   x_o    = A_oo^{-1} (b_o + kappa D_oe x_e)
 * Half-lattice vectors are full-lattice arrays that vanish on the other parity.
 * ---------------------------------------------------------------------------------------- */
static void mask_parity(const int *L, long V, int parity, cplx *v)
{
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++)
        if (site_parity(L, i) != parity)
            for (int k = 0; k < 12; k++) v[i * 12 + k] = 0;
}

/* out_p = D_{p,1-p} in_{1-p}: hop applied to the (1-p)-masked input, kept on parity p only */
void oracle_dslash_parity(const int *L, const int *bc, const double *U_, int out_parity,
                          const double *psi_, double *out_)
{
    dirac_t d;
    dirac_init(&d);
    long V = vol(L);
    cplx *out = (cplx *)out_;
    masked_field_t m = {(const cplx *)psi_, L, 1 - out_parity};
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) {
        if (site_parity(L, i) == out_parity)
            hop_site(&d, L, bc, (const cplx *)U_, masked_field_at, &m, i, out + i * 12);
        else
            for (int k = 0; k < 12; k++) out[i * 12 + k] = 0;
    }
}

static void schur_plain(const int *L, const int *bc, const double *U, const cplx *A, const cplx *Ainv,
                        double kappa, const cplx *x, cplx *out)
{
    long V = vol(L);
    cplx *t1 = (cplx *)malloc(sizeof(cplx) * 12 * V);
    cplx *t2 = (cplx *)malloc(sizeof(cplx) * 12 * V);
    cplx *xe = (cplx *)malloc(sizeof(cplx) * 12 * V);
    memcpy(xe, x, sizeof(cplx) * 12 * V);
    mask_parity(L, V, 0, xe);                                                   /* x_e            */
    oracle_dslash_parity(L, bc, U, 1, (double *)xe, (double *)t1);              /* D_oe x_e       */
    oracle_block_apply(V, (const double *)Ainv, (double *)t1, (double *)t2);    /* A^-1 (...)     */
    mask_parity(L, V, 1, t2);
    oracle_dslash_parity(L, bc, U, 0, (double *)t2, (double *)t1);              /* D_eo (...)     */
    oracle_block_apply(V, (const double *)A, (double *)xe, (double *)t2);       /* A_ee x_e       */
    mask_parity(L, V, 0, t2);
#pragma omp parallel for schedule(static)
    for (long k = 0; k < 12 * V; k++) out[k] = t2[k] - kappa * kappa * t1[k];
    free(t1); free(t2); free(xe);
}

/* out_e = S x_e (dagger: gamma_5 S gamma_5); odd sites of out are zero */
void oracle_schur(const int *L, const int *bc, const double *U_, const double *A_, const double *Ainv_,
                  double kappa, int dagger, const double *x_, double *out_)
{
    dirac_t d;
    dirac_init(&d);
    long V = vol(L);
    if (!dagger) {
        schur_plain(L, bc, U_, (const cplx *)A_, (const cplx *)Ainv_, kappa, (const cplx *)x_, (cplx *)out_);
        return;
    }
    cplx *t = (cplx *)malloc(sizeof(cplx) * 12 * V);
    gamma5_field(&d, V, (const cplx *)x_, t);
    schur_plain(L, bc, U_, (const cplx *)A_, (const cplx *)Ainv_, kappa, t, (cplx *)out_);
    gamma5_field(&d, V, (cplx *)out_, (cplx *)out_);
    free(t);
}

/* bhat_e = b_e + kappa D_eo A_oo^{-1} b_o  (odd sites of bhat are zero) */
void oracle_eo_prepare(const int *L, const int *bc, const double *U_, const double *Ainv_, double kappa,
                       const double *b_, double *bhat_)
{
    long V = vol(L);
    const cplx *b = (const cplx *)b_;
    cplx *bhat = (cplx *)bhat_;
    cplx *t1 = (cplx *)malloc(sizeof(cplx) * 12 * V);
    cplx *t2 = (cplx *)malloc(sizeof(cplx) * 12 * V);
    oracle_block_apply(V, Ainv_, b_, (double *)t1);
    mask_parity(L, V, 1, t1);                                                   /* A_oo^-1 b_o */
    oracle_dslash_parity(L, bc, U_, 0, (double *)t1, (double *)t2);             /* D_eo (...)  */
    for (long i = 0; i < V; i++)
        for (int k = 0; k < 12; k++)
            bhat[i * 12 + k] = (site_parity(L, i) == 0) ? b[i * 12 + k] + kappa * t2[i * 12 + k] : 0.0;
    free(t1); free(t2);
}

/* x_o = A_oo^{-1}(b_o + kappa D_oe x_e); x holds x_e on entry (odd part ignored), full x on exit */
void oracle_eo_reconstruct(const int *L, const int *bc, const double *U_, const double *Ainv_, double kappa,
                           const double *b_, double *x_)
{
    long V = vol(L);
    const cplx *b = (const cplx *)b_;
    cplx *x = (cplx *)x_;
    cplx *t1 = (cplx *)malloc(sizeof(cplx) * 12 * V);
    cplx *t2 = (cplx *)malloc(sizeof(cplx) * 12 * V);
    mask_parity(L, V, 0, x);
    oracle_dslash_parity(L, bc, U_, 1, x_, (double *)t1);                       /* D_oe x_e */
    for (long k = 0; k < 12 * V; k++) t1[k] = b[k] + kappa * t1[k];
    mask_parity(L, V, 1, t1);
    oracle_block_apply(V, Ainv_, (double *)t1, (double *)t2);
    for (long i = 0; i < V; i++)
        if (site_parity(L, i) == 1)
            for (int k = 0; k < 12; k++) x[i * 12 + k] = t2[i * 12 + k];
    free(t1); free(t2);
}

/* ------------------------------------------------------------------------------------------
 * O-L: evaluation at a list of sites (large lattices).  No full-lattice temporaries: the
 * clover block and its inverse are rebuilt from the links at each site that needs them.
 * ---------------------------------------------------------------------------------------- */
/* (gamma_5) psi on every site: gamma_5 is site-diagonal, so gamma_5 K gamma_5 at one site is K applied
 * to a field read through this provider, followed by gamma_5 on the single output site. */
typedef struct { const dirac_t *d; const cplx *psi; int g5; } g5_field_t;

static void g5_field_at(void *ctx, long site, cplx out[12])
{
    g5_field_t *g = (g5_field_t *)ctx;
    for (int s = 0; s < 4; s++)
        for (int a = 0; a < 3; a++) {
            cplx acc = 0;
            if (g->g5) for (int q = 0; q < 4; q++) acc += g->d->g[4][s][q] * g->psi[site * 12 + 3 * q + a];
            else acc = g->psi[site * 12 + 3 * s + a];
            out[3 * s + a] = acc;
        }
}

typedef struct {
    const dirac_t *d; const int *L; const int *bc; const cplx *U; g5_field_t x;
    double kappa, csw; int trace_sub;
} schur_inner_t;

/* x_e: the (gamma_5-multiplied) input on even sites, 0 on odd sites */
static void x_even_at(void *ctx, long site, cplx out[12])
{
    schur_inner_t *s = (schur_inner_t *)ctx;
    if (site_parity(s->L, site) != 0) { for (int k = 0; k < 12; k++) out[k] = 0; return; }
    g5_field_at(&s->x, site, out);
}

/* t(o) = A(o)^{-1} (D_oe x_e)(o) for odd o, 0 for even o */
static void schur_inner_at(void *ctx, long site, cplx out[12])
{
    schur_inner_t *s = (schur_inner_t *)ctx;
    if (site_parity(s->L, site) != 1) { for (int k = 0; k < 12; k++) out[k] = 0; return; }
    cplx h[12], A[144], Ainv[144];
    hop_site(s->d, s->L, s->bc, s->U, x_even_at, s, site, h);
    clover_site(s->d, s->L, s->U, site, s->kappa, s->csw, s->trace_sub, A);
    dense_inverse(12, A, Ainv, NULL);
    block12_apply(Ainv, h, out);
}

/* which: 0 = D (full hop), 1 = M, 2 = M^dagger, 3 = S, 4 = S^dagger.  out[n][12] complex.
 * For which >= 3 the listed sites must be even (odd ones return 0). */
void oracle_apply_sites(const int *L, const int *bc, const double *U_, double kappa, double csw,
                        int trace_sub, int which, const double *psi_, long n, const long *sites,
                        double *out_)
{
    const cplx *U = (const cplx *)U_, *psi = (const cplx *)psi_;
    cplx *out = (cplx *)out_;
    dirac_t d;
    dirac_init(&d);
    int dag = (which == 2 || which == 4);
#pragma omp parallel for schedule(dynamic, 16)
    for (long q = 0; q < n; q++) {
        long i = sites[q];
        cplx r[12], h[12], c[12], v[12], A[144];
        g5_field_t gf = {&d, psi, dag};
        if (which == 0) {
            hop_site(&d, L, bc, U, g5_field_at, &gf, i, r);
        } else if (which == 1 || which == 2) {
            hop_site(&d, L, bc, U, g5_field_at, &gf, i, h);
            g5_field_at(&gf, i, v);
            clover_site(&d, L, U, i, kappa, csw, trace_sub, A);
            block12_apply(A, v, c);
            for (int k = 0; k < 12; k++) r[k] = c[k] - kappa * h[k];
        } else {
            schur_inner_t s = {&d, L, bc, U, gf, kappa, csw, trace_sub};
            if (site_parity(L, i) != 0) {
                for (int k = 0; k < 12; k++) r[k] = 0;
            } else {
                hop_site(&d, L, bc, U, schur_inner_at, &s, i, h);      /* D_eo A_oo^-1 D_oe x_e */
                x_even_at(&s, i, v);
                clover_site(&d, L, U, i, kappa, csw, trace_sub, A);
                block12_apply(A, v, c);
                for (int k = 0; k < 12; k++) r[k] = c[k] - kappa * kappa * h[k];
            }
        }
        if (dag) {
            for (int s4 = 0; s4 < 4; s4++)
                for (int a = 0; a < 3; a++) {
                    cplx acc = 0;
                    for (int sp = 0; sp < 4; sp++) acc += d.g[4][s4][sp] * r[3 * sp + a];
                    out[q * 12 + 3 * s4 + a] = acc;
                }
        } else {
            memcpy(out + q * 12, r, sizeof(r));
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * O7: CGNR in CGLS form for K x = b, K = M (even_odd = 0) or K = S with b = bhat_e (even_odd = 1).
 *   x0 = 0; r0 = b; s0 = K^+ r0; p0 = s0; gamma0 = |s0|^2
 *   loop: q = K p; alpha = gamma/|q|^2; x += alpha p; r -= alpha q;
 *         stop if |r| <= tol*|b_full|; s = K^+ r; gamma' = |s|^2; beta = gamma'/gamma; p = s + beta p
 * Iteration count = number of passes (one K and one K^+ each).  resid_hist[k] = |r_{k+1}|/|b_full|.
 * After the loop the full-lattice true residual |b - M x|/|b| is recomputed with O5.
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    const int *L; const int *bc; const double *U; const double *A; const double *Ainv;
    double kappa; int even_odd;
} op_ctx_t;

static void apply_K(const op_ctx_t *o, int dagger, const cplx *in, cplx *out)
{
    if (o->even_odd) oracle_schur(o->L, o->bc, o->U, o->A, o->Ainv, o->kappa, dagger, (const double *)in, (double *)out);
    else oracle_M(o->L, o->bc, o->U, o->A, o->kappa, dagger, (const double *)in, (double *)out);
}

static double norm2(long n, const cplx *v)
{
    double s = 0;
    for (long k = 0; k < n; k++) s += creal(v[k]) * creal(v[k]) + cimag(v[k]) * cimag(v[k]);
    return s;
}

/* returns 0 if converged, 1 if max_iter was hit.  x is the FULL-lattice solution of M x = b. */
int oracle_cgnr(const int *L, const int *bc, const double *U_, const double *A_, const double *Ainv_,
                double kappa, int even_odd, const double *b_, double *x_, double tol, int max_iter,
                int *iters_out, double *resid_hist, double *true_resid_out)
{
    long V = vol(L), n = 12 * V;
    op_ctx_t o = {L, bc, U_, A_, Ainv_, kappa, even_odd};
    const cplx *b = (const cplx *)b_;
    cplx *x = (cplx *)x_;
    cplx *rhs = (cplx *)malloc(sizeof(cplx) * n), *r = (cplx *)malloc(sizeof(cplx) * n);
    cplx *p = (cplx *)malloc(sizeof(cplx) * n), *q = (cplx *)malloc(sizeof(cplx) * n);
    cplx *s = (cplx *)malloc(sizeof(cplx) * n);
    double bnorm = sqrt(norm2(n, b));
    if (even_odd) oracle_eo_prepare(L, bc, U_, Ainv_, kappa, b_, (double *)rhs);
    else memcpy(rhs, b, sizeof(cplx) * n);

    for (long k = 0; k < n; k++) x[k] = 0;
    memcpy(r, rhs, sizeof(cplx) * n);
    apply_K(&o, 1, r, s);
    memcpy(p, s, sizeof(cplx) * n);
    double gamma = norm2(n, s);
    int it = 0, status = 1;
    if (sqrt(norm2(n, r)) <= tol * bnorm) status = 0;
    while (status && it < max_iter) {
        apply_K(&o, 0, p, q);
        double alpha = gamma / norm2(n, q);
        for (long k = 0; k < n; k++) { x[k] += alpha * p[k]; r[k] -= alpha * q[k]; }
        double rn = sqrt(norm2(n, r));
        if (resid_hist) resid_hist[it] = rn / bnorm;
        it++;
        if (rn <= tol * bnorm) { status = 0; break; }
        apply_K(&o, 1, r, s);
        double gamma_new = norm2(n, s);
        double beta = gamma_new / gamma;
        gamma = gamma_new;
        for (long k = 0; k < n; k++) p[k] = s[k] + beta * p[k];
    }
    if (even_odd) oracle_eo_reconstruct(L, bc, U_, Ainv_, kappa, b_, x_);
    /* true residual on the full lattice, O5 */
    oracle_M(L, bc, U_, A_, kappa, 0, x_, (double *)q);
    for (long k = 0; k < n; k++) q[k] = b[k] - q[k];
    if (true_resid_out) *true_resid_out = sqrt(norm2(n, q)) / bnorm;
    if (iters_out) *iters_out = it;
    free(rhs); free(r); free(p); free(q); free(s);
    return status;
}

/* ------------------------------------------------------------------------------------------
 * O8: mixed-precision CGLS with reliable updates (32-bit inner, 64-bit outer).
 * The inner vectors p, q, s, r32, x32 are rounded to float after every update; the operator is
 * applied in double to the float-rounded vector and its result rounded to float (a model of an
 * fp32 operator good to one rounding; the GPU path does its arithmetic in float throughout).
 * Reductions in double.  r_max = max |r| since the last update; when |r32| < delta*r_max or
 * |r32| <= tol*|b|:  x64 += x32; x32 = 0; r64 = rhs - K x64 (double); r32 = float(r64);
 * r_max = |r64|; continue with the SAME p.  Terminate on the fp64 residual only.
 * Used for iteration-count comparison; reference results stay those of oracle_cgnr.
 * Outputs that expose the schedule (no effect on the arithmetic): resid_hist[k] = |r32_{k+1}|/|b| of the
 * recurrence as the delta test sees it (before an update replaces it), k < iterations; update_iters[j] = the
 * iteration count `it` (1-based) at which the j-th reliable update fired, j < min(updates, max_updates).
 * tests/test_oracle_pins.py pins the schedule against the rule applied to oracle_cgnr's fp64 history.
 * ---------------------------------------------------------------------------------------- */
static void round_to_float(long n, cplx *v)
{
    for (long k = 0; k < n; k++) v[k] = (double)(float)creal(v[k]) + I * (double)(float)cimag(v[k]);
}

int oracle_cgnr_mixed(const int *L, const int *bc, const double *U_, const double *A_, const double *Ainv_,
                      double kappa, int even_odd, const double *b_, double *x_, double tol, double delta,
                      int max_iter, int *iters_out, int *updates_out, double *true_resid_out,
                      double *resid_hist, int *update_iters, int max_updates)
{
    long V = vol(L), n = 12 * V;
    op_ctx_t o = {L, bc, U_, A_, Ainv_, kappa, even_odd};
    const cplx *b = (const cplx *)b_;
    cplx *x = (cplx *)x_;
    cplx *rhs = (cplx *)malloc(sizeof(cplx) * n), *r = (cplx *)malloc(sizeof(cplx) * n);
    cplx *p = (cplx *)malloc(sizeof(cplx) * n), *q = (cplx *)malloc(sizeof(cplx) * n);
    cplx *s = (cplx *)malloc(sizeof(cplx) * n), *xl = (cplx *)malloc(sizeof(cplx) * n);
    double bnorm = sqrt(norm2(n, b));
    if (even_odd) oracle_eo_prepare(L, bc, U_, Ainv_, kappa, b_, (double *)rhs);
    else memcpy(rhs, b, sizeof(cplx) * n);
    for (long k = 0; k < n; k++) { x[k] = 0; xl[k] = 0; }
    memcpy(r, rhs, sizeof(cplx) * n);
    double rmax = sqrt(norm2(n, r));
    round_to_float(n, r);
    apply_K(&o, 1, r, s); round_to_float(n, s);
    memcpy(p, s, sizeof(cplx) * n);
    double gamma = norm2(n, s);
    int it = 0, updates = 0, status = 1;
    while (status && it < max_iter) {
        apply_K(&o, 0, p, q); round_to_float(n, q);
        double alpha = gamma / norm2(n, q);
        for (long k = 0; k < n; k++) { xl[k] += alpha * p[k]; r[k] -= alpha * q[k]; }
        round_to_float(n, xl); round_to_float(n, r);
        double rn = sqrt(norm2(n, r));
        if (resid_hist) resid_hist[it] = rn / bnorm;
        it++;
        if (rn > rmax) rmax = rn;
        if (rn < delta * rmax || rn <= tol * bnorm) {
            if (update_iters && updates < max_updates) update_iters[updates] = it;
            for (long k = 0; k < n; k++) { x[k] += xl[k]; xl[k] = 0; }
            apply_K(&o, 0, x, q);                       /* double */
            for (long k = 0; k < n; k++) r[k] = rhs[k] - q[k];
            rn = sqrt(norm2(n, r));
            rmax = rn;
            updates++;
            if (rn <= tol * bnorm) { status = 0; break; }
            round_to_float(n, r);
        }
        apply_K(&o, 1, r, s); round_to_float(n, s);
        double gamma_new = norm2(n, s);
        double beta = gamma_new / gamma;
        gamma = gamma_new;
        for (long k = 0; k < n; k++) p[k] = s[k] + beta * p[k];
        round_to_float(n, p);
    }
    if (status) for (long k = 0; k < n; k++) x[k] += xl[k];
    if (even_odd) oracle_eo_reconstruct(L, bc, U_, Ainv_, kappa, b_, x_);
    oracle_M(L, bc, U_, A_, kappa, 0, x_, (double *)q);
    for (long k = 0; k < n; k++) q[k] = b[k] - q[k];
    if (true_resid_out) *true_resid_out = sqrt(norm2(n, q)) / bnorm;
    if (iters_out) *iters_out = it;
    if (updates_out) *updates_out = updates;
    free(rhs); free(r); free(p); free(q); free(s); free(xl);
    return status;
}

/* ------------------------------------------------------------------------------------------
 * BiCGStab ("other Krylov variants (BiCGStab on S)"; "solvers for linear systems") for
 * K x = b, K = M (even_odd = 0) or K = S with b = bhat_e (even_odd = 1), in van der Vorst's order, unpreconditioned,
 * x0 = 0, shadow residual rhat = r0:
 *   rho_0 = alpha = omega_0 = 1; v_0 = p_0 = 0
 *   for i = 1, 2, ...:
 *     rho_i = <rhat, r_{i-1}>;  beta = (rho_i / rho_{i-1}) (alpha / omega_{i-1});
 *     p_i = r_{i-1} + beta (p_{i-1} - omega_{i-1} v_{i-1});   v_i = K p_i;   alpha = rho_i / <rhat, v_i>;
 *     s = r_{i-1} - alpha v_i;   t = K s;   omega_i = <t, s> / <t, t>;
 *     x_i = x_{i-1} + alpha p_i + omega_i s;   r_i = s - omega_i t;   stop if |r_i| <= tol |b_full|
 * with <a, b> = sum conj(a) b.  One pass = two applications of K.  resid_hist[i-1] = |r_i| / |b_full|.  After the loop
 * the full-lattice true residual |b - M x| / |b| is recomputed with O5, as in oracle_cgnr.
 * returns 0 if converged, 1 if max_iter was hit, 2 on breakdown (rho, <rhat, v> or <t, t> exactly 0).
 * ---------------------------------------------------------------------------------------- */
static cplx cdot(long n, const cplx *a, const cplx *b)
{
    double re = 0, im = 0;
    for (long k = 0; k < n; k++) {
        re += creal(a[k]) * creal(b[k]) + cimag(a[k]) * cimag(b[k]);
        im += creal(a[k]) * cimag(b[k]) - cimag(a[k]) * creal(b[k]);
    }
    return re + I * im;
}

int oracle_bicgstab(const int *L, const int *bc, const double *U_, const double *A_, const double *Ainv_,
                    double kappa, int even_odd, const double *b_, double *x_, double tol, int max_iter,
                    int *iters_out, double *resid_hist, double *true_resid_out)
{
    long V = vol(L), n = 12 * V;
    op_ctx_t o = {L, bc, U_, A_, Ainv_, kappa, even_odd};
    const cplx *b = (const cplx *)b_;
    cplx *x = (cplx *)x_;
    cplx *r = (cplx *)malloc(sizeof(cplx) * n), *rhat = (cplx *)malloc(sizeof(cplx) * n);
    cplx *p = (cplx *)malloc(sizeof(cplx) * n), *v = (cplx *)malloc(sizeof(cplx) * n);
    cplx *sv = (cplx *)malloc(sizeof(cplx) * n), *t = (cplx *)malloc(sizeof(cplx) * n);
    double bnorm = sqrt(norm2(n, b));
    if (even_odd) oracle_eo_prepare(L, bc, U_, Ainv_, kappa, b_, (double *)r);
    else memcpy(r, b, sizeof(cplx) * n);
    memcpy(rhat, r, sizeof(cplx) * n);
    for (long k = 0; k < n; k++) { x[k] = 0; p[k] = 0; v[k] = 0; }
    cplx rho = 1, alpha = 1, omega = 1;
    int it = 0, status = 1;
    if (sqrt(norm2(n, r)) <= tol * bnorm) status = 0;
    while (status == 1 && it < max_iter) {
        cplx rho_new = cdot(n, rhat, r);
        if (rho_new == 0) { status = 2; break; }
        cplx beta = (rho_new / rho) * (alpha / omega);
        rho = rho_new;
        for (long k = 0; k < n; k++) p[k] = r[k] + beta * (p[k] - omega * v[k]);
        apply_K(&o, 0, p, v);
        cplx rv = cdot(n, rhat, v);
        if (rv == 0) { status = 2; break; }
        alpha = rho / rv;
        for (long k = 0; k < n; k++) sv[k] = r[k] - alpha * v[k];
        apply_K(&o, 0, sv, t);
        double tt = norm2(n, t);
        if (tt == 0) { status = 2; break; }
        omega = cdot(n, t, sv) / tt;
        for (long k = 0; k < n; k++) { x[k] += alpha * p[k] + omega * sv[k]; r[k] = sv[k] - omega * t[k]; }
        double rn = sqrt(norm2(n, r));
        if (resid_hist) resid_hist[it] = rn / bnorm;
        it++;
        if (rn <= tol * bnorm) { status = 0; break; }
    }
    if (even_odd) oracle_eo_reconstruct(L, bc, U_, Ainv_, kappa, b_, x_);
    oracle_M(L, bc, U_, A_, kappa, 0, x_, (double *)t);
    for (long k = 0; k < n; k++) t[k] = b[k] - t[k];
    if (true_resid_out) *true_resid_out = sqrt(norm2(n, t)) / bnorm;
    if (iters_out) *iters_out = it;
    free(r); free(rhat); free(p); free(v); free(sv); free(t);
    return status;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
