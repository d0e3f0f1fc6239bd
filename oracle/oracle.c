/*
 * oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the hot path computes: the hopping term Dphi of the
 * Wilson-Dirac operator for fermions in a representation R of SU(N), its even-odd restriction, the
 * full operator D = (4+m0) + Dphi, and the link map U -> U^R.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code, header, table or helper with the CUDA path (paper_2405_19294_b200/).
 *
 * Authority for each function:
 *   - operator:  BASELINE.json:north_star
 *                  out(x) = -1/2 sum_mu [ (1-gamma_mu) U^R_mu(x) psi(x+mu)
 *                                       + (1+gamma_mu) U^R_mu(x-mu)^dagger psi(x-mu) ],
 *                  D = (4+m0) + Dphi;  PAPER.md:70 (section 3.1: Wilson-Dirac operator, any SU(N_c),
 *                  any representation, even-odd), PAPER.md:90 (represented link is d_R x d_R).
 *   - conventions the paper is silent on: SURVEY.md section 8(c) readings C1..C12 (restated in
 *     DESIGN.md "Readings").
 *   - link map:  BASELINE.json:north_star / configs[2]: U^adj_ab = 2 tr(T_a U T_b U^dagger);
 *                configs[3]: two-index symmetric rep on the symmetric tensor basis (reading C8:
 *                R_ab = tr[(e_a)^dagger U e_b U^T]).
 *
 * The algorithm is deliberately the definition written out: full 4x4 gamma tables, the colour
 * matrix-vector product for all four spin components, explicit coordinate wrap and boundary sign,
 * trace definitions with explicit basis matrices for the representations.  No half-spinor trick,
 * no layout tricks, no blocking.  (OpenMP over output sites only.)
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Clifford algebra + printed gamma tables
 * (tests/golden/gamma_chiral.txt), free-field plane waves in closed form on a 4x2x6x8 lattice at
 * every momentum, gamma5-hermiticity, gauge covariance in every representation, brute-force dense
 * Kronecker assembly (oracle/dense.py, numpy) on 2^4 / 4.2^3 / 2^3.4, zero even-even/odd-odd blocks,
 * homomorphism / unitarity / characters / textbook special cases of the representation maps.
 * Pure conventions (basis ordering C4/C6/C8) are "parity unpinned by physics": fixed only through
 * the canonical layout shared with the CUDA path at the C-ABI boundary.
 *
 * Canonical layouts (reading C4):
 *   full-lattice site index i = ((t*X + x)*Y + y)*Z + z,  dims = {T,X,Y,Z}, mu = 0..3 = t,x,y,z
 *   parity(i) = (t+x+y+z) & 1;  a parity-p half field lists parity-p sites by increasing i
 *   (half index = i>>1 since Z is even);  an "eo full field" is [even half | odd half].
 *   spinor site: [spin alpha 0..3][colour a 0..d-1] complex;  link: [site i][mu][row][col] complex.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

enum { REP_FUND = 0, REP_ADJ = 1, REP_SYM = 2, REP_ASYM = 3 };

/* ------------------------------------------------------------------------------------------ */
/* gamma matrices, reading C1 (Hermitian chiral basis, mu = 0 is time)                         */
/* ------------------------------------------------------------------------------------------ */
static void gamma_table(int mu, cplx g[4][4])
{
    memset(g, 0, 16 * sizeof(cplx));
    switch (mu) {
    case 0:
        g[0][2] = -1; g[1][3] = -1; g[2][0] = -1; g[3][1] = -1;
        break;
    case 1:
        g[0][3] = -I; g[1][2] = -I; g[2][1] = I; g[3][0] = I;
        break;
    case 2:
        g[0][3] = -1; g[1][2] = 1; g[2][1] = 1; g[3][0] = -1;
        break;
    case 3:
        g[0][2] = -I; g[1][3] = I; g[2][0] = I; g[3][1] = -I;
        break;
    case 5: { /* gamma5 = gamma0 gamma1 gamma2 gamma3, computed, not typed in */
        cplx a[4][4], b[4][4], c[4][4], d[4][4], ab[4][4], abc[4][4];
        gamma_table(0, a); gamma_table(1, b); gamma_table(2, c); gamma_table(3, d);
        for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) {
            ab[i][j] = 0; for (int k = 0; k < 4; k++) ab[i][j] += a[i][k] * b[k][j]; }
        for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) {
            abc[i][j] = 0; for (int k = 0; k < 4; k++) abc[i][j] += ab[i][k] * c[k][j]; }
        for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) {
            g[i][j] = 0; for (int k = 0; k < 4; k++) g[i][j] += abc[i][k] * d[k][j]; }
        break; }
    default: break;
    }
}

void oracle_gamma(int mu, cplx *out16)
{
    cplx g[4][4];
    gamma_table(mu, g);
    memcpy(out16, g, sizeof g);
}

/* ------------------------------------------------------------------------------------------ */
/* representation maps from their trace definitions (readings C6, C7, C8)                      */
/* ------------------------------------------------------------------------------------------ */
int oracle_rep_dim(int N, int rep)
{
    switch (rep) {
    case REP_FUND: return N;
    case REP_ADJ:  return N * N - 1;
    case REP_SYM:  return N * (N + 1) / 2;
    case REP_ASYM: return N * (N - 1) / 2;
    }
    return -1;
}

/* generalised Gell-Mann matrices lambda_a (tr lambda^2 = 2), nested order (C6):
 * for m = 1..N-1: { for i < m: S_im, A_im } then the diagonal D_m.  Returns count. */
static int gellmann_basis(int N, cplx *lam /* [N*N-1][N][N] */)
{
    int a = 0;
    memset(lam, 0, (size_t)(N * N - 1) * N * N * sizeof(cplx));
    for (int m = 1; m < N; m++) {
        for (int i = 0; i < m; i++) {
            cplx *S = lam + (size_t)a * N * N; a++;
            S[i * N + m] = 1; S[m * N + i] = 1;
            cplx *A = lam + (size_t)a * N * N; a++;
            A[i * N + m] = -I; A[m * N + i] = I;
        }
        cplx *D = lam + (size_t)a * N * N; a++;
        double c = sqrt(2.0 / (m * (m + 1.0)));
        for (int k = 0; k < m; k++) D[k * N + k] = c;
        D[m * N + m] = -c * m;
    }
    return a;
}

/* two-index basis matrices e^(ij) (C8): pairs lexicographic with i<=j (sym) or i<j (asym);
 * e^(ii) = E_ii, e^(ij) = (E_ij +- E_ji)/sqrt2.  Returns count. */
static int twoindex_basis(int N, int sign, cplx *e /* [dim][N][N] */)
{
    int a = 0;
    for (int i = 0; i < N; i++)
        for (int j = i; j < N; j++) {
            if (i == j && sign < 0) continue;
            cplx *m = e + (size_t)a * N * N; a++;
            memset(m, 0, (size_t)N * N * sizeof(cplx));
            if (i == j) m[i * N + i] = 1;
            else { m[i * N + j] = 1.0 / sqrt(2.0); m[j * N + i] = sign / sqrt(2.0); }
        }
    return a;
}

static void matmul(int N, const cplx *A, const cplx *B, cplx *C)
{
    for (int i = 0; i < N; i++)
        for (int j = 0; j < N; j++) {
            cplx s = 0;
            for (int k = 0; k < N; k++) s += A[i * N + k] * B[k * N + j];
            C[i * N + j] = s;
        }
}

static cplx trace_prod(int N, const cplx *A, const cplx *B) /* tr(A B) */
{
    cplx s = 0;
    for (int i = 0; i < N; i++) for (int k = 0; k < N; k++) s += A[i * N + k] * B[k * N + i];
    return s;
}

/* One link.  U: N x N row-major.  R: d x d row-major complex (for the adjoint the imaginary parts are
 * rounding-level; *max_imag (if not NULL) is raised to max |Im R_ab| so the caller can assert C7). */
int oracle_represent(int N, int rep, const cplx *U, cplx *R, double *max_imag)
{
    int d = oracle_rep_dim(N, rep);
    if (d <= 0 || N < 2 || N > 8) return -1;
    cplx Ud[64], Ut[64], tmp1[64], tmp2[64];
    for (int i = 0; i < N; i++) for (int j = 0; j < N; j++) {
        Ud[i * N + j] = conj(U[j * N + i]);
        Ut[i * N + j] = U[j * N + i];
    }
    if (rep == REP_FUND) {
        memcpy(R, U, (size_t)N * N * sizeof(cplx));
        return d;
    }
    if (rep == REP_ADJ) {
        /* R_ab = 2 tr(T_a U T_b U^dagger), T = lambda/2  =>  R_ab = 1/2 tr(lambda_a U lambda_b U^dagger) */
        cplx *lam = malloc((size_t)d * N * N * sizeof(cplx));
        gellmann_basis(N, lam);
        for (int b = 0; b < d; b++) {
            matmul(N, U, lam + (size_t)b * N * N, tmp1);      /* U lambda_b */
            matmul(N, tmp1, Ud, tmp2);                          /* U lambda_b U^dagger */
            for (int a = 0; a < d; a++) {
                cplx r = 0.5 * trace_prod(N, lam + (size_t)a * N * N, tmp2);
                R[a * d + b] = r;
                if (max_imag && fabs(cimag(r)) > *max_imag) *max_imag = fabs(cimag(r));
            }
        }
        free(lam);
        return d;
    }
    /* two-index: R_ab = tr[(e_a)^dagger U e_b U^T] */
    int sign = (rep == REP_SYM) ? +1 : -1;
    cplx *e = malloc((size_t)d * N * N * sizeof(cplx));
    twoindex_basis(N, sign, e);
    for (int b = 0; b < d; b++) {
        matmul(N, U, e + (size_t)b * N * N, tmp1);              /* U e_b */
        matmul(N, tmp1, Ut, tmp2);                              /* U e_b U^T */
        for (int a = 0; a < d; a++) {
            cplx ead[64];
            const cplx *ea = e + (size_t)a * N * N;
            for (int i = 0; i < N; i++) for (int j = 0; j < N; j++) ead[i * N + j] = conj(ea[j * N + i]);
            R[a * d + b] = trace_prod(N, ead, tmp2);
        }
    }
    free(e);
    return d;
}

/* Whole field: nlinks consecutive links.  Returns max |Im| seen (adjoint), 0 otherwise, <0 on error. */
double oracle_represent_field(int N, int rep, long nlinks, const cplx *U, cplx *R)
{
    int d = oracle_rep_dim(N, rep);
    if (d <= 0) return -1.0;
    double worst = 0.0;
#pragma omp parallel for reduction(max : worst) schedule(static)
    for (long l = 0; l < nlinks; l++) {
        double mi = 0.0;
        oracle_represent(N, rep, U + (size_t)l * N * N, R + (size_t)l * d * d, &mi);
        if (mi > worst) worst = mi;
    }
    return worst;
}

/* ------------------------------------------------------------------------------------------ */
/* the hopping term at one site, straight from the definition                                   */
/* ------------------------------------------------------------------------------------------ */
enum { PSI_LEX = 0,   /* psi[i] for every full-lattice site i (lexicographic)                 */
       PSI_HALF = 1,  /* psi holds ONE parity; site i lives at i>>1 (caller guarantees parity)  */
       PSI_EO = 2 };  /* psi = [even half | odd half]; site i lives at parity(i)*V/2 + (i>>1)    */

typedef struct {
    int dims[4];
    int bc[4];
    int d;
    long V;
    const cplx *links; /* [V][4][d][d] represented links, canonical */
    const cplx *psi;
    int psi_mode;
    cplx P[4][2][4][4]; /* P[mu][0] = 1 - gamma_mu, P[mu][1] = 1 + gamma_mu */
} dphi_ctx;

static void ctx_init(dphi_ctx *c, const int *dims, const int *bc, int d, const cplx *links,
                     const cplx *psi, int psi_mode)
{
    for (int m = 0; m < 4; m++) { c->dims[m] = dims[m]; c->bc[m] = bc[m]; }
    c->d = d;
    c->V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    c->links = links; c->psi = psi; c->psi_mode = psi_mode;
    for (int mu = 0; mu < 4; mu++) {
        cplx g[4][4];
        gamma_table(mu, g);
        for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) {
            cplx one = (a == b) ? 1.0 : 0.0;
            c->P[mu][0][a][b] = one - g[a][b];
            c->P[mu][1][a][b] = one + g[a][b];
        }
    }
}

static long site_index(const int *dims, const int *x)
{
    return (((long)x[0] * dims[1] + x[1]) * dims[2] + x[2]) * dims[3] + x[3];
}

static void site_coords(const int *dims, long i, int *x)
{
    x[3] = (int)(i % dims[3]); i /= dims[3];
    x[2] = (int)(i % dims[2]); i /= dims[2];
    x[1] = (int)(i % dims[1]); i /= dims[1];
    x[0] = (int)i;
}

static const cplx *psi_at(const dphi_ctx *c, long i, const int *x)
{
    size_t per = (size_t)4 * c->d;
    switch (c->psi_mode) {
    case PSI_LEX:  return c->psi + (size_t)i * per;
    case PSI_HALF: return c->psi + (size_t)(i >> 1) * per;
    default: {
        int par = (x[0] + x[1] + x[2] + x[3]) & 1;
        return c->psi + ((size_t)par * (size_t)(c->V / 2) + (size_t)(i >> 1)) * per; }
    }
}

/* out[4*d] = Dphi psi (x), x given by coordinates */
static void dphi_site(const dphi_ctx *c, const int *x, cplx *out)
{
    const int d = c->d;
    cplx acc[4 * 64]; /* 4*d, d <= 64 is far more than ever used */
    cplx w[4 * 64];
    for (int k = 0; k < 4 * d; k++) acc[k] = 0;
    long ix = site_index(c->dims, x);
    for (int mu = 0; mu < 4; mu++) {
        const int L = c->dims[mu];
        /* forward hop: (1 - gamma_mu) * sigma+ * U_mu(x) * psi(x + mu) */
        {
            int y[4] = { x[0], x[1], x[2], x[3] };
            y[mu] = (x[mu] + 1) % L;
            double sgn = (x[mu] == L - 1) ? (double)c->bc[mu] : 1.0;
            long iy = site_index(c->dims, y);
            const cplx *U = c->links + ((size_t)ix * 4 + mu) * d * d;
            const cplx *p = psi_at(c, iy, y);
            for (int be = 0; be < 4; be++)           /* w_be = U psi_be  (colour mat-vec) */
                for (int a = 0; a < d; a++) {
                    cplx s = 0;
                    for (int b = 0; b < d; b++) s += U[a * d + b] * p[be * d + b];
                    w[be * d + a] = s;
                }
            for (int al = 0; al < 4; al++)
                for (int be = 0; be < 4; be++) {
                    cplx g = c->P[mu][0][al][be];
                    for (int a = 0; a < d; a++) acc[al * d + a] += sgn * g * w[be * d + a];
                }
        }
        /* backward hop: (1 + gamma_mu) * sigma- * U_mu(x - mu)^dagger * psi(x - mu) */
        {
            int y[4] = { x[0], x[1], x[2], x[3] };
            y[mu] = (x[mu] - 1 + L) % L;
            double sgn = (x[mu] == 0) ? (double)c->bc[mu] : 1.0;
            long iy = site_index(c->dims, y);
            const cplx *U = c->links + ((size_t)iy * 4 + mu) * d * d;
            const cplx *p = psi_at(c, iy, y);
            for (int be = 0; be < 4; be++)           /* w_be = U^dagger psi_be */
                for (int a = 0; a < d; a++) {
                    cplx s = 0;
                    for (int b = 0; b < d; b++) s += conj(U[b * d + a]) * p[be * d + b];
                    w[be * d + a] = s;
                }
            for (int al = 0; al < 4; al++)
                for (int be = 0; be < 4; be++) {
                    cplx g = c->P[mu][1][al][be];
                    for (int a = 0; a < d; a++) acc[al * d + a] += sgn * g * w[be * d + a];
                }
        }
    }
    for (int k = 0; k < 4 * d; k++) out[k] = -0.5 * acc[k];
}

/* ------------------------------------------------------------------------------------------ */
/* public entry points                                                                         */
/* ------------------------------------------------------------------------------------------ */
static int check_dims(const int *dims, const int *bc, int d)
{
    if (d < 1 || d > 64) return -1;
    for (int m = 0; m < 4; m++) {
        if (dims[m] < 2 || (dims[m] & 1)) return -1;   /* reading C11 */
        if (bc[m] != 1 && bc[m] != -1) return -1;
    }
    return 0;
}

/* Dphi on every site; psi and out are lexicographic full-lattice fields [V][4][d]. */
int oracle_dphi_lex(const int *dims, const int *bc, int d, const cplx *links, const cplx *psi, cplx *out)
{
    if (check_dims(dims, bc, d)) return -1;
    dphi_ctx c; ctx_init(&c, dims, bc, d, links, psi, PSI_LEX);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < c.V; i++) {
        int x[4]; site_coords(dims, i, x);
        dphi_site(&c, x, out + (size_t)i * 4 * d);
    }
    return 0;
}

/* Dphi_eo: out on the parity-`parity` sites (half field), psi_half given on parity 1-parity. */
int oracle_dphi_eo(const int *dims, const int *bc, int d, const cplx *links, int parity,
                   const cplx *psi_half, cplx *out_half)
{
    if (check_dims(dims, bc, d) || (parity != 0 && parity != 1)) return -1;
    dphi_ctx c; ctx_init(&c, dims, bc, d, links, psi_half, PSI_HALF);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < c.V; i++) {
        int x[4]; site_coords(dims, i, x);
        if (((x[0] + x[1] + x[2] + x[3]) & 1) != parity) continue;
        dphi_site(&c, x, out_half + (size_t)(i >> 1) * 4 * d);
    }
    return 0;
}

/* Same, for a list of output sites given by their half index h (site = the parity-`parity` site with
 * i>>1 == h).  out is [nsites][4][d].  Used for sampled parity at full benchmark volumes. */
int oracle_dphi_eo_sites(const int *dims, const int *bc, int d, const cplx *links, int parity,
                         const cplx *psi_half, long nsites, const long *half_index, cplx *out)
{
    if (check_dims(dims, bc, d) || (parity != 0 && parity != 1)) return -1;
    dphi_ctx c; ctx_init(&c, dims, bc, d, links, psi_half, PSI_HALF);
#pragma omp parallel for schedule(static)
    for (long n = 0; n < nsites; n++) {
        long i0 = 2 * half_index[n];
        int x[4]; site_coords(dims, i0, x);
        if (((x[0] + x[1] + x[2] + x[3]) & 1) != parity) { x[3] += 1; }
        dphi_site(&c, x, out + (size_t)n * 4 * d);
    }
    return 0;
}

/* D = (4+m0) + Dphi on eo full fields [even half | odd half]. */
int oracle_dirac(const int *dims, const int *bc, int d, const cplx *links, double m0,
                 const cplx *psi_eo, cplx *out_eo)
{
    if (check_dims(dims, bc, d)) return -1;
    dphi_ctx c; ctx_init(&c, dims, bc, d, links, psi_eo, PSI_EO);
    const size_t per = (size_t)4 * d;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < c.V; i++) {
        int x[4]; site_coords(dims, i, x);
        int par = (x[0] + x[1] + x[2] + x[3]) & 1;
        size_t pos = ((size_t)par * (size_t)(c.V / 2) + (size_t)(i >> 1)) * per;
        cplx hop[4 * 64];
        dphi_site(&c, x, hop);
        for (size_t k = 0; k < per; k++) out_eo[pos + k] = (4.0 + m0) * psi_eo[pos + k] + hop[k];
    }
    return 0;
}

int oracle_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}
