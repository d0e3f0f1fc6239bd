/*
 * gen.c -- seeded synthetic input generators shared by the tests, the oracle legs and bench.py.
 *
 * This module holds NONE of the method's arithmetic (no gamma matrices, no hopping term, no
 * representation map): only random numbers and random SU(N) matrices in the canonical layout
 *   links  [site i][mu][row][col] complex double,   spinors [site][spin][colour] complex double.
 * Recipes (BASELINE.json:configs, readings C16/C17 in DESIGN.md):
 *   - spinor components: i.i.d. unit Gaussian real and imaginary parts;
 *   - Haar SU(N): Z complex Ginibre (re, im ~ N(0,1)), Z = QR by Gram-Schmidt with positive diagonal R
 *     (this Q is Haar on U(N)), then U = Q * det(Q)^(-1/N) with the principal root;
 *   - near-identity SU(N): G Ginibre, H = (G + G^dagger)/2 - tr/N, U = exp(i eps H) by scaling and
 *     squaring of the Taylor series.
 * Random numbers: counter-based Philox4x32-10 (Salmon et al., SC'11), key = seed, counter = (element
 * index, stream), so any chunk of a field can be produced independently and the result does not
 * depend on the number of threads.  Normals by Box-Muller from two 32-bit-pair uniforms.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

static inline void philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1)
{
    for (int r = 0; r < 10; r++) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
}

/* two independent N(0,1) for (seed, stream, pair index) */
static inline void normal_pair(uint64_t seed, uint32_t stream, uint64_t pair, double *a, double *b)
{
    uint32_t c[4] = { (uint32_t)pair, (uint32_t)(pair >> 32), stream, 0x5eedu };
    philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
    uint64_t u0 = ((uint64_t)c[0] << 32) | c[1];
    uint64_t u1 = ((uint64_t)c[2] << 32) | c[3];
    double x0 = ((double)(u0 >> 11) + 0.5) * (1.0 / 9007199254740992.0); /* (0,1) */
    double x1 = ((double)(u1 >> 11) + 0.5) * (1.0 / 9007199254740992.0);
    double r = sqrt(-2.0 * log(x0));
    double th = 6.283185307179586476925286766559 * x1;
    *a = r * cos(th);
    *b = r * sin(th);
}

/* out[j] = complex unit Gaussian number `first + j` of stream `stream` */
void gen_gaussian_complex(uint64_t seed, uint32_t stream, int64_t first, int64_t count, cplx *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < count; j++) {
        double a, b;
        normal_pair(seed, stream, (uint64_t)(first + j), &a, &b);
        out[j] = a + I * b;
    }
}

static void ginibre(uint64_t seed, uint32_t stream, uint64_t mat, int N, cplx *Z)
{
    for (int e = 0; e < N * N; e++) {
        double a, b;
        normal_pair(seed, stream, mat * (uint64_t)(N * N) + (uint64_t)e, &a, &b);
        Z[e] = a + I * b;
    }
}

static cplx determinant(int N, const cplx *A)
{
    cplx M[64];
    memcpy(M, A, (size_t)N * N * sizeof(cplx));
    cplx det = 1;
    for (int k = 0; k < N; k++) {
        int piv = k; double best = cabs(M[k * N + k]);
        for (int r = k + 1; r < N; r++) if (cabs(M[r * N + k]) > best) { best = cabs(M[r * N + k]); piv = r; }
        if (piv != k) {
            for (int c = 0; c < N; c++) { cplx t = M[k * N + c]; M[k * N + c] = M[piv * N + c]; M[piv * N + c] = t; }
            det = -det;
        }
        det *= M[k * N + k];
        for (int r = k + 1; r < N; r++) {
            cplx f = M[r * N + k] / M[k * N + k];
            for (int c = k; c < N; c++) M[r * N + c] -= f * M[k * N + c];
        }
    }
    return det;
}

/* Haar SU(N) matrix number `mat` of stream `stream` */
static void haar_sun(uint64_t seed, uint32_t stream, uint64_t mat, int N, cplx *U)
{
    cplx Z[64];
    ginibre(seed, stream, mat, N, Z);
    /* modified Gram-Schmidt on the columns, twice for orthogonality to rounding */
    for (int pass = 0; pass < 2; pass++)
        for (int j = 0; j < N; j++) {
            for (int k = 0; k < j; k++) {
                cplx dot = 0;
                for (int r = 0; r < N; r++) dot += conj(Z[r * N + k]) * Z[r * N + j];
                for (int r = 0; r < N; r++) Z[r * N + j] -= dot * Z[r * N + k];
            }
            double nrm = 0;
            for (int r = 0; r < N; r++) nrm += creal(Z[r * N + j]) * creal(Z[r * N + j]) + cimag(Z[r * N + j]) * cimag(Z[r * N + j]);
            nrm = sqrt(nrm);
            for (int r = 0; r < N; r++) Z[r * N + j] /= nrm;
        }
    cplx det = determinant(N, Z);
    cplx ph = cexp(-I * carg(det) / N) * pow(cabs(det), -1.0 / N);
    for (int e = 0; e < N * N; e++) U[e] = Z[e] * ph;
}

static void matmul(int N, const cplx *A, const cplx *B, cplx *C)
{
    for (int i = 0; i < N; i++) for (int j = 0; j < N; j++) {
        cplx s = 0;
        for (int k = 0; k < N; k++) s += A[i * N + k] * B[k * N + j];
        C[i * N + j] = s;
    }
}

/* U = exp(i eps H), H = (G + G^dagger)/2 - tr/N */
static void near_identity_sun(uint64_t seed, uint32_t stream, uint64_t mat, int N, double eps, cplx *U)
{
    cplx G[64], A[64], T[64], S[64], W[64];
    ginibre(seed, stream, mat, N, G);
    cplx tr = 0;
    for (int i = 0; i < N; i++) for (int j = 0; j < N; j++) A[i * N + j] = 0.5 * (G[i * N + j] + conj(G[j * N + i]));
    for (int i = 0; i < N; i++) tr += A[i * N + i];
    for (int i = 0; i < N; i++) A[i * N + i] -= tr / N;
    const int squarings = 6;
    const double scale = eps / 64.0;
    for (int e = 0; e < N * N; e++) A[e] = I * scale * A[e];
    /* S = sum_{k=0}^{16} A^k / k! */
    memset(S, 0, sizeof S); memset(T, 0, sizeof T);
    for (int i = 0; i < N; i++) { S[i * N + i] = 1; T[i * N + i] = 1; }
    for (int k = 1; k <= 16; k++) {
        matmul(N, T, A, W);
        for (int e = 0; e < N * N; e++) { T[e] = W[e] / k; S[e] += T[e]; }
    }
    for (int s = 0; s < squarings; s++) { matmul(N, S, S, W); memcpy(S, W, (size_t)N * N * sizeof(cplx)); }
    memcpy(U, S, (size_t)N * N * sizeof(cplx));
}

/* kind: 0 = Haar, 1 = near identity exp(i eps H).  Matrices `first .. first+count-1` of `stream`. */
int gen_sun(uint64_t seed, uint32_t stream, int kind, double eps, int N, int64_t first, int64_t count, cplx *out)
{
    if (N < 1 || N > 8) return -1;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < count; m++) {
        cplx *U = out + (size_t)m * N * N;
        if (kind == 0) haar_sun(seed, stream, (uint64_t)(first + m), N, U);
        else near_identity_sun(seed, stream, (uint64_t)(first + m), N, eps, U);
    }
    return 0;
}
