/*
 * oracle/gvqe_oracle_t1.c -- CPU ORACLE tier T1 (second plain evaluator).  TEST INFRASTRUCTURE ONLY.
 *
 * T0 (gvqe_oracle.c) costs M * 2^n per energy, impractical for n >= 26 with M ~ 2*10^4.  T1 evaluates the
 * same number, Eq. 4 with Eq. 6, from two textbook identities, in complex128/float64:
 *   (i)  terms with no X/Y:  sum_k c_k (-1)^{popcount(x & z_k)}  for all x at once is the Walsh-Hadamard
 *        transform of the vector that holds c_k at index z_k; then E_Z = sum_x |psi[x]|^2 T[x];
 *   (ii) the remaining terms are summed flip mask by flip mask (Eq. 12: energies of any
 *        partition of the terms add), each term with its own sign loop.
 * T1 is NOT trusted on its own: tests/test_oracle_pins.py requires T1 == T0 to 1e-11 on configs 1-3-like
 * cases and on random Hamiltonians before T1 is used for n >= 26 checks.  Shares nothing with the CUDA path.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

static int t1_parse(int n, const char *s, uint64_t *xm, uint64_t *zm, int *ny)
{
    *xm = 0; *zm = 0; *ny = 0;
    for (int j = 0; j < n; ++j) {
        switch (s[j]) {
        case 'I': break;
        case 'X': *xm |= 1ull << j; break;
        case 'Z': *zm |= 1ull << j; break;
        case 'Y': *xm |= 1ull << j; *zm |= 1ull << j; ++*ny; break;
        default: return -1;
        }
    }
    return 0;
}

/* T[x] = sum_{k: x_mask_k = 0} c_k (-1)^{popcount(x & z_k)}; table: 2^n doubles (caller-owned). */
int orc_t1_diag_table(int n, int M, const char *paulis, const double *coeffs, double *table)
{
    const uint64_t dim = 1ull << n;
    memset(table, 0, sizeof(double) * dim);
    for (int k = 0; k < M; ++k) {
        uint64_t xm, zm; int ny;
        if (t1_parse(n, paulis + (size_t)k * n, &xm, &zm, &ny)) return -1;
        if (xm == 0) table[zm] += coeffs[k];
    }
    for (int q = 0; q < n; ++q) {                       /* in-place Walsh-Hadamard butterflies */
        const uint64_t b = 1ull << q;
#pragma omp parallel for schedule(static)
        for (uint64_t x = 0; x < dim; ++x) {
            if (x & b) continue;
            const double u = table[x], v = table[x | b];
            table[x] = u + v; table[x | b] = u - v;
        }
    }
    return 0;
}

/* E = sum_x |psi|^2 T[x]  +  sum over X/Y terms (mask by mask).  table may be NULL (built internally). */
double orc_t1_energy(int n, const cplx *psi, int M, const char *paulis, const double *coeffs, const double *table_in)
{
    const uint64_t dim = 1ull << n;
    double *table = (double *)table_in;
    if (!table) {
        table = (double *)malloc(sizeof(double) * dim);
        if (!table || orc_t1_diag_table(n, M, paulis, coeffs, table)) { free(table); return NAN; }
    }
    double E = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : E)
    for (uint64_t x = 0; x < dim; ++x)
        E += (creal(psi[x]) * creal(psi[x]) + cimag(psi[x]) * cimag(psi[x])) * table[x];
    if (!table_in) free(table);

    static const double pr[4] = {1, 0, -1, 0}, pi_[4] = {0, 1, 0, -1};
    for (int k = 0; k < M; ++k) {
        uint64_t xm, zm; int ny;
        if (t1_parse(n, paulis + (size_t)k * n, &xm, &zm, &ny)) return NAN;
        if (xm == 0) continue;
        const cplx ph = pr[ny & 3] + I * pi_[ny & 3];
        double s = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : s)
        for (uint64_t x = 0; x < dim; ++x) {
            const double sg = (__builtin_popcountll(x & zm) & 1) ? -1.0 : 1.0;
            s += sg * creal(conj(psi[x ^ xm]) * ph * psi[x]);
        }
        E += coeffs[k] * s;
    }
    return E;
}
