/*
 * oracle/gvqe_oracle.c -- CPU ORACLE (tier T0) for the Graph-VQE energy hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or
 * call this file.  It shares no code, header, table or helper with the CUDA library (paper_2607_02749_b200/csrc);
 * the two see the same INPUT arrays (workload/) and nothing else.
 *
 * What it computes is the plain definition, in complex128, in the paper's order, with no fusion, tiling,
 * tables or grouping (PAPER.md = /root/reference/PAPER.md, arxiv/paper_2607_02749):
 *   state   |psi(theta)> = U(theta)|0>^{(x)N}                           PAPER.md:179 (Sec. IV-B)
 *   gates   R_y, R_z exactly as Eq. 7
 *   H       = sum_k c_k P_k, c_k real, P_k in {I,X,Y,Z}^{(x)N}            PAPER.md:148-153 (Eq. 6)
 *   E       = <psi|H|psi> = sum_k c_k <psi|P_k|psi>                      PAPER.md:135 (Eq. 4)
 *   dE/dth_i = 1/2 [E(th + pi/2 e_i) - E(th - pi/2 e_i)]                 PAPER.md:221-225 (Eq. 13)
 *   restricted objective = same E with only masked coordinates moved     PAPER.md:207-212 (Eq. 11)
 * Readings where the paper is silent: qubit q <-> bit q of the amplitude index
 * (LSB = qubit 0); character j of a Pauli string acts on qubit j; Y = [[0,-i],[i,0]];
 * CNOT stored as (kind, target, control); ops are applied in list order.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): dense Kronecker brute force n<=8, closed forms
 * (n=1 Bloch vector, product states, GHZ), invariants (norm, theta=0, basis states, |E|<=sum|c|, Eq. 12
 * additivity, sinusoid in one parameter), parameter shift vs central differences, diagonal ground energy by
 * enumeration.  Every function below is covered by at least one of them.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

enum { ORC_RY = 0, ORC_RZ = 1, ORC_CZ = 2, ORC_CNOT = 3 };

/* ---- state preparation: PAPER.md:179, gates PAPER.md:171-173 (Eq. 7) ------------------------------- */

/* ops: int32 [n_ops][4] = (kind, q0, q1, param).  RY/RZ: qubit q0, angle theta[param].
 * CZ: qubits q0,q1.  CNOT: target q0, control q1.  psi: 2^n amplitudes, overwritten. */
void orc_state(int n, const int32_t *ops, int n_ops, const double *theta, cplx *psi)
{
    const uint64_t dim = 1ull << n;
#pragma omp parallel for schedule(static)
    for (uint64_t x = 0; x < dim; ++x) psi[x] = 0.0;
    psi[0] = 1.0;                                           /* |0...0> */
    for (int o = 0; o < n_ops; ++o) {
        const int kind = ops[4 * o], q0 = ops[4 * o + 1], q1 = ops[4 * o + 2], p = ops[4 * o + 3];
        const uint64_t b0 = 1ull << q0;
        if (kind == ORC_RY) {                               /* Eq. 7: [[c,-s],[s,c]], c=cos(th/2), s=sin(th/2) */
            const double c = cos(0.5 * theta[p]), s = sin(0.5 * theta[p]);
#pragma omp parallel for schedule(static)
            for (uint64_t x = 0; x < dim; ++x) {
                if (x & b0) continue;
                const cplx a = psi[x], b = psi[x | b0];
                psi[x] = c * a - s * b;
                psi[x | b0] = s * a + c * b;
            }
        } else if (kind == ORC_RZ) {                        /* Eq. 7: diag(e^{-i th/2}, e^{+i th/2}) */
            const cplx e0 = cexp(-0.5 * I * theta[p]), e1 = cexp(0.5 * I * theta[p]);
#pragma omp parallel for schedule(static)
            for (uint64_t x = 0; x < dim; ++x) psi[x] *= (x & b0) ? e1 : e0;
        } else if (kind == ORC_CZ) {                        /* diag(1,1,1,-1) on (q0,q1) */
            const uint64_t b1 = 1ull << q1;
#pragma omp parallel for schedule(static)
            for (uint64_t x = 0; x < dim; ++x)
                if ((x & b0) && (x & b1)) psi[x] = -psi[x];
        } else if (kind == ORC_CNOT) {                      /* control q1 set: X on target q0 */
            const uint64_t bc = 1ull << q1;
#pragma omp parallel for schedule(static)
            for (uint64_t x = 0; x < dim; ++x)
                if ((x & bc) && !(x & b0)) { const cplx t = psi[x]; psi[x] = psi[x | b0]; psi[x | b0] = t; }
        }
    }
}

/* ---- Pauli string -> integers (A4: char j acts on qubit j).  Returns 0 ok, -1 bad character. -------- */
static int orc_parse(int n, const char *s, uint64_t *xm, uint64_t *zm, int *ny)
{
    *xm = 0; *zm = 0; *ny = 0;
    for (int j = 0; j < n; ++j) {
        const char ch = s[j];
        if (ch == 'I') continue;
        else if (ch == 'X') *xm |= 1ull << j;
        else if (ch == 'Z') *zm |= 1ull << j;
        else if (ch == 'Y') { *xm |= 1ull << j; *zm |= 1ull << j; ++*ny; }
        else return -1;
    }
    return 0;
}

/* <psi|P|psi> for one string, from  P|x> = i^{nY} (-1)^{popcount(x & z)} |x ^ xmask>   (Y = i X Z),
 * hence <psi|P|psi> = sum_x conj(psi[x ^ xmask]) i^{nY} (-1)^{popcount(x&z)} psi[x]. */
static cplx orc_term(int n, const cplx *psi, uint64_t xm, uint64_t zm, int ny)
{
    const uint64_t dim = 1ull << n;
    static const double pr[4] = {1, 0, -1, 0}, pi_[4] = {0, 1, 0, -1};
    const cplx iy = pr[ny & 3] + I * pi_[ny & 3];
    double sr = 0.0, si = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : sr, si)
    for (uint64_t x = 0; x < dim; ++x) {
        const double sg = (__builtin_popcountll(x & zm) & 1) ? -1.0 : 1.0;
        const cplx v = conj(psi[x ^ xm]) * (iy * sg) * psi[x];
        sr += creal(v); si += cimag(v);
    }
    return sr + I * si;
}

/* E = sum_k c_k Re<P_k>  (Eq. 4 with Eq. 6), term by term.  term_re[M] (optional) receives <P_k>;
 * *max_imag (optional) receives max_k |Im<P_k>| (must be ~0: P_k Hermitian).
 * Returns NaN on a bad Pauli character. */
double orc_energy(int n, const cplx *psi, int M, const char *paulis, const double *coeffs,
                  double *term_re, double *max_imag)
{
    double E = 0.0, mi = 0.0;
    for (int k = 0; k < M; ++k) {
        uint64_t xm, zm; int ny;
        if (orc_parse(n, paulis + (size_t)k * n, &xm, &zm, &ny)) return NAN;
        const cplx v = orc_term(n, psi, xm, zm, ny);
        if (term_re) term_re[k] = creal(v);
        if (fabs(cimag(v)) > mi) mi = fabs(cimag(v));
        E += coeffs[k] * creal(v);
    }
    if (max_imag) *max_imag = mi;
    return E;
}

/* E[b] for every row of params[B][P]  (what gvqe_energy_batch must return). */
int orc_energy_batch(int n, const int32_t *ops, int n_ops, int P, const double *params, int B,
                     int M, const char *paulis, const double *coeffs, double *E)
{
    cplx *psi = (cplx *)malloc(sizeof(cplx) << n);
    if (!psi) return -1;
    for (int b = 0; b < B; ++b) {
        orc_state(n, ops, n_ops, params + (size_t)b * P, psi);
        E[b] = orc_energy(n, psi, M, paulis, coeffs, NULL, NULL);
    }
    free(psi);
    return 0;
}

/* Eq. 13 literally: two fresh evaluations per masked parameter; dE = 0 outside the mask (Eq. 11: the
 * restricted objective moves only the block's coordinates).  E0 (optional) = E(theta). */
int orc_param_shift_grad(int n, const int32_t *ops, int n_ops, int P, const double *theta,
                         const uint8_t *mask, int M, const char *paulis, const double *coeffs,
                         double *dE, double *E0)
{
    cplx *psi = (cplx *)malloc(sizeof(cplx) << n);
    double *th = (double *)malloc(sizeof(double) * (size_t)(P > 0 ? P : 1));
    if (!psi || !th) { free(psi); free(th); return -1; }
    memcpy(th, theta, sizeof(double) * (size_t)P);
    if (E0) { orc_state(n, ops, n_ops, th, psi); *E0 = orc_energy(n, psi, M, paulis, coeffs, NULL, NULL); }
    for (int p = 0; p < P; ++p) {
        dE[p] = 0.0;
        if (!mask[p]) continue;
        th[p] = theta[p] + M_PI / 2;
        orc_state(n, ops, n_ops, th, psi);
        const double ep = orc_energy(n, psi, M, paulis, coeffs, NULL, NULL);
        th[p] = theta[p] - M_PI / 2;
        orc_state(n, ops, n_ops, th, psi);
        const double em = orc_energy(n, psi, M, paulis, coeffs, NULL, NULL);
        th[p] = theta[p];
        dE[p] = 0.5 * (ep - em);
    }
    free(psi); free(th);
    return 0;
}

/* ---- integer side of "Hamiltonian batching" re-read as flip-mask grouping (reading A10) ----
 * per term (x_mask, z_mask, n_Y mod 4); groups = distinct x_mask values in ascending unsigned order;
 * group_of_term[k] = rank of x_mask_k.  Compared with gvqe_get_grouping by memcmp.  Deliberately naive
 * (insertion into a sorted list), nothing shared with the library's routine. */
int orc_grouping(int n, int M, const char *paulis, uint64_t *x_mask, uint64_t *z_mask, uint8_t *ny_mod4,
                 int32_t *group_of_term, int32_t *n_groups, uint64_t *group_mask)
{
    int ng = 0;
    for (int k = 0; k < M; ++k) {
        int ny;
        if (orc_parse(n, paulis + (size_t)k * n, &x_mask[k], &z_mask[k], &ny)) return -1;
        ny_mod4[k] = (uint8_t)(ny & 3);
        int lo = 0;
        while (lo < ng && group_mask[lo] < x_mask[k]) ++lo;
        if (lo == ng || group_mask[lo] != x_mask[k]) {
            memmove(group_mask + lo + 1, group_mask + lo, sizeof(uint64_t) * (size_t)(ng - lo));
            group_mask[lo] = x_mask[k];
            ++ng;
        }
    }
    for (int k = 0; k < M; ++k) {
        int g = 0;
        while (group_mask[g] != x_mask[k]) ++g;
        group_of_term[k] = g;
    }
    *n_groups = ng;
    return 0;
}

double orc_norm2(int n, const cplx *psi)
{
    const uint64_t dim = 1ull << n;
    double s = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : s)
    for (uint64_t x = 0; x < dim; ++x) s += creal(psi[x]) * creal(psi[x]) + cimag(psi[x]) * cimag(psi[x]);
    return s;
}
