/*
 * qmc_oracle.c -- CPU ORACLE for the batched Slater-Jastrow electron move.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or helper with the CUDA path (paper_2504_07948_b200/csrc); the only thing both
 * sides consume is the seeded input data made by qmc_inputs/.
 *
 * What it is: a plain, slow, step-by-step FP64 (or long double with -DORACLE_LONG_DOUBLE)
 * restatement of the method, in the paper's order and notation:
 *   - trial function  Psi = exp(J) * D_up * D_dn, phi_j = sum_l C_lj Phi_l       PAPER.md L125-127 (eq. 2)
 *   - Slater matrix   A_pj = phi_j(r_p), inverse A^-1
 *   - log-derivative  d ln D / d lambda = tr(A^-1 dA/d lambda)                    PAPER.md L173 (eq. 3)
 *   - fixed-node rejection of sign-changing moves
 *   - everything the paper leaves open (basis functional form, Pade Jastrow, drift-diffusion
 *     proposal, Philox stream, Sherman-Morrison / delayed update, local energy) follows
 *     BASELINE.json north_star + configs and the readings A1-A27 of SURVEY.md 8(c), each listed
 *     in DESIGN.md.
 * There is no blocking, fusion, screening or reordering beyond those definitions.  Sums run in
 * ascending index order.  One library primitive is used: libm exp/log/sqrt/sin/cos.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors; basis
 * derivatives vs finite differences and closed forms; unit self-overlap by quadrature; LU inverse
 * and determinant ratios vs numpy.linalg; Sherman-Morrison and delayed rank-k vs direct inverse;
 * Jastrow vs finite differences; hydrogen 1s E_L = -1/2; antisymmetry; eq. (3) by finite
 * differences; reverse-move symmetry of the acceptance; running log|Psi| vs from-scratch.
 * WHOLE TRAJECTORIES: parity unpinned by the paper (it prints no worked example); they are pinned
 * only through the invariants above.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORACLE_LONG_DOUBLE
typedef long double real;
#define R_EXP expl
#define R_LOG logl
#define R_SQRT sqrtl
#define R_COS cosl
#define R_SIN sinl
#define R_FABS fabsl
#else
typedef double real;
#define R_EXP exp
#define R_LOG log
#define R_SQRT sqrt
#define R_COS cos
#define R_SIN sin
#define R_FABS fabs
#endif

#define SQRT3 ((real)1.7320508075688772935274463415058723669428L)
#define TWO_PI ((real)6.283185307179586476925286766559005768394L)

/* ------------------------------------------------------------------ system */

typedef struct {
    int n_atoms;
    real *xyz; /* [n_atoms][3] */
    real *Z;
    int n_shells;
    int *sh_atom, *sh_l, *sh_nprim, *sh_off;
    real *alpha, *coef;
    int n_basis, n_up, n_dn;
    real *C[2]; /* [n_basis][n_s] row-major */
    real a_anti, a_para, b_ee, b_en;
} oracle_system;

static real *dup_real(const double *src, size_t n) {
    real *p = (real *)malloc((n ? n : 1) * sizeof(real));
    for (size_t i = 0; i < n; i++) p[i] = (real)src[i];
    return p;
}
static int *dup_int(const int *src, size_t n) {
    int *p = (int *)malloc((n ? n : 1) * sizeof(int));
    memcpy(p, src, n * sizeof(int));
    return p;
}

int oracle_real_bytes(void) { return (int)sizeof(real); }

oracle_system *oracle_system_create(int n_atoms, const double *xyz, const double *Z, int n_shells,
                                    const int *sh_atom, const int *sh_l, const int *sh_nprim,
                                    const int *sh_off, int n_prim_total, const double *alpha,
                                    const double *coef, int n_basis, int n_up, int n_dn,
                                    const double *C_up, const double *C_dn, double a_anti,
                                    double a_para, double b_ee, double b_en) {
    oracle_system *s = (oracle_system *)calloc(1, sizeof(*s));
    s->n_atoms = n_atoms;
    s->xyz = dup_real(xyz, (size_t)3 * n_atoms);
    s->Z = dup_real(Z, n_atoms);
    s->n_shells = n_shells;
    s->sh_atom = dup_int(sh_atom, n_shells);
    s->sh_l = dup_int(sh_l, n_shells);
    s->sh_nprim = dup_int(sh_nprim, n_shells);
    s->sh_off = dup_int(sh_off, n_shells);
    s->alpha = dup_real(alpha, n_prim_total);
    s->coef = dup_real(coef, n_prim_total);
    s->n_basis = n_basis;
    s->n_up = n_up;
    s->n_dn = n_dn;
    s->C[0] = dup_real(C_up, (size_t)n_basis * n_up);
    s->C[1] = dup_real(C_dn, (size_t)n_basis * n_dn);
    s->a_anti = a_anti;
    s->a_para = a_para;
    s->b_ee = b_ee;
    s->b_en = b_en;
    int nb = 0;
    for (int i = 0; i < n_shells; i++) {
        if (sh_l[i] < 0 || sh_l[i] > 2) { nb = -1; break; }
        nb += 2 * sh_l[i] + 1;
    }
    if (nb != n_basis) { /* inconsistent input */
        free(s);
        return NULL;
    }
    return s;
}

void oracle_system_destroy(oracle_system *s) {
    if (!s) return;
    free(s->xyz); free(s->Z); free(s->sh_atom); free(s->sh_l); free(s->sh_nprim); free(s->sh_off);
    free(s->alpha); free(s->coef); free(s->C[0]); free(s->C[1]); free(s);
}

/* ------------------------------------------------------------------ RNG
 * Philox4x32-10 (Salmon et al. 2011), keyed as BASELINE.json north_star item 4 / SURVEY 8(c).1:
 * key = (seed lo, seed hi), counter = (walker, step, electron, block). */

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; r++) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* word pair -> U in (0,1): odd integer times 2^-53, exact in FP64 */
static double u01(uint32_t w_even, uint32_t w_odd) {
    uint64_t x = ((uint64_t)w_even << 32) | (uint64_t)w_odd;
    return (double)(2 * (x >> 12) + 1) * 0x1.0p-53;
}

/* the five uniforms of one move: blocks 0,1,2 */
void oracle_move_uniforms(uint64_t seed, uint32_t walker, uint32_t step, uint32_t electron, double U[5]) {
    uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
    uint32_t ctr[4] = {walker, step, electron, 0}, o[4];
    oracle_philox4x32_10(ctr, key, o);
    U[0] = u01(o[0], o[1]); U[1] = u01(o[2], o[3]);
    ctr[3] = 1; oracle_philox4x32_10(ctr, key, o);
    U[2] = u01(o[0], o[1]); U[3] = u01(o[2], o[3]);
    ctr[3] = 2; oracle_philox4x32_10(ctr, key, o);
    U[4] = u01(o[0], o[1]);
}

/* Box-Muller normals chi[3] and the acceptance uniform u */
static void move_variates(uint64_t seed, uint32_t walker, uint32_t step, uint32_t electron, real chi[3], real *u) {
    double U[5];
    oracle_move_uniforms(seed, walker, step, electron, U);
    real r1 = R_SQRT((real)-2 * R_LOG((real)U[0]));
    real r2 = R_SQRT((real)-2 * R_LOG((real)U[2]));
    chi[0] = r1 * R_COS(TWO_PI * (real)U[1]);
    chi[1] = r1 * R_SIN(TWO_PI * (real)U[1]);
    chi[2] = r2 * R_COS(TWO_PI * (real)U[3]);
    *u = (real)U[4];
}

void oracle_move_variates(uint64_t seed, uint32_t walker, uint32_t step, uint32_t electron, double chi[3], double *u) {
    real c[3], uu;
    move_variates(seed, walker, step, electron, c, &uu);
    chi[0] = (double)c[0]; chi[1] = (double)c[1]; chi[2] = (double)c[2]; *u = (double)uu;
}

/* ------------------------------------------------------------------ basis functions
 * Phi = S_lm(x) g(t), t = |x|^2, x = r - R_I, g = sum_p d_p exp(-alpha_p t)   (A1)
 * grad Phi = g grad S + 2 g' S x ;  lap Phi = S [ (4l+6) g' + 4 t g'' ]
 * out arrays have n_basis entries; grad is [3][n_basis]. */

static void basis_eval(const oracle_system *s, const real r[3], real *phi, real *grad, real *lap) {
    int nb = s->n_basis;
    int f = 0;
    for (int sh = 0; sh < s->n_shells; sh++) {
        int a = s->sh_atom[sh], l = s->sh_l[sh];
        real x = r[0] - s->xyz[3 * a + 0];
        real y = r[1] - s->xyz[3 * a + 1];
        real z = r[2] - s->xyz[3 * a + 2];
        real t = x * x + y * y + z * z;
        real g = 0, g1 = 0, g2 = 0;
        for (int p = 0; p < s->sh_nprim[sh]; p++) {
            real al = s->alpha[s->sh_off[sh] + p];
            real e = s->coef[s->sh_off[sh] + p] * R_EXP(-al * t);
            g += e;
            g1 -= al * e;
            g2 += al * al * e;
        }
        int nf = 2 * l + 1;
        real S[5], Sx[5], Sy[5], Sz[5];
        if (l == 0) {
            S[0] = 1; Sx[0] = 0; Sy[0] = 0; Sz[0] = 0;
        } else if (l == 1) {
            S[0] = x; Sx[0] = 1; Sy[0] = 0; Sz[0] = 0;
            S[1] = y; Sx[1] = 0; Sy[1] = 1; Sz[1] = 0;
            S[2] = z; Sx[2] = 0; Sy[2] = 0; Sz[2] = 1;
        } else {
            S[0] = SQRT3 * x * y;                         Sx[0] = SQRT3 * y;  Sy[0] = SQRT3 * x;   Sz[0] = 0;
            S[1] = SQRT3 * y * z;                         Sx[1] = 0;          Sy[1] = SQRT3 * z;   Sz[1] = SQRT3 * y;
            S[2] = z * z - (real)0.5 * (x * x + y * y);   Sx[2] = -x;         Sy[2] = -y;          Sz[2] = 2 * z;
            S[3] = SQRT3 * x * z;                         Sx[3] = SQRT3 * z;  Sy[3] = 0;           Sz[3] = SQRT3 * x;
            S[4] = (SQRT3 / 2) * (x * x - y * y);         Sx[4] = SQRT3 * x;  Sy[4] = -SQRT3 * y;  Sz[4] = 0;
        }
        real lapfac = (real)(4 * l + 6) * g1 + 4 * t * g2;
        for (int m = 0; m < nf; m++, f++) {
            phi[f] = S[m] * g;
            grad[0 * nb + f] = g * Sx[m] + 2 * g1 * S[m] * x;
            grad[1 * nb + f] = g * Sy[m] + 2 * g1 * S[m] * y;
            grad[2 * nb + f] = g * Sz[m] + 2 * g1 * S[m] * z;
            lap[f] = S[m] * lapfac;
        }
    }
}

void oracle_basis_eval(const oracle_system *s, const double r[3], double *phi, double *grad, double *lap) {
    int nb = s->n_basis;
    real rr[3] = {r[0], r[1], r[2]};
    real *b = (real *)malloc((size_t)5 * nb * sizeof(real));
    basis_eval(s, rr, b, b + nb, b + 4 * nb);
    for (int i = 0; i < nb; i++) phi[i] = (double)b[i];
    for (int i = 0; i < 3 * nb; i++) grad[i] = (double)b[nb + i];
    for (int i = 0; i < nb; i++) lap[i] = (double)b[4 * nb + i];
    free(b);
}

/* ------------------------------------------------------------------ molecular-orbital rows
 * v_j = sum_l C_lj Phi_l(r), same for the three gradient components and the Laplacian
 * (PAPER.md L127).  out = [5][n_s]: value, d/dx, d/dy, d/dz, laplacian. */

static void mo_rows(const oracle_system *s, int spin, const real r[3], real *restrict out, real *restrict scratch /*[5*n_basis]*/) {
    int nb = s->n_basis, ns = spin == 0 ? s->n_up : s->n_dn;
    const real *restrict C = s->C[spin];
    basis_eval(s, r, scratch, scratch + nb, scratch + 4 * nb);
    for (int i = 0; i < 5 * ns; i++) out[i] = 0;
    for (int l = 0; l < nb; l++) {
        const real *restrict Cl = C + (size_t)l * ns;
        real b0 = scratch[l], b1 = scratch[nb + l], b2 = scratch[2 * nb + l], b3 = scratch[3 * nb + l], b4 = scratch[4 * nb + l];
        for (int j = 0; j < ns; j++) {
            out[j] += Cl[j] * b0;
            out[ns + j] += Cl[j] * b1;
            out[2 * ns + j] += Cl[j] * b2;
            out[3 * ns + j] += Cl[j] * b3;
            out[4 * ns + j] += Cl[j] * b4;
        }
    }
}

void oracle_mo_rows(const oracle_system *s, int spin, const double r[3], double *out) {
    int nb = s->n_basis, ns = spin == 0 ? s->n_up : s->n_dn;
    real rr[3] = {r[0], r[1], r[2]};
    real *scratch = (real *)malloc((size_t)5 * nb * sizeof(real));
    real *o = (real *)malloc((size_t)(5 * ns + 1) * sizeof(real));
    mo_rows(s, spin, rr, o, scratch);
    for (int i = 0; i < 5 * ns; i++) out[i] = (double)o[i];
    free(o); free(scratch);
}

/* ------------------------------------------------------------------ LU inverse
 * Doolittle LU with partial pivoting; inverse by forward/back substitution on the identity.
 * Returns 0, or -3 if a pivot is exactly zero.  Ainv[j][p]: row j, column p. */

static int lu_inverse(int n, const real *A, real *Ainv, real *logabsdet, int *sign) {
    *logabsdet = 0; *sign = 1;
    if (n == 0) return 0;
    real *LU = (real *)malloc((size_t)n * n * sizeof(real));
    int *piv = (int *)malloc(n * sizeof(int));
    memcpy(LU, A, (size_t)n * n * sizeof(real));
    for (int i = 0; i < n; i++) piv[i] = i;
    int sg = 1;
    real lad = 0;
    for (int k = 0; k < n; k++) {
        int pr = k;
        real best = R_FABS(LU[(size_t)k * n + k]);
        for (int i = k + 1; i < n; i++) {
            real v = R_FABS(LU[(size_t)i * n + k]);
            if (v > best) { best = v; pr = i; }
        }
        if (!(best > 0)) { free(LU); free(piv); return -3; }
        if (pr != k) {
            for (int j = 0; j < n; j++) { real t = LU[(size_t)k * n + j]; LU[(size_t)k * n + j] = LU[(size_t)pr * n + j]; LU[(size_t)pr * n + j] = t; }
            int t = piv[k]; piv[k] = piv[pr]; piv[pr] = t;
            sg = -sg;
        }
        real d = LU[(size_t)k * n + k];
        if (d < 0) sg = -sg;
        lad += R_LOG(R_FABS(d));
        for (int i = k + 1; i < n; i++) {
            real f = LU[(size_t)i * n + k] / d;
            LU[(size_t)i * n + k] = f;
            real *restrict ri = LU + (size_t)i * n;
            const real *restrict rk = LU + (size_t)k * n;
            for (int j = k + 1; j < n; j++) ri[j] -= f * rk[j];
        }
    }
    /* solve A X = I  ->  L U X = P I ; work on all right-hand sides at once, row-wise */
    real *X = Ainv;
    for (int i = 0; i < n; i++)
        for (int j = 0; j < n; j++) X[(size_t)i * n + j] = (piv[i] == j) ? 1 : 0;
    for (int i = 0; i < n; i++) /* forward: L has unit diagonal */
        for (int k = 0; k < i; k++) {
            real f = LU[(size_t)i * n + k];
            if (f != 0) {
                real *restrict xi = X + (size_t)i * n;
                const real *restrict xk = X + (size_t)k * n;
                for (int j = 0; j < n; j++) xi[j] -= f * xk[j];
            }
        }
    for (int i = n - 1; i >= 0; i--) { /* backward */
        real *restrict xi = X + (size_t)i * n;
        for (int k = i + 1; k < n; k++) {
            real f = LU[(size_t)i * n + k];
            const real *restrict xk = X + (size_t)k * n;
            for (int j = 0; j < n; j++) xi[j] -= f * xk[j];
        }
        real d = LU[(size_t)i * n + i];
        for (int j = 0; j < n; j++) xi[j] /= d;
    }
    *logabsdet = lad; *sign = sg;
    free(LU); free(piv);
    return 0;
}

int oracle_lu_inverse(int n, const double *A, double *Ainv, double *logabsdet, int *sign) {
    real *a = dup_real(A, (size_t)n * n), *ai = (real *)malloc(((size_t)n * n + 1) * sizeof(real)), lad;
    int rc = lu_inverse(n, a, ai, &lad, sign);
    if (rc == 0) for (size_t i = 0; i < (size_t)n * n; i++) Ainv[i] = (double)ai[i];
    *logabsdet = (double)lad;
    free(a); free(ai);
    return rc;
}

/* ------------------------------------------------------------------ Jastrow
 * J = sum_{i<k} u_ee(r_ik) + sum_i sum_I u_en(r_iI), u = a r / (1 + b r)         (A5)
 * a = a_anti (opposite spins) / a_para (same spin); e-n: a = -Z_I.  Psi ~ exp(+J). */

static real pade_u(real a, real b, real r) { return a * r / (1 + b * r); }
static real pade_du(real a, real b, real r) { real q = 1 + b * r; return a / (q * q); }
static real pade_d2u(real a, real b, real r) { real q = 1 + b * r; return -2 * a * b / (q * q * q); }

static int spin_of(const oracle_system *s, int i) { return i < s->n_up ? 0 : 1; }
static real a_ee(const oracle_system *s, int i, int k) { return spin_of(s, i) == spin_of(s, k) ? s->a_para : s->a_anti; }

/* sum over partners of electron i placed at ri (others from R): value, gradient, laplacian */
static void jastrow_one(const oracle_system *s, const real *R, int i, const real ri[3], real *val, real grad[3], real *lap) {
    int ne = s->n_up + s->n_dn;
    real v = 0, gx = 0, gy = 0, gz = 0, lp = 0;
    for (int k = 0; k < ne; k++) {
        if (k == i) continue;
        real dx = ri[0] - R[3 * k], dy = ri[1] - R[3 * k + 1], dz = ri[2] - R[3 * k + 2];
        real r = R_SQRT(dx * dx + dy * dy + dz * dz);
        real a = a_ee(s, i, k);
        real du = pade_du(a, s->b_ee, r);
        v += pade_u(a, s->b_ee, r);
        gx += du * dx / r; gy += du * dy / r; gz += du * dz / r;
        lp += pade_d2u(a, s->b_ee, r) + 2 * du / r;
    }
    for (int I = 0; I < s->n_atoms; I++) {
        real dx = ri[0] - s->xyz[3 * I], dy = ri[1] - s->xyz[3 * I + 1], dz = ri[2] - s->xyz[3 * I + 2];
        real r = R_SQRT(dx * dx + dy * dy + dz * dz);
        real a = -s->Z[I];
        real du = pade_du(a, s->b_en, r);
        v += pade_u(a, s->b_en, r);
        gx += du * dx / r; gy += du * dy / r; gz += du * dz / r;
        lp += pade_d2u(a, s->b_en, r) + 2 * du / r;
    }
    *val = v; grad[0] = gx; grad[1] = gy; grad[2] = gz; *lap = lp;
}

/* dJ = sum_{k!=i} [u_ee(|r'-r_k|) - u_ee(|r-r_k|)] + sum_I [u_en(|r'-R_I|) - u_en(|r-R_I|)], term by term */
static real jastrow_delta(const oracle_system *s, const real *R, int i, const real r[3], const real rp[3]) {
    int ne = s->n_up + s->n_dn;
    real dJ = 0;
    for (int k = 0; k < ne; k++) {
        if (k == i) continue;
        real dx = r[0] - R[3 * k], dy = r[1] - R[3 * k + 1], dz = r[2] - R[3 * k + 2];
        real ex = rp[0] - R[3 * k], ey = rp[1] - R[3 * k + 1], ez = rp[2] - R[3 * k + 2];
        real a = a_ee(s, i, k);
        dJ += pade_u(a, s->b_ee, R_SQRT(ex * ex + ey * ey + ez * ez)) - pade_u(a, s->b_ee, R_SQRT(dx * dx + dy * dy + dz * dz));
    }
    for (int I = 0; I < s->n_atoms; I++) {
        real dx = r[0] - s->xyz[3 * I], dy = r[1] - s->xyz[3 * I + 1], dz = r[2] - s->xyz[3 * I + 2];
        real ex = rp[0] - s->xyz[3 * I], ey = rp[1] - s->xyz[3 * I + 1], ez = rp[2] - s->xyz[3 * I + 2];
        real a = -s->Z[I];
        dJ += pade_u(a, s->b_en, R_SQRT(ex * ex + ey * ey + ez * ez)) - pade_u(a, s->b_en, R_SQRT(dx * dx + dy * dy + dz * dz));
    }
    return dJ;
}

static real jastrow_total(const oracle_system *s, const real *R) {
    int ne = s->n_up + s->n_dn;
    real J = 0;
    for (int i = 0; i < ne; i++) {
        for (int k = i + 1; k < ne; k++) {
            real dx = R[3 * i] - R[3 * k], dy = R[3 * i + 1] - R[3 * k + 1], dz = R[3 * i + 2] - R[3 * k + 2];
            J += pade_u(a_ee(s, i, k), s->b_ee, R_SQRT(dx * dx + dy * dy + dz * dz));
        }
        for (int I = 0; I < s->n_atoms; I++) {
            real dx = R[3 * i] - s->xyz[3 * I], dy = R[3 * i + 1] - s->xyz[3 * I + 1], dz = R[3 * i + 2] - s->xyz[3 * I + 2];
            J += pade_u(-s->Z[I], s->b_en, R_SQRT(dx * dx + dy * dy + dz * dz));
        }
    }
    return J;
}

/* J(R), grad_i J [n_e][3], lap_i J [n_e] */
void oracle_jastrow(const oracle_system *s, const double *Rd, double *J, double *grad, double *lap) {
    int ne = s->n_up + s->n_dn;
    real *R = dup_real(Rd, (size_t)3 * ne);
    *J = (double)jastrow_total(s, R);
    for (int i = 0; i < ne; i++) {
        real v, g[3], lp;
        jastrow_one(s, R, i, R + 3 * i, &v, g, &lp);
        grad[3 * i] = (double)g[0]; grad[3 * i + 1] = (double)g[1]; grad[3 * i + 2] = (double)g[2];
        lap[i] = (double)lp;
    }
    free(R);
}

/* ------------------------------------------------------------------ walker state */

typedef struct {
    int ne;
    real *R;        /* [n_e][3] */
    real *Ainv[2];  /* [n_s][n_s], Ainv[j][p] */
    real *orb[2];   /* [n_s(p)][5][n_s(j)]: value / gradient / laplacian rows of the orbitals at the
                       CURRENT position of electron p; bitwise what re-evaluation would give */
    real logabs;    /* log|Psi| running value */
    int sign;       /* sign of D_up D_dn */
    real *scratch;  /* [5*n_basis] */
    real *row;      /* [5*n_s_max] */
    real *tmp;      /* [n_s_max] */
} oracle_walker;

void oracle_walker_destroy(oracle_walker *w) {
    if (!w) return;
    free(w->R); free(w->Ainv[0]); free(w->Ainv[1]); free(w->orb[0]); free(w->orb[1]);
    free(w->scratch); free(w->row); free(w->tmp); free(w);
}

/* init(w) of SURVEY 8(c).2: A from positions, LU inverse, log|D|, sign, J by direct sums */
static int walker_rebuild(const oracle_system *s, oracle_walker *w) {
    real lad_tot = 0;
    int sg_tot = 1;
    for (int sp = 0; sp < 2; sp++) {
        int ns = sp == 0 ? s->n_up : s->n_dn, e0 = sp == 0 ? 0 : s->n_up;
        if (ns == 0) continue; /* empty determinant = 1 (A23) */
        real *A = (real *)malloc((size_t)ns * ns * sizeof(real));
        for (int p = 0; p < ns; p++) {
            real *o = w->orb[sp] + (size_t)p * 5 * ns;
            mo_rows(s, sp, w->R + 3 * (e0 + p), o, w->scratch);
            for (int j = 0; j < ns; j++) A[(size_t)p * ns + j] = o[j];
        }
        real lad; int sg;
        int rc = lu_inverse(ns, A, w->Ainv[sp], &lad, &sg);
        free(A);
        if (rc) return rc;
        lad_tot += lad; sg_tot *= sg;
    }
    w->logabs = lad_tot + jastrow_total(s, w->R);
    w->sign = sg_tot;
    return 0;
}

oracle_walker *oracle_walker_create(const oracle_system *s, const double *R) {
    oracle_walker *w = (oracle_walker *)calloc(1, sizeof(*w));
    int ne = s->n_up + s->n_dn, nsm = s->n_up > s->n_dn ? s->n_up : s->n_dn;
    w->ne = ne;
    w->R = dup_real(R, (size_t)3 * ne);
    for (int sp = 0; sp < 2; sp++) {
        size_t ns = sp == 0 ? s->n_up : s->n_dn;
        w->Ainv[sp] = (real *)calloc(ns * ns + 1, sizeof(real));
        w->orb[sp] = (real *)calloc(ns * 5 * ns + 1, sizeof(real));
    }
    w->scratch = (real *)malloc((size_t)5 * s->n_basis * sizeof(real));
    w->row = (real *)malloc((size_t)(5 * nsm + 1) * sizeof(real));
    w->tmp = (real *)malloc((size_t)(nsm + 1) * sizeof(real));
    if (walker_rebuild(s, w)) { oracle_walker_destroy(w); return NULL; }
    return w;
}

/* deep copy of a walker (the copies a DMC reconfiguration makes, row f1) */
oracle_walker *oracle_walker_clone(const oracle_system *s, const oracle_walker *w) {
    oracle_walker *c = (oracle_walker *)calloc(1, sizeof(oracle_walker));
    int nsm = s->n_up > s->n_dn ? s->n_up : s->n_dn;
    c->ne = w->ne;
    c->R = (real *)malloc((size_t)3 * w->ne * sizeof(real));
    memcpy(c->R, w->R, (size_t)3 * w->ne * sizeof(real));
    for (int sp = 0; sp < 2; sp++) {
        int ns = sp == 0 ? s->n_up : s->n_dn;
        c->Ainv[sp] = (real *)malloc(((size_t)ns * ns + 1) * sizeof(real));
        c->orb[sp] = (real *)malloc(((size_t)ns * 5 * ns + 1) * sizeof(real));
        memcpy(c->Ainv[sp], w->Ainv[sp], (size_t)ns * ns * sizeof(real));
        memcpy(c->orb[sp], w->orb[sp], (size_t)ns * 5 * ns * sizeof(real));
    }
    c->logabs = w->logabs;
    c->sign = w->sign;
    c->scratch = (real *)malloc((size_t)5 * s->n_basis * sizeof(real));
    c->row = (real *)malloc(((size_t)5 * nsm + 1) * sizeof(real));
    c->tmp = (real *)malloc(((size_t)nsm + 1) * sizeof(real));
    return c;
}

/* re-synchronise from externally supplied positions (comparison protocol) */
int oracle_walker_set_positions(const oracle_system *s, oracle_walker *w, const double *R) {
    for (int i = 0; i < 3 * w->ne; i++) w->R[i] = (real)R[i];
    return walker_rebuild(s, w);
}

void oracle_walker_get_positions(const oracle_walker *w, double *R) {
    for (int i = 0; i < 3 * w->ne; i++) R[i] = (double)w->R[i];
}

/* export orientation A18: out[p][j] = (A^-1)[j][p] */
void oracle_walker_get_Ainv(const oracle_system *s, const oracle_walker *w, int spin, double *out) {
    int ns = spin == 0 ? s->n_up : s->n_dn;
    for (int p = 0; p < ns; p++)
        for (int j = 0; j < ns; j++) out[(size_t)p * ns + j] = (double)w->Ainv[spin][(size_t)j * ns + p];
}

/* the Slater matrix itself, out[p][j] = A[p][j] = phi_j(r_p): the value rows of the walker's orbital cache (no arithmetic) */
void oracle_walker_get_A(const oracle_system *s, const oracle_walker *w, int spin, double *out) {
    int ns = spin == 0 ? s->n_up : s->n_dn;
    for (int p = 0; p < ns; p++)
        for (int j = 0; j < ns; j++) out[(size_t)p * ns + j] = (double)w->orb[spin][(size_t)p * 5 * ns + j];
}

/* Replace the inverse of one spin by a caller-supplied one (export orientation A18: in[p][j] = (A^-1)[j][p]).  No
 * arithmetic.  The tests use it to start a DOUBLE-precision walker from the LONG-DOUBLE LU inverse of its own Slater
 * matrix: how far such a walker's sweep lands from the plain double walker's is a measured conditioning floor (reading
 * A26) at sizes where a whole long-double sweep is out of reach (config 3). */
void oracle_walker_set_Ainv(const oracle_system *s, oracle_walker *w, int spin, const double *in) {
    int ns = spin == 0 ? s->n_up : s->n_dn;
    for (int p = 0; p < ns; p++)
        for (int j = 0; j < ns; j++) w->Ainv[spin][(size_t)j * ns + p] = (real)in[(size_t)p * ns + j];
}

void oracle_walker_get_logpsi(const oracle_walker *w, double *logabs, int *sign) {
    *logabs = (double)w->logabs; *sign = w->sign;
}

/* ------------------------------------------------------------------ one sweep
 * bits[i]: 1 = accepted, 2 = tie-flagged (A19).  ratio[i] = rho_D * exp(dJ), pacc[i] = p_acc
 * (0 when rejected by the fixed-node test).  Any of the log pointers may be NULL.
 * The _range form runs electrons e_begin..e_end-1 only (a full sweep is 0..n_e); it exists so that a
 * bounded sample of a sweep can be timed. */

/* Drift limiter of the DMC generation (row f1, reading A28; Umrigar, Nightingale, Runge 1993, eq. 35 with one
 * constant a): vbar = v * (-1 + sqrt(1 + 2 a v^2 tau)) / (a v^2 tau).  Written as 2 / (1 + sqrt(1 + 2x)), x = a v^2 tau,
 * which is the same number without the cancellation at small x ((sqrt(1+2x) - 1)(sqrt(1+2x) + 1) = 2x); a test pins it
 * to the literal form.  lim_a <= 0: no limiter (A6), the drift is used as it is. */
static void limit_drift(real G[3], real lim_a, real tau) {
    if (!(lim_a > 0)) return;
    real v2 = G[0] * G[0] + G[1] * G[1] + G[2] * G[2];
    real x = lim_a * v2 * tau;
    real sc = 2 / (1 + R_SQRT(1 + 2 * x));
    G[0] *= sc; G[1] *= sc; G[2] *= sc;
}
double oracle_drift_limiter_scale(double v2, double lim_a, double tau) {
    real G[3] = {R_SQRT((real)v2), 0, 0};
    limit_drift(G, (real)lim_a, (real)tau);
    return v2 > 0 ? (double)(G[0] / R_SQRT((real)v2)) : 1.0;
}

/* lim_a, dr2: see oracle_walker_dmc_generation; the plain sweep passes lim_a = 0 and dr2 = NULL. */
static void sweep_core(const oracle_system *s, oracle_walker *w, uint64_t seed, uint32_t walker_id,
                       uint32_t step, double tau_d, int e_begin, int e_end, uint8_t *bits, double *ratio,
                       double *pacc, real lim_a, real *dr2 /* [2]: accepted, proposed */) {
    real tau = (real)tau_d, sqrt_tau = R_SQRT(tau);
    for (int i = e_begin; i < e_end; i++) {
        int sp = spin_of(s, i), ns = sp == 0 ? s->n_up : s->n_dn, p = sp == 0 ? i : i - s->n_up;
        real *Ainv = w->Ainv[sp];
        real *orbp = w->orb[sp] + (size_t)p * 5 * ns;
        real *r = w->R + 3 * i;
        /* drift G = sum_j grad phi_j(r) Ainv[j][p] + grad_i J(R)   (A6: no limiter) */
        real G[3], Jold, gJ[3], lJ;
        jastrow_one(s, w->R, i, r, &Jold, gJ, &lJ);
        for (int d = 0; d < 3; d++) {
            real acc = 0;
            for (int j = 0; j < ns; j++) acc += orbp[(1 + d) * ns + j] * Ainv[(size_t)j * ns + p];
            G[d] = acc + gJ[d];
        }
        limit_drift(G, lim_a, tau);
        real chi[3], u;
        move_variates(seed, walker_id, step, (uint32_t)i, chi, &u);
        real rr = tau * (chi[0] * chi[0] + chi[1] * chi[1] + chi[2] * chi[2]); /* |diffusive displacement|^2 */
        if (dr2) dr2[1] += rr;
        real rp[3];
        for (int d = 0; d < 3; d++) rp[d] = r[d] + tau * G[d] + sqrt_tau * chi[d];
        /* orbital rows at r' */
        real *v = w->row;
        mo_rows(s, sp, rp, v, w->scratch);
        real rho = 0;
        for (int j = 0; j < ns; j++) rho += v[j] * Ainv[(size_t)j * ns + p];
        uint8_t b = 0;
        real pa = 0, jr = 0;
        if (R_FABS(rho) < (real)1e-12) b |= 2;
        int accept = 0;
        real dJ = 0;
        if (rho > 0) { /* fixed node: reject if rho_D <= 0 (A7); NaN rejects */
            real Jnew, gJn[3], lJn;
            jastrow_one(s, w->R, i, rp, &Jnew, gJn, &lJn);
            dJ = jastrow_delta(s, w->R, i, r, rp);
            real Gp[3];
            for (int d = 0; d < 3; d++) {
                real acc = 0;
                for (int j = 0; j < ns; j++) acc += v[(1 + d) * ns + j] * Ainv[(size_t)j * ns + p];
                Gp[d] = acc / rho + gJn[d];
            }
            limit_drift(Gp, lim_a, tau);
            real fwd = 0, rev = 0;
            for (int d = 0; d < 3; d++) {
                real a = rp[d] - r[d] - tau * G[d];
                real c = r[d] - rp[d] - tau * Gp[d];
                fwd += a * a; rev += c * c;
            }
            real Delta = (fwd - rev) / (2 * tau);
            pa = rho * rho * R_EXP(2 * dJ + Delta); /* A25 */
            jr = rho * R_EXP(dJ);
            if (R_FABS(u - pa) < (real)1e-12) b |= 2;
            accept = (u < pa);
        }
        if (accept) {
            b |= 1;
            if (dr2) dr2[0] += rr;
            r[0] = rp[0]; r[1] = rp[1]; r[2] = rp[2];
            /* Sherman-Morrison: Ainv[:,q] -= Ainv[:,p] (v.Ainv[:,q]) / rho (q != p); Ainv[:,p] /= rho */
            real *sq = w->tmp;
            for (int q = 0; q < ns; q++) sq[q] = 0;
            for (int j = 0; j < ns; j++) {
                const real *aj = Ainv + (size_t)j * ns;
                real vj = v[j];
                for (int q = 0; q < ns; q++) sq[q] += vj * aj[q];
            }
            for (int j = 0; j < ns; j++) {
                real *aj = Ainv + (size_t)j * ns;
                real cp = aj[p];
                for (int q = 0; q < ns; q++)
                    if (q != p) aj[q] -= cp * sq[q] / rho;
                aj[p] = cp / rho;
            }
            for (int c = 0; c < 5 * ns; c++) orbp[c] = v[c];
            w->logabs += R_LOG(rho) + dJ;
        }
        if (bits) bits[i] = b;
        if (ratio) ratio[i] = (double)jr;
        if (pacc) pacc[i] = (double)pa;
    }
}

void oracle_walker_sweep_range(const oracle_system *s, oracle_walker *w, uint64_t seed, uint32_t walker_id,
                               uint32_t step, double tau_d, int e_begin, int e_end, uint8_t *bits, double *ratio,
                               double *pacc) {
    sweep_core(s, w, seed, walker_id, step, tau_d, e_begin, e_end, bits, ratio, pacc, 0, NULL);
}

void oracle_walker_sweep(const oracle_system *s, oracle_walker *w, uint64_t seed, uint32_t walker_id,
                         uint32_t step, double tau_d, uint8_t *bits, double *ratio, double *pacc) {
    oracle_walker_sweep_range(s, w, seed, walker_id, step, tau_d, 0, w->ne, bits, ratio, pacc);
}

/* ------------------------------------------------------------------ local energy (A9)
 * K = -1/2 sum_i [ l_i - |g_i|^2 + lap_i J + |g_i + grad_i J|^2 ],
 * V = sum_{i<k} 1/r_ik - sum_{i,I} Z_I / r_iI + sum_{I<J} Z_I Z_J / R_IJ */

void oracle_walker_eloc(const oracle_system *s, const oracle_walker *w, double *eloc, double *ekin) {
    int ne = w->ne;
    real K = 0, V = 0;
    for (int i = 0; i < ne; i++) {
        int sp = spin_of(s, i), ns = sp == 0 ? s->n_up : s->n_dn, p = sp == 0 ? i : i - s->n_up;
        const real *Ainv = w->Ainv[sp];
        const real *orbp = w->orb[sp] + (size_t)p * 5 * ns;
        real g[3], l = 0;
        for (int d = 0; d < 3; d++) {
            real acc = 0;
            for (int j = 0; j < ns; j++) acc += orbp[(1 + d) * ns + j] * Ainv[(size_t)j * ns + p];
            g[d] = acc;
        }
        for (int j = 0; j < ns; j++) l += orbp[4 * ns + j] * Ainv[(size_t)j * ns + p];
        real Jv, gJ[3], lJ;
        jastrow_one(s, w->R, i, w->R + 3 * i, &Jv, gJ, &lJ);
        real g2 = g[0] * g[0] + g[1] * g[1] + g[2] * g[2];
        real t2 = (g[0] + gJ[0]) * (g[0] + gJ[0]) + (g[1] + gJ[1]) * (g[1] + gJ[1]) + (g[2] + gJ[2]) * (g[2] + gJ[2]);
        K += l - g2 + lJ + t2;
    }
    K *= (real)-0.5;
    for (int i = 0; i < ne; i++) {
        for (int k = i + 1; k < ne; k++) {
            real dx = w->R[3 * i] - w->R[3 * k], dy = w->R[3 * i + 1] - w->R[3 * k + 1], dz = w->R[3 * i + 2] - w->R[3 * k + 2];
            V += 1 / R_SQRT(dx * dx + dy * dy + dz * dz);
        }
        for (int I = 0; I < s->n_atoms; I++) {
            real dx = w->R[3 * i] - s->xyz[3 * I], dy = w->R[3 * i + 1] - s->xyz[3 * I + 1], dz = w->R[3 * i + 2] - s->xyz[3 * I + 2];
            V -= s->Z[I] / R_SQRT(dx * dx + dy * dy + dz * dz);
        }
    }
    for (int I = 0; I < s->n_atoms; I++)
        for (int J = I + 1; J < s->n_atoms; J++) {
            real dx = s->xyz[3 * I] - s->xyz[3 * J], dy = s->xyz[3 * I + 1] - s->xyz[3 * J + 1], dz = s->xyz[3 * I + 2] - s->xyz[3 * J + 2];
            V += s->Z[I] * s->Z[J] / R_SQRT(dx * dx + dy * dy + dz * dz);
        }
    *eloc = (double)(K + V);
    if (ekin) *ekin = (double)K;
}

/* ------------------------------------------------------------------ one DMC generation (row f1 of SURVEY 8(f))
 * The paper runs fixed-node DMC (eq. 1; tau = 0.01, 4096 walkers, L131) and says nothing about the
 * weights, so this follows the textbook algorithm (Umrigar, Nightingale, Runge, J. Chem. Phys. 99, 2865 (1993)),
 * readings A28-A30 of DESIGN.md:
 *   1. the sweep above with the drift of every proposal (forward and reverse) limited by limit_drift;
 *   2. tau_eff = tau * (sum over ACCEPTED moves of |sqrt(tau) chi|^2) / (sum over ALL proposed moves of it);
 *      tau if nothing was proposed;
 *   3. weight *= exp(-tau_eff * ((E_old + E_new) / 2 - E_T)),  E_old / E_new = E_L before / after the sweep.
 * e_io: in E_old, out E_new.  weight_io: in/out.  bits: accept log of the sweep, may be NULL. */
/* The sweep with the limited drift alone (no E_L, no weight), with its logs: lets a test recompute every p_acc of a
 * limited-drift sweep from first principles.  dr2: [accepted, proposed] sums of |sqrt(tau) chi|^2, may be NULL. */
void oracle_walker_sweep_limited(const oracle_system *s, oracle_walker *w, uint64_t seed, uint32_t walker_id,
                                 uint32_t step, double tau_d, double lim_a, uint8_t *bits, double *ratio, double *pacc,
                                 double *dr2_out) {
    real dr2[2] = {0, 0};
    sweep_core(s, w, seed, walker_id, step, tau_d, 0, w->ne, bits, ratio, pacc, (real)lim_a, dr2);
    if (dr2_out) { dr2_out[0] = (double)dr2[0]; dr2_out[1] = (double)dr2[1]; }
}

void oracle_walker_dmc_generation(const oracle_system *s, oracle_walker *w, uint64_t seed, uint32_t walker_id,
                                  uint32_t step, double tau_d, double lim_a, double E_T, double *e_io,
                                  double *weight_io, double *tau_eff_out, uint8_t *bits) {
    real dr2[2] = {0, 0};
    sweep_core(s, w, seed, walker_id, step, tau_d, 0, w->ne, bits, NULL, NULL, (real)lim_a, dr2);
    double e_new, e_kin;
    oracle_walker_eloc(s, w, &e_new, &e_kin);
    real tau_eff = dr2[1] > 0 ? (real)tau_d * dr2[0] / dr2[1] : (real)tau_d;
    real arg = -tau_eff * (((real)*e_io + (real)e_new) / 2 - (real)E_T);
    *weight_io = (double)((real)*weight_io * R_EXP(arg));
    *e_io = e_new;
    if (tau_eff_out) *tau_eff_out = (double)tau_eff;
}

/* ------------------------------------------------------------------ delayed rank-k update
 * Separate plain-loop routine (not used by the trajectory code above), SURVEY 8(c).2:
 * rows p_1..p_m of A replaced by v_1..v_m.  With E = [e_p1..e_pm], Vb = [v_1..v_m] (n x m),
 * Wb = A0inv E, S = Vb^T Wb, Y = Vb^T A0inv - E^T:   A'^-1 = A0inv - Wb S^-1 Y.
 * Also returns det S (= det A' / det A0).  A0inv, out: [n][n] with Ainv[j][p]. */

int oracle_delayed_update(int n, const double *A0inv_d, int m, const int *rows, const double *Vrows_d /*[m][n]*/,
                          double *out, double *detS_sign_logabs /*[2]*/) {
    real *A0inv = dup_real(A0inv_d, (size_t)n * n), *V = dup_real(Vrows_d, (size_t)m * n);
    real *Wb = (real *)malloc(((size_t)n * m + 1) * sizeof(real)); /* [n][m] */
    real *S = (real *)malloc(((size_t)m * m + 1) * sizeof(real)), *Sinv = (real *)malloc(((size_t)m * m + 1) * sizeof(real));
    real *Y = (real *)malloc(((size_t)m * n + 1) * sizeof(real)), *T = (real *)malloc(((size_t)m * n + 1) * sizeof(real));
    for (int j = 0; j < n; j++)
        for (int a = 0; a < m; a++) Wb[(size_t)j * m + a] = A0inv[(size_t)j * n + rows[a]];
    for (int a = 0; a < m; a++)
        for (int b = 0; b < m; b++) {
            real acc = 0;
            for (int j = 0; j < n; j++) acc += V[(size_t)a * n + j] * Wb[(size_t)j * m + b];
            S[(size_t)a * m + b] = acc;
        }
    real lad; int sg;
    int rc = lu_inverse(m, S, Sinv, &lad, &sg);
    if (rc == 0) {
        for (int a = 0; a < m; a++)
            for (int q = 0; q < n; q++) {
                real acc = 0;
                for (int j = 0; j < n; j++) acc += V[(size_t)a * n + j] * A0inv[(size_t)j * n + q];
                Y[(size_t)a * n + q] = acc - (q == rows[a] ? 1 : 0);
            }
        for (int a = 0; a < m; a++)
            for (int q = 0; q < n; q++) {
                real acc = 0;
                for (int b = 0; b < m; b++) acc += Sinv[(size_t)a * m + b] * Y[(size_t)b * n + q];
                T[(size_t)a * n + q] = acc;
            }
        for (int j = 0; j < n; j++)
            for (int q = 0; q < n; q++) {
                real acc = 0;
                for (int a = 0; a < m; a++) acc += Wb[(size_t)j * m + a] * T[(size_t)a * n + q];
                out[(size_t)j * n + q] = (double)(A0inv[(size_t)j * n + q] - acc);
            }
        if (detS_sign_logabs) { detS_sign_logabs[0] = (double)sg; detS_sign_logabs[1] = (double)lad; }
    }
    free(A0inv); free(V); free(Wb); free(S); free(Sinv); free(Y); free(T);
    return rc;
}

/* single Sherman-Morrison row replacement, exposed for the pins: row p of A replaced by v.
 * Ainv updated in place; returns rho = det A' / det A. */
double oracle_sherman_morrison(int n, double *Ainv_d, int p, const double *v_d) {
    real *Ainv = dup_real(Ainv_d, (size_t)n * n), *v = dup_real(v_d, n), *sq = (real *)calloc(n + 1, sizeof(real));
    real rho = 0;
    for (int j = 0; j < n; j++) rho += v[j] * Ainv[(size_t)j * n + p];
    for (int j = 0; j < n; j++)
        for (int q = 0; q < n; q++) sq[q] += v[j] * Ainv[(size_t)j * n + q];
    for (int j = 0; j < n; j++) {
        real cp = Ainv[(size_t)j * n + p];
        for (int q = 0; q < n; q++)
            if (q != p) Ainv[(size_t)j * n + q] -= cp * sq[q] / rho;
        Ainv[(size_t)j * n + p] = cp / rho;
    }
    for (size_t i = 0; i < (size_t)n * n; i++) Ainv_d[i] = (double)Ainv[i];
    free(Ainv); free(v); free(sq);
    return (double)rho;
}

/* ------------------------------------------------------------------ row f2 (first half): d ln|Psi| / d R_a
 * The paper's eq. (3) with lambda = a nuclear coordinate:  d ln D / d R_a = tr(A^-1 dA/dR_a).
 * A basis function centred on atom a depends on r - R_a only, so dPhi_l/dR_a = -grad Phi_l for l on a and 0 otherwise:
 *   (dA/dR_a,d)[p][j] = - sum_{l on a} C[l][j] d_d Phi_l(r_p),
 *   d ln D / d R_a,d   = - sum_p sum_j Ainv[j][p] sum_{l on a} C[l][j] d_d Phi_l(r_p)        (both spins added),
 * plus the Jastrow, where only the electron-nucleus term knows R_a:  dJ/dR_a = - sum_i u_en'(r_ia) (r_i - R_a)/r_ia.
 * This is the wave-function ("Pulay") term of a QMC force estimator; the derivative of E_L itself (eq. 4) is
 * oracle_walker_deloc_dR below.
 * out[n_atoms][3].  Plain loops in the order written; a test pins it to finite differences of log|Psi| under a
 * displacement of the nucleus together with its basis functions. */
void oracle_walker_dlogpsi_dR(const oracle_system *s, const oracle_walker *w, double *out) {
    int nb = s->n_basis;
    real *phi = (real *)malloc((size_t)5 * nb * sizeof(real));
    real *acc = (real *)calloc((size_t)3 * s->n_atoms, sizeof(real));
    for (int sp = 0; sp < 2; sp++) {
        int ns = sp == 0 ? s->n_up : s->n_dn, e0 = sp == 0 ? 0 : s->n_up;
        const real *Ainv = w->Ainv[sp];
        for (int p = 0; p < ns; p++) {
            basis_eval(s, w->R + 3 * (e0 + p), phi, phi + nb, phi + 4 * nb); /* phi | grad [3][nb] | lap */
            int f = 0;
            for (int sh = 0; sh < s->n_shells; sh++) {
                int a = s->sh_atom[sh], nf = 2 * s->sh_l[sh] + 1;
                for (int m = 0; m < nf; m++, f++) {
                    real cm = 0; /* (C A^-1)[l][p] = sum_j C[l][j] Ainv[j][p] */
                    for (int j = 0; j < ns; j++) cm += s->C[sp][(size_t)f * ns + j] * Ainv[(size_t)j * ns + p];
                    for (int d = 0; d < 3; d++) acc[3 * a + d] -= phi[(size_t)(1 + d) * nb + f] * cm;
                }
            }
        }
    }
    for (int i = 0; i < w->ne; i++)
        for (int a = 0; a < s->n_atoms; a++) {
            real dx = w->R[3 * i] - s->xyz[3 * a], dy = w->R[3 * i + 1] - s->xyz[3 * a + 1], dz = w->R[3 * i + 2] - s->xyz[3 * a + 2];
            real r = R_SQRT(dx * dx + dy * dy + dz * dz);
            real du = pade_du(-s->Z[a], s->b_en, r);
            acc[3 * a] -= du * dx / r; acc[3 * a + 1] -= du * dy / r; acc[3 * a + 2] -= du * dz / r;
        }
    for (int k = 0; k < 3 * s->n_atoms; k++) out[k] = (double)acc[k];
    free(phi); free(acc);
}

/* ------------------------------------------------------------------ row f2 (second half): d E_L / d R_a, eq. (4)
 * PAPER.md L177-181:  dE_L/dR_a = tr(A^-1 dB/dR_a - X dA/dR_a),  X = A^-1 B A^-1,  with (Filippi, Assaraf, Moroni 2016,
 * the "complete mathematical framework" the paper names) B the matrix whose trace with A^-1 is the local energy.  For
 * Psi = D_up D_dn exp(J) (reading A9):
 *     E_L = sum_spin tr(A^-1 B) + sum_i c_i + V,
 *     B[i][j] = -1/2 [ lap phi_j(r_i) + 2 gJ_i . grad phi_j(r_i) ],   c_i = -1/2 [ lap_i J + |gJ_i|^2 ],  gJ_i = grad_i J,
 * so that, with the electrons held fixed, MO coefficients and Jastrow parameters constant and every basis function and
 * electron-nucleus Jastrow term moving with its nucleus (reading A33),
 *     dE_L/dR_a = sum_spin tr(A^-1 dB/dR_a - X dA/dR_a) + sum_i dc_i/dR_a + dV/dR_a .
 * Pieces, d = x, y, z a component of R_a, x = r_i - R_a, r = |x|, u = u_en of atom a (u1, u2, u3 its derivatives):
 *     dA[i][j]   = - sum_{l on a} C[l][j] d_d Phi_l(r_i)
 *     dgJ_i,b    = - [ u2 x_d x_b / r^2 + u1 (delta_db / r - x_d x_b / r^3) ]                (= - d_d d_b u)
 *     dB[i][j]   = -1/2 [ - sum_{l on a} C[l][j] ( d_d lap Phi_l + 2 sum_b gJ_i,b d_d d_b Phi_l )(r_i)
 *                         + 2 sum_b dgJ_i,b d_b phi_j(r_i) ]
 *     dc_i       = -1/2 [ - (u3 + 2 u2 / r - 2 u1 / r^2) x_d / r + 2 sum_b gJ_i,b dgJ_i,b ]
 *     dV         = - Z_a sum_i x_d / r^3 - sum_{b != a} Z_a Z_b (R_a - R_b)_d / R_ab^3
 * Every matrix is built explicitly and multiplied by plain triple loops, one (atom, direction) at a time.
 * out[n_atoms][3].  Pinned by central finite differences of oracle_walker_eloc under a displacement of the nucleus. */

/* second derivatives and the gradient of the Laplacian of every basis function:
 *   Phi = S g(t):   d_a d_b Phi = g d_a d_b S + 2 g' (d_a S x_b + d_b S x_a + S delta_ab) + 4 g'' S x_a x_b
 *   lap Phi = S h,  h = (4l+6) g' + 4 t g'':   d_a lap Phi = h d_a S + 2 h' S x_a,   h' = (4l+10) g'' + 4 t g'''
 * hess [6][nb] in the order xx, yy, zz, xy, xz, yz;  glap [3][nb]. */
static void basis_eval_d3(const oracle_system *s, const real r[3], real *hess, real *glap) {
    int nb = s->n_basis;
    int f = 0;
    for (int sh = 0; sh < s->n_shells; sh++) {
        int a = s->sh_atom[sh], l = s->sh_l[sh];
        real x[3] = {r[0] - s->xyz[3 * a + 0], r[1] - s->xyz[3 * a + 1], r[2] - s->xyz[3 * a + 2]};
        real t = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
        real g = 0, g1 = 0, g2 = 0, g3 = 0;
        for (int p = 0; p < s->sh_nprim[sh]; p++) {
            real al = s->alpha[s->sh_off[sh] + p];
            real e = s->coef[s->sh_off[sh] + p] * R_EXP(-al * t);
            g += e;
            g1 -= al * e;
            g2 += al * al * e;
            g3 -= al * al * al * e;
        }
        int nf = 2 * l + 1;
        real S[5], dS[5][3], ddS[5][6];
        for (int m = 0; m < 5; m++) {
            S[m] = 0;
            for (int k = 0; k < 3; k++) dS[m][k] = 0;
            for (int k = 0; k < 6; k++) ddS[m][k] = 0;
        }
        if (l == 0) {
            S[0] = 1;
        } else if (l == 1) {
            for (int m = 0; m < 3; m++) { S[m] = x[m]; dS[m][m] = 1; }
        } else {
            S[0] = SQRT3 * x[0] * x[1];  dS[0][0] = SQRT3 * x[1]; dS[0][1] = SQRT3 * x[0];  ddS[0][3] = SQRT3;
            S[1] = SQRT3 * x[1] * x[2];  dS[1][1] = SQRT3 * x[2]; dS[1][2] = SQRT3 * x[1];  ddS[1][5] = SQRT3;
            S[2] = x[2] * x[2] - (real)0.5 * (x[0] * x[0] + x[1] * x[1]);
            dS[2][0] = -x[0]; dS[2][1] = -x[1]; dS[2][2] = 2 * x[2];   ddS[2][0] = -1; ddS[2][1] = -1; ddS[2][2] = 2;
            S[3] = SQRT3 * x[0] * x[2];  dS[3][0] = SQRT3 * x[2]; dS[3][2] = SQRT3 * x[0];  ddS[3][4] = SQRT3;
            S[4] = (SQRT3 / 2) * (x[0] * x[0] - x[1] * x[1]);
            dS[4][0] = SQRT3 * x[0]; dS[4][1] = -SQRT3 * x[1];         ddS[4][0] = SQRT3; ddS[4][1] = -SQRT3;
        }
        real h = (real)(4 * l + 6) * g1 + 4 * t * g2;
        real h1 = (real)(4 * l + 10) * g2 + 4 * t * g3;
        static const int pa[6] = {0, 1, 2, 0, 0, 1}, pb[6] = {0, 1, 2, 1, 2, 2};
        for (int m = 0; m < nf; m++, f++) {
            for (int k = 0; k < 6; k++) {
                int ia = pa[k], ib = pb[k];
                real v = g * ddS[m][k] + 2 * g1 * (dS[m][ia] * x[ib] + dS[m][ib] * x[ia]) + 4 * g2 * S[m] * x[ia] * x[ib];
                if (ia == ib) v += 2 * g1 * S[m];
                hess[(size_t)k * nb + f] = v;
            }
            for (int d = 0; d < 3; d++) glap[(size_t)d * nb + f] = h * dS[m][d] + 2 * h1 * S[m] * x[d];
        }
    }
}

void oracle_basis_eval_d3(const oracle_system *s, const double r[3], double *hess, double *glap) {
    int nb = s->n_basis;
    real rr[3] = {r[0], r[1], r[2]};
    real *b = (real *)malloc((size_t)9 * nb * sizeof(real));
    basis_eval_d3(s, rr, b, b + 6 * nb);
    for (int i = 0; i < 6 * nb; i++) hess[i] = (double)b[i];
    for (int i = 0; i < 3 * nb; i++) glap[i] = (double)b[6 * nb + i];
    free(b);
}

static real pade_d3u(real a, real b, real r) { real q = 1 + b * r; return 6 * a * b * b / (q * q * q * q); }

/* the atoms sel[0..n_sel) only (out[n_sel][3]): every atom's derivative is computed independently of the others, so a
 * test at full size can afford a few of them */
void oracle_walker_deloc_dR_atoms(const oracle_system *s, const oracle_walker *w, int n_sel, const int *sel, double *out) {
    int nb = s->n_basis, ne = w->ne, na = s->n_atoms;
    static const int hidx[3][3] = {{0, 3, 4}, {3, 1, 5}, {4, 5, 2}};
    real *acc = (real *)calloc((size_t)3 * n_sel, sizeof(real));
    int *flist = (int *)malloc((size_t)nb * sizeof(int)); /* functions of the current atom */
    real *gJ = (real *)malloc((size_t)3 * ne * sizeof(real));
    for (int i = 0; i < ne; i++) {
        real v, lp;
        jastrow_one(s, w->R, i, w->R + 3 * i, &v, gJ + 3 * i, &lp);
    }
    /* function -> atom */
    int *f_atom = (int *)malloc((size_t)nb * sizeof(int));
    for (int sh = 0, f = 0; sh < s->n_shells; sh++)
        for (int m = 0; m < 2 * s->sh_l[sh] + 1; m++, f++) f_atom[f] = s->sh_atom[sh];
    for (int sp = 0; sp < 2; sp++) {
        int ns = sp == 0 ? s->n_up : s->n_dn, e0 = sp == 0 ? 0 : s->n_up;
        if (ns == 0) continue;
        const real *Ainv = w->Ainv[sp]; /* Ainv[j][i] */
        const real *C = s->C[sp];
        size_t nn = (size_t)ns * ns;
        real *B = (real *)malloc(nn * sizeof(real)), *T = (real *)malloc(nn * sizeof(real)), *X = (real *)malloc(nn * sizeof(real));
        real *dA = (real *)malloc(nn * sizeof(real)), *dB = (real *)malloc(nn * sizeof(real));
        /* derivatives of the basis functions at every electron of this spin: [i][14][nb] = grad 0..2 | hess 3..8 | glap 9..11 | value 12 | lap 13 */
        real *bas = (real *)malloc((size_t)ns * 14 * nb * sizeof(real));
        for (int i = 0; i < ns; i++) {
            real *bi = bas + (size_t)i * 14 * nb;
            basis_eval(s, w->R + 3 * (e0 + i), bi + (size_t)12 * nb, bi, bi + (size_t)13 * nb);
            basis_eval_d3(s, w->R + 3 * (e0 + i), bi + (size_t)3 * nb, bi + (size_t)9 * nb);
        }
        /* B[i][j] from the walker's orbital rows */
        for (int i = 0; i < ns; i++) {
            const real *o = w->orb[sp] + (size_t)i * 5 * ns;
            const real *g = gJ + 3 * (e0 + i);
            for (int j = 0; j < ns; j++)
                B[(size_t)i * ns + j] = (real)-0.5 * (o[4 * ns + j] + 2 * (g[0] * o[ns + j] + g[1] * o[2 * ns + j] + g[2] * o[3 * ns + j]));
        }
        /* X = A^-1 B A^-1:  T[j][k] = sum_i Ainv[j][i] B[i][k];  X[j][i] = sum_k T[j][k] Ainv[k][i] */
        for (int j = 0; j < ns; j++)
            for (int k = 0; k < ns; k++) {
                real a = 0;
                for (int i = 0; i < ns; i++) a += Ainv[(size_t)j * ns + i] * B[(size_t)i * ns + k];
                T[(size_t)j * ns + k] = a;
            }
        for (int j = 0; j < ns; j++)
            for (int i = 0; i < ns; i++) {
                real a = 0;
                for (int k = 0; k < ns; k++) a += T[(size_t)j * ns + k] * Ainv[(size_t)k * ns + i];
                X[(size_t)j * ns + i] = a;
            }
        for (int ia = 0; ia < n_sel; ia++) {
            int a = sel[ia], nfa = 0;
            for (int l = 0; l < nb; l++)
                if (f_atom[l] == a) flist[nfa++] = l;
            for (int d = 0; d < 3; d++) {
                for (int i = 0; i < ns; i++) {
                    const real *bi = bas + (size_t)i * 14 * nb;
                    const real *o = w->orb[sp] + (size_t)i * 5 * ns;
                    const real *g = gJ + 3 * (e0 + i);
                    const real *ri = w->R + 3 * (e0 + i);
                    real x[3] = {ri[0] - s->xyz[3 * a], ri[1] - s->xyz[3 * a + 1], ri[2] - s->xyz[3 * a + 2]};
                    real r = R_SQRT(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
                    real u1 = pade_du(-s->Z[a], s->b_en, r), u2 = pade_d2u(-s->Z[a], s->b_en, r);
                    real dg[3];
                    for (int b = 0; b < 3; b++) dg[b] = -(u2 * x[d] * x[b] / (r * r) + u1 * ((d == b ? 1 / r : 0) - x[d] * x[b] / (r * r * r)));
                    for (int j = 0; j < ns; j++) {
                        real sa = 0, sb = 0;
                        for (int li = 0; li < nfa; li++) {
                            int l = flist[li];
                            real c = C[(size_t)l * ns + j];
                            sa += c * bi[(size_t)d * nb + l];
                            real hg = 0;
                            for (int b = 0; b < 3; b++) hg += g[b] * bi[(size_t)(3 + hidx[d][b]) * nb + l];
                            sb += c * (bi[(size_t)(9 + d) * nb + l] + 2 * hg);
                        }
                        real dgo = dg[0] * o[ns + j] + dg[1] * o[2 * ns + j] + dg[2] * o[3 * ns + j];
                        dA[(size_t)i * ns + j] = -sa;
                        dB[(size_t)i * ns + j] = (real)-0.5 * (-sb + 2 * dgo);
                    }
                }
                real tr = 0;
                for (int i = 0; i < ns; i++)
                    for (int j = 0; j < ns; j++)
                        tr += Ainv[(size_t)j * ns + i] * dB[(size_t)i * ns + j] - X[(size_t)j * ns + i] * dA[(size_t)i * ns + j];
                acc[3 * ia + d] += tr;
            }
        }
        free(B); free(T); free(X); free(dA); free(dB); free(bas);
    }
    /* dc_i and dV */
    for (int ia = 0; ia < n_sel; ia++)
        for (int d = 0; d < 3; d++) {
            int a = sel[ia];
            real sum = 0;
            for (int i = 0; i < ne; i++) {
                const real *g = gJ + 3 * i;
                real x[3] = {w->R[3 * i] - s->xyz[3 * a], w->R[3 * i + 1] - s->xyz[3 * a + 1], w->R[3 * i + 2] - s->xyz[3 * a + 2]};
                real r = R_SQRT(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
                real u1 = pade_du(-s->Z[a], s->b_en, r), u2 = pade_d2u(-s->Z[a], s->b_en, r), u3 = pade_d3u(-s->Z[a], s->b_en, r);
                real gdg = 0;
                for (int b = 0; b < 3; b++) {
                    real dgb = -(u2 * x[d] * x[b] / (r * r) + u1 * ((d == b ? 1 / r : 0) - x[d] * x[b] / (r * r * r)));
                    gdg += g[b] * dgb;
                }
                sum += (real)-0.5 * (-(u3 + 2 * u2 / r - 2 * u1 / (r * r)) * x[d] / r + 2 * gdg);
                sum -= s->Z[a] * x[d] / (r * r * r);
            }
            for (int b = 0; b < na; b++) {
                if (b == a) continue;
                real y[3] = {s->xyz[3 * a] - s->xyz[3 * b], s->xyz[3 * a + 1] - s->xyz[3 * b + 1], s->xyz[3 * a + 2] - s->xyz[3 * b + 2]};
                real rr = R_SQRT(y[0] * y[0] + y[1] * y[1] + y[2] * y[2]);
                sum -= s->Z[a] * s->Z[b] * y[d] / (rr * rr * rr);
            }
            acc[3 * ia + d] += sum;
        }
    for (int k = 0; k < 3 * n_sel; k++) out[k] = (double)acc[k];
    free(acc); free(gJ); free(f_atom); free(flist);
}

void oracle_walker_deloc_dR(const oracle_system *s, const oracle_walker *w, double *out) {
    int *all = (int *)malloc((size_t)s->n_atoms * sizeof(int));
    for (int a = 0; a < s->n_atoms; a++) all[a] = a;
    oracle_walker_deloc_dR_atoms(s, w, s->n_atoms, all, out);
    free(all);
}

/* ------------------------------------------------------------------ row f3: non-local pseudopotential energy
 * PAPER.md L129 ("ccECP pseudopotentials"), L180 ("the non-local pseudopotential contribution").  The paper prints no
 * formula; this is the standard semi-local form evaluated by spherical quadrature (Fahy, Wang, Louie 1990; Mitas,
 * Shirley, Ceperley 1991), reading A34 of DESIGN.md.  Atom I carries channels l with radial functions
 * v_l(r) = beta_l exp(-alpha_l r^2), cut at rcut_I.  For every electron i with r = |r_i - R_I| < rcut_I,
 *     (V_nl Psi / Psi)_iI = sum_l (2l+1) v_l(r) sum_q w_q P_l(cos th_q) Psi(.., r_q, ..) / Psi(.., r_i, ..),
 *     r_q = R_I + r O_q,   cos th_q = O_q . (r_i - R_I) / r,
 * O_q = Rot * (vertex q of the icosahedron), w_q = 1/12 (exact for spherical polynomials up to degree 5), Rot a
 * uniformly random rotation drawn per (walker, step, electron) from Philox blocks 4 and 5.  The wave-function ratio
 * is the determinant ratio (orbital values at r_q against column i of A^-1) times exp(J(r_q) - J(r_i)).
 * V_nl = sum_i (ascending) sum_I (ascending) of that.  l <= 2. */

/* vertex q = 4 c + 2 a + b  (c = 0,1,2; a, b in {0,1}):  coordinate c is 0, coordinate c+1 is (+/-) n, coordinate c+2 is (+/-) phi n,
 * the first sign from a, the second from b (0: +, 1: -);  phi = (1 + sqrt 5)/2,  n = 1/sqrt(1 + phi^2) */
static void icosahedron_vertex(int q, real v[3]) {
    real phi = ((real)1 + R_SQRT((real)5)) / 2;
    real n = 1 / R_SQRT(1 + phi * phi);
    int c = q / 4, a = (q / 2) % 2, b = q % 2;
    v[c] = 0;
    v[(c + 1) % 3] = a ? -n : n;
    v[(c + 2) % 3] = b ? -phi * n : phi * n;
}

/* uniformly random rotation (Shoemake 1992): three uniforms -> unit quaternion (x, y, z, w) -> matrix, row-major */
static void quadrature_rotation(uint64_t seed, uint32_t walker, uint32_t step, uint32_t electron, real rot[9]) {
    uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
    uint32_t ctr[4] = {walker, step, electron, 4}, o[4];
    oracle_philox4x32_10(ctr, key, o);
    real u1 = (real)u01(o[0], o[1]), u2 = (real)u01(o[2], o[3]);
    ctr[3] = 5; oracle_philox4x32_10(ctr, key, o);
    real u3 = (real)u01(o[0], o[1]);
    real a = R_SQRT(1 - u1), b = R_SQRT(u1);
    real x = a * R_SIN(TWO_PI * u2), y = a * R_COS(TWO_PI * u2), z = b * R_SIN(TWO_PI * u3), w = b * R_COS(TWO_PI * u3);
    rot[0] = 1 - 2 * (y * y + z * z); rot[1] = 2 * (x * y - z * w);     rot[2] = 2 * (x * z + y * w);
    rot[3] = 2 * (x * y + z * w);     rot[4] = 1 - 2 * (x * x + z * z); rot[5] = 2 * (y * z - x * w);
    rot[6] = 2 * (x * z - y * w);     rot[7] = 2 * (y * z + x * w);     rot[8] = 1 - 2 * (x * x + y * y);
}

void oracle_quadrature_directions(uint64_t seed, uint32_t walker, uint32_t step, uint32_t electron, double dirs[36]) {
    real rot[9];
    quadrature_rotation(seed, walker, step, electron, rot);
    for (int q = 0; q < 12; q++) {
        real v[3];
        icosahedron_vertex(q, v);
        for (int d = 0; d < 3; d++) dirs[3 * q + d] = (double)(rot[3 * d] * v[0] + rot[3 * d + 1] * v[1] + rot[3 * d + 2] * v[2]);
    }
}

/* returns V_nl of the walker.  Optional outputs for the pins (may be NULL; at most max_pairs pairs are recorded, all are counted):
 * pair_i, pair_I [max_pairs], pts [max_pairs][12][3], ratios [max_pairs][12], n_pairs. */
double oracle_walker_vnl(const oracle_system *s, const oracle_walker *w, uint64_t seed, uint32_t walker_id, uint32_t step,
                         int n_ch, const int *ch_atom, const int *ch_l, const double *ch_beta, const double *ch_alpha,
                         const double *rcut, int max_pairs, int *pair_i, int *pair_I, double *pts, double *ratios, int *n_pairs) {
    int ne = w->ne, np = 0;
    real vnl = 0;
    real *row = (real *)malloc((size_t)5 * (s->n_up > s->n_dn ? s->n_up : s->n_dn) * sizeof(real) + 8);
    for (int i = 0; i < ne; i++) {
        int sp = spin_of(s, i), ns = sp == 0 ? s->n_up : s->n_dn, p = sp == 0 ? i : i - s->n_up;
        const real *ri = w->R + 3 * i;
        real rot[9];
        quadrature_rotation(seed, walker_id, step, (uint32_t)i, rot);
        for (int I = 0; I < s->n_atoms; I++) {
            real x[3] = {ri[0] - s->xyz[3 * I], ri[1] - s->xyz[3 * I + 1], ri[2] - s->xyz[3 * I + 2]};
            real r = R_SQRT(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
            if (!(r < (real)rcut[I])) continue;
            real vl[3] = {0, 0, 0};  /* (2l+1) v_l(r) */
            int any = 0;
            for (int c = 0; c < n_ch; c++)
                if (ch_atom[c] == I) {
                    vl[ch_l[c]] += (real)(2 * ch_l[c] + 1) * (real)ch_beta[c] * R_EXP(-(real)ch_alpha[c] * r * r);
                    any = 1;
                }
            if (!any) continue;
            real pair_sum = 0;
            for (int q = 0; q < 12; q++) {
                real v[3], o[3], rq[3];
                icosahedron_vertex(q, v);
                for (int d = 0; d < 3; d++) o[d] = rot[3 * d] * v[0] + rot[3 * d + 1] * v[1] + rot[3 * d + 2] * v[2];
                for (int d = 0; d < 3; d++) rq[d] = s->xyz[3 * I + d] + r * o[d];
                real c = (o[0] * x[0] + o[1] * x[1] + o[2] * x[2]) / r;
                mo_rows(s, sp, rq, row, w->scratch);
                real det = 0;
                for (int j = 0; j < ns; j++) det += row[j] * w->Ainv[sp][(size_t)j * ns + p];
                real rho = det * R_EXP(jastrow_delta(s, w->R, i, ri, rq));
                real ang = vl[0] + vl[1] * c + vl[2] * ((real)1.5 * c * c - (real)0.5);
                pair_sum += ang * rho / 12;
                if (np < max_pairs) {
                    if (pts) for (int d = 0; d < 3; d++) pts[((size_t)np * 12 + q) * 3 + d] = (double)rq[d];
                    if (ratios) ratios[(size_t)np * 12 + q] = (double)rho;
                }
            }
            if (np < max_pairs) {
                if (pair_i) pair_i[np] = i;
                if (pair_I) pair_I[np] = I;
            }
            np++;
            vnl += pair_sum;
        }
    }
    free(row);
    if (n_pairs) *n_pairs = np;
    return (double)vnl;
}

/* from-scratch log|Psi| and sign at the walker's current positions (pin for the running value) */
int oracle_walker_logpsi_scratch(const oracle_system *s, const oracle_walker *w, double *logabs, int *sign) {
    real lad_tot = 0; int sg_tot = 1;
    real *scratch = (real *)malloc((size_t)5 * s->n_basis * sizeof(real));
    for (int sp = 0; sp < 2; sp++) {
        int ns = sp == 0 ? s->n_up : s->n_dn, e0 = sp == 0 ? 0 : s->n_up;
        if (ns == 0) continue;
        real *A = (real *)malloc((size_t)ns * ns * sizeof(real)), *Ai = (real *)malloc((size_t)ns * ns * sizeof(real));
        real *o = (real *)malloc((size_t)5 * ns * sizeof(real));
        for (int p = 0; p < ns; p++) {
            mo_rows(s, sp, w->R + 3 * (e0 + p), o, scratch);
            for (int j = 0; j < ns; j++) A[(size_t)p * ns + j] = o[j];
        }
        real lad; int sg;
        int rc = lu_inverse(ns, A, Ai, &lad, &sg);
        free(A); free(Ai); free(o);
        if (rc) { free(scratch); return rc; }
        lad_tot += lad; sg_tot *= sg;
    }
    free(scratch);
    *logabs = (double)(lad_tot + jastrow_total(s, w->R)); *sign = sg_tot;
    return 0;
}
