/*
 * pcm_oracle.c -- CPU ORACLE for the C-PCM hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, fp64 restatement of what arxiv 1505.07851 defines:
 *   - the smeared-charge one-electron integrals of Eq. 6 / Eq. 12 (Obara-Saika
 *     recursion, series-evaluated Boys function),
 *   - the two contractions  v_k = sum_{mu,nu} P_mu,nu (mu|J_k|nu)   (Eq. 5, c_k = -v_k)
 *                           F_mu,nu = sum_k q_k (mu|J_k|nu)          (Eq. 10, dF^S = -F),
 *   - the matrix A of Eq. 2 / 3 / 8 and the product A q,
 *   - textbook preconditioned CG (section 4b) with the Jacobi and the randomized
 *     block-Jacobi (RBJ, section 4b-ii) preconditioners,
 *   - the rest of a C-PCM step: B z (Eq. 4), the right-hand side of Eq. 1, the energy of Eq. 13,
 *     the dynamic CG threshold of Eq. 21                       (pins: tests/test_oracle_glue.py),
 *   - the gradient of E = v.q with respect to shell centres and surface points, i.e. the
 *     one-electron term of Eq. 14 / Eq. 22                     (pins: tests/test_oracle_gradient.py),
 *   - the ISWIG switching function of Eq. 9 and the surface terms of Eq. 14 (grad B, grad A
 *     including A_kk through S_k)                              (pins: tests/test_oracle_surface.py),
 *   - the ISWIG cavity construction itself: sphere points per atom from a given unit-sphere
 *     quadrature, zeta_k of Eq. 7, S_k of Eq. 9, the S_k >= 1e-8 screening of PAPER.md:106
 *                                                              (pins: tests/test_oracle_cavity.py).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this file.  It shares no code, table, constant generator or helper with
 * the CUDA path under paper_1505_07851_b200/ and neither includes the other.
 *
 * Pins (tests/test_oracle_*.py, all run with -m "not gpu"): every function below is pinned
 * against something other than itself -- closed forms, library special functions,
 * brute-force quadrature, limits and invariants; nothing here is "parity unpinned".
 *
 * Readings of the paper (it is silent or garbled there; listed in DESIGN.md):
 *   R1  Eq. 3 prints zeta_k/sqrt(2 pi); the self-energy of a unit Gaussian charge and the
 *       r->0 limit of Eq. 2 are zeta_k*sqrt(2/pi); BASELINE.json configs[4] says the same.
 *   R2  library sign: v and F are the unsigned quantities; the paper's c = -v, dF^S = -F.
 *   R3  prim_coef multiplies RAW Cartesian primitives x^i y^j z^k exp(-a r^2); pure d =
 *       (sqrt3 xy, sqrt3 yz, zz-(xx+yy)/2, sqrt3 xz, (sqrt3/2)(xx-yy)); Cartesian d =
 *       (xx,xy,xz,yy,yz,zz); p = (x,y,z).
 *   R4  the oracle does not screen with Eq. 15; it skips only primitive pairs with
 *       |c_i c_j| K_AB < cutoff (default 1e-20, 0 switches it off).
 *   R5  PCG: x0 = 0 unless given, r = b - A x, Euclidean absolute norm, the recurrence
 *       residual decides.  RBJ: pivot = first still-unassigned index in a given pivot
 *       order; the block is the pivot plus the l-1 unassigned indices with largest
 *       |A_kj| (ties -> lower index); last block takes the remainder.
 *
 * Build:  gcc -O2 -fopenmp -shared -fPIC -o libpcm_oracle.so pcm_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288
#define LMAX_SHELL 2          /* s, p, d */
#define LTAB (LMAX_SHELL + 1) /* the recursion tables go one power further: derivative integrals raise one side */
#define LSUM (2 * LMAX_SHELL + 1) /* l_a + l_b <= 4, + 1 for a raised side */
#define NA (LSUM + 1)         /* 0..5 per Cartesian power in the recursion tables */

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Neumaier compensated accumulation: (*s) + (*c) carries the running sum. */
static void nsum(double *s, double *c, double x) {
    double t = *s + x;
    if (fabs(*s) >= fabs(x)) *c += (*s - t) + x; else *c += (x - t) + *s;
    *s = t;
}

/* ------------------------------------------------------------------------------------
 * Boys function F_n(T) = int_0^1 t^{2n} exp(-T t^2) dt, n = 0..nmax.
 * The paper does not say how it is evaluated (PAPER.md:122 cites refs 19, 48 only).
 * T < 35 : series for the highest order
 *            F_n(T) = exp(-T) sum_{k>=0} (2T)^k / [(2n+1)(2n+3)...(2n+2k+1)]
 *          (all terms positive), then downward  F_{n-1} = (2T F_n + exp(-T)) / (2n-1).
 * T >= 35: F_0 = (1/2) sqrt(pi/T) erf(sqrt T), then upward
 *            F_{n+1} = ((2n+1) F_n - exp(-T)) / (2T), keeping the exp(-T) term.
 * ---------------------------------------------------------------------------------- */
void orc_boys(int nmax, double T, double *F) {
    double eT = exp(-T);
    if (T < 35.0) {
        double term = 1.0 / (2.0 * nmax + 1.0), sum = term;
        for (int k = 0; k < 2000; ++k) {
            term *= 2.0 * T / (2.0 * nmax + 2.0 * k + 3.0);
            sum += term;
            if (term < 1e-17 * sum) break;
        }
        F[nmax] = eT * sum;
        for (int n = nmax; n >= 1; --n) F[n - 1] = (2.0 * T * F[n] + eT) / (2.0 * n - 1.0);
    } else {
        F[0] = 0.5 * sqrt(ORC_PI / T) * erf(sqrt(T));
        for (int n = 0; n < nmax; ++n) F[n + 1] = ((2.0 * n + 1.0) * F[n] - eT) / (2.0 * T);
    }
}

/* ------------------------------------------------------------------------------------
 * Primitive integrals [chi_a | erf(zeta |r-C|)/|r-C| | chi_b]  (Eq. 6 integrand, Eq. 12
 * bracket) for RAW Cartesian primitives chi_a = (x-Ax)^ax (y-Ay)^ay (z-Az)^az exp(-alpha|r-A|^2).
 *
 * Obara-Saika.  With p = alpha+beta, P = (alpha A + beta B)/p, K_AB = exp(-alpha beta/p |A-B|^2),
 * rho = p zeta^2/(p+zeta^2), T = rho |P-C|^2  (from erf(zeta r)/r = (2/sqrt pi) int_0^zeta exp(-t^2 r^2) dt
 * and u^2 = t^2/(p+t^2), upper limit u_max^2 = rho/p):
 *   Theta^N_{0,0}      = (2 pi/p) K_AB (rho/p)^{N+1/2} F_N(T)
 *   Theta^N_{a+1_i,0}  = (P-A)_i Theta^N_{a,0} - (P-C)_i Theta^{N+1}_{a,0}
 *                        + a_i/(2p) (Theta^N_{a-1_i,0} - Theta^{N+1}_{a-1_i,0})
 *   Theta_{a,b+1_i}    = Theta_{a+1_i,b} + (A-B)_i Theta_{a,b}          (horizontal transfer)
 * `path` picks which Cartesian direction the vertical step lowers when several are possible
 * (0: first non-zero power, 1: last non-zero power) -- the result must not depend on it.
 *
 * tab[(bx,by,bz)][(ax,ay,az)] is filled for |b| <= lb and la <= |a| <= la+lb-|b|; the caller
 * reads |a| = la, |b| = lb.
 * ---------------------------------------------------------------------------------- */
#define AIDX(x, y, z) (((x) * NA + (y)) * NA + (z))
#define NB (LTAB + 1)
#define BIDX(x, y, z) (((x) * NB + (y)) * NB + (z))

static void os_tables(int la, double alpha, const double *A, int lb, double beta, const double *B,
                      double zeta, const double *C, int path, double hrr[NB * NB * NB][NA * NA * NA]) {
    const int L = la + lb;
    const double p = alpha + beta;
    double P[3], PA[3], PC[3], AB[3];
    double r2ab = 0.0, r2pc = 0.0;
    for (int i = 0; i < 3; ++i) {
        P[i] = (alpha * A[i] + beta * B[i]) / p;
        PA[i] = P[i] - A[i];
        PC[i] = P[i] - C[i];
        AB[i] = A[i] - B[i];
        r2ab += AB[i] * AB[i];
        r2pc += PC[i] * PC[i];
    }
    const double KAB = exp(-alpha * beta / p * r2ab);
    const double rho = p * zeta * zeta / (p + zeta * zeta);
    const double T = rho * r2pc;
    double F[LSUM + 1];
    orc_boys(L, T, F);

    /* vertical recursion: th[N][a] for |a| <= L, N <= L - |a| */
    static const int dirs[2][3] = {{0, 1, 2}, {2, 1, 0}};
    double th[LSUM + 1][NA * NA * NA];
    const double w = rho / p;
    for (int N = 0; N <= L; ++N) th[N][AIDX(0, 0, 0)] = (2.0 * ORC_PI / p) * KAB * pow(w, N + 0.5) * F[N];
    for (int n = 1; n <= L; ++n)
        for (int ax = 0; ax <= n; ++ax)
            for (int ay = 0; ay <= n - ax; ++ay) {
                int a[3] = {ax, ay, n - ax - ay};
                int i = -1;
                for (int d = 0; d < 3; ++d)
                    if (a[dirs[path ? 1 : 0][d]] > 0) { i = dirs[path ? 1 : 0][d]; break; }
                int am[3] = {a[0], a[1], a[2]};
                am[i] -= 1; /* a = am + 1_i */
                int amm[3] = {am[0], am[1], am[2]};
                amm[i] -= 1;
                for (int N = 0; N <= L - n; ++N) {
                    double v = PA[i] * th[N][AIDX(am[0], am[1], am[2])] - PC[i] * th[N + 1][AIDX(am[0], am[1], am[2])];
                    if (am[i] > 0)
                        v += am[i] / (2.0 * p) *
                             (th[N][AIDX(amm[0], amm[1], amm[2])] - th[N + 1][AIDX(amm[0], amm[1], amm[2])]);
                    th[N][AIDX(a[0], a[1], a[2])] = v;
                }
            }

    /* horizontal transfer */
    for (int n = la; n <= L; ++n)
        for (int ax = 0; ax <= n; ++ax)
            for (int ay = 0; ay <= n - ax; ++ay)
                hrr[BIDX(0, 0, 0)][AIDX(ax, ay, n - ax - ay)] = th[0][AIDX(ax, ay, n - ax - ay)];
    for (int m = 1; m <= lb; ++m)
        for (int bx = 0; bx <= m; ++bx)
            for (int by = 0; by <= m - bx; ++by) {
                int b[3] = {bx, by, m - bx - by};
                int i = -1;
                for (int d = 0; d < 3; ++d)
                    if (b[dirs[path ? 1 : 0][d]] > 0) { i = dirs[path ? 1 : 0][d]; break; }
                int bm[3] = {b[0], b[1], b[2]};
                bm[i] -= 1;
                for (int n = la; n <= L - m; ++n)
                    for (int ax = 0; ax <= n; ++ax)
                        for (int ay = 0; ay <= n - ax; ++ay) {
                            int a[3] = {ax, ay, n - ax - ay};
                            int ap[3] = {a[0], a[1], a[2]};
                            ap[i] += 1;
                            hrr[BIDX(b[0], b[1], b[2])][AIDX(a[0], a[1], a[2])] =
                                hrr[BIDX(bm[0], bm[1], bm[2])][AIDX(ap[0], ap[1], ap[2])] +
                                AB[i] * hrr[BIDX(bm[0], bm[1], bm[2])][AIDX(a[0], a[1], a[2])];
                        }
            }
}

/* Cartesian component lists: s; p = x,y,z; d = xx,xy,xz,yy,yz,zz  (reading R3) */
static const int CART[3][6][3] = {
    {{0, 0, 0}},
    {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}},
    {{2, 0, 0}, {1, 1, 0}, {1, 0, 1}, {0, 2, 0}, {0, 1, 1}, {0, 0, 2}},
};
static const int NCART[3] = {1, 3, 6};

/* one primitive integral with explicit powers (any |a|,|b| <= 3, |a| + |b| <= 5) */
double orc_prim_integral(const int *a, double alpha, const double *A, const int *b, double beta, const double *B,
                         double zeta, const double *C, int path) {
    int la = a[0] + a[1] + a[2], lb = b[0] + b[1] + b[2];
    double hrr[NB * NB * NB][NA * NA * NA];
    os_tables(la, alpha, A, lb, beta, B, zeta, C, path, hrr);
    return hrr[BIDX(b[0], b[1], b[2])][AIDX(a[0], a[1], a[2])];
}

/* whole Cartesian primitive batch: out[ia*NCART[lb] + ib] */
void orc_prim_block(int la, double alpha, const double *A, int lb, double beta, const double *B, double zeta,
                    const double *C, int path, double *out) {
    double hrr[NB * NB * NB][NA * NA * NA];
    os_tables(la, alpha, A, lb, beta, B, zeta, C, path, hrr);
    for (int ia = 0; ia < NCART[la]; ++ia)
        for (int ib = 0; ib < NCART[lb]; ++ib) {
            const int *a = CART[la][ia], *b = CART[lb][ib];
            out[ia * NCART[lb] + ib] = hrr[BIDX(b[0], b[1], b[2])][AIDX(a[0], a[1], a[2])];
        }
}

/* ------------------------------------------------------------------------------------
 * Contracted basis (Eq. 11 / 12).  Layout = include/pcm.h's pcm_setup arguments.
 * ---------------------------------------------------------------------------------- */
typedef struct {
    int nshell;
    const int *l;         /* [nshell] */
    const double *xyz;    /* [3 nshell] */
    const int *nprim;     /* [nshell] */
    const double *ex;     /* [sum nprim] */
    const double *co;     /* [sum nprim] */
    int d_pure;
} orc_basis;

static int ncomp_of(int l, int d_pure) { return l == 0 ? 1 : (l == 1 ? 3 : (d_pure ? 5 : 6)); }

/* rows: pure component, cols: Cartesian d component (xx,xy,xz,yy,yz,zz)  (reading R3) */
static void pure_d_matrix(double m[5][6]) {
    const double s3 = sqrt(3.0);
    memset(m, 0, sizeof(double) * 30);
    m[0][1] = s3;                                /* sqrt3 xy */
    m[1][4] = s3;                                /* sqrt3 yz */
    m[2][5] = 1.0; m[2][0] = -0.5; m[2][3] = -0.5; /* zz - (xx+yy)/2 */
    m[3][2] = s3;                                /* sqrt3 xz */
    m[4][0] = 0.5 * s3; m[4][3] = -0.5 * s3;     /* (sqrt3/2)(xx-yy) */
}

/* Cartesian block [6x6 max] -> component block (pure d transform on either side) */
static void to_components(int la, int lb, int d_pure, const double *cart, double *out) {
    int nca = NCART[la], ncb = NCART[lb];
    int na = ncomp_of(la, d_pure), nb = ncomp_of(lb, d_pure);
    double m[5][6];
    pure_d_matrix(m);
    double tmp[6 * 6];
    /* left side */
    for (int i = 0; i < na; ++i)
        for (int j = 0; j < ncb; ++j) {
            if (la == 2 && d_pure) {
                double s = 0.0;
                for (int c = 0; c < 6; ++c) s += m[i][c] * cart[c * ncb + j];
                tmp[i * ncb + j] = s;
            } else tmp[i * ncb + j] = cart[i * ncb + j];
        }
    (void)nca;
    for (int i = 0; i < na; ++i)
        for (int j = 0; j < nb; ++j) {
            if (lb == 2 && d_pure) {
                double s = 0.0;
                for (int c = 0; c < 6; ++c) s += m[j][c] * tmp[i * ncb + c];
                out[i * nb + j] = s;
            } else out[i * nb + j] = tmp[i * ncb + j];
        }
}

static void offsets(const orc_basis *bs, long *prim_off, long *bf_off) {
    prim_off[0] = 0; bf_off[0] = 0;
    for (int s = 0; s < bs->nshell; ++s) {
        prim_off[s + 1] = prim_off[s] + bs->nprim[s];
        bf_off[s + 1] = bf_off[s] + ncomp_of(bs->l[s], bs->d_pure);
    }
}

/* which primitive pairs of shell pair (I,J) are kept: |c_i c_j| K_AB >= cutoff (reading R4) */
static int keep_mask(const orc_basis *bs, const long *po, int I, int J, double cutoff, unsigned char *keep) {
    const double *A = bs->xyz + 3 * I, *B = bs->xyz + 3 * J;
    double r2 = 0.0;
    for (int d = 0; d < 3; ++d) r2 += (A[d] - B[d]) * (A[d] - B[d]);
    int any = 0;
    for (int i = 0; i < bs->nprim[I]; ++i)
        for (int j = 0; j < bs->nprim[J]; ++j) {
            double a = bs->ex[po[I] + i], b = bs->ex[po[J] + j];
            double k = fabs(bs->co[po[I] + i] * bs->co[po[J] + j]) * exp(-a * b / (a + b) * r2);
            unsigned char kp = (cutoff <= 0.0) || (k >= cutoff);
            keep[i * bs->nprim[J] + j] = kp;
            any |= kp;
        }
    return any;
}

/* contracted component block (mu in I, nu in J | J_k) at one point; out[ncompI*ncompJ] */
static void shell_block(const orc_basis *bs, const long *po, int I, int J, const unsigned char *keep, double zeta,
                        const double *C, double *out) {
    int la = bs->l[I], lb = bs->l[J];
    double cart[36], prim[36];
    int n = NCART[la] * NCART[lb];
    for (int c = 0; c < n; ++c) cart[c] = 0.0;
    for (int i = 0; i < bs->nprim[I]; ++i)
        for (int j = 0; j < bs->nprim[J]; ++j) {
            if (keep && !keep[i * bs->nprim[J] + j]) continue;
            orc_prim_block(la, bs->ex[po[I] + i], bs->xyz + 3 * I, lb, bs->ex[po[J] + j], bs->xyz + 3 * J, zeta, C, 0,
                           prim);
            double cc = bs->co[po[I] + i] * bs->co[po[J] + j];
            for (int c = 0; c < n; ++c) cart[c] += cc * prim[c];
        }
    to_components(la, lb, bs->d_pure, cart, out);
}

/* public: one contracted shell-pair block at one point (no cutoff) */
void orc_shell_block(int nshell, const int *l, const double *xyz, const int *nprim, const double *ex, const double *co,
                     int d_pure, int I, int J, double zeta, const double *C, double *out) {
    orc_basis bs = {nshell, l, xyz, nprim, ex, co, d_pure};
    long *po = malloc(sizeof(long) * (nshell + 1)), *bo = malloc(sizeof(long) * (nshell + 1));
    offsets(&bs, po, bo);
    shell_block(&bs, po, I, J, NULL, zeta, C, out);
    free(po); free(bo);
}

/* ------------------------------------------------------------------------------------
 * v_k = sum_{mu,nu} P_mu,nu (mu|J_k|nu)  over the FULL square (both (mu,nu) and (nu,mu)),
 * Eq. 5 with reading R2 (c_k = -v_k), for the selected points sel[0..nsel).
 * sel == NULL means points 0..nsel-1.  P is row-major nbf x nbf with leading dimension ldp.
 * ---------------------------------------------------------------------------------- */
void orc_potential(int nshell, const int *l, const double *xyz, const int *nprim, const double *ex, const double *co,
                   int d_pure, const double *pt_xyz, const double *pt_zeta, const double *P, long ldp, double cutoff,
                   long nsel, const long *sel, double *v_out) {
    orc_basis bs = {nshell, l, xyz, nprim, ex, co, d_pure};
    long *po = malloc(sizeof(long) * (nshell + 1)), *bo = malloc(sizeof(long) * (nshell + 1));
    offsets(&bs, po, bo);
    /* hoist the point-independent keep decision: per ordered shell pair a mask offset, -1 = nothing kept */
    long *moff = malloc(sizeof(long) * (size_t)nshell * nshell);
    long tot = 0;
    for (int I = 0; I < nshell; ++I)
        for (int J = 0; J < nshell; ++J) { moff[(long)I * nshell + J] = tot; tot += nprim[I] * nprim[J]; }
    unsigned char *mask = malloc((size_t)tot);
#pragma omp parallel for schedule(dynamic, 8)
    for (int I = 0; I < nshell; ++I)
        for (int J = 0; J < nshell; ++J) {
            long o = moff[(long)I * nshell + J];
            if (!keep_mask(&bs, po, I, J, cutoff, mask + o)) moff[(long)I * nshell + J] = -1;
        }
#pragma omp parallel for schedule(dynamic, 1)
    for (long s = 0; s < nsel; ++s) {
        long k = sel ? sel[s] : s;
        double sum = 0.0, comp = 0.0, blk[36];
        for (int I = 0; I < nshell; ++I)
            for (int J = 0; J < nshell; ++J) {
                long o = moff[(long)I * nshell + J];
                if (o < 0) continue;
                shell_block(&bs, po, I, J, mask + o, pt_zeta[k], pt_xyz + 3 * k, blk);
                int na = ncomp_of(l[I], d_pure), nb = ncomp_of(l[J], d_pure);
                for (int i = 0; i < na; ++i)
                    for (int j = 0; j < nb; ++j) nsum(&sum, &comp, P[(bo[I] + i) * ldp + bo[J] + j] * blk[i * nb + j]);
            }
        v_out[s] = sum + comp;
    }
    free(mask); free(moff); free(po); free(bo);
}

/* ------------------------------------------------------------------------------------
 * F_mu,nu = sum_k q_k (mu|J_k|nu), Eq. 10 with reading R2 (dF^S = -F), for the listed ORDERED
 * shell pairs (pI[n], pJ[n]); blocks are written back to back into out (block n has
 * ncomp(I)*ncomp(J) doubles, row-major).  (J,I) is computed independently of (I,J) when both
 * are listed, so F = F^T is a property to be tested, not a construction.
 * ---------------------------------------------------------------------------------- */
void orc_fock_blocks(int nshell, const int *l, const double *xyz, const int *nprim, const double *ex, const double *co,
                     int d_pure, long npt, const double *pt_xyz, const double *pt_zeta, const double *q, double cutoff,
                     long npair, const int *pI, const int *pJ, double *out) {
    orc_basis bs = {nshell, l, xyz, nprim, ex, co, d_pure};
    long *po = malloc(sizeof(long) * (nshell + 1)), *bo = malloc(sizeof(long) * (nshell + 1));
    offsets(&bs, po, bo);
    long *ooff = malloc(sizeof(long) * (npair + 1));
    ooff[0] = 0;
    for (long n = 0; n < npair; ++n) ooff[n + 1] = ooff[n] + ncomp_of(l[pI[n]], d_pure) * ncomp_of(l[pJ[n]], d_pure);
#pragma omp parallel for schedule(dynamic, 1)
    for (long n = 0; n < npair; ++n) {
        int I = pI[n], J = pJ[n];
        int nc = (int)(ooff[n + 1] - ooff[n]);
        double sum[36], comp[36], blk[36];
        unsigned char keep[64 * 64];
        unsigned char *kp = keep;
        if (nprim[I] * nprim[J] > 64 * 64) kp = malloc((size_t)nprim[I] * nprim[J]);
        for (int c = 0; c < nc; ++c) { sum[c] = 0.0; comp[c] = 0.0; }
        if (keep_mask(&bs, po, I, J, cutoff, kp)) {
            for (long k = 0; k < npt; ++k) {
                shell_block(&bs, po, I, J, kp, pt_zeta[k], pt_xyz + 3 * k, blk);
                for (int c = 0; c < nc; ++c) nsum(&sum[c], &comp[c], q[k] * blk[c]);
            }
        }
        for (int c = 0; c < nc; ++c) out[ooff[n] + c] = sum[c] + comp[c];
        if (kp != keep) free(kp);
    }
    free(ooff); free(po); free(bo);
}

/* ------------------------------------------------------------------------------------
 * A matrix (Eq. 2, 3, 8 with reading R1):
 *   A_kl = erf(zeta'_kl r_kl)/r_kl,  zeta'_kl = zeta_k zeta_l / sqrt(zeta_k^2 + zeta_l^2),
 *   A_kk = zeta_k sqrt(2/pi) / S_k.   Coincident points (r = 0, a caller error) -> 2 zeta'/sqrt(pi).
 * ---------------------------------------------------------------------------------- */
double orc_a_entry(const double *pt_xyz, const double *pt_zeta, const double *pt_switch, long i, long j) {
    if (i == j) return pt_zeta[i] * sqrt(2.0 / ORC_PI) / (pt_switch ? pt_switch[i] : 1.0);
    double dx = pt_xyz[3 * i] - pt_xyz[3 * j], dy = pt_xyz[3 * i + 1] - pt_xyz[3 * j + 1],
           dz = pt_xyz[3 * i + 2] - pt_xyz[3 * j + 2];
    double r = sqrt(dx * dx + dy * dy + dz * dz);
    double zi = pt_zeta[i], zj = pt_zeta[j];
    double zp = zi * zj / sqrt(zi * zi + zj * zj);
    if (r == 0.0) return 2.0 * zp / sqrt(ORC_PI);
    return erf(zp * r) / r;
}

/* dense A, row-major M x M */
void orc_amatrix(long M, const double *pt_xyz, const double *pt_zeta, const double *pt_switch, double *A) {
#pragma omp parallel for schedule(static)
    for (long i = 0; i < M; ++i)
        for (long j = 0; j < M; ++j) A[i * M + j] = orc_a_entry(pt_xyz, pt_zeta, pt_switch, i, j);
}

/* y_i = sum_j A_ij q_j for rows sel[0..nsel) (NULL: rows 0..nsel-1), on the fly */
void orc_amatvec(long M, const double *pt_xyz, const double *pt_zeta, const double *pt_switch, const double *q, long nsel,
                 const long *sel, double *y) {
#pragma omp parallel for schedule(static)
    for (long s = 0; s < nsel; ++s) {
        long i = sel ? sel[s] : s;
        double sum = 0.0, comp = 0.0;
        for (long j = 0; j < M; ++j) nsum(&sum, &comp, orc_a_entry(pt_xyz, pt_zeta, pt_switch, i, j) * q[j]);
        y[s] = sum + comp;
    }
}

/* ------------------------------------------------------------------------------------
 * Pivot order from a seed: a counter-based generator both sides implement on their own.
 * key_i = splitmix64 finaliser of (seed + (i+1)*0x9E3779B97F4A7C15); perm = indices sorted by (key, index).
 * ---------------------------------------------------------------------------------- */
static uint64_t mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
typedef struct { uint64_t key; long idx; } keyidx;
static int cmp_keyidx(const void *a, const void *b) {
    const keyidx *x = a, *y = b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    return x->idx < y->idx ? -1 : (x->idx > y->idx);
}
void orc_pivot_order(uint64_t seed, long M, long *perm) {
    keyidx *k = malloc(sizeof(keyidx) * (size_t)M);
    for (long i = 0; i < M; ++i) { k[i].key = mix64(seed + (uint64_t)(i + 1) * 0x9E3779B97F4A7C15ULL); k[i].idx = i; }
    qsort(k, (size_t)M, sizeof(keyidx), cmp_keyidx);
    for (long i = 0; i < M; ++i) perm[i] = k[i].idx;
    free(k);
}

/* ------------------------------------------------------------------------------------
 * Randomized block-Jacobi: "randomly select a pivot A_kk, sort the elements of the
 * kth row by descending magnitude, pick the first l column indices and form the first diagonal block
 * of M with the corresponding elements, repeating the procedure for the remaining indices until all
 * rows of A have been accounted for.  The inverse M^-1 is then calculated and its non-zero entries
 * (diagonal blocks) are stored".  Reading R5 for what the text leaves open.
 *   order[M]        : indices, block after block (pivot first, then by descending |A_kj|)
 *   bstart[nb+1]    : block boundaries in order[];  returns nb = ceil(M/l)
 *   inv             : the l_b x l_b inverse blocks, row-major, back to back (sum l_b^2 doubles)
 * ---------------------------------------------------------------------------------- */
typedef struct { double val; long idx; } validx;
static int cmp_validx(const void *a, const void *b) {
    const validx *x = a, *y = b;
    if (x->val != y->val) return x->val > y->val ? -1 : 1; /* descending magnitude */
    return x->idx < y->idx ? -1 : (x->idx > y->idx);       /* ties -> lower index */
}

/* in-place inverse of an SPD n x n matrix through its Cholesky factor; returns 0 on success */
static int spd_inverse(int n, double *a) {
    double *Lm = calloc((size_t)n * n, sizeof(double));
    for (int j = 0; j < n; ++j) {
        double d = a[j * n + j];
        for (int k = 0; k < j; ++k) d -= Lm[j * n + k] * Lm[j * n + k];
        if (!(d > 0.0)) { free(Lm); return -1; }
        Lm[j * n + j] = sqrt(d);
        for (int i = j + 1; i < n; ++i) {
            double s = a[i * n + j];
            for (int k = 0; k < j; ++k) s -= Lm[i * n + k] * Lm[j * n + k];
            Lm[i * n + j] = s / Lm[j * n + j];
        }
    }
    /* solve L L^T X = I column by column */
    double *y = malloc(sizeof(double) * n);
    for (int c = 0; c < n; ++c) {
        for (int i = 0; i < n; ++i) {
            double s = (i == c) ? 1.0 : 0.0;
            for (int k = 0; k < i; ++k) s -= Lm[i * n + k] * y[k];
            y[i] = s / Lm[i * n + i];
        }
        for (int i = n - 1; i >= 0; --i) {
            double s = y[i];
            for (int k = i + 1; k < n; ++k) s -= Lm[k * n + i] * a[k * n + c];
            a[i * n + c] = s / Lm[i * n + i];
        }
    }
    free(y); free(Lm);
    return 0;
}

long orc_rbj_build(long M, const double *pt_xyz, const double *pt_zeta, const double *pt_switch, int l,
                   const long *pivot_order, long *order, long *bstart, double *inv) {
    unsigned char *assigned = calloc((size_t)M, 1);
    validx *cand = malloc(sizeof(validx) * (size_t)M);
    long nb = 0, filled = 0, pos = 0, ioff = 0;
    bstart[0] = 0;
    while (filled < M) {
        while (assigned[pivot_order[pos]]) ++pos;
        long k = pivot_order[pos];
        long nc = 0;
        for (long j = 0; j < M; ++j)
            if (!assigned[j] && j != k) { cand[nc].val = fabs(orc_a_entry(pt_xyz, pt_zeta, pt_switch, k, j)); cand[nc].idx = j; ++nc; }
        qsort(cand, (size_t)nc, sizeof(validx), cmp_validx);
        long take = nc < l - 1 ? nc : l - 1;
        order[filled] = k; assigned[k] = 1;
        for (long t = 0; t < take; ++t) { order[filled + 1 + t] = cand[t].idx; assigned[cand[t].idx] = 1; }
        int n = (int)(take + 1);
        double *blk = inv + ioff;
        for (int r = 0; r < n; ++r)
            for (int c = 0; c < n; ++c)
                blk[r * n + c] = orc_a_entry(pt_xyz, pt_zeta, pt_switch, order[filled + r], order[filled + c]);
        if (spd_inverse(n, blk)) { free(assigned); free(cand); return -1; }
        ioff += (long)n * n;
        filled += n;
        bstart[++nb] = filled;
    }
    free(assigned); free(cand);
    return nb;
}

/* z = C r : precond 0 none, 1 Jacobi (C = diag(A)^-1), 2 RBJ (C = P M^-1 P) */
static void apply_precond(int precond, long M, const double *diagA, long nb, const long *order, const long *bstart,
                          const double *inv, const double *r, double *z) {
    if (precond == 0) { memcpy(z, r, sizeof(double) * (size_t)M); return; }
    if (precond == 1) { for (long i = 0; i < M; ++i) z[i] = r[i] / diagA[i]; return; }
    long ioff = 0;
    for (long b = 0; b < nb; ++b) {
        long n = bstart[b + 1] - bstart[b];
        const long *idx = order + bstart[b];
        for (long i = 0; i < n; ++i) {
            double s = 0.0, c = 0.0;
            for (long j = 0; j < n; ++j) nsum(&s, &c, inv[ioff + i * n + j] * r[idx[j]]);
            z[idx[i]] = s + c;
        }
        ioff += n * n;
    }
}

static double dotc(long n, const double *a, const double *b) {
    double s = 0.0, c = 0.0;
    for (long i = 0; i < n; ++i) nsum(&s, &c, a[i] * b[i]);
    return s + c;
}

static void matvec(long M, const double *Adense, const double *pt_xyz, const double *pt_zeta, const double *pt_switch,
                   const double *x, double *y) {
    if (!Adense) { orc_amatvec(M, pt_xyz, pt_zeta, pt_switch, x, M, NULL, y); return; }
#pragma omp parallel for schedule(static)
    for (long i = 0; i < M; ++i) {
        double s = 0.0, c = 0.0;
        for (long j = 0; j < M; ++j) nsum(&s, &c, Adense[i * M + j] * x[j]);
        y[i] = s + c;
    }
}

/* ------------------------------------------------------------------------------------
 * Preconditioned conjugate gradient on A x = b (textbook PCG, the paper's ref. 33):
 *   r0 = b - A x0, z0 = C r0, p0 = z0
 *   repeat: stop if ||r||_2 <= tol;  alpha = (r.z)/(p.Ap);  x += alpha p;  r -= alpha Ap;
 *           z = C r;  beta = (r.z)_new/(r.z)_old;  p = z + beta p
 * Adense (row-major M x M, the paper's stored A) may be NULL -> entries on the fly.
 * Returns the number of iterations (matrix-vector products after the initial residual);
 * resid[0] = final recurrence ||r||, resid[1] = true ||b - A x||.  -1: max_iter reached is NOT an
 * error here: the count returned is then max_iter and resid says how far it got.
 * ---------------------------------------------------------------------------------- */
long orc_pcg(long M, const double *Adense, const double *pt_xyz, const double *pt_zeta, const double *pt_switch,
             const double *b, double *x, int use_x0, double tol, long max_iter, int precond, long nb, const long *order,
             const long *bstart, const double *inv, double *resid, double *resid_history) {
    double *r = malloc(sizeof(double) * M), *z = malloc(sizeof(double) * M), *p = malloc(sizeof(double) * M),
           *Ap = malloc(sizeof(double) * M), *dg = malloc(sizeof(double) * M);
    for (long i = 0; i < M; ++i) dg[i] = orc_a_entry(pt_xyz, pt_zeta, pt_switch, i, i);
    if (!use_x0) memset(x, 0, sizeof(double) * (size_t)M);
    if (use_x0) {
        matvec(M, Adense, pt_xyz, pt_zeta, pt_switch, x, Ap);
        for (long i = 0; i < M; ++i) r[i] = b[i] - Ap[i];
    } else memcpy(r, b, sizeof(double) * (size_t)M);
    apply_precond(precond, M, dg, nb, order, bstart, inv, r, z);
    memcpy(p, z, sizeof(double) * (size_t)M);
    double rz = dotc(M, r, z);
    long it = 0;
    double rn = sqrt(dotc(M, r, r));
    if (resid_history) resid_history[0] = rn;
    while (rn > tol && it < max_iter) {
        matvec(M, Adense, pt_xyz, pt_zeta, pt_switch, p, Ap);
        double alpha = rz / dotc(M, p, Ap);
        for (long i = 0; i < M; ++i) { x[i] += alpha * p[i]; r[i] -= alpha * Ap[i]; }
        apply_precond(precond, M, dg, nb, order, bstart, inv, r, z);
        double rz_new = dotc(M, r, z);
        double beta = rz_new / rz;
        for (long i = 0; i < M; ++i) p[i] = z[i] + beta * p[i];
        rz = rz_new;
        ++it;
        rn = sqrt(dotc(M, r, r));
        if (resid_history) resid_history[it] = rn;
    }
    resid[0] = rn;
    matvec(M, Adense, pt_xyz, pt_zeta, pt_switch, x, Ap);
    double s = 0.0, c = 0.0;
    for (long i = 0; i < M; ++i) nsum(&s, &c, (b[i] - Ap[i]) * (b[i] - Ap[i]));
    resid[1] = sqrt(s + c);
    free(r); free(z); free(p); free(Ap); free(dg);
    return it;
}

/* ------------------------------------------------------------------------------------
 * The rest of one C-PCM step around the hot path.
 *   B z  (Eq. 4):  u_k = sum_J z_J erf(zeta_k |r_k - R_J|)/|r_k - R_J|; a nucleus is a point
 *        charge, so the exponent is the surface point's own zeta_k.  r = 0 -> 2 zeta_k/sqrt(pi) (the limit).
 *   right-hand side of Eq. 1 with the library's sign (reading R2: c = -v):  b = -f (B z - v),  f = (eps-1)/(eps+k)
 *   Delta G_els (Eq. 13):  (B z).q + c.q + (1/2f) q.A q  with c = -v; out[0..2] the three terms, out[3] the sum
 *   dynamic CG threshold (Eq. 21; reading R10 in DESIGN.md): the delta for which
 *        Err(delta) = 0.01 delta^1.07 equals 1e-3 x the previous SCF step's DIIS error; delta = 1 on the first SCF
 *        iteration (no previous error: diis_prev <= 0); never tighter than delta_min, never looser than 1.
 * ---------------------------------------------------------------------------------- */
void orc_bz(long M, const double *pt_xyz, const double *pt_zeta, long N, const double *atom_xyz, const double *z, double *u) {
#pragma omp parallel for schedule(static)
    for (long k = 0; k < M; ++k) {
        double sum = 0.0, comp = 0.0;
        for (long J = 0; J < N; ++J) {
            double dx = pt_xyz[3 * k] - atom_xyz[3 * J], dy = pt_xyz[3 * k + 1] - atom_xyz[3 * J + 1],
                   dz = pt_xyz[3 * k + 2] - atom_xyz[3 * J + 2];
            double r = sqrt(dx * dx + dy * dy + dz * dz);
            double B = r == 0.0 ? 2.0 * pt_zeta[k] / sqrt(ORC_PI) : erf(pt_zeta[k] * r) / r;
            nsum(&sum, &comp, z[J] * B);
        }
        u[k] = sum + comp;
    }
}

void orc_rhs(long M, const double *u, const double *v, double f, double *b) {
    for (long k = 0; k < M; ++k) b[k] = -f * (u[k] - v[k]);
}

void orc_energy(long M, const double *u, const double *v, const double *q, const double *Aq, double f, double *out) {
    double s0 = 0, c0 = 0, s1 = 0, c1 = 0, s2 = 0, c2 = 0;
    for (long k = 0; k < M; ++k) {
        nsum(&s0, &c0, u[k] * q[k]);
        nsum(&s1, &c1, -v[k] * q[k]);
        nsum(&s2, &c2, q[k] * Aq[k]);
    }
    out[0] = s0 + c0;
    out[1] = s1 + c1;
    out[2] = (s2 + c2) / (2.0 * f);
    out[3] = out[0] + out[1] + out[2];
}

double orc_cg_threshold(double diis_prev, double delta_min) {
    if (!(diis_prev > 0.0)) return 1.0;
    double delta = pow(1e-3 * diis_prev / 0.01, 1.0 / 1.07);
    if (delta > 1.0) delta = 1.0;
    if (delta < delta_min) delta = delta_min;
    return delta;
}

/* ------------------------------------------------------------------------------------
 * Gradient of E = v.q = sum_k q_k sum_{mu,nu} P_mu,nu (mu|J_k|nu) with respect to the shell centres and the
 * surface points at fixed P and q: the one-electron part (grad* c^T) q of Eq. 14, PAPER.md:202-218 (Eq. 22:
 * ga, gb per primitive pair, gc per point).  Library sign (reading R2): the paper's c = -v, so its term is -E.
 *   [d/dA_x chi_a | J | chi_b] = 2 alpha [a+1_x|J|b] - a_x [a-1_x|J|b]      (derivative of a Cartesian Gaussian)
 *   [chi_a | J | d/dB_x chi_b] = 2 beta  [a|J|b+1_x] - b_x [a|J|b-1_x]
 *   [chi_a | d/dC_x J | chi_b] = -(d/dA_x + d/dB_x)[a|J|b]                  (the integral depends on A-C, B-C only)
 * each bracket on the right by the Obara-Saika tables above.  zeta_k does not move with the point (Eq. 7).
 *   g_shell[S] = sum_J sum_k q_k ( P_{S,J} . d/dA (S J|J_k)  +  P_{J,S} . d/dB (J S|J_k) )     (S as bra and as ket)
 *   g_point[k] = q_k sum_{I,J} P_{I,J} . d/dC (I J|J_k)
 * ---------------------------------------------------------------------------------- */
typedef double hrr_table[NB * NB * NB][NA * NA * NA];

/* Cartesian derivative blocks of one primitive pair at one point: dA[x][ia*NCART[lb]+ib], dB likewise */
static void prim_deriv_blocks(int la, double alpha, const double *A, int lb, double beta, const double *B, double zeta,
                              const double *C, double dA[3][36], double dB[3][36]) {
    static _Thread_local hrr_table up, dn;
    /* bra raised / lowered */
    os_tables(la + 1, alpha, A, lb, beta, B, zeta, C, 0, up);
    if (la > 0) os_tables(la - 1, alpha, A, lb, beta, B, zeta, C, 0, dn);
    for (int ia = 0; ia < NCART[la]; ++ia)
        for (int ib = 0; ib < NCART[lb]; ++ib) {
            const int *a = CART[la][ia], *b = CART[lb][ib];
            for (int x = 0; x < 3; ++x) {
                int ap[3] = {a[0], a[1], a[2]}, am[3] = {a[0], a[1], a[2]};
                ap[x] += 1; am[x] -= 1;
                double v = 2.0 * alpha * up[BIDX(b[0], b[1], b[2])][AIDX(ap[0], ap[1], ap[2])];
                if (a[x] > 0) v -= a[x] * dn[BIDX(b[0], b[1], b[2])][AIDX(am[0], am[1], am[2])];
                dA[x][ia * NCART[lb] + ib] = v;
            }
        }
    /* ket raised / lowered */
    os_tables(la, alpha, A, lb + 1, beta, B, zeta, C, 0, up);
    if (lb > 0) os_tables(la, alpha, A, lb - 1, beta, B, zeta, C, 0, dn);
    for (int ia = 0; ia < NCART[la]; ++ia)
        for (int ib = 0; ib < NCART[lb]; ++ib) {
            const int *a = CART[la][ia], *b = CART[lb][ib];
            for (int x = 0; x < 3; ++x) {
                int bp[3] = {b[0], b[1], b[2]}, bm[3] = {b[0], b[1], b[2]};
                bp[x] += 1; bm[x] -= 1;
                double v = 2.0 * beta * up[BIDX(bp[0], bp[1], bp[2])][AIDX(a[0], a[1], a[2])];
                if (b[x] > 0) v -= b[x] * dn[BIDX(bm[0], bm[1], bm[2])][AIDX(a[0], a[1], a[2])];
                dB[x][ia * NCART[lb] + ib] = v;
            }
        }
}

/* public: the derivative blocks of one primitive pair (for the pins) */
void orc_prim_deriv(int la, double alpha, const double *A, int lb, double beta, const double *B, double zeta, const double *C,
                    double *dA_out, double *dB_out) {
    double dA[3][36], dB[3][36];
    prim_deriv_blocks(la, alpha, A, lb, beta, B, zeta, C, dA, dB);
    int n = NCART[la] * NCART[lb];
    for (int x = 0; x < 3; ++x)
        for (int c = 0; c < n; ++c) { dA_out[x * n + c] = dA[x][c]; dB_out[x * n + c] = dB[x][c]; }
}

/* contracted component blocks of d/dA and d/dB of (mu in I, nu in J | J_k): outA[x][ncompI*ncompJ], outB likewise */
static void shell_deriv_block(const orc_basis *bs, const long *po, int I, int J, const unsigned char *keep, double zeta,
                              const double *C, double outA[3][36], double outB[3][36]) {
    int la = bs->l[I], lb = bs->l[J];
    double cA[3][36], cB[3][36], pA[3][36], pB[3][36];
    int n = NCART[la] * NCART[lb];
    for (int x = 0; x < 3; ++x)
        for (int c = 0; c < n; ++c) { cA[x][c] = 0.0; cB[x][c] = 0.0; }
    for (int i = 0; i < bs->nprim[I]; ++i)
        for (int j = 0; j < bs->nprim[J]; ++j) {
            if (keep && !keep[i * bs->nprim[J] + j]) continue;
            prim_deriv_blocks(la, bs->ex[po[I] + i], bs->xyz + 3 * I, lb, bs->ex[po[J] + j], bs->xyz + 3 * J, zeta, C, pA, pB);
            double cc = bs->co[po[I] + i] * bs->co[po[J] + j];
            for (int x = 0; x < 3; ++x)
                for (int c = 0; c < n; ++c) { cA[x][c] += cc * pA[x][c]; cB[x][c] += cc * pB[x][c]; }
        }
    for (int x = 0; x < 3; ++x) {
        to_components(la, lb, bs->d_pure, cA[x], outA[x]);
        to_components(la, lb, bs->d_pure, cB[x], outB[x]);
    }
}

/* g_shell_out[3*nselS]: gradient with respect to the centres of the shells selS[0..nselS) (NULL: shells 0..nselS-1);
 * g_point_out[3*nselK]: gradient with respect to the positions of the points selK[0..nselK) (NULL: 0..nselK-1).
 * Every sum runs over the full square of shell pairs and over all npt points. */
void orc_gradient(int nshell, const int *l, const double *xyz, const int *nprim, const double *ex, const double *co,
                  int d_pure, long npt, const double *pt_xyz, const double *pt_zeta, const double *q, const double *P,
                  long ldp, double cutoff, long nselS, const long *selS, long nselK, const long *selK,
                  double *g_shell_out, double *g_point_out) {
    orc_basis bs = {nshell, l, xyz, nprim, ex, co, d_pure};
    long *po = malloc(sizeof(long) * (nshell + 1)), *bo = malloc(sizeof(long) * (nshell + 1));
    offsets(&bs, po, bo);
    long *moff = malloc(sizeof(long) * (size_t)nshell * nshell);
    long tot = 0;
    for (int I = 0; I < nshell; ++I)
        for (int J = 0; J < nshell; ++J) { moff[(long)I * nshell + J] = tot; tot += nprim[I] * nprim[J]; }
    unsigned char *mask = malloc((size_t)tot + 1);
#pragma omp parallel for schedule(dynamic, 8)
    for (int I = 0; I < nshell; ++I)
        for (int J = 0; J < nshell; ++J) {
            long o = moff[(long)I * nshell + J];
            if (!keep_mask(&bs, po, I, J, cutoff, mask + o)) moff[(long)I * nshell + J] = -1;
        }
    /* shells: one (selected shell, partner shell) pair per task, partner sums added in order afterwards */
    double *part = calloc((size_t)(nselS > 0 ? nselS : 1) * nshell * 3, sizeof(double));
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (long s = 0; s < nselS; ++s)
        for (int J = 0; J < nshell; ++J) {
            int S = (int)(selS ? selS[s] : s);
            int nS = ncomp_of(l[S], d_pure), nJ = ncomp_of(l[J], d_pure);
            long o_sj = moff[(long)S * nshell + J], o_js = moff[(long)J * nshell + S];
            double sum[3] = {0, 0, 0}, comp[3] = {0, 0, 0}, dA[3][36], dB[3][36];
            for (long k = 0; k < npt; ++k) {
                if (o_sj >= 0) {   /* S as the bra */
                    shell_deriv_block(&bs, po, S, J, mask + o_sj, pt_zeta[k], pt_xyz + 3 * k, dA, dB);
                    for (int x = 0; x < 3; ++x)
                        for (int i = 0; i < nS; ++i)
                            for (int j = 0; j < nJ; ++j)
                                nsum(&sum[x], &comp[x], q[k] * P[(bo[S] + i) * ldp + bo[J] + j] * dA[x][i * nJ + j]);
                }
                if (o_js >= 0) {   /* S as the ket */
                    shell_deriv_block(&bs, po, J, S, mask + o_js, pt_zeta[k], pt_xyz + 3 * k, dA, dB);
                    for (int x = 0; x < 3; ++x)
                        for (int j = 0; j < nJ; ++j)
                            for (int i = 0; i < nS; ++i)
                                nsum(&sum[x], &comp[x], q[k] * P[(bo[J] + j) * ldp + bo[S] + i] * dB[x][j * nS + i]);
                }
            }
            for (int x = 0; x < 3; ++x) part[((size_t)s * nshell + J) * 3 + x] = sum[x] + comp[x];
        }
    for (long s = 0; s < nselS; ++s)
        for (int x = 0; x < 3; ++x) {
            double sum = 0.0, comp = 0.0;
            for (int J = 0; J < nshell; ++J) nsum(&sum, &comp, part[((size_t)s * nshell + J) * 3 + x]);
            g_shell_out[3 * s + x] = sum + comp;
        }
    free(part);
    /* points */
#pragma omp parallel for schedule(dynamic, 1)
    for (long s = 0; s < nselK; ++s) {
        long k = selK ? selK[s] : s;
        double sum[3] = {0, 0, 0}, comp[3] = {0, 0, 0}, dA[3][36], dB[3][36];
        for (int I = 0; I < nshell; ++I)
            for (int J = 0; J < nshell; ++J) {
                long o = moff[(long)I * nshell + J];
                if (o < 0) continue;
                shell_deriv_block(&bs, po, I, J, mask + o, pt_zeta[k], pt_xyz + 3 * k, dA, dB);
                int na = ncomp_of(l[I], d_pure), nb = ncomp_of(l[J], d_pure);
                for (int x = 0; x < 3; ++x)
                    for (int i = 0; i < na; ++i)
                        for (int j = 0; j < nb; ++j)
                            nsum(&sum[x], &comp[x], -P[(bo[I] + i) * ldp + bo[J] + j] * (dA[x][i * nb + j] + dB[x][i * nb + j]));
            }
        for (int x = 0; x < 3; ++x) g_point_out[3 * s + x] = q[k] * (sum[x] + comp[x]);
    }
    free(mask); free(moff); free(po); free(bo);
}

/* ------------------------------------------------------------------------------------
 * ISWIG switching function (Eq. 9) and the surface terms of the gradient (Eq. 14):
 *   S_k = prod_{J != I(k)} S_wf(r_k, R_J),   I(k) = the atom that owns point k,
 *   S_wf = 1 - (1/2) { erf[zeta_k (R_J - d)] + erf[zeta_k (R_J + d)] },  d = |r_k - R_J|, R_J = cavity radius of atom J.
 * Gradient of  E_s = (B z).q + (1/2f) q.A q  at fixed q with respect to point positions r_k and atom positions R_J
 * (as nuclei and as sphere centres), everything else held fixed -- the caller adds a point's row to its owning atom,
 * because "each MS point only moves with the atom on which it is centered".  With g(z', r) =
 * d/dr [erf(z' r)/r] = (2 z'/sqrt pi) exp(-z'^2 r^2)/r - erf(z' r)/r^2   (0 at r = 0):
 *   B term      z_J q_k g(zeta_k, d_kJ) (r_k - R_J)/d_kJ                      -> + point k, - atom J
 *   A, k != l   (1/f) q_k q_l g(zeta'_kl, r_kl) (r_k - r_l)/r_kl             -> point k  (both orders of the pair)
 *   A_kk        -(1/2f) q_k^2 A_kk (dS_wf/dd)/S_wf (r_k - R_J)/d_kJ, J != I(k) -> + point k, - atom J,
 *               dS_wf/dd = (zeta_k/sqrt pi) { exp[-zeta_k^2 (R_J - d)^2] - exp[-zeta_k^2 (R_J + d)^2] }
 * ---------------------------------------------------------------------------------- */
static double swf(double zeta, double R, double d) { return 1.0 - 0.5 * (erf(zeta * (R - d)) + erf(zeta * (R + d))); }
static double dswf(double zeta, double R, double d) {
    return zeta / sqrt(ORC_PI) * (exp(-zeta * zeta * (R - d) * (R - d)) - exp(-zeta * zeta * (R + d) * (R + d)));
}
static double dcoul(double zp, double r) {
    if (r == 0.0) return 0.0;
    return 2.0 * zp / sqrt(ORC_PI) * exp(-zp * zp * r * r) / r - erf(zp * r) / (r * r);
}

void orc_switching(long M, const double *pt_xyz, const double *pt_zeta, const long *pt_atom, long N, const double *atom_xyz,
                   const double *atom_radius, double *S) {
#pragma omp parallel for schedule(static)
    for (long k = 0; k < M; ++k) {
        double s = 1.0;
        for (long J = 0; J < N; ++J) {
            if (J == pt_atom[k]) continue;
            double dx = pt_xyz[3 * k] - atom_xyz[3 * J], dy = pt_xyz[3 * k + 1] - atom_xyz[3 * J + 1],
                   dz = pt_xyz[3 * k + 2] - atom_xyz[3 * J + 2];
            s *= swf(pt_zeta[k], atom_radius[J], sqrt(dx * dx + dy * dy + dz * dz));
        }
        S[k] = s;
    }
}

void orc_surface_gradient(long M, const double *pt_xyz, const double *pt_zeta, const long *pt_atom, long N,
                          const double *atom_xyz, const double *atom_radius, const double *z, const double *q, double f,
                          double *g_point, double *g_atom) {
    double *S = malloc(sizeof(double) * (size_t)(M > 0 ? M : 1));
    orc_switching(M, pt_xyz, pt_zeta, pt_atom, N, atom_xyz, atom_radius, S);
    /* per (point, atom) pair force, kept so that the atom rows can be summed in point order afterwards */
    double *pa = calloc((size_t)(M > 0 ? M : 1) * (size_t)(N > 0 ? N : 1) * 3, sizeof(double));
#pragma omp parallel for schedule(static)
    for (long k = 0; k < M; ++k) {
        double sum[3] = {0, 0, 0}, comp[3] = {0, 0, 0};
        const double zk = pt_zeta[k], akk = zk * sqrt(2.0 / ORC_PI) / S[k];
        for (long J = 0; J < N; ++J) {
            double e[3] = {pt_xyz[3 * k] - atom_xyz[3 * J], pt_xyz[3 * k + 1] - atom_xyz[3 * J + 1], pt_xyz[3 * k + 2] - atom_xyz[3 * J + 2]};
            double d = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]);
            if (d == 0.0) continue;
            double w = z[J] * q[k] * dcoul(zk, d);
            if (J != pt_atom[k]) w += -0.5 / f * q[k] * q[k] * akk * dswf(zk, atom_radius[J], d) / swf(zk, atom_radius[J], d);
            for (int x = 0; x < 3; ++x) {
                double t = w * e[x] / d;
                nsum(&sum[x], &comp[x], t);
                pa[((size_t)k * N + J) * 3 + x] = t;
            }
        }
        for (long l = 0; l < M; ++l) {
            if (l == k) continue;
            double e[3] = {pt_xyz[3 * k] - pt_xyz[3 * l], pt_xyz[3 * k + 1] - pt_xyz[3 * l + 1], pt_xyz[3 * k + 2] - pt_xyz[3 * l + 2]};
            double r = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]);
            if (r == 0.0) continue;
            double zl = pt_zeta[l], zp = zk * zl / sqrt(zk * zk + zl * zl);
            double w = q[k] * q[l] / f * dcoul(zp, r);
            for (int x = 0; x < 3; ++x) nsum(&sum[x], &comp[x], w * e[x] / r);
        }
        for (int x = 0; x < 3; ++x) g_point[3 * k + x] = sum[x] + comp[x];
    }
    for (long J = 0; J < N; ++J)
        for (int x = 0; x < 3; ++x) {
            double s = 0.0, c = 0.0;
            for (long k = 0; k < M; ++k) nsum(&s, &c, -pa[((size_t)k * N + J) * 3 + x]);
            g_atom[3 * J + x] = s + c;
        }
    free(pa); free(S);
}

/* ------------------------------------------------------------------------------------
 * ISWIG cavity construction (Eq. 7 and Eq. 9, PAPER.md:106 the 1e-8 screening).
 * Every atom I (centre R_I, cavity radius rad_I) carries the same unit-sphere quadrature: nodes u_g, |u_g| = 1, with
 * weights w_g, sum_g w_g = 4 pi (the paper uses Lebedev grids; the grid is an INPUT here).  For every (I, g):
 *     r     = R_I + rad_I u_g
 *     zeta  = zeta_tab / (rad_I sqrt(w_g))                                     Eq. 7
 *     S     = prod_{J != I} S_wf(r, R_J)                                       Eq. 9 (reading R13: J runs over the other atoms)
 * and the point is kept iff S >= s_min ("MS points with a switching function value less than this threshold are
 * ignored"; the paper's threshold is 1e-8).  Output order: atom after atom, node index ascending.
 * The arrays must hold N*G entries; the return value is the number of points kept.
 * Pins: tests/test_oracle_cavity.py.
 * ---------------------------------------------------------------------------------- */
long orc_build_cavity(long N, const double *atom_xyz, const double *atom_radius, long G, const double *unit, const double *w,
                      double zeta_tab, double s_min, double *pt_xyz, double *pt_zeta, double *pt_S, long *pt_atom, long *pt_node) {
    long n = 0;
    for (long I = 0; I < N; ++I)
        for (long g = 0; g < G; ++g) {
            double r[3];
            for (int x = 0; x < 3; ++x) r[x] = atom_xyz[3 * I + x] + atom_radius[I] * unit[3 * g + x];
            double zeta = zeta_tab / (atom_radius[I] * sqrt(w[g]));
            double S = 1.0;
            for (long J = 0; J < N; ++J) {
                if (J == I) continue;
                double dx = r[0] - atom_xyz[3 * J], dy = r[1] - atom_xyz[3 * J + 1], dz = r[2] - atom_xyz[3 * J + 2];
                S *= swf(zeta, atom_radius[J], sqrt(dx * dx + dy * dy + dz * dz));
            }
            if (!(S >= s_min)) continue;
            pt_xyz[3 * n] = r[0]; pt_xyz[3 * n + 1] = r[1]; pt_xyz[3 * n + 2] = r[2];
            pt_zeta[n] = zeta; pt_S[n] = S; pt_atom[n] = I; pt_node[n] = g;
            ++n;
        }
    return n;
}
