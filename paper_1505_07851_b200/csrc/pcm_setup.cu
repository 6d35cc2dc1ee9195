// pcm_setup.cu -- host side of step a1: shell-pair enumeration, Eq. 15 screening,
// Hermite Gaussian product merging, class sort, SoA packing and upload.  Also the Boys tables.
#include <algorithm>
#include <chrono>
#include <array>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "pcm_internal.h"

namespace pcm {

static thread_local std::string g_setup_error;

int set_error(pcm_ctx *ctx, int code, const std::string &msg) {
    if (ctx) ctx->err = msg; else g_setup_error = msg;
    return code;
}
const char *setup_error_text() { return g_setup_error.c_str(); }

int dev_alloc(pcm_ctx *ctx, void **p, size_t bytes) {
    *p = nullptr;
    if (bytes == 0) bytes = 8;
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) return set_error(ctx, PCM_ERR_ALLOC, std::string("cudaMalloc: ") + cudaGetErrorString(e));
    ctx->allocs.push_back(*p);
    ctx->device_bytes += (int64_t)bytes;
    return PCM_OK;
}

// ---------------------------------------------------------------------------------------------
// Boys tables.  F_n(T) = int_0^1 t^2n exp(-T t^2) dt.  Highest order by the all-positive series
//   F_n(T) = exp(-T) sum_k (2T)^k / ((2n+1)(2n+3)...(2n+2k+1))
// in long double, lower orders by downward recursion F_{n-1} = (2T F_n + exp(-T))/(2n-1).
// Row i of table L holds c_k = (-1)^k F_{L+k}(T_i)/k!, k = 0..7 (Taylor coefficients of F_L about T_i:
// dF_n/dT = -F_{n+1}), then exp(-T_i).
// ---------------------------------------------------------------------------------------------
void build_boys_tables(std::vector<double> &tab) {
    const int nmax = MAXLG + BOYS_TERMS - 1;
    tab.assign((size_t)(MAXLG + 1) * BOYS_ROWS * BOYS_STRIDE, 0.0);
    std::vector<long double> F(nmax + 1);
    for (int i = 0; i < BOYS_ROWS; ++i) {
        const long double T = (long double)i / 16.0L;
        const long double eT = expl(-T);
        long double term = 1.0L / (2.0L * nmax + 1.0L), sum = term;
        for (int k = 1; k < 4000; ++k) {
            term *= 2.0L * T / (2.0L * nmax + 2.0L * k + 1.0L);
            sum += term;
            if (term < 1e-22L * sum) break;
        }
        F[nmax] = eT * sum;
        for (int n = nmax; n >= 1; --n) F[n - 1] = (2.0L * T * F[n] + eT) / (2.0L * n - 1.0L);
        for (int L = 0; L <= MAXLG; ++L) {
            double *row = &tab[((size_t)L * BOYS_ROWS + i) * BOYS_STRIDE];
            long double fact = 1.0L;
            for (int k = 0; k < BOYS_TERMS; ++k) {
                if (k > 0) fact *= k;
                row[k] = (double)(((k & 1) ? -1.0L : 1.0L) * F[L + k] / fact);
            }
            row[BOYS_TERMS] = (double)eT;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// One-dimensional Hermite expansion coefficients E^{ij}_t, i, j <= 2 (McMurchie-Davidson):
//   E^{00}_0 = exp(-mu X_AB^2),  E^{i+1,j}_t = E^{ij}_{t-1}/2p + X_PA E^{ij}_t + (t+1) E^{ij}_{t+1}
// ---------------------------------------------------------------------------------------------
struct E1D {
    double e[3][3][5];
};
static void hermite_E(double a, double b, double Ax, double Bx, int la, int lb, E1D &E) {
    const double p = a + b, mu = a * b / p;
    const double Px = (a * Ax + b * Bx) / p;
    const double XPA = Px - Ax, XPB = Px - Bx, XAB = Ax - Bx, h = 0.5 / p;
    std::memset(&E, 0, sizeof(E));
    E.e[0][0][0] = std::exp(-mu * XAB * XAB);
    for (int i = 0; i < la; ++i)
        for (int t = 0; t <= i + 1; ++t)
            E.e[i + 1][0][t] = (t > 0 ? h * E.e[i][0][t - 1] : 0.0) + XPA * E.e[i][0][t] + (t + 1) * (t + 1 <= i ? E.e[i][0][t + 1] : 0.0);
    for (int i = 0; i <= la; ++i)
        for (int j = 0; j < lb; ++j)
            for (int t = 0; t <= i + j + 1; ++t)
                E.e[i][j + 1][t] = (t > 0 ? h * E.e[i][j][t - 1] : 0.0) + XPB * E.e[i][j][t] + (t + 1) * (t + 1 <= i + j ? E.e[i][j][t + 1] : 0.0);
}

// dE^{ij}_t/dX_AB at fixed P (X_PA = -(b/p) X_AB, X_PB = (a/p) X_AB, E^{00}_0 = exp(-mu X_AB^2)): the recursion differentiated
static void hermite_dE(double a, double b, double Ax, double Bx, int la, int lb, const E1D &E, E1D &D) {
    const double p = a + b, mu = a * b / p;
    const double Px = (a * Ax + b * Bx) / p;
    const double XPA = Px - Ax, XPB = Px - Bx, XAB = Ax - Bx, h = 0.5 / p;
    const double dXPA = -b / p, dXPB = a / p;
    std::memset(&D, 0, sizeof(D));
    D.e[0][0][0] = -2.0 * mu * XAB * E.e[0][0][0];
    for (int i = 0; i < la; ++i)
        for (int t = 0; t <= i + 1; ++t)
            D.e[i + 1][0][t] = (t > 0 ? h * D.e[i][0][t - 1] : 0.0) + dXPA * E.e[i][0][t] + XPA * D.e[i][0][t] +
                               (t + 1) * (t + 1 <= i ? D.e[i][0][t + 1] : 0.0);
    for (int i = 0; i <= la; ++i)
        for (int j = 0; j < lb; ++j)
            for (int t = 0; t <= i + j + 1; ++t)
                D.e[i][j + 1][t] = (t > 0 ? h * D.e[i][j][t - 1] : 0.0) + dXPB * E.e[i][j][t] + XPB * D.e[i][j][t] +
                                   (t + 1) * (t + 1 <= i + j ? D.e[i][j][t + 1] : 0.0);
}

static const int CARTS[3][6][3] = {{{0, 0, 0}},
                                   {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}},
                                   {{2, 0, 0}, {1, 1, 0}, {1, 0, 1}, {0, 2, 0}, {0, 1, 1}, {0, 0, 2}}};
static const int NCART[3] = {1, 3, 6};

static double dfact_m1(int T) {  // (T-1)!! for even T >= 0
    double r = 1.0;
    for (int k = T - 1; k > 1; k -= 2) r *= k;
    return r;
}

// max over Cartesian components of [chi_a chi_b|chi_a chi_b]^{1/2} for raw primitives (Eq. 15; closed form
// SURVEY.md 8(c4)): (ab|ab) = 2 pi^{5/2}/(p^2 sqrt(2p)) sum E_tuv E_t'u'v' (-1)^{t'+u'+v'} R_{t+t',u+u',v+v'}(p/2, 0)
double schwarz_bound(int la, double alpha, const double *A, int lb, double beta, const double *B) {
    const double p = alpha + beta;
    E1D Ex, Ey, Ez;
    hermite_E(alpha, beta, A[0], B[0], la, lb, Ex);
    hermite_E(alpha, beta, A[1], B[1], la, lb, Ey);
    hermite_E(alpha, beta, A[2], B[2], la, lb, Ez);
    const double pref = 2.0 * std::pow(M_PI, 2.5) / (p * p * std::sqrt(2.0 * p));
    double best = 0.0;
    for (int ia = 0; ia < NCART[la]; ++ia)
        for (int ib = 0; ib < NCART[lb]; ++ib) {
            const int *a = CARTS[la][ia], *b = CARTS[lb][ib];
            const int nx = a[0] + b[0], ny = a[1] + b[1], nz = a[2] + b[2];
            double s = 0.0;
            for (int t = 0; t <= nx; ++t)
                for (int u = 0; u <= ny; ++u)
                    for (int v = 0; v <= nz; ++v) {
                        const double e1 = Ex.e[a[0]][b[0]][t] * Ey.e[a[1]][b[1]][u] * Ez.e[a[2]][b[2]][v];
                        if (e1 == 0.0) continue;
                        for (int t2 = (t & 1); t2 <= nx; t2 += 2)
                            for (int u2 = (u & 1); u2 <= ny; u2 += 2)
                                for (int v2 = (v & 1); v2 <= nz; v2 += 2) {
                                    const double e2 = Ex.e[a[0]][b[0]][t2] * Ey.e[a[1]][b[1]][u2] * Ez.e[a[2]][b[2]][v2];
                                    const int T = t + t2, U = u + u2, V = v + v2, n = (T + U + V) / 2;
                                    const double R = std::pow(-p, n) * dfact_m1(T) * dfact_m1(U) * dfact_m1(V) / (2.0 * n + 1.0);
                                    s += (((t2 + u2 + v2) & 1) ? -1.0 : 1.0) * e1 * e2 * R;
                                }
                    }
            best = std::max(best, pref * s);
        }
    return std::sqrt(std::max(best, 0.0));
}

// rows: pure component, cols: Cartesian d (xx,xy,xz,yy,yz,zz); identity-like for s, p and Cartesian d
static void component_matrix(int l, int d_pure, double m[6][6], int &ncomp) {
    std::memset(m, 0, sizeof(double) * 36);
    if (l < 2 || !d_pure) {
        ncomp = NCART[l];
        for (int i = 0; i < ncomp; ++i) m[i][i] = 1.0;
        return;
    }
    const double s3 = std::sqrt(3.0);
    ncomp = 5;
    m[0][1] = s3;
    m[1][4] = s3;
    m[2][5] = 1.0; m[2][0] = -0.5; m[2][3] = -0.5;
    m[3][2] = s3;
    m[4][0] = 0.5 * s3; m[4][3] = -0.5 * s3;
}

static inline uint64_t spread21(uint64_t x) {
    x &= 0x1fffff;
    x = (x | x << 32) & 0x1f00000000ffffULL;
    x = (x | x << 16) & 0x1f0000ff0000ffULL;
    x = (x | x << 8) & 0x100f00f00f00f00fULL;
    x = (x | x << 4) & 0x10c30c30c30c30c3ULL;
    x = (x | x << 2) & 0x1249249249249249ULL;
    return x;
}

// Hilbert-curve key of a cell (x, y, z), 21 bits per axis (Skilling's transpose algorithm): unlike the Morton order,
// consecutive keys are always adjacent cells, so 32 consecutive objects of the sorted order stay compact in space.
static inline uint64_t hilbert_key(uint64_t x, uint64_t y, uint64_t z) {
    uint64_t X[3] = {x & 0x1fffff, y & 0x1fffff, z & 0x1fffff};
    const uint64_t Mb = 1ULL << 20;
    for (uint64_t Q = Mb; Q > 1; Q >>= 1) {
        const uint64_t P = Q - 1;
        for (int i = 0; i < 3; ++i) {
            if (X[i] & Q) X[0] ^= P;
            else { const uint64_t t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
        }
    }
    X[1] ^= X[0];
    X[2] ^= X[1];
    uint64_t t = 0;
    for (uint64_t Q = Mb; Q > 1; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1;
    for (int i = 0; i < 3; ++i) X[i] ^= t;
    return (spread21(X[0]) << 2) | (spread21(X[1]) << 1) | spread21(X[2]);
}

struct HostMember {
    int32_t sp;       // shell pair (final index)
    int32_t prod;     // product (temporary index, remapped after the sort)
    int8_t L;         // la + lb
    int64_t goff;
};
struct HostPair {
    int I, J, cls;
    std::vector<std::pair<int, int>> prims;  // surviving (i, j)
};

template <class T>
static int upload(pcm_ctx *ctx, T **dst, const std::vector<T> &src) {
    int rc = dev_alloc_t(ctx, dst, src.size());
    if (rc) return rc;
    if (!src.empty()) PCM_CUDA(ctx, cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return PCM_OK;
}

// Group boxes: 7 doubles per group of 32 sorted objects -- lo xyz, hi xyz, largest far-field radius^2 in the group.
struct GroupBoxes {
    std::vector<double> b;
    int64_t n() const { return (int64_t)b.size() / 7; }
};
static double box_gap2(const double *a, const double *b) {
    double s = 0.0;
    for (int d = 0; d < 3; ++d) {
        const double g = std::max(std::max(a[d] - b[3 + d], b[d] - a[3 + d]), 0.0);
        s += g * g;
    }
    return s;
}
// patch (rg, cg) is far when the boxes are further apart than both groups' far-field radii (1 % margin)
static int build_patch_map(pcm_ctx *ctx, const GroupBoxes &rows, const GroupBoxes &cols, PatchMap &pm, bool keep_host = false) {
    const int64_t nrg = rows.n(), ncg = cols.n(), nbyte = (ncg + 7) / 8;
    pm.nrg = nrg; pm.ncg = ncg; pm.nbyte = nbyte;
    std::vector<uint8_t> far((size_t)std::max<int64_t>(nrg * nbyte, 1), 0);
    std::vector<int64_t> start((size_t)nrg + 1, 0);
#pragma omp parallel for schedule(static)
    for (int64_t rg = 0; rg < nrg; ++rg) {
        const double *a = &rows.b[(size_t)rg * 7];
        int64_t cnt = 0;
        for (int64_t cg = 0; cg < ncg; ++cg) {
            const double *c = &cols.b[(size_t)cg * 7];
            if (box_gap2(a, c) > 1.01 * std::max(a[6], c[6])) far[(size_t)rg * nbyte + cg / 8] |= (uint8_t)(1u << (cg & 7));
            else ++cnt;
        }
        start[rg + 1] = cnt;
    }
    for (int64_t rg = 0; rg < nrg; ++rg) start[rg + 1] += start[rg];
    std::vector<int32_t> list((size_t)std::max<int64_t>(start[nrg], 1), 0);
#pragma omp parallel for schedule(static)
    for (int64_t rg = 0; rg < nrg; ++rg) {
        int64_t o = start[rg];
        for (int64_t cg = 0; cg < ncg; ++cg)
            if (!((far[(size_t)rg * nbyte + cg / 8] >> (cg & 7)) & 1)) list[o++] = (int32_t)cg;
    }
    pm.nnear = start[nrg];
    // near-kernel work items: each row group's list is cut into pieces of at most NEAR_PIECE patches
    std::vector<int64_t> pstart((size_t)nrg + 1, 0);
    for (int64_t rg = 0; rg < nrg; ++rg) pstart[rg + 1] = pstart[rg] + (start[rg + 1] - start[rg] + NEAR_PIECE - 1) / NEAR_PIECE;
    pm.npiece = pstart[nrg];
    std::vector<int32_t> piece_rg((size_t)std::max<int64_t>(pm.npiece, 1), 0);
    for (int64_t rg = 0; rg < nrg; ++rg)
        for (int64_t q = pstart[rg]; q < pstart[rg + 1]; ++q) piece_rg[q] = (int32_t)rg;
    if (getenv("PCM_VERBOSE")) {
        int64_t mx = 0;
        for (int64_t rg = 0; rg < nrg; ++rg) mx = std::max(mx, start[rg + 1] - start[rg]);
        fprintf(stderr, "[pcm] patch map %lld x %lld: near %lld (%.2f %%), longest list %lld\n", (long long)nrg, (long long)ncg,
                (long long)pm.nnear, 100.0 * (double)pm.nnear / std::max<double>(1.0, (double)nrg * (double)ncg), (long long)mx);
    }
    int rc;
    if ((rc = upload(ctx, &pm.far, far))) return rc;
    if ((rc = upload(ctx, &pm.start, start))) return rc;
    if ((rc = upload(ctx, &pm.pstart, pstart))) return rc;
    if ((rc = upload(ctx, &pm.piece_rg, piece_rg))) return rc;
    if ((rc = upload(ctx, &pm.list, list))) return rc;
    if (keep_host) { pm.far_host = std::move(far); pm.start_host = std::move(start); pm.pstart_host = std::move(pstart); pm.piece_rg_host = std::move(piece_rg); }
    return PCM_OK;
}

static int class_of(int la, int lb) {
    int lo = std::min(la, lb), hi = std::max(la, lb);
    static const int tab[3][3] = {{0, 1, 3}, {1, 2, 4}, {3, 4, 5}};
    return tab[lo][hi];
}

// PCM_VERBOSE: wall time of the stages of pcm_setup
void setup_stage(const char *name) {
    static const bool verbose = getenv("PCM_VERBOSE") != nullptr;
    static std::chrono::steady_clock::time_point last;
    if (!verbose) return;
    const auto now = std::chrono::steady_clock::now();
    if (name) fprintf(stderr, "[pcm] setup: %-40s %8.1f ms\n", name, std::chrono::duration<double, std::milli>(now - last).count());
    last = now;
}

int build_context(pcm_ctx *ctx, int nshell, const int *shell_l, const double *shell_xyz, const int *shell_nprim,
                  const double *prim_exp, const double *prim_coef, int64_t npoint, const double *pt_xyz,
                  const double *pt_zeta, const double *pt_switch) {
    const pcm_options &opt = ctx->opt;
    setup_stage(nullptr);
    // ------------------------------------------------------------------ points (Hilbert order, boxes of 32)
    ctx->M = npoint;
    GroupBoxes ptboxes;  // radius^2 entry 0: the product groups carry the far-field radius of a (product, point) pair
    {
        double zmin = 1e300, zmax = 0.0;
        double plo[3] = {1e300, 1e300, 1e300}, phi[3] = {-1e300, -1e300, -1e300};
        for (int64_t k = 0; k < npoint; ++k) {
            zmin = std::min(zmin, pt_zeta[k]);
            zmax = std::max(zmax, pt_zeta[k]);
            for (int d = 0; d < 3; ++d) { plo[d] = std::min(plo[d], pt_xyz[3 * k + d]); phi[d] = std::max(phi[d], pt_xyz[3 * k + d]); }
        }
        if (npoint == 0) zmin = zmax = 1.0;
        ctx->zeta_min = zmin;
        ctx->zeta_max = zmax;
        const double pspan = npoint ? std::max({phi[0] - plo[0], phi[1] - plo[1], phi[2] - plo[2], 1e-9}) : 1.0;
        const double pcell = std::max(pspan / 2097151.0, 0.25);
        std::vector<uint64_t> key((size_t)npoint);
#pragma omp parallel for schedule(static)
        for (int64_t k = 0; k < npoint; ++k)
            key[k] = hilbert_key((uint64_t)((pt_xyz[3 * k] - plo[0]) / pcell), (uint64_t)((pt_xyz[3 * k + 1] - plo[1]) / pcell),
                                 (uint64_t)((pt_xyz[3 * k + 2] - plo[2]) / pcell));
        std::vector<int32_t> &s2c = ctx->s2c_host, &c2s = ctx->c2s_host;
        s2c.resize((size_t)npoint);
        c2s.resize((size_t)npoint);
        for (int64_t k = 0; k < npoint; ++k) s2c[k] = (int32_t)k;
        std::sort(s2c.begin(), s2c.end(), [&](int32_t a, int32_t b) { return key[a] != key[b] ? key[a] < key[b] : a < b; });
        for (int64_t s = 0; s < npoint; ++s) c2s[s2c[s]] = (int32_t)s;
        std::vector<double4> pt((size_t)npoint);
        std::vector<double> diag((size_t)npoint);
        const int64_t ng = (npoint + 31) / 32;
        ptboxes.b.assign((size_t)ng * 7, 0.0);
        std::vector<double> &box = ptboxes.b;
        for (int64_t s = 0; s < npoint; ++s) {
            const int64_t k = s2c[s];
            const double z = pt_zeta[k];
            pt[s] = make_double4(pt_xyz[3 * k], pt_xyz[3 * k + 1], pt_xyz[3 * k + 2], 1.0 / (z * z));
            diag[s] = z * std::sqrt(2.0 / M_PI) / (pt_switch ? pt_switch[k] : 1.0);
            double *bx = &box[(size_t)(s / 32) * 7];
            if (s % 32 == 0) { for (int d = 0; d < 3; ++d) { bx[d] = 1e300; bx[3 + d] = -1e300; } }
            for (int d = 0; d < 3; ++d) { bx[d] = std::min(bx[d], pt_xyz[3 * k + d]); bx[3 + d] = std::max(bx[3 + d], pt_xyz[3 * k + d]); }
        }
        int rc = upload(ctx, &ctx->pt, pt);
        if (rc) return rc;
        if ((rc = upload(ctx, &ctx->pt_diag, diag))) return rc;
        if ((rc = upload(ctx, &ctx->s2c, s2c))) return rc;
        // A q patches: far-field radius^2 of a pair of points is at most TFAR_AMAT (1/zeta_i^2 + 1/zeta_j^2)
        {   // bounding boxes of the groups of 32 sorted points (lo xyz, hi xyz) for the RBJ neighbourhood search
            std::vector<double> b6((size_t)std::max<int64_t>(ng, 1) * 6, 0.0);
            for (int64_t g = 0; g < ng; ++g)
                for (int d = 0; d < 6; ++d) b6[(size_t)g * 6 + d] = box[(size_t)g * 7 + d];
            if ((rc = upload(ctx, &ctx->pt_boxes, b6))) return rc;
        }
        GroupBoxes amat_boxes = ptboxes;
        for (int64_t g = 0; g < ng; ++g) amat_boxes.b[(size_t)g * 7 + 6] = TFAR_AMAT * 2.0 / (zmin * zmin);
        if ((rc = build_patch_map(ctx, amat_boxes, amat_boxes, ctx->amat_map, npoint < 4 * AMAT_PERSIST_MAX))) return rc;
    }
    setup_stage("points, A q patch map");
    {
        std::vector<double> tab;
        build_boys_tables(tab);
        int rc = upload(ctx, &ctx->boys, tab);
        if (rc) return rc;
    }

    setup_stage("Boys tables");
    // ------------------------------------------------------------------ shells
    std::vector<int64_t> poff(nshell + 1, 0), boff(nshell + 1, 0);
    std::vector<double> amin(nshell), cmax(nshell);
    for (int s = 0; s < nshell; ++s) {
        int nc = shell_l[s] == 0 ? 1 : (shell_l[s] == 1 ? 3 : (opt.d_pure ? 5 : 6));
        poff[s + 1] = poff[s] + shell_nprim[s];
        boff[s + 1] = boff[s] + nc;
        double am = 1e300, cm = 0.0;
        for (int64_t i = poff[s]; i < poff[s + 1]; ++i) { am = std::min(am, prim_exp[i]); cm = std::max(cm, std::fabs(prim_coef[i])); }
        amin[s] = am;
        cmax[s] = cm;
    }
    ctx->nbf = boff[nshell];
    const double eps = opt.screen_eps;

    // ------------------------------------------------------------------ shell pairs + Eq. 15 screening
    std::vector<std::vector<HostPair>> per_row(nshell);
    int64_t unscreened = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : unscreened)
    for (int I = 0; I < nshell; ++I) {
        const double *A = shell_xyz + 3 * I;
        for (int J = I; J < nshell; ++J) {
            const double *B = shell_xyz + 3 * J;
            const int la = shell_l[I], lb = shell_l[J];
            const int64_t npp = (I == J) ? (int64_t)shell_nprim[I] * (shell_nprim[I] + 1) / 2 : (int64_t)shell_nprim[I] * shell_nprim[J];
            unscreened += npp;
            const double r2 = (A[0] - B[0]) * (A[0] - B[0]) + (A[1] - B[1]) * (A[1] - B[1]) + (A[2] - B[2]) * (A[2] - B[2]);
            // shell-level upper bound of |c c| [ab|ab]^{1/2}: every factor is an upper bound over the primitive pairs
            const double mu_min = amin[I] * amin[J] / (amin[I] + amin[J]);
            if (eps > 0.0) {
                if (mu_min * r2 > 200.0) continue;
                const double pmin = amin[I] + amin[J];
                const double reach = std::sqrt(r2) + std::sqrt(2.0 / pmin);
                const double ub = cmax[I] * cmax[J] * std::exp(-mu_min * r2) * 50.0 * std::pow(pmin, -1.25) * std::pow(std::max(reach, 1.0), la + lb);
                if (ub < eps) continue;
            }
            HostPair hp;
            hp.I = I; hp.J = J; hp.cls = class_of(la, lb);
            for (int i = 0; i < shell_nprim[I]; ++i)
                for (int j = (I == J ? i : 0); j < shell_nprim[J]; ++j) {
                    const double a = prim_exp[poff[I] + i], b = prim_exp[poff[J] + j];
                    const double cc = std::fabs(prim_coef[poff[I] + i] * prim_coef[poff[J] + j]);
                    if (eps > 0.0) {
                        const double mu = a * b / (a + b);
                        if (mu * r2 > 200.0) continue;
                        if (cc * schwarz_bound(la, a, A, lb, b, B) < eps) continue;
                    }
                    hp.prims.emplace_back(i, j);
                }
            if (!hp.prims.empty()) per_row[I].push_back(std::move(hp));
        }
    }
    setup_stage("shell pairs, Eq. 15 screening");
    std::vector<HostPair> pairs;
    for (auto &row : per_row) for (auto &hp : row) pairs.push_back(std::move(hp));
    per_row.clear();
    std::stable_sort(pairs.begin(), pairs.end(), [](const HostPair &x, const HostPair &y) { return x.cls < y.cls; });
    ctx->nsp = (int64_t)pairs.size();

    pcm_info &info = ctx->info;
    std::memset(&info, 0, sizeof(info));
    info.nbf = ctx->nbf; info.nshell = nshell; info.npoint = npoint;
    info.prim_pairs_unscreened = unscreened;
    info.zeta_min = ctx->zeta_min; info.zeta_max = ctx->zeta_max;

    setup_stage("pair list by class");
    // ------------------------------------------------------------------ members, products, G matrices
    std::vector<HostMember> members;
    std::vector<double> G, dG, m_ap;
    const bool want_grad = opt.gradient != 0;
    std::vector<int64_t> sp_mstart(pairs.size() + 1, 0);
    std::vector<int32_t> sp_i0(pairs.size()), sp_j0(pairs.size()), sp_dims(pairs.size());
    std::vector<int32_t> c_sp, c_ab;
    struct HostProd { double p, x, y, z; int L; };
    std::vector<HostProd> prods;
    auto bits = [](double d) { uint64_t u; std::memcpy(&u, &d, 8); return u; };

    // pass 1 (serial, light): offsets of every shell pair's members and G blocks, component list, counts
    std::vector<int64_t> sp_goff(pairs.size() + 1, 0);
    for (size_t sp = 0; sp < pairs.size(); ++sp) {
        const HostPair &hp = pairs[sp];
        const int I = hp.I, J = hp.J, la = shell_l[I], lb = shell_l[J], nh = nherm(la + lb);
        const int na = la == 2 ? (opt.d_pure ? 5 : 6) : NCART[la], nb = lb == 2 ? (opt.d_pure ? 5 : 6) : NCART[lb];
        sp_i0[sp] = (int32_t)boff[I]; sp_j0[sp] = (int32_t)boff[J];
        sp_dims[sp] = na | (nb << 8) | ((I == J ? 1 : 0) << 16);
        for (int ab = 0; ab < na * nb; ++ab) { c_sp.push_back((int32_t)sp); c_ab.push_back(ab); }
        info.shell_pairs[hp.cls] += 1;
        info.prim_pairs[hp.cls] += (int64_t)hp.prims.size();
        sp_mstart[sp + 1] = sp_mstart[sp] + (int64_t)hp.prims.size();
        sp_goff[sp + 1] = sp_goff[sp] + (int64_t)hp.prims.size() * na * nb * nh;
    }
    members.resize((size_t)sp_mstart[pairs.size()]);
    G.assign((size_t)sp_goff[pairs.size()], 0.0);
    if (want_grad) { dG.assign(3 * G.size(), 0.0); m_ap.resize(members.size()); }
    std::vector<HostProd> mprod(members.size());       // the Gaussian product of every member, before merging
    // pass 2 (all host threads): the G (and dG) block of every member -- independent of one another
#pragma omp parallel for schedule(dynamic, 256)
    for (size_t sp = 0; sp < pairs.size(); ++sp) {
        const HostPair &hp = pairs[sp];
        const int I = hp.I, J = hp.J, la = shell_l[I], lb = shell_l[J], L = la + lb, nh = nherm(L);
        const double *A = shell_xyz + 3 * I, *B = shell_xyz + 3 * J;
        double Ta[6][6], Tb[6][6];
        int na, nb;
        component_matrix(la, opt.d_pure, Ta, na);
        component_matrix(lb, opt.d_pure, Tb, nb);
        for (size_t k = 0; k < hp.prims.size(); ++k) {
            const auto ij = hp.prims[k];
            const double a = prim_exp[poff[I] + ij.first], b = prim_exp[poff[J] + ij.second];
            const double cc = prim_coef[poff[I] + ij.first] * prim_coef[poff[J] + ij.second] * ((I == J && ij.first != ij.second) ? 2.0 : 1.0);
            const double p = a + b;
            const double Px = (a * A[0] + b * B[0]) / p, Py = (a * A[1] + b * B[1]) / p, Pz = (a * A[2] + b * B[2]) / p;
            const size_t mi = (size_t)sp_mstart[sp] + k;
            mprod[mi] = {p, Px, Py, Pz, L};
            HostMember &m = members[mi];
            m.sp = (int32_t)sp; m.prod = -1; m.L = (int8_t)L; m.goff = sp_goff[sp] + (int64_t)k * na * nb * nh;
            // G[ab][h] = cc (pi/p)^{3/2} sum_cart Ta[a][ca] Tb[b][cb] Ex Ey Ez   (K_AB is inside E^{00}_0)
            E1D Ex, Ey, Ez;
            hermite_E(a, b, A[0], B[0], la, lb, Ex);
            hermite_E(a, b, A[1], B[1], la, lb, Ey);
            hermite_E(a, b, A[2], B[2], la, lb, Ez);
            const double pref = cc * std::pow(M_PI / p, 1.5);
            double *g = G.data() + m.goff;
            E1D Dx, Dy, Dz;
            double *dg = nullptr;
            if (want_grad) {
                hermite_dE(a, b, A[0], B[0], la, lb, Ex, Dx);
                hermite_dE(a, b, A[1], B[1], la, lb, Ey, Dy);
                hermite_dE(a, b, A[2], B[2], la, lb, Ez, Dz);
                dg = dG.data() + 3 * m.goff;
                m_ap[mi] = a / p;
            }
            for (int ca = 0; ca < NCART[la]; ++ca)
                for (int cb = 0; cb < NCART[lb]; ++cb) {
                    const int *pa = CARTS[la][ca], *pb = CARTS[lb][cb];
                    for (int t = 0; t <= pa[0] + pb[0]; ++t)
                        for (int u = 0; u <= pa[1] + pb[1]; ++u)
                            for (int v = 0; v <= pa[2] + pb[2]; ++v) {
                                const double e = pref * Ex.e[pa[0]][pb[0]][t] * Ey.e[pa[1]][pb[1]][u] * Ez.e[pa[2]][pb[2]][v];
                                const int h = hidx(t, u, v);
                                double de[3] = {0.0, 0.0, 0.0};
                                if (want_grad) {
                                    de[0] = pref * Dx.e[pa[0]][pb[0]][t] * Ey.e[pa[1]][pb[1]][u] * Ez.e[pa[2]][pb[2]][v];
                                    de[1] = pref * Ex.e[pa[0]][pb[0]][t] * Dy.e[pa[1]][pb[1]][u] * Ez.e[pa[2]][pb[2]][v];
                                    de[2] = pref * Ex.e[pa[0]][pb[0]][t] * Ey.e[pa[1]][pb[1]][u] * Dz.e[pa[2]][pb[2]][v];
                                }
                                for (int x = 0; x < na; ++x) {
                                    if (Ta[x][ca] == 0.0) continue;
                                    for (int y = 0; y < nb; ++y)
                                        if (Tb[y][cb] != 0.0) {
                                            const double w = Ta[x][ca] * Tb[y][cb];
                                            g[(size_t)(x * nb + y) * nh + h] += w * e;
                                            if (want_grad)
                                                for (int d = 0; d < 3; ++d) dg[((size_t)(x * nb + y) * 3 + d) * nh + h] += w * de[d];
                                        }
                                }
                            }
                }
        }
    }
    setup_stage("G matrices of the members");
    // pass 3 (serial, in member order: the product numbering is that of the first member that carries it): members with
    // bit-identical (p, P) share one product
    // (an open-addressing table of product indices keyed by the four bit patterns: one allocation, linear probing)
    size_t cap = 16;
    while (cap < 2 * members.size() + 1) cap <<= 1;
    std::vector<int32_t> table(opt.merge_products ? cap : 0, -1);
    for (size_t mi = 0; mi < members.size(); ++mi) {
        const HostProd &q = mprod[mi];
        int32_t prod = -1;
        if (opt.merge_products) {
            const uint64_t kp = bits(q.p), kx = bits(q.x), ky = bits(q.y), kz = bits(q.z);
            uint64_t hsh = kp * 0x9E3779B97F4A7C15ull;
            hsh = (hsh ^ (hsh >> 29) ^ kx) * 0xBF58476D1CE4E5B9ull;
            hsh = (hsh ^ (hsh >> 31) ^ ky) * 0x94D049BB133111EBull;
            hsh = (hsh ^ (hsh >> 30) ^ kz) * 0x9E3779B97F4A7C15ull;
            size_t slot = (size_t)(hsh >> 17) & (cap - 1);
            for (;; slot = (slot + 1) & (cap - 1)) {
                const int32_t cand = table[slot];
                if (cand < 0) break;
                const HostProd &r = prods[cand];
                if (bits(r.p) == kp && bits(r.x) == kx && bits(r.y) == ky && bits(r.z) == kz) { prod = cand; break; }
            }
            if (prod < 0) {
                prod = (int32_t)prods.size();
                table[slot] = prod;
                prods.push_back(q);
            } else {
                prods[prod].L = std::max(prods[prod].L, q.L);
            }
        } else {
            prod = (int32_t)prods.size();
            prods.push_back(q);
        }
        members[mi].prod = prod;
    }
    mprod.clear(); mprod.shrink_to_fit();
    sp_mstart[pairs.size()] = (int64_t)members.size();
    ctx->nmember = (int64_t)members.size();
    ctx->ncomp = (int64_t)c_sp.size();
    for (int c = 0; c < PCM_NCLASS; ++c) info.prim_pairs_total += info.prim_pairs[c];

    setup_stage("members, products, G matrices");
    // ------------------------------------------------------------------ sort products by (L, reach, Hilbert(P), p)
    // "reach" = binary order of magnitude of 1/p + 1/zeta_min^2, which the far-field radius^2 is proportional to:
    // tight products (far from every surface point) and diffuse ones end up in different groups of 32, so that the
    // box test of the hot kernels classifies whole groups.
    const int64_t np = (int64_t)prods.size();
    ctx->nprod = np;
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (auto &q : prods) {
        lo[0] = std::min(lo[0], q.x); hi[0] = std::max(hi[0], q.x);
        lo[1] = std::min(lo[1], q.y); hi[1] = std::max(hi[1], q.y);
        lo[2] = std::min(lo[2], q.z); hi[2] = std::max(hi[2], q.z);
    }
    const double span = std::max({hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2], 1e-9});
    const double cell = std::max(span / 2097151.0, 0.25);
    const double izmin2 = 1.0 / (ctx->zeta_min * ctx->zeta_min);
    std::vector<uint64_t> mort(np);
    std::vector<int> reach(np);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < np; ++i) {
        mort[i] = hilbert_key((uint64_t)((prods[i].x - lo[0]) / cell), (uint64_t)((prods[i].y - lo[1]) / cell),
                              (uint64_t)((prods[i].z - lo[2]) / cell));
        reach[i] = std::min(std::max(std::ilogb(1.0 / prods[i].p + izmin2), -6), 4);
    }
    std::vector<int32_t> order(np);
    {   // the keys travel with the index: the comparisons stay in one array instead of chasing three
        struct SortKey { uint64_t mort; double p; int32_t cls_reach, idx; };
        std::vector<SortKey> sk((size_t)np);
        for (int64_t i = 0; i < np; ++i) sk[i] = {mort[i], prods[i].p, (prods[i].L << 8) | (reach[i] + 16), (int32_t)i};
        std::sort(sk.begin(), sk.end(), [](const SortKey &x, const SortKey &y) {
            if (x.cls_reach != y.cls_reach) return x.cls_reach < y.cls_reach;
            if (x.mort != y.mort) return x.mort < y.mort;
            if (x.p != y.p) return x.p > y.p;
            return x.idx < y.idx;
        });
        for (int64_t i = 0; i < np; ++i) order[i] = sk[i].idx;
    }
    std::vector<int32_t> newidx(np);
    for (int64_t i = 0; i < np; ++i) newidx[order[i]] = (int32_t)i;

    setup_stage("product sort");
    // per class SoA
    int64_t first = 0;
    for (int L = 0; L <= MAXL; ++L) {
        int64_t n = 0;
        while (first + n < np && prods[order[first + n]].L == L) ++n;
        ClassData &c = ctx->cls[L];
        c.n = n; c.first = first; c.npad = (n + 127) / 128 * 128;
        info.products[L] = n;
        std::vector<double4> pa((size_t)c.npad);
        std::vector<double2> pb((size_t)c.npad);
        GroupBoxes pboxes;
        pboxes.b.assign((size_t)(c.npad / 32) * 7, 0.0);
        std::vector<double> &box = pboxes.b;
        for (int64_t i = 0; i < c.npad; ++i) {
            // padding repeats the last product: it never carries density (D = 0) and its sums are never read
            const HostProd &q = prods[order[first + std::min(i, n - 1)]];
            // far-field radius for one order more than L, so that pcm_gradient (orders 0..L+1) can share the patch maps
            pa[i] = make_double4(q.x, q.y, q.z, tfar(L + 1) * (1.0 / q.p + izmin2));
            pb[i] = make_double2(q.p, 2.0 * std::sqrt(q.p / M_PI));
            double *bx = &box[(size_t)(i / 32) * 7];
            if (i % 32 == 0) { for (int d = 0; d < 3; ++d) { bx[d] = 1e300; bx[3 + d] = -1e300; } bx[6] = 0.0; }
            bx[0] = std::min(bx[0], q.x); bx[1] = std::min(bx[1], q.y); bx[2] = std::min(bx[2], q.z);
            bx[3] = std::max(bx[3], q.x); bx[4] = std::max(bx[4], q.y); bx[5] = std::max(bx[5], q.z);
            bx[6] = std::max(bx[6], pa[i].w);
        }
        int rc = upload(ctx, &c.prodA, pa);
        if (rc) return rc;
        rc = upload(ctx, &c.prodB, pb);
        if (rc) return rc;
        if ((rc = build_patch_map(ctx, ptboxes, pboxes, c.pot_map))) return rc;
        if ((rc = build_patch_map(ctx, pboxes, ptboxes, c.fock_map))) return rc;
        first += n;
    }
    info.products_total = np;
    info.prim_pair_points = (double)info.prim_pairs_total * (double)npoint;
    info.product_points = (double)np * (double)npoint;

    setup_stage("class arrays, patch maps");
    // members: remap products, CSR product -> members
    std::vector<int32_t> m_prod(members.size()), m_cls(members.size()), m_sp(members.size());
    std::vector<int64_t> m_goff(members.size());
    std::vector<int64_t> pm_start(np + 1, 0);
    for (size_t m = 0; m < members.size(); ++m) {
        const int32_t g = newidx[members[m].prod];
        m_prod[m] = g;
        m_cls[m] = members[m].L | (prods[members[m].prod].L << 8);
        m_goff[m] = members[m].goff;
        m_sp[m] = members[m].sp;
        pm_start[g + 1] += 1;
    }
    for (int64_t i = 0; i < np; ++i) pm_start[i + 1] += pm_start[i];
    std::vector<int32_t> pm_list(members.size());
    {
        std::vector<int64_t> fill(pm_start.begin(), pm_start.end() - 1);
        for (size_t m = 0; m < members.size(); ++m) pm_list[fill[m_prod[m]]++] = (int32_t)m;
    }
    int rc;
    if ((rc = upload(ctx, &ctx->m_prod, m_prod))) return rc;
    if ((rc = upload(ctx, &ctx->m_cls, m_cls))) return rc;
    if ((rc = upload(ctx, &ctx->m_sp, m_sp))) return rc;
    if ((rc = upload(ctx, &ctx->m_goff, m_goff))) return rc;
    if ((rc = upload(ctx, &ctx->G, G))) return rc;
    if ((rc = upload(ctx, &ctx->pm_start, pm_start))) return rc;
    if ((rc = upload(ctx, &ctx->pm_list, pm_list))) return rc;
    if ((rc = upload(ctx, &ctx->sp_mstart, sp_mstart))) return rc;
    if ((rc = upload(ctx, &ctx->sp_i0, sp_i0))) return rc;
    if ((rc = upload(ctx, &ctx->sp_j0, sp_j0))) return rc;
    if ((rc = upload(ctx, &ctx->sp_dims, sp_dims))) return rc;
    if ((rc = upload(ctx, &ctx->c_sp, c_sp))) return rc;
    if ((rc = upload(ctx, &ctx->c_ab, c_ab))) return rc;
    {   // element of every component, for the compact transfers of the host-buffer calls
        const size_t nc = c_sp.size();
        ctx->comp_mu_host.resize(nc); ctx->comp_nu_host.resize(nc); ctx->comp_diag_host.resize(nc);
        for (size_t c = 0; c < nc; ++c) {
            const int sp = c_sp[c], dims = sp_dims[sp], nb = (dims >> 8) & 0xff;
            const int a = c_ab[c] / nb, b = c_ab[c] - a * nb;
            ctx->comp_mu_host[c] = sp_i0[sp] + a;
            ctx->comp_nu_host[c] = sp_j0[sp] + b;
            ctx->comp_diag_host[c] = (uint8_t)(dims >> 16);
        }
        if ((rc = upload(ctx, &ctx->comp_mu, ctx->comp_mu_host))) return rc;
        if ((rc = upload(ctx, &ctx->comp_nu, ctx->comp_nu_host))) return rc;
        if ((rc = upload(ctx, &ctx->comp_diag, ctx->comp_diag_host))) return rc;
    }
    setup_stage("member tables, uploads");
    ctx->nshell = nshell;
    if (want_grad) {
        std::vector<int32_t> shI(pairs.size()), shJ(pairs.size());
        std::vector<int64_t> cstart(pairs.size() + 1, 0), sh_start((size_t)nshell + 1, 0);
        for (size_t sp = 0; sp < pairs.size(); ++sp) {
            shI[sp] = pairs[sp].I; shJ[sp] = pairs[sp].J;
            cstart[sp + 1] = cstart[sp] + (sp_dims[sp] & 0xff) * ((sp_dims[sp] >> 8) & 0xff);
            sh_start[pairs[sp].I + 1] += 1;
            sh_start[pairs[sp].J + 1] += 1;   // a diagonal shell pair is listed as bra and as ket of its shell
        }
        for (int sidx = 0; sidx < nshell; ++sidx) sh_start[sidx + 1] += sh_start[sidx];
        std::vector<int32_t> sh_list((size_t)std::max<int64_t>(sh_start[nshell], 1), 0);
        {
            std::vector<int64_t> fill(sh_start.begin(), sh_start.end() - 1);
            for (size_t sp = 0; sp < pairs.size(); ++sp) {
                sh_list[fill[pairs[sp].I]++] = (int32_t)(2 * sp);
                sh_list[fill[pairs[sp].J]++] = (int32_t)(2 * sp + 1);
            }
        }
        std::vector<int32_t> hshift((size_t)3 * nherm(MAXL), 0);
        for (int t = 0; t <= MAXL; ++t)
            for (int u = 0; t + u <= MAXL; ++u)
                for (int v = 0; t + u + v <= MAXL; ++v) {
                    hshift[0 * nherm(MAXL) + hidx(t, u, v)] = hidx(t + 1, u, v);
                    hshift[1 * nherm(MAXL) + hidx(t, u, v)] = hidx(t, u + 1, v);
                    hshift[2 * nherm(MAXL) + hidx(t, u, v)] = hidx(t, u, v + 1);
                }
        if ((rc = upload(ctx, &ctx->dG, dG))) return rc;
        if ((rc = upload(ctx, &ctx->m_ap, m_ap))) return rc;
        if ((rc = upload(ctx, &ctx->sp_shI, shI))) return rc;
        if ((rc = upload(ctx, &ctx->sp_shJ, shJ))) return rc;
        if ((rc = upload(ctx, &ctx->sp_cstart, cstart))) return rc;
        if ((rc = upload(ctx, &ctx->sh_start, sh_start))) return rc;
        if ((rc = upload(ctx, &ctx->sh_list, sh_list))) return rc;
        if ((rc = upload(ctx, &ctx->hshift, hshift))) return rc;
    }
    return PCM_OK;
}

}  // namespace pcm
