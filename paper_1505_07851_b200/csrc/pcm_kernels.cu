// pcm_kernels.cu -- the three hot kernels (a2 pcm_potential, a3 pcm_fock, a4 pcm_amatvec of SURVEY.md 8(a))
// and the small transforms around them.  All arithmetic fp64 on the plain FP64 pipe; no tensor cores (these are
// not dense contractions), no atomics (every reduction has a fixed order, results are bit-reproducible).
//
// Formulation: a primitive pair (or several sharing exponent sum p and centre P)
// is one Hermite Gaussian product.  For point k at C with exponent zeta:
//   [chi_a|J_k|chi_b] = (pi/p)^{3/2} sum_tuv E^{ab}_tuv Rt_tuv(P - C),   Rt = far-normalised Hermite Coulomb integrals
// (pcm_device.cuh).  Everything that depends on the basis functions (E, contraction coefficients, the pure-d
// transform, the factor 2 of off-diagonal pairs) is folded into the per-member matrices G (pcm_setup.cu), so
//   potential:  D_h(product) = sum_members sum_ab G[ab][h] P_ab ;  v_k = sum_products sum_h D_h Rt_h(P - C_k)
//   Fock:       H_h(product) = sum_k q_k Rt_h(P - C_k)          ;  F_ab = sum_members sum_h G[ab][h] H_h
#include <algorithm>
#include <cstdio>

#include "pcm_device.cuh"

namespace pcm {

constexpr int TPB = 128;        // threads per block of the hot kernels ("1 x 128", still a good size)
constexpr int FOCK_TILE = 256;  // points staged per shared-memory tile
constexpr int POT_TILE = 64;    // products staged per shared-memory tile
constexpr int AMAT_TILE = 256;

// ---------------------------------------------------------------------------------------------
// work partition: how many chunks the reduction dimension is split into (fixed by sizes only)
// ---------------------------------------------------------------------------------------------
static int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

int64_t fock_chunks(const pcm_ctx *ctx, int L) {
    const int64_t xb = ceil_div(ctx->cls[L].n, TPB);
    if (xb == 0 || ctx->M == 0) return 1;
    const int64_t target = (int64_t)ctx->sm_count * 8;
    int64_t c = ceil_div(target, xb);
    c = std::min<int64_t>(c, ceil_div(ctx->M, FOCK_TILE));
    return std::max<int64_t>(c, 1);
}
int pot_ppt(int L) { return L <= 2 ? 2 : 1; }
int64_t pot_chunks(const pcm_ctx *ctx, int L) {
    const int64_t xb = ceil_div(ctx->M, (int64_t)TPB * pot_ppt(L));
    if (xb == 0 || ctx->cls[L].n == 0) return 1;
    const int64_t target = (int64_t)ctx->sm_count * 8;
    int64_t c = ceil_div(target, xb);
    c = std::min<int64_t>(c, ceil_div(ctx->cls[L].n, POT_TILE));
    return std::max<int64_t>(c, 1);
}
int64_t amat_chunks(const pcm_ctx *ctx) {
    const int64_t xb = ceil_div(ctx->M, (int64_t)TPB * 2);
    if (xb == 0) return 1;
    const int64_t target = (int64_t)ctx->sm_count * 8;
    int64_t c = ceil_div(target, xb);
    c = std::min<int64_t>(c, ceil_div(ctx->M, AMAT_TILE));
    return std::max<int64_t>(c, 1);
}

// ---------------------------------------------------------------------------------------------
// a4: y = A q on the fly (Eq. 2, 3, 8).  Thread = 2 rows, the column points stream through shared memory.
//   far (zeta'^2 r^2 >= 38, erf = 1 to fp64):  A_ij = 1/r                       -- 12 FP64 instructions + MUFU
//   general:  A_ij = (2 zeta'/sqrt pi) F_0(zeta'^2 r^2), zeta'^2 = 1/(1/zeta_i^2 + 1/zeta_j^2); A_ii from pt_diag
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double amat_general(double r2, double izi, double izj, const double *__restrict__ boys0) {
    const double zp = rsqrt_fast(izi + izj);
    const double T = r2 * zp * zp;
    if (T >= TFAR_AMAT) return rsqrt_fast(r2);
    const int i = __double2int_rn(T * 16.0);
    const double d = T - (double)i * 0.0625;
    const double *row = boys0 + (size_t)i * BOYS_STRIDE;
    double f = __ldg(row + BOYS_TERMS - 1);
#pragma unroll
    for (int k = BOYS_TERMS - 2; k >= 0; --k) f = fma(f, d, __ldg(row + k));
    return 1.1283791670955125739 * zp * f;  // 2/sqrt(pi)
}

__global__ void __launch_bounds__(TPB) amatvec_kernel(const double4 *__restrict__ pt, const double *__restrict__ diag,
                                                      const double *__restrict__ q, int M, int chunk_len,
                                                      double *__restrict__ out, const double *__restrict__ boys0,
                                                      int thr_hi) {
    __shared__ double4 s_pt[AMAT_TILE];   // x, y, z, q
    __shared__ double s_iz[AMAT_TILE];
    const int i0 = blockIdx.x * (2 * TPB) + threadIdx.x, i1 = i0 + TPB;
    const double4 a0 = pt[min(i0, M - 1)], a1 = pt[min(i1, M - 1)];
    double y0 = 0.0, y1 = 0.0;
    const int jbeg = blockIdx.y * chunk_len, jend = min(M, jbeg + chunk_len);
    for (int base = jbeg; base < jend; base += AMAT_TILE) {
        __syncthreads();
        for (int t = threadIdx.x; t < AMAT_TILE; t += TPB) {
            const int j = base + t;
            if (j < jend) {
                const double4 b = pt[j];
                s_pt[t] = make_double4(b.x, b.y, b.z, q[j]);
                s_iz[t] = b.w;
            } else {  // padding: far away, zero charge
                s_pt[t] = make_double4(3e8, 3e8, 3e8, 0.0);
                s_iz[t] = 1.0;
            }
        }
        __syncthreads();
        const int cnt = min(AMAT_TILE, jend - base);
#pragma unroll 2
        for (int t = 0; t < cnt; ++t) {
            const double4 b = s_pt[t];
            const double dx0 = a0.x - b.x, dy0 = a0.y - b.y, dz0 = a0.z - b.z;
            const double dx1 = a1.x - b.x, dy1 = a1.y - b.y, dz1 = a1.z - b.z;
            const double r20 = fma(dz0, dz0, fma(dy0, dy0, dx0 * dx0));
            const double r21 = fma(dz1, dz1, fma(dy1, dy1, dx1 * dx1));
            if (min(hi32(r20), hi32(r21)) > thr_hi) {
                y0 = fma(b.w, rsqrt_fast(r20), y0);
                y1 = fma(b.w, rsqrt_fast(r21), y1);
            } else {
                const int j = base + t;
                const double izj = s_iz[t];
                const double e0 = (j == i0) ? diag[j] : amat_general(r20, a0.w, izj, boys0);
                const double e1 = (j == i1) ? diag[j] : amat_general(r21, a1.w, izj, boys0);
                y0 = fma(b.w, e0, y0);
                y1 = fma(b.w, e1, y1);
            }
        }
    }
    if (i0 < M) out[(size_t)blockIdx.y * M + i0] = y0;
    if (i1 < M) out[(size_t)blockIdx.y * M + i1] = y1;
}

// out[k] = sum_slots part[slot][k]  (fixed order)
__global__ void reduce_slots_kernel(const double *__restrict__ part, int64_t n, int slots, double *__restrict__ out) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    double s = 0.0;
    for (int c = 0; c < slots; ++c) s += part[(size_t)c * n + k];
    out[k] = s;
}

// ---------------------------------------------------------------------------------------------
// a3 main kernel: H_h(product) = sum_k q_k Rt_h(P - C_k).  Thread = product (NHERM(L) register accumulators),
// the points stream through shared memory, two points per step for instruction-level parallelism.
// ---------------------------------------------------------------------------------------------
template <int L>
struct FockSink {
    double acc[nherm(L)];
    __device__ __forceinline__ void value(int h, double v) { acc[h] += v; }
    __device__ __forceinline__ void product(int h, double a, double b) { acc[h] = fma(a, b, acc[h]); }
};

template <int L>
__global__ void __launch_bounds__(TPB) fock_kernel(const double4 *__restrict__ prodA, const double2 *__restrict__ prodB,
                                                   int64_t npad, const double4 *__restrict__ pt, const double *__restrict__ q,
                                                   int M, int chunk_len, double *__restrict__ herm,
                                                   const double *__restrict__ boysL) {
    constexpr int NH = nherm(L);
    __shared__ double4 s_pt[FOCK_TILE];  // x, y, z, q
    __shared__ double s_iz[FOCK_TILE];
    const int64_t ip = (int64_t)blockIdx.x * TPB + threadIdx.x;  // < npad by construction
    const double4 A = prodA[ip];
    const double2 B = prodB[ip];
    const int thr_hi = hi32(A.w);
    FockSink<L> sink;
#pragma unroll
    for (int h = 0; h < NH; ++h) sink.acc[h] = 0.0;
    const int kbeg = blockIdx.y * chunk_len, kend = min(M, kbeg + chunk_len);
    for (int base = kbeg; base < kend; base += FOCK_TILE) {
        __syncthreads();
        for (int t = threadIdx.x; t < FOCK_TILE; t += TPB) {
            const int k = base + t;
            if (k < kend) {
                const double4 c = pt[k];
                s_pt[t] = make_double4(c.x, c.y, c.z, q[k]);
                s_iz[t] = c.w;
            } else {
                s_pt[t] = make_double4(-3e8, -3e8, -3e8, 0.0);
                s_iz[t] = 1.0;
            }
        }
        __syncthreads();
        const int cnt = min(FOCK_TILE, kend - base);  // an odd count runs one padding point (zero charge)
        for (int t = 0; t < cnt; t += 2) {
            const double4 c0 = s_pt[t], c1 = s_pt[t + 1];
            const double x0 = A.x - c0.x, y0 = A.y - c0.y, z0 = A.z - c0.z;
            const double x1 = A.x - c1.x, y1 = A.y - c1.y, z1 = A.z - c1.z;
            const double r20 = fma(z0, z0, fma(y0, y0, x0 * x0));
            const double r21 = fma(z1, z1, fma(y1, y1, x1 * x1));
            double g0[L + 1], g1[L + 1];
            if (min(hi32(r20), hi32(r21)) > thr_hi) {
                seeds_far<L>(r20, g0);
                seeds_far<L>(r21, g1);
            } else {
                seeds_general<L>(r20, B.x, B.y, s_iz[t], boysL, g0);
                seeds_general<L>(r21, B.x, B.y, s_iz[t + 1], boysL, g1);
            }
#pragma unroll
            for (int n = 0; n <= L; ++n) { g0[n] *= c0.w; g1[n] *= c1.w; }
            hermite_R<L>(x0, y0, z0, g0, sink);
            hermite_R<L>(x1, y1, z1, g1, sink);
        }
    }
    double *out = herm + (size_t)blockIdx.y * NH * npad + ip;
#pragma unroll
    for (int h = 0; h < NH; ++h) out[(size_t)h * npad] = sink.acc[h];
}

// herm[0][h][i] += sum_{c>=1} herm[c][h][i]
__global__ void reduce_herm_kernel(double *__restrict__ herm, int64_t plane, int chunks) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= plane) return;
    double s = herm[k];
    for (int c = 1; c < chunks; ++c) s += herm[(size_t)c * plane + k];
    herm[k] = s;
}

// ---------------------------------------------------------------------------------------------
// a2 main kernel: v_k = sum_products sum_h D_h Rt_h(P - C_k).  Thread = PPT points (register accumulators),
// the products (centre, threshold, Hermite density) stream through shared memory.
// ---------------------------------------------------------------------------------------------
template <int L>
struct PotSink {
    const double *D;
    double v;
    __device__ __forceinline__ void value(int h, double x) { v = fma(D[h], x, v); }
    __device__ __forceinline__ void product(int h, double a, double b) { v = fma(D[h], a * b, v); }
};

template <int L>
__host__ __device__ constexpr int pot_rec() { return (4 + nherm(L) + 2 + 1) / 2 * 2; }  // doubles per staged product

template <int L, int PPT>
__global__ void __launch_bounds__(TPB) potential_kernel(const double4 *__restrict__ prodA, const double2 *__restrict__ prodB,
                                                        const double *__restrict__ herm, int64_t npad, int64_t nprod,
                                                        int chunk_len, const double4 *__restrict__ pt, int M,
                                                        double *__restrict__ vpart, const double *__restrict__ boysL) {
    constexpr int NH = nherm(L);
    constexpr int REC = pot_rec<L>();
    __shared__ __align__(16) double s_rec[POT_TILE * REC];
    double4 c[PPT];
    int kk[PPT];
    double v[PPT];
#pragma unroll
    for (int r = 0; r < PPT; ++r) {
        kk[r] = blockIdx.x * (TPB * PPT) + r * TPB + threadIdx.x;
        c[r] = pt[min(kk[r], M - 1)];
        v[r] = 0.0;
    }
    const int64_t pbeg = (int64_t)blockIdx.y * chunk_len, pend = min(nprod, pbeg + (int64_t)chunk_len);
    for (int64_t base = pbeg; base < pend; base += POT_TILE) {
        const int cnt = (int)min((int64_t)POT_TILE, pend - base);
        __syncthreads();
        // stage: header (Px,Py,Pz,thr), D_0..D_{NH-1}, (p, 1/kappa)
        for (int t = threadIdx.x; t < cnt; t += TPB) {
            const double4 a = prodA[base + t];
            const double2 b = prodB[base + t];
            double *r = s_rec + t * REC;
            r[0] = a.x; r[1] = a.y; r[2] = a.z; r[3] = a.w;
            r[4 + NH] = b.x; r[5 + NH] = b.y;
        }
        for (int t = threadIdx.x; t < cnt * NH; t += TPB) {
            const int h = t / cnt, i = t - h * cnt;  // consecutive threads read consecutive products of one component
            s_rec[i * REC + 4 + h] = herm[(size_t)h * npad + base + i];
        }
        __syncthreads();
        for (int t = 0; t < cnt; ++t) {
            const double *r = s_rec + t * REC;
            const double2 h01 = *reinterpret_cast<const double2 *>(r);
            const double2 h23 = *reinterpret_cast<const double2 *>(r + 2);
            const int thr_hi = hi32(h23.y);
            double x[PPT], y[PPT], z[PPT], r2[PPT];
            int mn = 0x7fffffff;
#pragma unroll
            for (int s = 0; s < PPT; ++s) {
                x[s] = h01.x - c[s].x; y[s] = h01.y - c[s].y; z[s] = h23.x - c[s].z;
                r2[s] = fma(z[s], z[s], fma(y[s], y[s], x[s] * x[s]));
                mn = min(mn, hi32(r2[s]));
            }
            double g[PPT][L + 1];
            if (mn > thr_hi) {
#pragma unroll
                for (int s = 0; s < PPT; ++s) seeds_far<L>(r2[s], g[s]);
            } else {
                const double p = r[4 + NH], invk = r[5 + NH];
#pragma unroll
                for (int s = 0; s < PPT; ++s) seeds_general<L>(r2[s], p, invk, c[s].w, boysL, g[s]);
            }
#pragma unroll
            for (int s = 0; s < PPT; ++s) {
                PotSink<L> sink{r + 4, v[s]};
                hermite_R<L>(x[s], y[s], z[s], g[s], sink);
                v[s] = sink.v;
            }
        }
    }
#pragma unroll
    for (int s = 0; s < PPT; ++s)
        if (kk[s] < M) vpart[(size_t)blockIdx.y * M + kk[s]] = v[s];
}

// ---------------------------------------------------------------------------------------------
// transforms between the basis-function and the Hermite-product representations
// ---------------------------------------------------------------------------------------------
struct ClassPtrs {
    double *herm[MAXL + 1];
    int64_t npad[MAXL + 1];
    int64_t first[MAXL + 1];
};

// D_h(product) = sum_members sum_ab G[ab][h] Pw_ab,  Pw = P_ab + P_ba for an off-diagonal shell pair (the sum of
// Eq. 5 runs over the full square), P_ab inside a diagonal one.  Thread = product; fixed member order.
template <int L>
__global__ void density_to_hermite_kernel(int64_t n, int64_t first, int64_t npad, const int64_t *__restrict__ pm_start,
                                          const int32_t *__restrict__ pm_list, const int32_t *__restrict__ m_sp,
                                          const int32_t *__restrict__ m_cls, const int64_t *__restrict__ m_goff,
                                          const double *__restrict__ G, const int32_t *__restrict__ sp_i0,
                                          const int32_t *__restrict__ sp_j0, const int32_t *__restrict__ sp_dims,
                                          const double *__restrict__ P, int64_t ldp, double *__restrict__ herm) {
    constexpr int NH = nherm(L);
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npad) return;
    double D[NH];
#pragma unroll
    for (int h = 0; h < NH; ++h) D[h] = 0.0;
    if (i < n) {
        const int64_t g = first + i;
        for (int64_t e = pm_start[g]; e < pm_start[g + 1]; ++e) {
            const int m = pm_list[e];
            const int sp = m_sp[m];
            const int dims = sp_dims[sp], na = dims & 0xff, nb = (dims >> 8) & 0xff, diag = dims >> 16;
            const int i0 = sp_i0[sp], j0 = sp_j0[sp];
            const int Lm = m_cls[m] & 0xff;
            const int nhm = (Lm + 1) * (Lm + 2) * (Lm + 3) / 6;
            const double *gm = G + m_goff[m];
            for (int a = 0; a < na; ++a)
                for (int b = 0; b < nb; ++b) {
                    double pw = P[(size_t)(i0 + a) * ldp + j0 + b];
                    if (!diag) pw += P[(size_t)(j0 + b) * ldp + i0 + a];
                    const double *row = gm + (size_t)(a * nb + b) * nhm;
#pragma unroll
                    for (int h = 0; h < NH; ++h)
                        if (h < nhm) D[h] = fma(row[h], pw, D[h]);
                }
        }
    }
#pragma unroll
    for (int h = 0; h < NH; ++h) herm[(size_t)h * npad + i] = D[h];
}

// F_ab (+)= sum_members sum_h G[ab][h] H_h(product of the member).  Thread = one component (a,b) of one shell pair;
// it writes F_mu,nu and, for an off-diagonal shell pair, F_nu,mu.  No two threads touch the same element.
__global__ void hermite_to_fock_kernel(int64_t ncomp, const int32_t *__restrict__ c_sp, const int32_t *__restrict__ c_ab,
                                       const int64_t *__restrict__ sp_mstart, const int32_t *__restrict__ m_prod,
                                       const int32_t *__restrict__ m_cls, const int64_t *__restrict__ m_goff,
                                       const double *__restrict__ G, const int32_t *__restrict__ sp_i0,
                                       const int32_t *__restrict__ sp_j0, const int32_t *__restrict__ sp_dims,
                                       ClassPtrs cp, double *__restrict__ F, int64_t ldf, int accumulate) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncomp) return;
    const int sp = c_sp[c], ab = c_ab[c];
    const int dims = sp_dims[sp], nb = (dims >> 8) & 0xff, diag = dims >> 16;
    const int a = ab / nb, b = ab - a * nb;
    // a diagonal shell pair's block is symmetric: (a,b) with a > b evaluates the (b,a) sum, so F = F^T bit for bit
    const int abg = (diag && a > b) ? b * nb + a : ab;
    double s = 0.0;
    for (int64_t m = sp_mstart[sp]; m < sp_mstart[sp + 1]; ++m) {
        const int cl = m_cls[m], Lm = cl & 0xff, Lp = cl >> 8;
        const int nhm = (Lm + 1) * (Lm + 2) * (Lm + 3) / 6;
        const double *row = G + m_goff[m] + (size_t)abg * nhm;
        const double *H = cp.herm[Lp] + (m_prod[m] - cp.first[Lp]);
        const int64_t np = cp.npad[Lp];
        double sm = 0.0;
        for (int h = 0; h < nhm; ++h) sm = fma(row[h], H[(size_t)h * np], sm);
        s += sm;
    }
    const size_t mu = (size_t)sp_i0[sp] + a, nu = (size_t)sp_j0[sp] + b;
    if (accumulate) {
        F[mu * ldf + nu] += s;
        if (!diag) F[nu * ldf + mu] += s;
    } else {
        F[mu * ldf + nu] = s;
        if (!diag) F[nu * ldf + mu] = s;
    }
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
#define PCM_LAUNCH_CHECK(ctx)                                                                      \
    do {                                                                                           \
        cudaError_t e__ = cudaGetLastError();                                                      \
        if (e__ != cudaSuccess) return set_error(ctx, PCM_ERR_CUDA, std::string("kernel launch: ") + cudaGetErrorString(e__)); \
    } while (0)

static int mark(pcm_ctx *ctx, int i, cudaStream_t s) {
    if (ctx->timing) PCM_CUDA(ctx, cudaEventRecord(ctx->ev[8 * ctx->cur_op + i], s));
    return PCM_OK;
}

int launch_amatvec(pcm_ctx *ctx, const double *q, double *y, cudaStream_t s) {
    ctx->cur_op = 2;
    ctx->launches[2] = 0;
    ctx->timed[2] = ctx->timing != 0;
    const int M = (int)ctx->M;
    if (M == 0) return PCM_OK;
    const int64_t chunks = amat_chunks(ctx);
    const int chunk_len = (int)(ceil_div(ceil_div(M, chunks), 2) * 2);
    const double thr = TFAR_AMAT * 2.0 / (ctx->zeta_min * ctx->zeta_min);
    int64_t thr_bits;
    memcpy(&thr_bits, &thr, 8);
    const int thr_hi = (int)(thr_bits >> 32);
    dim3 grid((unsigned)ceil_div(M, 2 * TPB), (unsigned)chunks);
    int rc;
    if ((rc = mark(ctx, 0, s))) return rc;
    if ((rc = mark(ctx, 1, s))) return rc;
    amatvec_kernel<<<grid, TPB, 0, s>>>(ctx->pt, ctx->pt_diag, q, M, chunk_len, chunks > 1 ? ctx->ypart : y, ctx->boys, thr_hi);
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    for (int i = 2; i <= 6; ++i)
        if ((rc = mark(ctx, i, s))) return rc;
    if (chunks > 1) {
        reduce_slots_kernel<<<(unsigned)ceil_div(M, 256), 256, 0, s>>>(ctx->ypart, M, (int)chunks, y);
        PCM_LAUNCH_CHECK(ctx);
        { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    }
    return mark(ctx, 7, s);
}

template <int L>
static int launch_fock_class(pcm_ctx *ctx, const double *q, cudaStream_t s) {
    ClassData &c = ctx->cls[L];
    if (c.n == 0) return PCM_OK;
    const int64_t chunks = fock_chunks(ctx, L);
    const int chunk_len = (int)(ceil_div(ceil_div(ctx->M, chunks), 2) * 2);
    dim3 grid((unsigned)(c.npad / TPB), (unsigned)chunks);
    fock_kernel<L><<<grid, TPB, 0, s>>>(c.prodA, c.prodB, c.npad, ctx->pt, q, (int)ctx->M, chunk_len, c.herm,
                                        ctx->boys + (size_t)L * BOYS_ROWS * BOYS_STRIDE);
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    return PCM_OK;
}

template <int L>
static int reduce_fock_class(pcm_ctx *ctx, cudaStream_t s) {
    ClassData &c = ctx->cls[L];
    const int64_t chunks = fock_chunks(ctx, L);
    if (c.n == 0 || chunks <= 1) return PCM_OK;
    const int64_t plane = (int64_t)nherm(L) * c.npad;
    reduce_herm_kernel<<<(unsigned)ceil_div(plane, 256), 256, 0, s>>>(c.herm, plane, (int)chunks);
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    return PCM_OK;
}

int launch_fock(pcm_ctx *ctx, const double *q, double *F, int64_t ldf, int accumulate, cudaStream_t s) {
    ctx->cur_op = 1;
    ctx->launches[1] = 0;
    ctx->timed[1] = ctx->timing != 0;
    int rc;
    if ((rc = mark(ctx, 0, s))) return rc;
    if ((rc = mark(ctx, 1, s))) return rc;
    if (ctx->M > 0) {
        if ((rc = launch_fock_class<0>(ctx, q, s)) || (rc = mark(ctx, 2, s))) return rc;
        if ((rc = launch_fock_class<1>(ctx, q, s)) || (rc = mark(ctx, 3, s))) return rc;
        if ((rc = launch_fock_class<2>(ctx, q, s)) || (rc = mark(ctx, 4, s))) return rc;
        if ((rc = launch_fock_class<3>(ctx, q, s)) || (rc = mark(ctx, 5, s))) return rc;
        if ((rc = launch_fock_class<4>(ctx, q, s)) || (rc = mark(ctx, 6, s))) return rc;
    } else {
        for (int i = 2; i <= 6; ++i)
            if ((rc = mark(ctx, i, s))) return rc;
    }
    if (!accumulate && ctx->nbf > 0)
        PCM_CUDA(ctx, cudaMemset2DAsync(F, (size_t)ldf * 8, 0, (size_t)ctx->nbf * 8, (size_t)ctx->nbf, s));
    if (ctx->M > 0 && ctx->ncomp > 0) {
        if ((rc = reduce_fock_class<0>(ctx, s))) return rc;
        if ((rc = reduce_fock_class<1>(ctx, s))) return rc;
        if ((rc = reduce_fock_class<2>(ctx, s))) return rc;
        if ((rc = reduce_fock_class<3>(ctx, s))) return rc;
        if ((rc = reduce_fock_class<4>(ctx, s))) return rc;
        ClassPtrs cp;
        for (int L = 0; L <= MAXL; ++L) { cp.herm[L] = ctx->cls[L].herm; cp.npad[L] = ctx->cls[L].npad; cp.first[L] = ctx->cls[L].first; }
        hermite_to_fock_kernel<<<(unsigned)ceil_div(ctx->ncomp, 128), 128, 0, s>>>(
            ctx->ncomp, ctx->c_sp, ctx->c_ab, ctx->sp_mstart, ctx->m_prod, ctx->m_cls, ctx->m_goff, ctx->G, ctx->sp_i0,
            ctx->sp_j0, ctx->sp_dims, cp, F, ldf, accumulate);
        PCM_LAUNCH_CHECK(ctx);
        { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    }
    return mark(ctx, 7, s);
}

template <int L>
static int launch_density_class(pcm_ctx *ctx, const double *P, int64_t ldp, cudaStream_t s) {
    ClassData &c = ctx->cls[L];
    if (c.n == 0) return PCM_OK;
    density_to_hermite_kernel<L><<<(unsigned)(c.npad / 128), 128, 0, s>>>(
        c.n, c.first, c.npad, ctx->pm_start, ctx->pm_list, ctx->m_sp, ctx->m_cls, ctx->m_goff, ctx->G, ctx->sp_i0,
        ctx->sp_j0, ctx->sp_dims, P, ldp, c.herm);
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    return PCM_OK;
}

template <int L, int PPT>
static int launch_potential_class(pcm_ctx *ctx, int64_t &slot, cudaStream_t s) {
    ClassData &c = ctx->cls[L];
    if (c.n == 0) return PCM_OK;
    const int64_t chunks = pot_chunks(ctx, L);
    const int chunk_len = (int)ceil_div(c.n, chunks);
    dim3 grid((unsigned)ceil_div(ctx->M, (int64_t)TPB * PPT), (unsigned)chunks);
    potential_kernel<L, PPT><<<grid, TPB, 0, s>>>(c.prodA, c.prodB, c.herm, c.npad, c.n, chunk_len, ctx->pt, (int)ctx->M,
                                                  ctx->vpart + (size_t)slot * ctx->M,
                                                  ctx->boys + (size_t)L * BOYS_ROWS * BOYS_STRIDE);
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    slot += chunks;
    return PCM_OK;
}

int launch_potential(pcm_ctx *ctx, const double *P, int64_t ldp, double *v, cudaStream_t s) {
    ctx->cur_op = 0;
    ctx->launches[0] = 0;
    ctx->timed[0] = ctx->timing != 0;
    int rc;
    if (ctx->M == 0) return PCM_OK;
    if ((rc = mark(ctx, 0, s))) return rc;
    if ((rc = launch_density_class<0>(ctx, P, ldp, s))) return rc;
    if ((rc = launch_density_class<1>(ctx, P, ldp, s))) return rc;
    if ((rc = launch_density_class<2>(ctx, P, ldp, s))) return rc;
    if ((rc = launch_density_class<3>(ctx, P, ldp, s))) return rc;
    if ((rc = launch_density_class<4>(ctx, P, ldp, s))) return rc;
    if ((rc = mark(ctx, 1, s))) return rc;
    int64_t slot = 0;
    if ((rc = launch_potential_class<0, 2>(ctx, slot, s)) || (rc = mark(ctx, 2, s))) return rc;
    if ((rc = launch_potential_class<1, 2>(ctx, slot, s)) || (rc = mark(ctx, 3, s))) return rc;
    if ((rc = launch_potential_class<2, 2>(ctx, slot, s)) || (rc = mark(ctx, 4, s))) return rc;
    if ((rc = launch_potential_class<3, 1>(ctx, slot, s)) || (rc = mark(ctx, 5, s))) return rc;
    if ((rc = launch_potential_class<4, 1>(ctx, slot, s)) || (rc = mark(ctx, 6, s))) return rc;
    if (slot == 0) {
        PCM_CUDA(ctx, cudaMemsetAsync(v, 0, (size_t)ctx->M * 8, s));
    } else {
        reduce_slots_kernel<<<(unsigned)ceil_div(ctx->M, 256), 256, 0, s>>>(ctx->vpart, ctx->M, (int)slot, v);
        PCM_LAUNCH_CHECK(ctx);
        { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    }
    return mark(ctx, 7, s);
}

// ---------------------------------------------------------------------------------------------
// FP64 peak: 8 independent DFMA chains per thread, 2048 resident threads per SM
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dfma_peak_kernel(double *out, int iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

int fp64_peak(pcm_ctx *ctx, int reps, double *tflops) {
    const int blocks = ctx->sm_count * 8, threads = 256, iters = 4096;
    double *out = nullptr;
    PCM_CUDA(ctx, cudaMalloc(&out, (size_t)blocks * threads * 8));
    cudaStream_t s = ctx->own_stream;
    double best_ms = 1e30;
    for (int r = 0; r < std::max(reps, 1) + 1; ++r) {
        cudaEventRecord(ctx->ev[25], s);
        dfma_peak_kernel<<<blocks, threads, 0, s>>>(out, iters, 0.999999, 1e-9);
        cudaEventRecord(ctx->ev[26], s);
        cudaError_t e = cudaEventSynchronize(ctx->ev[26]);
        if (e != cudaSuccess) { cudaFree(out); return set_error(ctx, PCM_ERR_CUDA, cudaGetErrorString(e)); }
        float ms = 0;
        cudaEventElapsedTime(&ms, ctx->ev[25], ctx->ev[26]);
        if (r > 0) best_ms = std::min(best_ms, (double)ms);
    }
    cudaFree(out);
    const double flops = 2.0 * 64.0 * iters * (double)blocks * threads;
    *tflops = flops / (best_ms * 1e-3) * 1e-12;
    return PCM_OK;
}

}  // namespace pcm
