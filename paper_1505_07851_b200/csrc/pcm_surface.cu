// pcm_surface.cu -- the ISWIG switching function S_k (Eq. 9) and the surface terms of the PCM gradient
// (Eq. 14): z^T (grad B^T) q and q^T (grad A) q / 2f, the latter including A_kk = zeta_k sqrt(2/pi)/S_k.
// With g(z', r) = d/dr [erf(z' r)/r]:  g/r = -(4 z'^3/sqrt pi) F_1(z'^2 r^2)  (-> -1/r^3 in the far field), F_1 from the
// same Boys table the integral kernels use.  Every sum has a fixed order.
#include <algorithm>
#include <cmath>
#include <vector>

#include "pcm_device.cuh"

namespace pcm {

constexpr int SF_TPB = 128;
constexpr int SF_TILE = 256;
constexpr double SF_SWITCH_CUT = 6.2;   // zeta (d - R) beyond which S_wf = 1 and dS_wf/dd = 0 to fp64 (erfc(6.2) = 2e-18)

// (1/r) d/dr [erf(z' r)/r] with z'^2 = 1/iz2: far field -1/r^3, otherwise the Boys table of order 1
__device__ __forceinline__ double dcoul_over_r(double r2, double iz2, const double *__restrict__ boys1) {
    const double zp = rsqrt_fast(iz2);
    const double T = r2 * zp * zp;
    if (T >= tfar(1)) {
        const double ri = rsqrt_fast(r2);
        return -ri * ri * ri;
    }
    const int i = __double2int_rn(T * 16.0);
    const double d = T - (double)i * 0.0625;
    const double *row = boys1 + (size_t)i * BOYS_STRIDE;
    double f = __ldg(row + BOYS_TERMS - 1);
#pragma unroll
    for (int k = BOYS_TERMS - 2; k >= 0; --k) f = fma(f, d, __ldg(row + k));
    return -2.2567583341910251478 * zp * zp * zp * f;   // 4/sqrt(pi)
}

// S_wf and (dS_wf/dd)/S_wf of one (point, atom) pair (Eq. 9)
__device__ __forceinline__ void switch_pair(double zeta, double R, double d, double &s, double &dlog) {
    if (zeta * (d - R) > SF_SWITCH_CUT) { s = 1.0; dlog = 0.0; return; }
    const double a = zeta * (R - d), b = zeta * (R + d);
    s = 1.0 - 0.5 * (erf(a) + erf(b));
    dlog = 0.56418958354775628695 * zeta * (exp(-a * a) - exp(-b * b)) / s;   // 1/sqrt(pi)
}

// force of atom J on point k per unit displacement vector: w such that the pair's gradient is w (r_k - R_J)
// (B term + the A_kk term through S_k); 0 at d = 0
__device__ __forceinline__ double point_atom_weight(double r2, double izk, double qk, double akk, bool owner, double zJ, double RJ,
                                                    double half_over_f, const double *__restrict__ boys1) {
    if (r2 == 0.0) return 0.0;
    double w = zJ * qk * dcoul_over_r(r2, izk, boys1);
    if (!owner) {
        const double d = sqrt(r2), zeta = rsqrt_fast(izk);
        double s, dlog;
        switch_pair(zeta, RJ, d, s, dlog);
        w -= half_over_f * qk * qk * akk * dlog / d;
    }
    return w;
}

// S_k = prod_{J != owner(k)} S_wf (caller order; thread = point)
__global__ void switching_kernel(int64_t M, const double *__restrict__ xyz, const double *__restrict__ zeta,
                                 const int32_t *__restrict__ owner, int natom, const double4 *__restrict__ atoms /* x,y,z,R */,
                                 double *__restrict__ S) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= M) return;
    const double x = xyz[3 * k], y = xyz[3 * k + 1], z = xyz[3 * k + 2], zk = zeta[k];
    const int own = owner[k];
    double s = 1.0;
    for (int J = 0; J < natom; ++J) {
        if (J == own) continue;
        const double4 a = atoms[J];
        const double dx = x - a.x, dy = y - a.y, dz = z - a.z;
        const double d = sqrt(fma(dz, dz, fma(dy, dy, dx * dx)));
        double sw, dl;
        switch_pair(zk, a.w, d, sw, dl);
        s *= sw;
    }
    S[k] = s;
}

// point side of the point-atom terms: thread = point (sorted order), atoms in order; gpa[d][k]
__global__ void __launch_bounds__(SF_TPB) surf_point_atom_kernel(const double4 *__restrict__ pt, const double *__restrict__ diag, int M,
                                                                 const double *__restrict__ q, const int32_t *__restrict__ s2c,
                                                                 const int32_t *__restrict__ owner_sorted,
                                                                 const double4 *__restrict__ atoms, const double *__restrict__ radius,
                                                                 int natom, double half_over_f, const double *__restrict__ boys1,
                                                                 double *__restrict__ gpa) {
    __shared__ double4 s_at[SF_TILE];
    __shared__ double s_rad[SF_TILE];
    const int k = blockIdx.x * SF_TPB + threadIdx.x;
    const double4 a = pt[min(k, M - 1)];
    const double qk = k < M ? q[s2c[k]] : 0.0, akk = diag[min(k, M - 1)];
    const int own = owner_sorted[min(k, M - 1)];
    double g[3] = {0.0, 0.0, 0.0};
    for (int base = 0; base < natom; base += SF_TILE) {
        const int cnt = min(SF_TILE, natom - base);
        __syncthreads();
        for (int t = threadIdx.x; t < cnt; t += SF_TPB) { s_at[t] = atoms[base + t]; s_rad[t] = radius[base + t]; }
        __syncthreads();
        for (int t = 0; t < cnt; ++t) {
            const double4 b = s_at[t];
            const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
            const double w = point_atom_weight(fma(dz, dz, fma(dy, dy, dx * dx)), a.w, qk, akk, base + t == own, b.w, s_rad[t],
                                               half_over_f, boys1);
            g[0] = fma(w, dx, g[0]); g[1] = fma(w, dy, g[1]); g[2] = fma(w, dz, g[2]);
        }
    }
    if (k < M) {
#pragma unroll
        for (int d = 0; d < 3; ++d) gpa[(size_t)d * M + k] = g[d];
    }
}

// atom side: one CTA per atom J, g_atom[J] = -sum_k (pair gradient); per-thread sums over k = tid, tid + 256, ...,
// then a fixed-order tree over the threads
__global__ void __launch_bounds__(256) surf_atom_kernel(const double4 *__restrict__ pt, const double *__restrict__ diag, int M,
                                                        const double *__restrict__ q, const int32_t *__restrict__ s2c,
                                                        const int32_t *__restrict__ owner_sorted,
                                                        const double4 *__restrict__ atoms, const double *__restrict__ radius,
                                                        double half_over_f, const double *__restrict__ boys1,
                                                        double *__restrict__ g_atom) {
    __shared__ double s_red[3][256];
    const int J = blockIdx.x;
    const double4 b = atoms[J];
    const double RJ = radius[J];
    double g[3] = {0.0, 0.0, 0.0};
    for (int k = threadIdx.x; k < M; k += 256) {
        const double4 a = pt[k];
        const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
        const double w = point_atom_weight(fma(dz, dz, fma(dy, dy, dx * dx)), a.w, q[s2c[k]], diag[k], owner_sorted[k] == J, b.w, RJ,
                                           half_over_f, boys1);
        g[0] = fma(-w, dx, g[0]); g[1] = fma(-w, dy, g[1]); g[2] = fma(-w, dz, g[2]);
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) s_red[d][threadIdx.x] = g[d];
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
#pragma unroll
            for (int d = 0; d < 3; ++d) s_red[d][threadIdx.x] += s_red[d][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x < 3) g_atom[(size_t)J * 3 + threadIdx.x] = s_red[threadIdx.x][0];
}

// A, k != l: thread = row point k, column points staged in shared memory; gaa[chunk][d][k] =
// sum_{l in chunk} q_l (g/r)(zeta'_kl, r_kl) (r_k - r_l); the self term vanishes with r_k - r_l (F_1(0) is finite)
__global__ void __launch_bounds__(SF_TPB) surf_aa_kernel(const double4 *__restrict__ pt, int M, const double *__restrict__ q,
                                                         const int32_t *__restrict__ s2c, int chunk_len, double thr,
                                                         const double *__restrict__ boys1, double *__restrict__ gaa) {
    __shared__ double4 s_pt[SF_TILE];
    __shared__ double s_q[SF_TILE];
    const int k = blockIdx.x * SF_TPB + threadIdx.x;
    const double4 a = pt[min(k, M - 1)];
    const int jbeg = blockIdx.y * chunk_len, jend = min(M, jbeg + chunk_len);
    const int thr_hi = hi32(thr);
    double g[3] = {0.0, 0.0, 0.0};
    for (int base = jbeg; base < jend; base += SF_TILE) {
        const int cnt = min(SF_TILE, jend - base);
        __syncthreads();
        for (int t = threadIdx.x; t < cnt; t += SF_TPB) { s_pt[t] = pt[base + t]; s_q[t] = q[s2c[base + t]]; }
        __syncthreads();
#pragma unroll 2
        for (int t = 0; t < cnt; ++t) {
            const double4 b = s_pt[t];
            const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            double w;
            if (hi32(r2) > thr_hi) {
                const double ri = rsqrt_fast(r2);
                w = -ri * ri * ri;
            } else {
                w = dcoul_over_r(r2, a.w + b.w, boys1);
            }
            w *= s_q[t];
            g[0] = fma(w, dx, g[0]); g[1] = fma(w, dy, g[1]); g[2] = fma(w, dz, g[2]);
        }
    }
    if (k < M) {
#pragma unroll
        for (int d = 0; d < 3; ++d) gaa[((size_t)blockIdx.y * 3 + d) * M + k] = g[d];
    }
}

// g_point[3 s2c[k] + d] = gpa[d][k] + (q_k / f) sum_chunks gaa[chunk][d][k]
__global__ void surf_point_reduce_kernel(int M, const double *__restrict__ gpa, const double *__restrict__ gaa, int chunks,
                                         const double *__restrict__ q, const int32_t *__restrict__ s2c, double inv_f,
                                         double *__restrict__ g_point) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= M) return;
    const int kc = s2c[k];
    const double qf = q[kc] * inv_f;
    for (int d = 0; d < 3; ++d) {
        double s = 0.0;
        for (int c = 0; c < chunks; ++c) s += gaa[((size_t)c * 3 + d) * M + k];
        g_point[(size_t)kc * 3 + d] = fma(qf, s, gpa[(size_t)d * M + k]);
    }
}

static int64_t sdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

int launch_surface_gradient(pcm_ctx *ctx, const double *q, double f, double *g_point, double *g_atom, cudaStream_t s) {
    const int M = (int)ctx->M;
    const int natom = (int)ctx->natom;
    const double *boys1 = ctx->boys + (size_t)1 * BOYS_ROWS * BOYS_STRIDE;
    if (g_atom && natom > 0) {
        if (M == 0) PCM_CUDA(ctx, cudaMemsetAsync(g_atom, 0, (size_t)natom * 24, s));
        else {
            surf_atom_kernel<<<natom, 256, 0, s>>>(ctx->pt, ctx->pt_diag, M, q, ctx->s2c, ctx->pt_owner, ctx->atoms, ctx->atom_radius,
                                                   0.5 / f, boys1, g_atom);
            ctx->launch_total += 1;
        }
    }
    if (!g_point || M == 0) { PCM_CUDA(ctx, cudaGetLastError()); return PCM_OK; }
    // scratch: gpa [3][M], then gaa [chunks][3][M]
    const int64_t rowblocks = sdiv(M, SF_TPB), tiles = sdiv(M, SF_TILE);
    const int64_t chunks = std::max<int64_t>(1, std::min<int64_t>(tiles, sdiv(4 * ctx->sm_count * 4, rowblocks)));
    const int64_t chunk_len = sdiv(tiles, chunks) * SF_TILE;
    const int64_t nch = sdiv(M, chunk_len);
    const size_t need = (size_t)(3 + 3 * nch) * M;
    if (need > ctx->surf_scratch_n) {
        int rc = dev_alloc_t(ctx, &ctx->surf_scratch, need);   // grow-only; the old buffer is freed with the context
        if (rc) return rc;
        ctx->surf_scratch_n = need;
    }
    double *gpa = ctx->surf_scratch, *gaa = gpa + (size_t)3 * M;
    surf_point_atom_kernel<<<(unsigned)rowblocks, SF_TPB, 0, s>>>(ctx->pt, ctx->pt_diag, M, q, ctx->s2c, ctx->pt_owner, ctx->atoms,
                                                                  ctx->atom_radius, natom, 0.5 / f, boys1, gpa);
    const double thr = tfar(1) * 2.0 / (ctx->zeta_min * ctx->zeta_min);
    surf_aa_kernel<<<dim3((unsigned)rowblocks, (unsigned)nch), SF_TPB, 0, s>>>(ctx->pt, M, q, ctx->s2c, (int)chunk_len, thr, boys1, gaa);
    surf_point_reduce_kernel<<<(unsigned)sdiv(M, 256), 256, 0, s>>>(M, gpa, gaa, (int)nch, q, ctx->s2c, 1.0 / f, g_point);
    ctx->launch_total += 3;
    PCM_CUDA(ctx, cudaGetLastError());
    return PCM_OK;
}

// standalone: S_k on the device from host arrays (used before pcm_setup, which takes S_k as an input)
int switching_host(int64_t M, const double *xyz, const double *zeta, const int32_t *owner, int natom, const double *atom_xyz,
                   const double *atom_radius, double *S) {
    if (M == 0) return PCM_OK;
    std::vector<double4> at((size_t)std::max(natom, 1));
    for (int j = 0; j < natom; ++j) at[j] = make_double4(atom_xyz[3 * j], atom_xyz[3 * j + 1], atom_xyz[3 * j + 2], atom_radius[j]);
    double *d_xyz = nullptr, *d_zeta = nullptr, *d_S = nullptr;
    int32_t *d_own = nullptr;
    double4 *d_at = nullptr;
    cudaError_t e = cudaMalloc(&d_xyz, (size_t)M * 24);
    if (e == cudaSuccess) e = cudaMalloc(&d_zeta, (size_t)M * 8);
    if (e == cudaSuccess) e = cudaMalloc(&d_S, (size_t)M * 8);
    if (e == cudaSuccess) e = cudaMalloc(&d_own, (size_t)M * 4);
    if (e == cudaSuccess) e = cudaMalloc(&d_at, at.size() * sizeof(double4));
    if (e == cudaSuccess) e = cudaMemcpy(d_xyz, xyz, (size_t)M * 24, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d_zeta, zeta, (size_t)M * 8, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d_own, owner, (size_t)M * 4, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d_at, at.data(), at.size() * sizeof(double4), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        switching_kernel<<<(unsigned)sdiv(M, 128), 128>>>(M, d_xyz, d_zeta, d_own, natom, d_at, d_S);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(S, d_S, (size_t)M * 8, cudaMemcpyDeviceToHost);
    cudaFree(d_xyz); cudaFree(d_zeta); cudaFree(d_S); cudaFree(d_own); cudaFree(d_at);
    return e == cudaSuccess ? PCM_OK : set_error(nullptr, PCM_ERR_CUDA, std::string("pcm_switching: ") + cudaGetErrorString(e));
}

}  // namespace pcm
