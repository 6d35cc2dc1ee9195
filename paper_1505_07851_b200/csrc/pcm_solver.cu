// pcm_solver.cu -- steps a5 (randomized block-Jacobi build) and a6 (preconditioned CG,
// PAPER.md:164-170) of SURVEY.md 8(a).  The matrix-vector product is pcm_kernels.cu's on-the-fly A q.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

#include "pcm_device.cuh"

namespace pcm {

static int64_t cdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

#define PCM_LAUNCH_CHECK(ctx)                                                                      \
    do {                                                                                           \
        cudaError_t e__ = cudaGetLastError();                                                      \
        if (e__ != cudaSuccess) return set_error(ctx, PCM_ERR_CUDA, std::string("kernel launch: ") + cudaGetErrorString(e__)); \
    } while (0)

// ---------------------------------------------------------------------------------------------
// seeded pivot order: indices sorted by (splitmix64 finaliser(seed + (i+1) golden), i)
// ---------------------------------------------------------------------------------------------
static inline uint64_t mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
void pivot_order(uint64_t seed, int64_t M, int64_t *perm) {
    std::vector<uint64_t> key((size_t)M);
    for (int64_t i = 0; i < M; ++i) key[i] = mix64(seed + (uint64_t)(i + 1) * 0x9E3779B97F4A7C15ULL);
    std::iota(perm, perm + M, (int64_t)0);
    std::sort(perm, perm + M, [&](int64_t a, int64_t b) { return key[a] != key[b] ? key[a] < key[b] : a < b; });
}

// ---------------------------------------------------------------------------------------------
// A_ij for arbitrary i, j (Eq. 2, 3, 8)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double a_entry(const double4 *__restrict__ pt, const double *__restrict__ diag, int i, int j,
                                          const double *__restrict__ boys0) {
    if (i == j) return diag[i];
    const double4 a = pt[i], b = pt[j];
    const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const double zp = rsqrt_fast(a.w + b.w);
    const double T = r2 * zp * zp;
    if (T >= TFAR_AMAT) return rsqrt_fast(r2);
    const int t = __double2int_rn(T * 16.0);
    const double d = T - (double)t * 0.0625;
    const double *row = boys0 + (size_t)t * BOYS_STRIDE;
    double f = __ldg(row + BOYS_TERMS - 1);
#pragma unroll
    for (int k = BOYS_TERMS - 2; k >= 0; --k) f = fma(f, d, __ldg(row + k));
    return 1.1283791670955125739 * zp * f;
}

// ---------------------------------------------------------------------------------------------
// RBJ block selection.  One step = one block: three small kernels over device-resident state.
//   state[0] = pos (next position in the pivot order), [1] = filled, [2] = pivot, [3] = candidate count,
//   [4] = error flag, [5] = take (block size - 1 for this step)
// Keys are A_kj > 0, compared as 64-bit integers.  Buckets = the top 16 bits of the key (sign, exponent,
// 4 mantissa bits) shifted into [0, 1023]: a monotone map, so "bucket >= b*" is a superset of the top `take`.
// ---------------------------------------------------------------------------------------------
constexpr int RBJ_BINS = 1024;
constexpr int RBJ_BIN_BASE = 0x3e00;  // bucket of 2^-31

__device__ __forceinline__ int rbj_bucket(double a) {
    const int b = (int)((unsigned long long)__double_as_longlong(a) >> 48) - RBJ_BIN_BASE;
    return min(max(b, 0), RBJ_BINS - 1);
}

__global__ void rbj_keys_kernel(const double4 *__restrict__ pt, const double *__restrict__ diag, int M,
                                const int32_t *__restrict__ perm, const unsigned char *__restrict__ assigned,
                                long long *__restrict__ state, double *__restrict__ keys, int *__restrict__ hist,
                                const double *__restrict__ boys0) {
    __shared__ int s_hist[RBJ_BINS];
    __shared__ int s_pivot;
    // every block finds the same pivot: the first unassigned index of the pivot order at or after pos
    if (threadIdx.x == 0) s_pivot = M;
    for (int t = threadIdx.x; t < RBJ_BINS; t += blockDim.x) s_hist[t] = 0;
    __syncthreads();
    long long pos = state[0];
    while (true) {
        const long long p = pos + threadIdx.x;
        if (p < M && !assigned[perm[p]]) atomicMin(&s_pivot, (int)p);
        __syncthreads();
        if (s_pivot < M || pos + blockDim.x >= M) break;
        pos += blockDim.x;
        __syncthreads();
    }
    const int ppos = s_pivot;
    if (ppos >= M) return;  // nothing left (not reached in a correct schedule)
    const int k = perm[ppos];
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < M; j += gridDim.x * blockDim.x) {
        double a = 0.0;
        if (!assigned[j] && j != k) {
            a = a_entry(pt, diag, k, j, boys0);
            atomicAdd(&s_hist[rbj_bucket(a)], 1);
        }
        keys[j] = a;
    }
    __syncthreads();
    for (int t = threadIdx.x; t < RBJ_BINS; t += blockDim.x)
        if (s_hist[t]) atomicAdd(&hist[t], s_hist[t]);
    if (blockIdx.x == 0 && threadIdx.x == 0) { state[0] = ppos; state[2] = k; }
}

__global__ void rbj_collect_kernel(int M, int block, const long long *__restrict__ state, const double *__restrict__ keys,
                                   const int *__restrict__ hist, int *__restrict__ cand_count, int2 *__restrict__ cand_meta,
                                   double *__restrict__ cand_key) {
    __shared__ int s_bstar;
    if (threadIdx.x == 0) {
        const long long remaining = M - state[1] - 1;  // unassigned other than the pivot
        const long long take = min((long long)block - 1, remaining);
        int b = RBJ_BINS, cum = 0;
        while (b > 0 && cum < take) { --b; cum += hist[b]; }
        s_bstar = (take > 0) ? b : RBJ_BINS;
    }
    __syncthreads();
    const int bstar = s_bstar;
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < M; j += gridDim.x * blockDim.x) {
        const double a = keys[j];
        if (a > 0.0 && rbj_bucket(a) >= bstar) {
            const int slot = atomicAdd(cand_count, 1);
            cand_meta[slot] = make_int2(j, 0);
            cand_key[slot] = a;
        }
    }
}

// single block: rank the candidates by (key descending, index ascending), keep the first `take`
__global__ void rbj_select_kernel(int M, int block, long long *__restrict__ state, int *__restrict__ cand_count,
                                  const int2 *__restrict__ cand_meta, const double *__restrict__ cand_key,
                                  int *__restrict__ hist, unsigned char *__restrict__ assigned, int32_t *__restrict__ order,
                                  const int32_t *__restrict__ s2c) {
    const long long filled = state[1];
    const int k = (int)state[2];
    const long long remaining = M - filled - 1;
    const int take = (int)min((long long)block - 1, remaining);
    const int n = *cand_count;
    for (int c = threadIdx.x; c < n; c += blockDim.x) {
        const double key = cand_key[c];
        const int idx = cand_meta[c].x, cidx = s2c[idx];  // ties -> lower index in the caller's numbering
        int rank = 0;
        for (int o = 0; o < n; ++o) {
            const double ko = cand_key[o];
            rank += (ko > key) || (ko == key && s2c[cand_meta[o].x] < cidx);
        }
        if (rank < take) {
            order[filled + 1 + rank] = idx;
            assigned[idx] = 1;
        }
    }
    for (int t = threadIdx.x; t < RBJ_BINS; t += blockDim.x) hist[t] = 0;
    __syncthreads();
    if (threadIdx.x == 0) {
        order[filled] = k;
        assigned[k] = 1;
        state[0] = state[0] + 1;
        state[1] = filled + 1 + take;
        *cand_count = 0;
        if (n < take) state[4] = 1;  // cannot happen: the bucket cut keeps at least `take`
    }
}

// ---------------------------------------------------------------------------------------------
// Block inversion: one thread block per diagonal block.  fill -> Cholesky (right-looking, in place, lower)
// -> W = L^-1 (one column per thread) -> inv = W^T W.  n x n row-major, in global memory (L2 resident).
// ---------------------------------------------------------------------------------------------
__global__ void rbj_invert_kernel(const double4 *__restrict__ pt, const double *__restrict__ diag, int M, int block,
                                  const int32_t *__restrict__ order, double *__restrict__ inv, double *__restrict__ work,
                                  int *__restrict__ err, const double *__restrict__ boys0) {
    const long long start = (long long)blockIdx.x * block;
    const int n = (int)min((long long)block, (long long)M - start);
    double *a = inv + (size_t)blockIdx.x * block * block;
    double *w = work + (size_t)blockIdx.x * block * block;
    const int32_t *idx = order + start;
    for (int e = threadIdx.x; e < n * n; e += blockDim.x) {
        const int r = e / n, c = e - r * n;
        a[e] = a_entry(pt, diag, idx[r], idx[c], boys0);
        w[e] = 0.0;
    }
    __syncthreads();
    for (int j = 0; j < n; ++j) {
        const double d = a[(size_t)j * n + j];
        if (!(d > 0.0)) {
            if (threadIdx.x == 0) *err = 1;
            return;
        }
        const double s = sqrt(d), is = 1.0 / s;
        __syncthreads();
        for (int i = j + threadIdx.x; i < n; i += blockDim.x) a[(size_t)i * n + j] = (i == j) ? s : a[(size_t)i * n + j] * is;
        __syncthreads();
        const int m = n - j - 1;  // trailing update a[i][c] -= L[i][j] L[c][j], j < c <= i
        for (int e = threadIdx.x; e < m * m; e += blockDim.x) {
            const int i = j + 1 + e / m, c = j + 1 + e % m;
            if (c <= i) a[(size_t)i * n + c] -= a[(size_t)i * n + j] * a[(size_t)c * n + j];
        }
        __syncthreads();
    }
    // W = L^-1: column c by forward substitution, x_i = (delta_ic - sum_{c<=k<i} L[i][k] x_k)/L[i][i]
    for (int c = threadIdx.x; c < n; c += blockDim.x) {
        for (int i = c; i < n; ++i) {
            double s = (i == c) ? 1.0 : 0.0;
            for (int k = c; k < i; ++k) s -= a[(size_t)i * n + k] * w[(size_t)k * n + c];
            w[(size_t)i * n + c] = s / a[(size_t)i * n + i];
        }
    }
    __syncthreads();
    // inv = W^T W (symmetric; both triangles from the same sum)
    for (int e = threadIdx.x; e < n * n; e += blockDim.x) {
        const int r = e / n, c = e - r * n;
        if (c > r) continue;
        double s = 0.0;
        for (int k = r; k < n; ++k) s = fma(w[(size_t)k * n + r], w[(size_t)k * n + c], s);
        a[(size_t)r * n + c] = s;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < n * n; e += blockDim.x) {
        const int r = e / n, c = e - r * n;
        if (c > r) a[(size_t)r * n + c] = a[(size_t)c * n + r];
    }
}

// z = C r = scatter( blockdiag(M_b^-1) gather(r) ); one thread block per diagonal block
__global__ void rbj_apply_kernel(int M, int block, const int32_t *__restrict__ order, const double *__restrict__ inv,
                                 const double *__restrict__ r, double *__restrict__ z) {
    extern __shared__ double s_r[];
    const long long start = (long long)blockIdx.x * block;
    const int n = (int)min((long long)block, (long long)M - start);
    const double *a = inv + (size_t)blockIdx.x * block * block;
    const int32_t *idx = order + start;
    for (int j = threadIdx.x; j < n; j += blockDim.x) s_r[j] = r[idx[j]];
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        double s = 0.0;
        for (int j = 0; j < n; ++j) s = fma(a[(size_t)j * n + i], s_r[j], s);  // inv is symmetric: column read is coalesced
        z[idx[i]] = s;
    }
}

// ---------------------------------------------------------------------------------------------
// CG vector kernels.  Dot products: fixed-shape two-stage reduction (DOT_BLOCKS partials, then one block).
// scal[]: 0 rz, 1 pAp, 2 rr, 3 rz_new, 4 bAx2
// ---------------------------------------------------------------------------------------------
constexpr int DOT_BLOCKS = 296;
constexpr int DOT_THREADS = 256;

__device__ __forceinline__ double block_sum(double v) {
    __shared__ double s_w[DOT_THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x < DOT_THREADS / 32) t = s_w[threadIdx.x];
    if (threadIdx.x < 32) {
#pragma unroll
        for (int o = DOT_THREADS / 64; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    return t;  // valid in thread 0
}

// partial[blockIdx] = sum a.b over this block's grid-stride slice;  partial2 likewise for c.d when c != nullptr
__global__ void __launch_bounds__(DOT_THREADS) dot_partial_kernel(int M, const double *__restrict__ a, const double *__restrict__ b,
                                                                  const double *__restrict__ c, const double *__restrict__ d,
                                                                  double *__restrict__ partial) {
    double s1 = 0.0, s2 = 0.0;
    for (int i = blockIdx.x * DOT_THREADS + threadIdx.x; i < M; i += DOT_BLOCKS * DOT_THREADS) {
        s1 = fma(a[i], b[i], s1);
        if (c) s2 = fma(c[i], d[i], s2);
    }
    s1 = block_sum(s1);
    s2 = block_sum(s2);
    if (threadIdx.x == 0) { partial[blockIdx.x] = s1; partial[DOT_BLOCKS + blockIdx.x] = s2; }
}
// scal[o1] = sum partial[0..), scal[o2] = sum partial[DOT_BLOCKS..)
__global__ void __launch_bounds__(DOT_THREADS) dot_final_kernel(const double *__restrict__ partial, double *__restrict__ scal,
                                                                int o1, int o2) {
    double s1 = 0.0, s2 = 0.0;
    for (int i = threadIdx.x; i < DOT_BLOCKS; i += DOT_THREADS) { s1 += partial[i]; s2 += partial[DOT_BLOCKS + i]; }
    s1 = block_sum(s1);
    s2 = block_sum(s2);
    if (threadIdx.x == 0) { scal[o1] = s1; if (o2 >= 0) scal[o2] = s2; }
}
// x += alpha p; r -= alpha Ap with alpha = rz/pAp; partial sums of r.r
__global__ void __launch_bounds__(DOT_THREADS) cg_update_kernel(int M, const double *__restrict__ scal, const double *__restrict__ p,
                                                                const double *__restrict__ Ap, double *__restrict__ x,
                                                                double *__restrict__ r, double *__restrict__ partial) {
    const double alpha = scal[0] / scal[1];
    double s = 0.0;
    for (int i = blockIdx.x * DOT_THREADS + threadIdx.x; i < M; i += DOT_BLOCKS * DOT_THREADS) {
        x[i] = fma(alpha, p[i], x[i]);
        const double ri = fma(-alpha, Ap[i], r[i]);
        r[i] = ri;
        s = fma(ri, ri, s);
    }
    s = block_sum(s);
    if (threadIdx.x == 0) { partial[blockIdx.x] = s; partial[DOT_BLOCKS + blockIdx.x] = 0.0; }
}
// p = z + beta p, beta = rz_new/rz; then rz <- rz_new (done by the last step of the single-thread tail kernel)
__global__ void cg_direction_kernel(int M, const double *__restrict__ scal, const double *__restrict__ z, double *__restrict__ p) {
    const double beta = scal[3] / scal[0];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) p[i] = fma(beta, p[i], z[i]);
}
__global__ void cg_shift_kernel(double *scal) { scal[0] = scal[3]; }
__global__ void jacobi_kernel(int M, const double *__restrict__ diag, const double *__restrict__ r, double *__restrict__ z) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) z[i] = r[i] / diag[i];
}
__global__ void residual_kernel(int M, const double *__restrict__ b, const double *__restrict__ Ax, double *__restrict__ r) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) r[i] = b[i] - Ax[i];
}

// caller order <-> sorted order
__global__ void gather_kernel(int M, const int32_t *__restrict__ s2c, const double *__restrict__ src, double *__restrict__ dst) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) dst[i] = src[s2c[i]];
}
__global__ void scatter_kernel(int M, const int32_t *__restrict__ s2c, const double *__restrict__ src, double *__restrict__ dst) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) dst[s2c[i]] = src[i];
}

// ---------------------------------------------------------------------------------------------
// host drivers
// ---------------------------------------------------------------------------------------------
int rbj_build(pcm_ctx *ctx, int block, uint64_t seed, const int64_t *pivot_order_host, cudaStream_t s) {
    const int64_t M = ctx->M;
    if (block < 1) return set_error(ctx, PCM_ERR_ARG, "pcm_rbj_build: block < 1");
    if (M == 0) { ctx->rbj_block = block; ctx->rbj_nblocks = 0; return PCM_OK; }
    if ((int64_t)block > M) block = (int)M;
    std::vector<int64_t> perm64((size_t)M);
    if (pivot_order_host) {
        std::vector<char> seen((size_t)M, 0);
        for (int64_t i = 0; i < M; ++i) {
            const int64_t v = pivot_order_host[i];
            if (v < 0 || v >= M || seen[v]) return set_error(ctx, PCM_ERR_ARG, "pcm_rbj_build: pivot order is not a permutation");
            seen[v] = 1;
            perm64[i] = v;
        }
    } else {
        pivot_order(seed, M, perm64.data());
    }
    std::vector<int32_t> perm((size_t)M);  // pivot order in the library's sorted point numbering
    for (int64_t i = 0; i < M; ++i) perm[i] = ctx->c2s_host[(size_t)perm64[i]];

    const int64_t nb = cdiv(M, block);
    // (re)allocate RBJ storage; earlier builds are released
    auto release = [&](void *p) {
        if (!p) return;
        auto it = std::find(ctx->allocs.begin(), ctx->allocs.end(), p);
        if (it != ctx->allocs.end()) ctx->allocs.erase(it);
        cudaFree(p);
    };
    release(ctx->rbj_order); release(ctx->rbj_inv);
    ctx->rbj_order = nullptr; ctx->rbj_inv = nullptr; ctx->rbj_block = 0; ctx->rbj_nblocks = 0;
    int rc;
    if ((rc = dev_alloc_t(ctx, &ctx->rbj_order, (size_t)M))) return rc;
    if ((rc = dev_alloc_t(ctx, &ctx->rbj_inv, (size_t)nb * block * block))) return rc;

    // scratch for the build
    int32_t *d_perm = nullptr; unsigned char *d_assigned = nullptr; long long *d_state = nullptr; double *d_keys = nullptr;
    int *d_hist = nullptr, *d_count = nullptr, *d_err = nullptr; int2 *d_meta = nullptr; double *d_ckey = nullptr, *d_work = nullptr;
    auto cleanup = [&]() {
        cudaFree(d_perm); cudaFree(d_assigned); cudaFree(d_state); cudaFree(d_keys); cudaFree(d_hist);
        cudaFree(d_count); cudaFree(d_err); cudaFree(d_meta); cudaFree(d_ckey); cudaFree(d_work);
    };
#define RBJ_TRY(call)                                                                                     \
    do {                                                                                                  \
        cudaError_t e__ = (call);                                                                         \
        if (e__ != cudaSuccess) { cleanup(); return set_error(ctx, PCM_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__)); } \
    } while (0)
    RBJ_TRY(cudaMalloc(&d_perm, (size_t)M * 4));
    RBJ_TRY(cudaMalloc(&d_assigned, (size_t)M));
    RBJ_TRY(cudaMalloc(&d_state, 8 * sizeof(long long)));
    RBJ_TRY(cudaMalloc(&d_keys, (size_t)M * 8));
    RBJ_TRY(cudaMalloc(&d_hist, RBJ_BINS * 4));
    RBJ_TRY(cudaMalloc(&d_count, 4));
    RBJ_TRY(cudaMalloc(&d_err, 4));
    RBJ_TRY(cudaMalloc(&d_meta, (size_t)M * sizeof(int2)));
    RBJ_TRY(cudaMalloc(&d_ckey, (size_t)M * 8));
    RBJ_TRY(cudaMalloc(&d_work, (size_t)nb * block * block * 8));
    RBJ_TRY(cudaMemcpyAsync(d_perm, perm.data(), (size_t)M * 4, cudaMemcpyHostToDevice, s));
    RBJ_TRY(cudaMemsetAsync(d_assigned, 0, (size_t)M, s));
    RBJ_TRY(cudaMemsetAsync(d_state, 0, 8 * sizeof(long long), s));
    RBJ_TRY(cudaMemsetAsync(d_hist, 0, RBJ_BINS * 4, s));
    RBJ_TRY(cudaMemsetAsync(d_count, 0, 4, s));
    RBJ_TRY(cudaMemsetAsync(d_err, 0, 4, s));

    const int threads = 256;
    const int grid = (int)std::min<int64_t>(cdiv(M, threads), (int64_t)ctx->sm_count * 4);
    for (int64_t b = 0; b < nb; ++b) {
        rbj_keys_kernel<<<grid, threads, 0, s>>>(ctx->pt, ctx->pt_diag, (int)M, d_perm, d_assigned, d_state, d_keys, d_hist, ctx->boys);
        rbj_collect_kernel<<<grid, threads, 0, s>>>((int)M, block, d_state, d_keys, d_hist, d_count, d_meta, d_ckey);
        rbj_select_kernel<<<1, 1024, 0, s>>>((int)M, block, d_state, d_count, d_meta, d_ckey, d_hist, d_assigned, ctx->rbj_order, ctx->s2c);
        ctx->launch_total += 3;
    }
    ctx->launch_total += 1;
    RBJ_TRY(cudaGetLastError());
    rbj_invert_kernel<<<(unsigned)nb, 256, 0, s>>>(ctx->pt, ctx->pt_diag, (int)M, block, ctx->rbj_order, ctx->rbj_inv, d_work, d_err, ctx->boys);
    RBJ_TRY(cudaGetLastError());
    long long h_state[8];
    int h_err = 0;
    RBJ_TRY(cudaMemcpyAsync(h_state, d_state, sizeof(h_state), cudaMemcpyDeviceToHost, s));
    RBJ_TRY(cudaMemcpyAsync(&h_err, d_err, 4, cudaMemcpyDeviceToHost, s));
    RBJ_TRY(cudaStreamSynchronize(s));
    cleanup();
#undef RBJ_TRY
    if (h_state[1] != M || h_state[4] != 0) return set_error(ctx, PCM_ERR_STATE, "pcm_rbj_build: block selection did not cover all points");
    if (h_err) return set_error(ctx, PCM_ERR_NUMERIC, "pcm_rbj_build: a diagonal block of A is not positive definite");
    ctx->rbj_block = block;
    ctx->rbj_nblocks = nb;
    ctx->info.rbj_block = block;
    ctx->info.rbj_nblocks = nb;
    return PCM_OK;
}

static int apply_precond(pcm_ctx *ctx, int precond, const double *r, double *z, cudaStream_t s) {
    const int M = (int)ctx->M;
    if (precond == 0) {
        PCM_CUDA(ctx, cudaMemcpyAsync(z, r, (size_t)M * 8, cudaMemcpyDeviceToDevice, s));
    } else if (precond == 1) {
        jacobi_kernel<<<(unsigned)cdiv(M, 256), 256, 0, s>>>(M, ctx->pt_diag, r, z);
        PCM_LAUNCH_CHECK(ctx);
        ctx->launch_total += 1;
    } else {
        const int block = (int)ctx->rbj_block;
        const int threads = std::min(256, std::max(32, (block + 31) / 32 * 32));
        rbj_apply_kernel<<<(unsigned)ctx->rbj_nblocks, threads, (size_t)block * 8, s>>>(M, block, ctx->rbj_order, ctx->rbj_inv, r, z);
        PCM_LAUNCH_CHECK(ctx);
        ctx->launch_total += 1;
    }
    return PCM_OK;
}

static int dot2(pcm_ctx *ctx, const double *a, const double *b, const double *c, const double *d, int o1, int o2, cudaStream_t s) {
    double *partial = ctx->cg_scal + 16;
    dot_partial_kernel<<<DOT_BLOCKS, DOT_THREADS, 0, s>>>((int)ctx->M, a, b, c, d, partial);
    dot_final_kernel<<<1, DOT_THREADS, 0, s>>>(partial, ctx->cg_scal, o1, o2);
    PCM_LAUNCH_CHECK(ctx);
    ctx->launch_total += 2;
    return PCM_OK;
}

int cg_solve(pcm_ctx *ctx, const double *b_caller, double *x_caller, double tol, int max_iter, int precond, int use_x0,
             int *iters, double *resid, cudaStream_t s) {
    const int M = (int)ctx->M;
    if (precond < 0 || precond > 2) return set_error(ctx, PCM_ERR_ARG, "pcm_cg_solve: precond must be 0, 1 or 2");
    if (precond == 2 && ctx->rbj_block == 0) return set_error(ctx, PCM_ERR_STATE, "pcm_cg_solve: RBJ requested before pcm_rbj_build");
    if (M == 0) { if (iters) *iters = 0; if (resid) resid[0] = resid[1] = 0.0; return PCM_OK; }
    // all solver vectors live in the library's sorted point order; b is gathered on entry, x scattered on exit
    double *r = ctx->cg_vec, *z = r + M, *p = z + M, *Ap = p + M, *x = Ap + M, *b = x + M;
    double *scal = ctx->cg_scal, *partial = scal + 16;
    double *h = ctx->cg_scal_host;
    int rc;
    const int saved_timing = ctx->timing;
    ctx->timing = 0;
    const unsigned gb = (unsigned)cdiv(M, 256);
#define CG_TRY(expr) do { rc = (expr); if (rc) { ctx->timing = saved_timing; return rc; } } while (0)
#define CG_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { ctx->timing = saved_timing; \
        return set_error(ctx, PCM_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__)); } } while (0)
    gather_kernel<<<gb, 256, 0, s>>>(M, ctx->s2c, b_caller, b);
    ctx->launch_total += 1;
    if (use_x0) {
        gather_kernel<<<gb, 256, 0, s>>>(M, ctx->s2c, x_caller, x);
        CG_TRY(launch_amatvec_sorted(ctx, x, Ap, s));
        residual_kernel<<<gb, 256, 0, s>>>(M, b, Ap, r);
        ctx->launch_total += 2;
    } else {
        CG_CUDA(cudaMemsetAsync(x, 0, (size_t)M * 8, s));
        CG_CUDA(cudaMemcpyAsync(r, b, (size_t)M * 8, cudaMemcpyDeviceToDevice, s));
    }
    CG_TRY(apply_precond(ctx, precond, r, z, s));
    CG_CUDA(cudaMemcpyAsync(p, z, (size_t)M * 8, cudaMemcpyDeviceToDevice, s));
    CG_TRY(dot2(ctx, r, z, r, r, 0, 2, s));  // rz, rr
    CG_CUDA(cudaMemcpyAsync(h, scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, s));
    CG_CUDA(cudaStreamSynchronize(s));
    double rn = std::sqrt(h[2]);
    int it = 0;
    while (rn > tol && it < max_iter) {
        CG_TRY(launch_amatvec_sorted(ctx, p, Ap, s));
        CG_TRY(dot2(ctx, p, Ap, nullptr, nullptr, 1, -1, s));  // pAp
        cg_update_kernel<<<DOT_BLOCKS, DOT_THREADS, 0, s>>>(M, scal, p, Ap, x, r, partial);
        dot_final_kernel<<<1, DOT_THREADS, 0, s>>>(partial, scal, 2, -1);  // rr
        CG_CUDA(cudaMemcpyAsync(h, scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, s));
        CG_CUDA(cudaEventRecord(ctx->ev[24], s));
        // queue the rest of the iteration before looking at the residual
        CG_TRY(apply_precond(ctx, precond, r, z, s));
        CG_TRY(dot2(ctx, r, z, nullptr, nullptr, 3, -1, s));  // rz_new
        cg_direction_kernel<<<gb, 256, 0, s>>>(M, scal, z, p);
        cg_shift_kernel<<<1, 1, 0, s>>>(scal);
        ctx->launch_total += 4;  // update, rr reduction, direction, shift
        CG_CUDA(cudaGetLastError());
        CG_CUDA(cudaEventSynchronize(ctx->ev[24]));
        ++it;
        rn = std::sqrt(h[2]);
    }
    // true residual
    CG_TRY(launch_amatvec_sorted(ctx, x, Ap, s));
    residual_kernel<<<gb, 256, 0, s>>>(M, b, Ap, z);
    CG_TRY(dot2(ctx, z, z, nullptr, nullptr, 4, -1, s));
    scatter_kernel<<<gb, 256, 0, s>>>(M, ctx->s2c, x, x_caller);
    ctx->launch_total += 2;
    CG_CUDA(cudaMemcpyAsync(h, scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, s));
    CG_CUDA(cudaStreamSynchronize(s));
#undef CG_TRY
#undef CG_CUDA
    ctx->timing = saved_timing;
    if (iters) *iters = it;
    if (resid) { resid[0] = rn; resid[1] = std::sqrt(h[4]); }
    return rn > tol ? PCM_NOT_CONVERGED : PCM_OK;
}

}  // namespace pcm
