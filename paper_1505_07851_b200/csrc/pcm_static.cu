// pcm_static.cu -- pcm_amatvec_static: y = A q (Eq. 2, 3, 8) for callers that may not allocate.
//
// No context, no cudaMalloc / cudaFree / allocating library routine anywhere on this path: the caller passes the points, q and
// y as device pointers, and the one piece of scratch the product needs -- the partial row sums of the column chunks, which a
// second kernel adds in a fixed order, as every reduction of this library does -- lives in a file-scope __device__ array of a
// fixed, modest size: ST_CHUNKS x PCM_STATIC_MAX_POINTS doubles = 2 MiB, held by every GPU that loads the library until the
// process exits.  Code under CUDA graph capture, serving loops and harnesses that forbid allocation can call it; everything
// else should use pcm_setup + pcm_amatvec, which is several times faster (symmetric sweep, stored near patches).
//
// The array is SHARED by every call on a device and keeps the last call's contents.  Nothing in it has to start at zero: a
// call writes every slot (chunk, row < npoint) it later reads -- chunks that lie beyond the last column write 0.0 -- so stale
// values of an earlier, larger call are never read.  Calls that overlap on one GPU (two streams, two host threads) race on it.
//
// In host code the array's name is a host-side stand-in, not a device address; the address comes from cudaGetSymbolAddress,
// once per device, with that device current (static_scratch below), and is what the kernels are given.
#include <mutex>
#include <string>

#include "pcm_internal.h"

namespace pcm {

constexpr int ST_MAX_POINTS = PCM_STATIC_MAX_POINTS;
constexpr int ST_CHUNKS = 16;      // column chunks = partial sums per row
constexpr int ST_ROWS = 128;       // rows (threads) of a CTA
constexpr int ST_TILE = 256;       // columns staged in shared memory at a time
constexpr int ST_MAX_DEVICES = 64;

static __device__ __align__(256) double g_static_scratch[(size_t)ST_CHUNKS * ST_MAX_POINTS];

// A_ij as the paper prints it: A_ii = zeta_i sqrt(2/pi) / S_i (R1), A_ij = erf(zeta' r)/r with
// zeta' = zeta_i zeta_j / sqrt(zeta_i^2 + zeta_j^2); r = 0 (coincident points, R9) -> the limit 2 zeta'/sqrt(pi).
// erf(x) rounds to 1 in fp64 from x = 5.93 on, so beyond zeta' r = 6 the entry is 1/r.
__device__ __forceinline__ double static_a_entry(bool diag, double dx, double dy, double dz, double zi, double zj, double si) {
    if (diag) return zi * 0.79788456080286535588 / si;
    const double zp = zi * zj / sqrt(fma(zi, zi, zj * zj));
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    if (r2 == 0.0) return zp * 1.12837916709551257390;
    const double r = sqrt(r2), x = zp * r;
    return (x >= 6.0 ? 1.0 : erf(x)) / r;
}

// part[chunk][i] = sum over the columns j of the chunk of A_ij q_j, in column order; thread = row, columns staged in tiles
__global__ void __launch_bounds__(ST_ROWS) amatvec_static_sweep_kernel(int M, int chunk_len, const double *__restrict__ xyz,
                                                                       const double *__restrict__ zeta, const double *__restrict__ sw,
                                                                       const double *__restrict__ q, double *__restrict__ part) {
    __shared__ double4 s_c[ST_TILE];     // (x, y, z, zeta) of a column
    __shared__ double s_q[ST_TILE];
    const int i = blockIdx.x * ST_ROWS + threadIdx.x, ic = min(i, M - 1);
    const int c0 = blockIdx.y * chunk_len, c1 = min(M, c0 + chunk_len);
    const double xi = xyz[3 * (size_t)ic], yi = xyz[3 * (size_t)ic + 1], zi3 = xyz[3 * (size_t)ic + 2];
    const double zi = zeta[ic], si = sw[ic];
    double acc = 0.0;
    for (int j0 = c0; j0 < c1; j0 += ST_TILE) {
        __syncthreads();
        for (int t = threadIdx.x; t < ST_TILE; t += ST_ROWS) {
            const int j = j0 + t;
            if (j < c1) {
                s_c[t] = make_double4(xyz[3 * (size_t)j], xyz[3 * (size_t)j + 1], xyz[3 * (size_t)j + 2], zeta[j]);
                s_q[t] = q[j];
            }
        }
        __syncthreads();
        const int n = min(ST_TILE, c1 - j0);
        for (int t = 0; t < n; ++t) {
            const double4 c = s_c[t];
            acc = fma(static_a_entry(j0 + t == i, xi - c.x, yi - c.y, zi3 - c.z, zi, c.w, si), s_q[t], acc);
        }
    }
    if (i < M) part[(size_t)blockIdx.y * ST_MAX_POINTS + i] = acc;       // chunks beyond the last column leave 0.0 here
}

// y_i = the chunks' partial sums of row i, added in chunk order
__global__ void amatvec_static_reduce_kernel(int M, const double *__restrict__ part, double *__restrict__ y) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < ST_CHUNKS; ++c) s += part[(size_t)c * ST_MAX_POINTS + i];
    y[i] = s;
}

// Device address of the scratch array on the current device, resolved once per device (cudaGetSymbolAddress allocates
// nothing: the array is part of the loaded module).
static int static_scratch(double **out) {
    static std::mutex mu;
    static double *ptr[ST_MAX_DEVICES] = {};
    int dev = 0;
    PCM_CUDA(nullptr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= ST_MAX_DEVICES) return set_error(nullptr, PCM_ERR_ARG, "pcm_amatvec_static: device index beyond 63");
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        double *p = nullptr;
        PCM_CUDA(nullptr, cudaGetSymbolAddress((void **)&p, g_static_scratch));
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return PCM_OK;
}

}  // namespace pcm

using namespace pcm;

extern "C" {

int pcm_amatvec_static_init(void) {
    double *p = nullptr;
    return static_scratch(&p);
}

int pcm_amatvec_static(int64_t npoint, const double *pt_xyz_dev, const double *pt_zeta_dev, const double *pt_switch_dev,
                       const double *q_dev, double *y_dev, void *stream) {
    if (npoint < 0) return set_error(nullptr, PCM_ERR_ARG, "pcm_amatvec_static: npoint < 0");
    if (npoint > ST_MAX_POINTS)
        return set_error(nullptr, PCM_ERR_ARG, "pcm_amatvec_static: npoint = " + std::to_string(npoint) + " exceeds PCM_STATIC_MAX_POINTS = " +
                                                   std::to_string(ST_MAX_POINTS) + " (the static scratch array is sized for that; use pcm_setup + pcm_amatvec)");
    if (npoint == 0) return PCM_OK;
    if (!pt_xyz_dev || !pt_zeta_dev || !pt_switch_dev || !q_dev || !y_dev) return set_error(nullptr, PCM_ERR_ARG, "pcm_amatvec_static: NULL pointer");
    double *part = nullptr;
    int rc = static_scratch(&part);
    if (rc) return rc;
    const int M = (int)npoint;
    const int chunk_len = ((M + ST_CHUNKS - 1) / ST_CHUNKS + 31) / 32 * 32;
    cudaStream_t s = (cudaStream_t)stream;
    amatvec_static_sweep_kernel<<<dim3((unsigned)((M + ST_ROWS - 1) / ST_ROWS), ST_CHUNKS), ST_ROWS, 0, s>>>(M, chunk_len, pt_xyz_dev, pt_zeta_dev,
                                                                                                              pt_switch_dev, q_dev, part);
    amatvec_static_reduce_kernel<<<(unsigned)((M + 255) / 256), 256, 0, s>>>(M, part, y_dev);
    PCM_CUDA(nullptr, cudaGetLastError());
    return PCM_OK;
}

}  // extern "C"
