// pcm_cavity.cu -- ISWIG cavity construction on the device.
// Every atom I carries the same unit-sphere quadrature (nodes u_g, weights w_g; an input -- the paper uses Lebedev grids):
//   r = R_I + rad_I u_g,  zeta = zeta_tab/(rad_I sqrt(w_g)) (Eq. 7),  S = prod_{J != I} S_wf(r, R_J) (Eq. 9),
// and a point is kept iff S >= s_min (the paper's 1e-8 screening).  One thread per (atom, node) evaluates S with the atoms
// staged through shared memory; the survivors are compacted in (atom, node) order by a block-count / scan / scatter pass,
// so the point order is fixed.  The result stays on the device (pcm_cavity) and feeds pcm_setup_cavity.
#include <algorithm>
#include <cmath>
#include <new>
#include <vector>

#include "pcm_internal.h"

struct pcm_cavity {
    int device = 0;
    int natom = 0, ngrid = 0;
    int64_t npoint = 0;
    double *xyz = nullptr, *zeta = nullptr, *S = nullptr;   // device: [3 n], [n], [n]
    int32_t *atom = nullptr, *node = nullptr;              // device: [n], [n]
    std::vector<double> atom_xyz, atom_radius;             // host copies (pcm_setup_cavity registers them with the context)
};

namespace pcm {

constexpr int CV_TPB = 128;
constexpr int CV_TILE = 256;
constexpr double CV_SWITCH_CUT = 6.2;   // zeta (d - R) beyond which S_wf = 1 to fp64 (erfc(6.2) = 2e-18)

// S of every candidate (atom I, node g), candidate index c = I G + g; flag[c] = S >= s_min
__global__ void __launch_bounds__(CV_TPB) cavity_eval_kernel(int natom, int ngrid, const double4 *__restrict__ atoms /* x, y, z, radius */,
                                                             const double4 *__restrict__ grid /* u, w */, double zeta_tab, double s_min,
                                                             double4 *__restrict__ cand /* x, y, z, zeta */, double *__restrict__ candS,
                                                             int32_t *__restrict__ flag) {
    __shared__ double4 s_at[CV_TILE];
    const int64_t ncand = (int64_t)natom * ngrid;
    const int64_t c = (int64_t)blockIdx.x * CV_TPB + threadIdx.x;
    const int I = (int)(min(c, ncand - 1) / ngrid), g = (int)(min(c, ncand - 1) - (int64_t)I * ngrid);
    const double4 a = atoms[I], u = grid[g];
    const double x = a.x + a.w * u.x, y = a.y + a.w * u.y, z = a.z + a.w * u.z;
    const double zeta = zeta_tab / (a.w * sqrt(u.w));
    double S = 1.0;
    for (int base = 0; base < natom; base += CV_TILE) {
        const int cnt = min(CV_TILE, natom - base);
        __syncthreads();
        for (int t = threadIdx.x; t < cnt; t += CV_TPB) s_at[t] = atoms[base + t];
        __syncthreads();
        for (int t = 0; t < cnt; ++t) {
            if (base + t == I) continue;
            const double4 b = s_at[t];
            const double dx = x - b.x, dy = y - b.y, dz = z - b.z;
            const double d = sqrt(dx * dx + dy * dy + dz * dz);
            if (zeta * (d - b.w) > CV_SWITCH_CUT) continue;     // S_wf = 1
            S *= 1.0 - 0.5 * (erf(zeta * (b.w - d)) + erf(zeta * (b.w + d)));
        }
    }
    if (c < ncand) {
        cand[c] = make_double4(x, y, z, zeta);
        candS[c] = S;
        flag[c] = (S >= s_min) ? 1 : 0;
    }
}

// kept candidates per block of CV_SCAN candidates
constexpr int CV_SCAN = 1024;
__global__ void __launch_bounds__(256) cavity_count_kernel(int64_t ncand, const int32_t *__restrict__ flag, int32_t *__restrict__ bcount) {
    __shared__ int s_w[8];
    const int64_t base = (int64_t)blockIdx.x * CV_SCAN;
    int n = 0;
    for (int t = threadIdx.x; t < CV_SCAN; t += 256)
        if (base + t < ncand) n += flag[base + t];
    for (int o = 16; o > 0; o >>= 1) n += __shfl_down_sync(0xffffffffu, n, o);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = n;
    __syncthreads();
    if (threadIdx.x == 0) {
        int s = 0;
        for (int w = 0; w < 8; ++w) s += s_w[w];
        bcount[blockIdx.x] = s;
    }
}
// exclusive scan of the block counts (one CTA; the count array is a few thousand entries at most); total -> boff[nblk]
__global__ void __launch_bounds__(1024) cavity_scan_kernel(int nblk, const int32_t *__restrict__ bcount, int64_t *__restrict__ boff) {
    __shared__ int64_t s_part[1024];
    const int per = (nblk + 1023) / 1024;
    const int b0 = threadIdx.x * per, b1 = min(nblk, b0 + per);
    int64_t s = 0;
    for (int b = b0; b < b1; ++b) s += bcount[b];
    s_part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        int64_t run = 0;
        for (int t = 0; t < 1024; ++t) { const int64_t v = s_part[t]; s_part[t] = run; run += v; }
        boff[nblk] = run;
    }
    __syncthreads();
    int64_t run = s_part[threadIdx.x];
    for (int b = b0; b < b1; ++b) { boff[b] = run; run += bcount[b]; }
}
// survivors to their final slots, candidate order preserved (one warp walks its 32-candidate strips in order)
__global__ void __launch_bounds__(256) cavity_scatter_kernel(int64_t ncand, int ngrid, const int32_t *__restrict__ flag,
                                                             const int64_t *__restrict__ boff, const double4 *__restrict__ cand,
                                                             const double *__restrict__ candS, double *__restrict__ xyz,
                                                             double *__restrict__ zeta, double *__restrict__ S,
                                                             int32_t *__restrict__ atom, int32_t *__restrict__ node) {
    __shared__ int s_cnt[CV_SCAN / 32 + 1];
    const int64_t base = (int64_t)blockIdx.x * CV_SCAN;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // strip s = candidates base + 32 s .. : count per strip, then a serial scan over the 32 strips, then the scatter
    for (int s = warp; s < CV_SCAN / 32; s += 8) {
        const int64_t c = base + s * 32 + lane;
        const unsigned m = __ballot_sync(0xffffffffu, c < ncand && flag[c]);
        if (lane == 0) s_cnt[s] = __popc(m);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int run = 0;
        for (int s = 0; s < CV_SCAN / 32; ++s) { const int v = s_cnt[s]; s_cnt[s] = run; run += v; }
    }
    __syncthreads();
    for (int s = warp; s < CV_SCAN / 32; s += 8) {
        const int64_t c = base + s * 32 + lane;
        const bool keep = c < ncand && flag[c];
        const unsigned m = __ballot_sync(0xffffffffu, keep);
        if (keep) {
            const int64_t o = boff[blockIdx.x] + s_cnt[s] + __popc(m & ((1u << lane) - 1u));
            const double4 p = cand[c];
            xyz[3 * o] = p.x; xyz[3 * o + 1] = p.y; xyz[3 * o + 2] = p.z;
            zeta[o] = p.w;
            S[o] = candS[c];
            atom[o] = (int32_t)(c / ngrid);
            node[o] = (int32_t)(c - (c / ngrid) * ngrid);
        }
    }
}

static void cavity_free(pcm_cavity *c) {
    if (!c) return;
    cudaSetDevice(c->device);
    cudaFree(c->xyz); cudaFree(c->zeta); cudaFree(c->S); cudaFree(c->atom); cudaFree(c->node);
    delete c;
}

int build_context(pcm_ctx *ctx, int nshell, const int *shell_l, const double *shell_xyz, const int *shell_nprim,
                  const double *prim_exp, const double *prim_coef, int64_t npoint, const double *pt_xyz,
                  const double *pt_zeta, const double *pt_switch);

}  // namespace pcm

using namespace pcm;

extern "C" {

int pcm_build_cavity(pcm_cavity **out, int natom, const double *atom_xyz_host, const double *atom_radius_host, int ngrid,
                     const double *grid_xyz_host, const double *grid_weight_host, double zeta_tab, double s_min, int device) {
    if (!out) return set_error(nullptr, PCM_ERR_ARG, "pcm_build_cavity: out is NULL");
    *out = nullptr;
    if (natom < 0 || ngrid < 0 || (natom > 0 && (!atom_xyz_host || !atom_radius_host)) || (ngrid > 0 && (!grid_xyz_host || !grid_weight_host)) ||
        !(zeta_tab > 0.0) || !(s_min >= 0.0))
        return set_error(nullptr, PCM_ERR_ARG, "pcm_build_cavity: bad argument");
    for (int j = 0; j < natom; ++j)
        if (!(atom_radius_host[j] > 0.0) || !std::isfinite(atom_radius_host[j])) return set_error(nullptr, PCM_ERR_ARG, "pcm_build_cavity: radii must be positive");
    for (int g = 0; g < ngrid; ++g)
        if (!(grid_weight_host[g] > 0.0) || !std::isfinite(grid_weight_host[g])) return set_error(nullptr, PCM_ERR_ARG, "pcm_build_cavity: weights must be positive");
    const int64_t ncand = (int64_t)natom * ngrid;
    if (ncand > 0x7fffffff) return set_error(nullptr, PCM_ERR_ARG, "pcm_build_cavity: natom * ngrid too large");
    pcm_cavity *cav = new (std::nothrow) pcm_cavity();
    if (!cav) return set_error(nullptr, PCM_ERR_ALLOC, "pcm_build_cavity: out of host memory");
    cudaError_t e = cudaSuccess;
    if (device < 0) e = cudaGetDevice(&device);
    if (e == cudaSuccess) e = cudaSetDevice(device);
    cav->device = device;
    cav->natom = natom;
    cav->ngrid = ngrid;
    cav->atom_xyz.assign(atom_xyz_host, atom_xyz_host + 3 * (size_t)natom);
    cav->atom_radius.assign(atom_radius_host, atom_radius_host + (size_t)natom);
    double4 *d_at = nullptr, *d_grid = nullptr, *d_cand = nullptr;
    double *d_S = nullptr;
    int32_t *d_flag = nullptr, *d_bcount = nullptr;
    int64_t *d_boff = nullptr;
    auto done = [&](int rc, const std::string &msg) {
        cudaFree(d_at); cudaFree(d_grid); cudaFree(d_cand); cudaFree(d_S); cudaFree(d_flag); cudaFree(d_bcount); cudaFree(d_boff);
        if (rc != PCM_OK) { cavity_free(cav); return set_error(nullptr, rc, msg); }
        *out = cav;
        return PCM_OK;
    };
    if (e != cudaSuccess) return done(PCM_ERR_CUDA, std::string("pcm_build_cavity: ") + cudaGetErrorString(e));
    if (ncand == 0) return done(PCM_OK, "");
    std::vector<double4> at((size_t)natom), gr((size_t)ngrid);
    for (int j = 0; j < natom; ++j) at[j] = make_double4(atom_xyz_host[3 * j], atom_xyz_host[3 * j + 1], atom_xyz_host[3 * j + 2], atom_radius_host[j]);
    for (int g = 0; g < ngrid; ++g) gr[g] = make_double4(grid_xyz_host[3 * g], grid_xyz_host[3 * g + 1], grid_xyz_host[3 * g + 2], grid_weight_host[g]);
    const int nblk = (int)((ncand + CV_SCAN - 1) / CV_SCAN);
    e = cudaMalloc(&d_at, at.size() * sizeof(double4));
    if (e == cudaSuccess) e = cudaMalloc(&d_grid, gr.size() * sizeof(double4));
    if (e == cudaSuccess) e = cudaMalloc(&d_cand, (size_t)ncand * sizeof(double4));
    if (e == cudaSuccess) e = cudaMalloc(&d_S, (size_t)ncand * 8);
    if (e == cudaSuccess) e = cudaMalloc(&d_flag, (size_t)ncand * 4);
    if (e == cudaSuccess) e = cudaMalloc(&d_bcount, (size_t)nblk * 4);
    if (e == cudaSuccess) e = cudaMalloc(&d_boff, (size_t)(nblk + 1) * 8);
    if (e != cudaSuccess) return done(PCM_ERR_ALLOC, std::string("pcm_build_cavity: cudaMalloc: ") + cudaGetErrorString(e));
    e = cudaMemcpy(d_at, at.data(), at.size() * sizeof(double4), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d_grid, gr.data(), gr.size() * sizeof(double4), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        cavity_eval_kernel<<<(unsigned)((ncand + CV_TPB - 1) / CV_TPB), CV_TPB>>>(natom, ngrid, d_at, d_grid, zeta_tab, s_min, d_cand, d_S, d_flag);
        cavity_count_kernel<<<(unsigned)nblk, 256>>>(ncand, d_flag, d_bcount);
        cavity_scan_kernel<<<1, 1024>>>(nblk, d_bcount, d_boff);
        e = cudaGetLastError();
    }
    int64_t n = 0;
    if (e == cudaSuccess) e = cudaMemcpy(&n, d_boff + nblk, 8, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return done(PCM_ERR_CUDA, std::string("pcm_build_cavity: ") + cudaGetErrorString(e));
    cav->npoint = n;
    if (n > 0) {
        e = cudaMalloc(&cav->xyz, (size_t)n * 24);
        if (e == cudaSuccess) e = cudaMalloc(&cav->zeta, (size_t)n * 8);
        if (e == cudaSuccess) e = cudaMalloc(&cav->S, (size_t)n * 8);
        if (e == cudaSuccess) e = cudaMalloc(&cav->atom, (size_t)n * 4);
        if (e == cudaSuccess) e = cudaMalloc(&cav->node, (size_t)n * 4);
        if (e != cudaSuccess) return done(PCM_ERR_ALLOC, std::string("pcm_build_cavity: cudaMalloc: ") + cudaGetErrorString(e));
        cavity_scatter_kernel<<<(unsigned)nblk, 256>>>(ncand, ngrid, d_flag, d_boff, d_cand, d_S, cav->xyz, cav->zeta, cav->S, cav->atom, cav->node);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        if (e != cudaSuccess) return done(PCM_ERR_CUDA, std::string("pcm_build_cavity: ") + cudaGetErrorString(e));
    }
    return done(PCM_OK, "");
}

int pcm_cavity_size(const pcm_cavity *cav, int64_t *npoint) {
    if (!cav || !npoint) return PCM_ERR_ARG;
    *npoint = cav->npoint;
    return PCM_OK;
}

int pcm_cavity_get(const pcm_cavity *cav, double *pt_xyz_host, double *pt_zeta_host, double *pt_switch_host, int32_t *pt_atom_host,
                   int32_t *pt_node_host) {
    if (!cav) return PCM_ERR_ARG;
    const size_t n = (size_t)cav->npoint;
    if (n == 0) return PCM_OK;
    cudaError_t e = cudaSetDevice(cav->device);
    if (e == cudaSuccess && pt_xyz_host) e = cudaMemcpy(pt_xyz_host, cav->xyz, n * 24, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && pt_zeta_host) e = cudaMemcpy(pt_zeta_host, cav->zeta, n * 8, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && pt_switch_host) e = cudaMemcpy(pt_switch_host, cav->S, n * 8, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && pt_atom_host) e = cudaMemcpy(pt_atom_host, cav->atom, n * 4, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && pt_node_host) e = cudaMemcpy(pt_node_host, cav->node, n * 4, cudaMemcpyDeviceToHost);
    return e == cudaSuccess ? PCM_OK : set_error(nullptr, PCM_ERR_CUDA, std::string("pcm_cavity_get: ") + cudaGetErrorString(e));
}

int pcm_cavity_device(const pcm_cavity *cav, const double **xyz_dev, const double **zeta_dev, const double **switch_dev,
                      const int32_t **atom_dev, const int32_t **node_dev) {
    if (!cav) return PCM_ERR_ARG;
    if (xyz_dev) *xyz_dev = cav->xyz;
    if (zeta_dev) *zeta_dev = cav->zeta;
    if (switch_dev) *switch_dev = cav->S;
    if (atom_dev) *atom_dev = cav->atom;
    if (node_dev) *node_dev = cav->node;
    return PCM_OK;
}

int pcm_cavity_destroy(pcm_cavity *cav) {
    cavity_free(cav);
    return PCM_OK;
}

// pcm_setup with the points, exponents and switching values of a built cavity.  pcm_setup sorts the points and classifies
// the patches on the host, so the cavity arrays are read back once, inside the library; the caller never handles them.
int pcm_setup_cavity(pcm_ctx **out, int nshell, const int *shell_l, const double *shell_xyz, const int *shell_nprim,
                     const double *prim_exp, const double *prim_coef, const pcm_cavity *cav, const pcm_options *opt) {
    if (!out) return set_error(nullptr, PCM_ERR_ARG, "pcm_setup_cavity: out is NULL");
    *out = nullptr;
    if (!cav) return set_error(nullptr, PCM_ERR_ARG, "pcm_setup_cavity: cav is NULL");
    const size_t n = (size_t)cav->npoint;
    std::vector<double> xyz(3 * n + 1), zeta(n + 1), S(n + 1);
    std::vector<int32_t> own(n + 1);
    int rc = pcm_cavity_get(cav, xyz.data(), zeta.data(), S.data(), own.data(), nullptr);
    if (rc) return rc;
    pcm_options o;
    if (opt) o = *opt; else pcm_options_default(&o);
    if (o.device < 0) o.device = cav->device;
    rc = pcm_setup(out, nshell, shell_l, shell_xyz, shell_nprim, prim_exp, prim_coef, (int64_t)n, xyz.data(), zeta.data(), S.data(), &o);
    if (rc) return rc;
    pcm_ctx *ctx = *out;
    ctx->cav_natom = cav->natom;
    ctx->cav_radius_host = cav->atom_radius;
    ctx->cav_owner_host.assign(own.begin(), own.begin() + n);
    return PCM_OK;
}

}  // extern "C"
