// pcm_solver.cu -- steps a5 (randomized block-Jacobi build) and a6 (preconditioned CG,
// PAPER.md:164-170) of SURVEY.md 8(a).  The matrix-vector product is pcm_kernels.cu's on-the-fly A q.
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdlib>
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
    std::vector<std::pair<uint64_t, int64_t>> key((size_t)M);
    for (int64_t i = 0; i < M; ++i) key[i] = {mix64(seed + (uint64_t)(i + 1) * 0x9E3779B97F4A7C15ULL), i};
    std::sort(key.begin(), key.end());  // by key, ties by index
    for (int64_t i = 0; i < M; ++i) perm[i] = key[i].second;
}

// ---------------------------------------------------------------------------------------------
// A_ij for arbitrary i, j (Eq. 2, 3, 8)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double amat_entry(double r2, double izi, double izj, const double *__restrict__ boys0) {
    const double zp = rsqrt_fast(izi + izj);
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
__device__ __forceinline__ double a_entry(const double4 *__restrict__ pt, const double *__restrict__ diag, int i, int j,
                                          const double *__restrict__ boys0) {
    if (i == j) return diag[i];
    const double4 a = pt[i], b = pt[j];
    const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
    return amat_entry(fma(dz, dz, fma(dy, dy, dx * dx)), a.w, b.w, boys0);
}

// ---------------------------------------------------------------------------------------------
// RBJ block selection: ONE persistent cooperative kernel for the whole sequence of blocks.  The blocks
// are inherently sequential (the next pivot depends on what the previous blocks took), a step's work -- one row of A
// over the unassigned points, then the l-1 largest -- is tiny, so the cost is synchronisation: two grid barriers per
// step instead of three kernel launches.
//   phase A  every CTA finds the step's pivot (first unassigned index of the pivot order; same answer everywhere),
//            evaluates A_kj for its own unassigned j, keeps the keys, histograms them (1024 buckets of the top 16
//            key bits, a monotone map)                                                     -- grid barrier 1
//   phase B  every CTA reads the histogram, finds the cut bucket b* (the top `take` keys all have bucket >= b*) and
//            appends its own candidates (bucket >= b*) to the step's candidate list        -- grid barrier 2
//   phase C  every CTA ranks the (few) candidates by (key descending, caller index ascending) and marks the first
//            `take` as assigned: all CTAs compute the same set and write the same flags, so no third barrier is
//            needed; CTA 0 also writes the block to `order`.
// Histograms are triple-buffered, candidate lists double-buffered; CTA 0 clears a buffer two phases after its last
// reader.  Keys are A_kj > 0 compared as doubles.
// ---------------------------------------------------------------------------------------------
constexpr int RBJ_BINS = 1024;
constexpr int RBJ_BIN_BASE = 0x3e00;  // bucket of 2^-31
constexpr int RBJ_THREADS = 512;
constexpr int RBJ_CAP = 1536;         // candidates ranked from shared memory; more (many near-ties) take the global path

__device__ __forceinline__ int rbj_bucket(double a) {
    const int b = (int)((unsigned long long)__double_as_longlong(a) >> 48) - RBJ_BIN_BASE;
    return min(max(b, 0), RBJ_BINS - 1);
}

struct RbjWork {
    int *hist;                 // [3][RBJ_BINS]
    int *cand_count;           // [2]
    double *cand_key;          // [2][M]
    int *cand_idx;             // [2][M]
    double *keys;              // [M]
    unsigned char *assigned;   // [M]
    unsigned long long *bar;   // grid barrier counter
    int *err;
};

__device__ __forceinline__ void grid_barrier(unsigned long long *bar, unsigned long long &target, unsigned nblocks) {
    __syncthreads();
    if (threadIdx.x == 0) {
        target += nblocks;
        __threadfence();
        atomicAdd(bar, 1ULL);
        while (*((volatile unsigned long long *)bar) < target) { }
        __threadfence();
    }
    __syncthreads();
}

__global__ void __launch_bounds__(RBJ_THREADS) rbj_select_kernel(const double4 *__restrict__ pt, const double *__restrict__ diag,
                                                                 int M, int block, const int32_t *__restrict__ perm,
                                                                 const int32_t *__restrict__ s2c, int32_t *__restrict__ order,
                                                                 RbjWork w, const double *__restrict__ boys0) {
    __shared__ int s_hist[RBJ_BINS];
    __shared__ int s_scan[RBJ_THREADS];
    __shared__ double s_key[RBJ_CAP];
    __shared__ int s_idx[RBJ_CAP];
    __shared__ int s_cidx[RBJ_CAP];
    __shared__ int s_pivot, s_bstar;
    const unsigned nblocks = gridDim.x;
    const int tid = threadIdx.x, gtid = blockIdx.x * RBJ_THREADS + tid, gstride = nblocks * RBJ_THREADS;
    unsigned long long target = 0;
    long long pos = 0, filled = 0;
    for (long long step = 0; filled < M; ++step) {
        int *hist = w.hist + (step % 3) * RBJ_BINS;
        int *cnt = w.cand_count + (step & 1);
        double *ckey = w.cand_key + (size_t)(step & 1) * M;
        int *cidx = w.cand_idx + (size_t)(step & 1) * M;
        // ---- phase A: pivot, keys, histogram
        if (tid == 0) s_pivot = M;
        for (int t = tid; t < RBJ_BINS; t += RBJ_THREADS) s_hist[t] = 0;
        __syncthreads();
        while (true) {
            const long long p = pos + tid;
            if (p < M && !w.assigned[perm[p]]) atomicMin(&s_pivot, (int)p);
            __syncthreads();
            if (s_pivot < M || pos + RBJ_THREADS >= M) break;
            pos += RBJ_THREADS;
            __syncthreads();
        }
        const int ppos = s_pivot;
        if (ppos >= M) { if (gtid == 0) *w.err = 2; return; }  // cannot happen while filled < M (uniform exit)
        pos = ppos;
        const int k = perm[ppos];
        const long long remaining = M - filled - 1;
        const int take = (int)min((long long)block - 1, remaining);
        const double4 pk = pt[k];
        for (int j = gtid; j < M; j += gstride) {
            double a = 0.0;
            if (!w.assigned[j] && j != k) {
                const double4 b = pt[j];
                const double dx = pk.x - b.x, dy = pk.y - b.y, dz = pk.z - b.z;
                a = amat_entry(fma(dz, dz, fma(dy, dy, dx * dx)), pk.w, b.w, boys0);
                atomicAdd(&s_hist[rbj_bucket(a)], 1);
            }
            w.keys[j] = a;
        }
        __syncthreads();
        if (take > 0)
            for (int t = tid; t < RBJ_BINS; t += RBJ_THREADS)
                if (s_hist[t]) atomicAdd(&hist[t], s_hist[t]);
        if (blockIdx.x == 0) {  // clear what step + 1 will accumulate into (last read in phase B of step - 2)
            int *nh = w.hist + ((step + 1) % 3) * RBJ_BINS;
            for (int t = tid; t < RBJ_BINS; t += RBJ_THREADS) nh[t] = 0;
        }
        grid_barrier(w.bar, target, nblocks);
        // ---- phase B: cut bucket, candidates
        if (take > 0) {
            // suffix counts: s_scan[t] = keys in buckets >= 2t (two buckets per thread)
            const int h0 = __ldcg(hist + 2 * tid), h1 = __ldcg(hist + 2 * tid + 1);
            s_scan[tid] = h0 + h1;
            __syncthreads();
            for (int o = 1; o < RBJ_THREADS; o <<= 1) {
                const int v = (tid + o < RBJ_THREADS) ? s_scan[tid + o] : 0;
                __syncthreads();
                s_scan[tid] += v;
                __syncthreads();
            }
            // b* = the largest bucket b with count(bucket >= b) >= take
            const int above = (tid + 1 < RBJ_THREADS) ? s_scan[tid + 1] : 0;  // buckets >= 2 tid + 2
            if (above < take && above + h1 >= take) s_bstar = 2 * tid + 1;
            else if (above + h1 < take && above + h1 + h0 >= take) s_bstar = 2 * tid;
            __syncthreads();
            const int bstar = s_bstar;
            for (int j = gtid; j < M; j += gstride) {
                const double a = w.keys[j];
                if (a > 0.0 && rbj_bucket(a) >= bstar) {
                    const int slot = atomicAdd(cnt, 1);
                    ckey[slot] = a;
                    cidx[slot] = j;
                }
            }
        }
        if (blockIdx.x == 0 && tid == 0) w.cand_count[(step + 1) & 1] = 0;  // last read in phase C of step - 1
        grid_barrier(w.bar, target, nblocks);
        // ---- phase C: rank, mark, record (every CTA computes the same selection)
        if (take > 0) {
            const int n = *((volatile int *)cnt);
            if (n < take) { if (gtid == 0) *w.err = 1; return; }  // cannot happen: the cut keeps at least `take`
            if (n <= RBJ_CAP) {
                for (int c = tid; c < n; c += RBJ_THREADS) {
                    const int j = __ldcg(cidx + c);
                    s_key[c] = __ldcg(ckey + c);
                    s_idx[c] = j;
                    s_cidx[c] = s2c[j];
                }
                __syncthreads();
                for (int c = tid; c < n; c += RBJ_THREADS) {
                    const double key = s_key[c];
                    const int ci = s_cidx[c];  // ties -> lower index in the caller's numbering
                    int rank = 0;
                    for (int o = 0; o < n; ++o) rank += (s_key[o] > key) || (s_key[o] == key && s_cidx[o] < ci);
                    if (rank < take) {
                        w.assigned[s_idx[c]] = 1;
                        if (blockIdx.x == 0) order[filled + 1 + rank] = s_idx[c];
                    }
                }
            } else {
                for (int c = tid; c < n; c += RBJ_THREADS) {
                    const double key = __ldcg(ckey + c);
                    const int j = __ldcg(cidx + c), ci = s2c[j];
                    int rank = 0;
                    for (int o = 0; o < n; ++o) {
                        const double ko = __ldcg(ckey + o);
                        rank += (ko > key) || (ko == key && s2c[__ldcg(cidx + o)] < ci);
                    }
                    if (rank < take) {
                        w.assigned[j] = 1;
                        if (blockIdx.x == 0) order[filled + 1 + rank] = j;
                    }
                }
            }
        }
        if (tid == 0) {
            w.assigned[k] = 1;
            if (blockIdx.x == 0) order[filled] = k;
        }
        filled += 1 + take;
        pos += 1;
        __syncthreads();  // this CTA's own flag writes are visible to its own threads in the next phase A
    }
}

// ---------------------------------------------------------------------------------------------
// RBJ block selection, neighbourhood version: ONE CTA, no grid barrier.  A_kj = erf(zeta' r)/r <= 1/r, so if every
// unassigned point within a radius rho of the pivot is a candidate and the take-th largest candidate key tau exceeds
// 1/rho, no point outside can enter the block: the l-1 largest over the candidates are the l-1 largest over all
// unassigned points -- the same block the global row scan of rbj_select_kernel finds, for a few hundred evaluations
// and a few block-level barriers per step instead of M evaluations and two grid barriers.  The candidates are the
// unassigned points of the groups of 32 (Hilbert order) whose bounding box is closer than rho; rho adapts from step to
// step (1.25/tau of the previous block) and grows when the test fails or too few candidates are found.  Selection among
// the candidates is the same as in rbj_select_kernel: histogram cut on the top 16 key bits, then ranking by (key
// descending, caller index ascending).  Used for block sizes <= 256; err = 3 asks the host to fall back.
// ---------------------------------------------------------------------------------------------
constexpr int RBL_THREADS = 1024;
constexpr int64_t RBJ_LOCAL_MAX = 150000;   // points up to which pcm_rbj_build uses this form
constexpr int RBL_RAW = 3072;   // candidate capacity (raw)
constexpr int RBL_CAP = 1024;   // candidates above the histogram cut that are ranked
constexpr int RBL_GL = 1024;    // candidate groups kept in shared memory (more: the global list)

struct RblShared {
    int hist[RBJ_BINS];
    int scan[RBJ_BINS];
    double rkey[RBL_RAW];
    int ridx[RBL_RAW];
    int rcal[RBL_RAW];          // caller index of a raw candidate (tie-break key)
    int sgl[RBL_GL];            // candidate groups (shared-memory copy of glist while they fit)
    double ckey[RBL_CAP];
    int cidx[RBL_CAP];
    int ccal[RBL_CAP];
    int crank[RBL_CAP];
    int pivot, nraw, ncut, bstar, ngl, all_in, ok;
    double rho, tau;
};

__global__ void __launch_bounds__(RBL_THREADS) rbj_select_local_kernel(const double4 *__restrict__ pt, int M, int block,
                                                                       const int32_t *__restrict__ perm,
                                                                       const int32_t *__restrict__ s2c,
                                                                       int32_t *__restrict__ order,
                                                                       unsigned char *__restrict__ assigned,
                                                                       const double *__restrict__ boxes, int ng,
                                                                       int *__restrict__ gcount, int *__restrict__ glist,
                                                                       int *__restrict__ err, const double *__restrict__ boys0,
                                                                       int cache) {
    extern __shared__ __align__(16) unsigned char rbl_smem[];
    RblShared &S = *reinterpret_cast<RblShared *>(rbl_smem);
    const int tid = threadIdx.x;
    // cache != 0: the assigned flags, the per-group counts and the group boxes live in shared memory behind S
    // (every step reads them several times in dependent order; from L2 that is most of a step's latency)
    double *s_bx = reinterpret_cast<double *>(rbl_smem + (sizeof(RblShared) + 15) / 16 * 16);
    int *s_gc = reinterpret_cast<int *>(s_bx + (size_t)6 * ng);
    unsigned char *s_asg = reinterpret_cast<unsigned char *>(s_gc + ng);
    unsigned char *asg = cache ? s_asg : assigned;
    int *gc = cache ? s_gc : gcount;
    const double *bx = cache ? s_bx : boxes;
    if (cache) {
        for (int i = tid; i < 6 * ng; i += RBL_THREADS) s_bx[i] = boxes[i];
        for (int i = tid; i < M; i += RBL_THREADS) s_asg[i] = 0;
    }
    for (int g = tid; g < ng; g += RBL_THREADS) gc[g] = min(32, M - g * 32);
    if (tid == 0) S.rho = 6.0;
    __syncthreads();
    long long pos = 0, filled = 0;
    while (filled < M) {
        // ---- pivot: first unassigned index of the pivot order
        if (tid == 0) S.pivot = M;
        __syncthreads();
        while (true) {
            const long long p = pos + tid;
            if (p < M && !asg[perm[p]]) atomicMin(&S.pivot, (int)p);
            __syncthreads();
            if (S.pivot < M || pos + RBL_THREADS >= M) break;
            pos += RBL_THREADS;
            __syncthreads();
        }
        const int ppos = S.pivot;
        if (ppos >= M) { if (tid == 0) *err = 2; return; }
        pos = ppos;
        const int k = perm[ppos];
        const int take = (int)min((long long)block - 1, (long long)M - filled - 1);
        const double4 pk = pt[k];
        __syncthreads();
        if (tid == 0) { asg[k] = 1; atomicSub(&gc[k >> 5], 1); }
        __syncthreads();
        if (take > 0) {
            // this step's bracket of the radius: lo = a radius that was not enough, hi = one whose candidates overflowed the
            // store (unassigned points are unevenly spread late in the selection: one growth step can take in a whole
            // untouched region); between them the radius is bisected.  Uniform over the CTA.
            double lo = 0.0, hi = 0.0;
            int tries = 0;
            while (true) {
                // ---- candidate groups: bounding box closer than rho and something unassigned in it
                const double rho = S.rho, rho2 = rho * rho;
                if (tid == 0) { S.ngl = 0; S.nraw = 0; S.ncut = 0; S.all_in = 1; S.ok = 0; }
                for (int t = tid; t < RBJ_BINS; t += RBL_THREADS) S.hist[t] = 0;
                __syncthreads();
                for (int g = tid; g < ng; g += RBL_THREADS) {
                    if (gc[g] <= 0) continue;
                    const double *b = bx + (size_t)g * 6;
                    const double gx = fmax(fmax(b[0] - pk.x, pk.x - b[3]), 0.0), gy = fmax(fmax(b[1] - pk.y, pk.y - b[4]), 0.0),
                                 gz = fmax(fmax(b[2] - pk.z, pk.z - b[5]), 0.0);
                    if (gx * gx + gy * gy + gz * gz < rho2) {
                        const int slot = atomicAdd(&S.ngl, 1);
                        if (slot < RBL_GL) S.sgl[slot] = g;
                        glist[slot] = g;
                    } else S.all_in = 0;
                }
                __syncthreads();
                const int ngl = S.ngl;
                // ---- keys of the unassigned points of those groups
                for (int t = tid; t < ngl * 32; t += RBL_THREADS) {
                    const int j = (ngl <= RBL_GL ? S.sgl[t >> 5] : glist[t >> 5]) * 32 + (t & 31);
                    // whole warps run this loop (ngl * 32 items): one slot reservation per warp instead of one per candidate
                    const bool live = j < M && !asg[j];
                    const unsigned live_mask = __ballot_sync(0xffffffffu, live);
                    int wbase = 0;
                    if ((tid & 31) == 0 && live_mask) wbase = atomicAdd(&S.nraw, __popc(live_mask));
                    wbase = __shfl_sync(0xffffffffu, wbase, 0);
                    if (live) {
                        const int cal = s2c[j];
                        const double4 b = pt[j];
                        const double dx = pk.x - b.x, dy = pk.y - b.y, dz = pk.z - b.z;
                        const double a = amat_entry(fma(dz, dz, fma(dy, dy, dx * dx)), pk.w, b.w, boys0);
                        const int slot = wbase + __popc(live_mask & ((1u << (tid & 31)) - 1u));
                        if (slot < RBL_RAW) { S.rkey[slot] = a; S.ridx[slot] = j; S.rcal[slot] = cal; }
                        atomicAdd(&S.hist[rbj_bucket(a)], 1);
                    }
                }
                __syncthreads();
                const int nraw = S.nraw;
                if (nraw > RBL_RAW) {   // more candidates than the store holds: a smaller radius
                    hi = rho;
                    if (++tries > 64 || !(hi - lo > 1e-9 * hi)) { if (tid == 0) *err = 3; return; }
                    __syncthreads();
                    if (tid == 0) { S.rho = lo > 0.0 ? 0.5 * (lo + hi) : rho / 1.6; err[1] += 1; }
                    __syncthreads();
                    continue;
                }
                if (nraw < take) {   // not enough unassigned points within rho (all_in cannot be set: take <= unassigned)
                    lo = rho;
                    __syncthreads();
                    if (tid == 0) { S.rho = hi > 0.0 ? 0.5 * (lo + hi) : rho * 1.6; err[1] += 1; }
                    __syncthreads();
                    continue;
                }
                // ---- histogram cut: b* = the largest bucket b with count(bucket >= b) >= take
                {
                    const int lane = tid & 31, warp = tid >> 5;
                    const int h = S.hist[tid];
                    int v = h;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_down_sync(0xffffffffu, v, o); if (lane + o < 32) v += u; }
                    if (lane == 0) S.scan[warp] = v;
                    __syncthreads();
                    if (warp == 0) {
                        const int w = S.scan[lane];
                        int x = w;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_down_sync(0xffffffffu, x, o); if (lane + o < 32) x += u; }
                        S.scan[32 + lane] = x - w;   // keys in the buckets of the higher warps
                    }
                    __syncthreads();
                    const int ge = v + S.scan[32 + warp], gt = ge - h;
                    if (gt < take && ge >= take) S.bstar = tid;
                }
                __syncthreads();
                const int bstar = S.bstar;
                for (int c = tid; c < nraw; c += RBL_THREADS) {
                    const double a = S.rkey[c];
                    if (rbj_bucket(a) >= bstar) {
                        const int slot = atomicAdd(&S.ncut, 1);
                        if (slot < RBL_CAP) { S.ckey[slot] = a; S.cidx[slot] = S.ridx[c]; S.ccal[slot] = S.rcal[c]; }
                    }
                }
                __syncthreads();
                const int n = S.ncut;
                if (n < take) { if (tid == 0) *err = 1; return; }
                if (n > RBL_CAP) {      // too many keys in the cut bucket to rank: a smaller radius, as above
                    hi = rho;
                    if (++tries > 64 || !(hi - lo > 1e-9 * hi)) { if (tid == 0) *err = 3; return; }
                    __syncthreads();
                    if (tid == 0) { S.rho = lo > 0.0 ? 0.5 * (lo + hi) : rho / 1.6; err[1] += 1; }
                    __syncthreads();
                    continue;
                }
                // ---- rank by (key descending, caller index ascending); tau = the take-th largest key
                // one warp per candidate, the lanes stride over the others (n^2 / 1024 comparisons per thread)
                for (int cand = tid >> 5; cand < n; cand += RBL_THREADS / 32) {
                    const double key = S.ckey[cand];
                    const int ci = S.ccal[cand];
                    int cnt = 0;
                    for (int o = tid & 31; o < n; o += 32) cnt += (S.ckey[o] > key) || (S.ckey[o] == key && S.ccal[o] < ci);
                    cnt = __reduce_add_sync(0xffffffffu, cnt);
                    if ((tid & 31) == 0) {
                        S.crank[cand] = cnt;
                        if (cnt == take - 1) S.tau = key;
                    }
                }
                __syncthreads();
                const int rank = tid < n ? S.crank[tid] : n;
                if (tid == 0) {
                    const double tau = S.tau;
                    S.ok = S.all_in || tau * rho > 1.0;          // tau > 1/rho: nothing outside rho can reach the block
                    S.rho = S.ok ? fmax(1.25 / tau, 1.0) : hi > 0.0 ? 0.5 * (rho + hi) : fmax(rho * 1.6, 1.0001 / tau);
                }
                __syncthreads();
                if (!S.ok) {
                    lo = rho;
                    if (++tries > 64 || (hi > 0.0 && !(hi - lo > 1e-9 * hi))) { if (tid == 0) *err = 3; return; }
                    if (tid == 0) err[1] += 1;
                    continue;
                }
                if (tid == 0) { err[2] += n; err[3] += nraw; }
                if (rank < take) {
                    const int j = S.cidx[tid];
                    asg[j] = 1;
                    order[filled + 1 + rank] = j;
                    atomicSub(&gc[j >> 5], 1);
                }
                break;
            }
        }
        if (tid == 0) order[filled] = k;
        filled += 1 + take;
        pos += 1;
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// Block inversion: one thread block per diagonal block.  fill -> Cholesky (right-looking, in place, lower)
// -> W = L^-1 (one column per thread) -> inv = W^T W.  n x n row-major; the two n x n work arrays live in shared memory
// when they fit (use_smem: 2 n^2 doubles of dynamic shared memory, block sizes up to ~100), otherwise in global memory
// (L2 resident).  Same arithmetic either way.
// ---------------------------------------------------------------------------------------------
__global__ void rbj_invert_kernel(const double4 *__restrict__ pt, const double *__restrict__ diag, int M, int block,
                                  const int32_t *__restrict__ order, double *__restrict__ inv, double *__restrict__ work,
                                  int *__restrict__ err, const double *__restrict__ boys0, int use_smem) {
    extern __shared__ double s_blk[];
    const long long start = (long long)blockIdx.x * block;
    const int n = (int)min((long long)block, (long long)M - start);
    double *ga = inv + (size_t)blockIdx.x * block * block;
    double *a = use_smem ? s_blk : ga;
    double *w = use_smem ? s_blk + (size_t)block * block : work + (size_t)blockIdx.x * block * block;
    const int32_t *idx = order + start;
    {   // a failed selection (asynchronous build: the host has not looked yet) leaves `order` undefined
        const int e0 = *((volatile int *)err);
        if (e0 == 1 || e0 == 2 || e0 == 3) return;
    }
    for (int e = threadIdx.x; e < n * n; e += blockDim.x) {
        const int r = e / n, c = e - r * n;
        a[e] = a_entry(pt, diag, idx[r], idx[c], boys0);
        w[e] = 0.0;
    }
    __syncthreads();
    for (int j = 0; j < n; ++j) {
        const double d = a[(size_t)j * n + j];
        if (!(d > 0.0)) {
            if (threadIdx.x == 0) *err = 4;   // not positive definite (1, 2: selection failed; 3: selection capacity, host falls back)
            return;
        }
        const double s = sqrt(d), is = 1.0 / s;
        __syncthreads();
        for (int i = j + threadIdx.x; i < n; i += blockDim.x) a[(size_t)i * n + j] = (i == j) ? s : a[(size_t)i * n + j] * is;
        __syncthreads();
        // trailing update a[i][c] -= L[i][j] L[c][j], j < c <= i: 16 x 16 threads stride over (i, c), no integer division
        for (int i = j + 1 + (int)(threadIdx.x >> 4); i < n; i += (int)(blockDim.x >> 4)) {
            const double lij = a[(size_t)i * n + j];
            for (int c = j + 1 + (int)(threadIdx.x & 15); c <= i; c += 16) a[(size_t)i * n + c] -= lij * a[(size_t)c * n + j];
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
    if (use_smem) {
        __syncthreads();
        for (int e = threadIdx.x; e < n * n; e += blockDim.x) ga[e] = a[e];
    }
}

// ---------------------------------------------------------------------------------------------
// PCG (textbook recurrences).  One iteration is five kernels on device-resident scalars:
//   A q main + near (pcm_kernels.cu)  ->  cg_matvec_reduce (Ap = sum of the partial-sum slots, p.Ap)
//   ->  cg_update_* (x += alpha p, r -= alpha Ap, z = C r, r.r, r.z, beta, convergence test)  ->  cg_direction.
// Dot products are two-stage and fixed-order: per-CTA partials, then the last CTA to finish (atomic ticket) sums
// them in index order.  The convergence test runs on the device: when ||r|| <= tol (or max_iter is reached) it raises
// ctl[STOP] and every later kernel of the solve returns at once, so the host can queue iterations in batches without
// changing what is computed.
// scal: 0 rz, 1 pAp, 2 rr, 4 |b - Ax|^2, 5 beta.   ctl: 0 stop, 1 iterations, 2 ticket
// ---------------------------------------------------------------------------------------------
constexpr int DOT_BLOCKS = 296;
constexpr int DOT_THREADS = 256;
enum { CTL_STOP = 0, CTL_ITERS = 1, CTL_TICKET = 2 };

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

// true for the last CTA of the grid to get here; its threads then see every other CTA's partials
__device__ __forceinline__ bool last_block(int *ctl) {
    __shared__ int s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(&ctl[CTL_TICKET], 1) == (int)gridDim.x - 1);
    __syncthreads();
    if (s_last) __threadfence();
    return s_last != 0;
}
// sum of partial[0..n) in a fixed order (valid in thread 0); blockDim.x == DOT_THREADS
__device__ __forceinline__ double ordered_sum(const double *partial, int n) {
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += DOT_THREADS) s += __ldcg(partial + i);
    return block_sum(s);
}

// Ap = sum of the A q partial sums (sorted order), pAp = p.Ap.  One CTA per 32 rows (amat_row_sum_block); the per-CTA
// dot products go to partial[blockIdx.x], the last CTA adds them in index order.
__global__ void __launch_bounds__(DOT_THREADS) cg_matvec_reduce_kernel(int M, AmatParts parts,
                                                                       const double *__restrict__ p, double *__restrict__ Ap,
                                                                       double *__restrict__ scal, double *__restrict__ partial,
                                                                       int *__restrict__ ctl) {
    __shared__ double s_tmp[AMAT_RED_PARTS * 32];
    if (*((volatile int *)&ctl[CTL_STOP])) return;
    const double t = amat_row_sum_block(parts, M, blockIdx.x * 32, s_tmp);
    const int k = blockIdx.x * 32 + threadIdx.x;
    if (threadIdx.x < 32) {
        double dot = 0.0;
        if (k < M) { Ap[k] = t; dot = p[k] * t; }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dot += __shfl_down_sync(0xffffffffu, dot, o);
        if (threadIdx.x == 0) partial[blockIdx.x] = dot;
    }
    if (last_block(ctl)) {
        const double pAp = ordered_sum(partial, (int)gridDim.x);
        if (threadIdx.x == 0) { scal[1] = pAp; ctl[CTL_TICKET] = 0; }
    }
}

// what the last CTA of an update kernel does with the two fixed-order sums
__device__ __forceinline__ void cg_finish(double rr, double rz_new, double *scal, int *ctl, double tol, int max_iter, int init) {
    if (threadIdx.x != 0) return;
    if (!init) {
        scal[5] = rz_new / scal[0];
        ctl[CTL_ITERS] += 1;
    }
    scal[0] = rz_new;
    scal[2] = rr;
    if (!(sqrt(rr) > tol) || ctl[CTL_ITERS] >= max_iter) ctl[CTL_STOP] = 1;
    ctl[CTL_TICKET] = 0;
}

// RBJ: one CTA per diagonal block b (a partition of the points): x += alpha p, r -= alpha Ap on the block's points,
// z = M_b^-1 r (C = scatter o blockdiag(M_b^-1) o gather), partial r.r and r.z.  init: r is given, no update.
__global__ void __launch_bounds__(DOT_THREADS) cg_update_rbj_kernel(int M, int block, const int32_t *__restrict__ order,
                                                                    const double *__restrict__ inv, const double *__restrict__ p,
                                                                    const double *__restrict__ Ap, double *__restrict__ x,
                                                                    double *__restrict__ r, double *__restrict__ z,
                                                                    double *__restrict__ scal, double *__restrict__ partial,
                                                                    int *__restrict__ ctl, double tol, int max_iter, int init) {
    extern __shared__ double s_r[];
    if (*((volatile int *)&ctl[CTL_STOP])) return;
    const long long start = (long long)blockIdx.x * block;
    const int n = (int)min((long long)block, (long long)M - start);
    const double *a = inv + (size_t)blockIdx.x * block * block;
    const int32_t *idx = order + start;
    const double alpha = init ? 0.0 : scal[0] / scal[1];
    double rr = 0.0, rz = 0.0;
    for (int j = threadIdx.x; j < n; j += DOT_THREADS) {
        const int i = idx[j];
        double ri = r[i];
        if (!init) {
            x[i] = fma(alpha, p[i], x[i]);
            ri = fma(-alpha, Ap[i], ri);
            r[i] = ri;
        }
        s_r[j] = ri;
        rr = fma(ri, ri, rr);
    }
    __syncthreads();
    // z = M_b^-1 r: np threads per row, each over every np-th column (inv is symmetric: the column read is coalesced
    // across the rows), the np partial sums added in order through shared memory
    const int np = n >= DOT_THREADS ? 1 : DOT_THREADS / n;
    const int rpp = DOT_THREADS / np;            // rows per pass (>= n when n < DOT_THREADS)
    const int part = threadIdx.x / rpp, il = threadIdx.x - part * rpp;
    double *s_part = s_r + block;                // [np][rpp] <= DOT_THREADS doubles
    for (int i0 = 0; i0 < n; i0 += rpp) {
        const int i = i0 + il;
        double s = 0.0;
        if (i < n && part < np) {
            int j = part;
            for (; j + 7 * np < n; j += 8 * np) {
                double v[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) v[u] = __ldg(a + (size_t)(j + u * np) * n + i);
#pragma unroll
                for (int u = 0; u < 8; ++u) s = fma(v[u], s_r[j + u * np], s);
            }
            for (; j < n; j += np) s = fma(__ldg(a + (size_t)j * n + i), s_r[j], s);
        }
        s_part[threadIdx.x] = s;
        __syncthreads();
        if (part == 0 && i < n) {
            double t = 0.0;
            for (int q = 0; q < np; ++q) t += s_part[q * rpp + il];
            z[idx[i]] = t;
            rz = fma(s_r[i], t, rz);
        }
        __syncthreads();
    }
    rr = block_sum(rr);
    rz = block_sum(rz);
    if (threadIdx.x == 0) { partial[blockIdx.x] = rr; partial[gridDim.x + blockIdx.x] = rz; }
    if (last_block(ctl)) {
        const double srr = ordered_sum(partial, gridDim.x);
        const double srz = ordered_sum(partial + gridDim.x, gridDim.x);
        cg_finish(srr, srz, scal, ctl, tol, max_iter, init);
    }
}

// ---------------------------------------------------------------------------------------------
// One cooperative kernel for everything of a PCG iteration that follows the A q sweep (RBJ preconditioner):
//   phase 1  Ap = row sums of the sweep's partial sums, per-task p.Ap        -- grid barrier --
//   phase 2  alpha; x += alpha p, r -= alpha Ap, z = M_b^-1 r per RBJ block, per-block r.r and r.z   -- grid barrier --
//   phase 3  beta, convergence test (CTA 0 records them), p = z + beta p
// Every CTA adds the per-task partial sums itself, in index order, so all of them hold the same alpha and beta without a
// broadcast, and the numbers are those of the three separate kernels (cg_matvec_reduce, cg_update_rbj, cg_direction)
// bit for bit.  At M ~ 10^4 those three launches and their tails cost as much as half an A q sweep; here they are two
// barriers.  The barrier is sense-reversing and self-resetting (count, generation in ctl[3], ctl[4]); the launch is
// cooperative, so all CTAs are resident; the spin is bounded and raises ctl[5] instead of hanging.
// ---------------------------------------------------------------------------------------------
enum { CTL_BAR_COUNT = 3, CTL_BAR_GEN = 4, CTL_BAR_ERR = 5 };

__device__ __forceinline__ void grid_sync(int *ctl, unsigned G) {
    __syncthreads();
    if (threadIdx.x == 0) {
        volatile int *gen = ctl + CTL_BAR_GEN;
        const int g = *gen;
        __threadfence();
        if (atomicAdd(ctl + CTL_BAR_COUNT, 1) == (int)G - 1) {
            ctl[CTL_BAR_COUNT] = 0;
            __threadfence();
            atomicAdd(ctl + CTL_BAR_GEN, 1);
        } else {
            long long spins = 0;
            while (*gen == g) {
                if (++spins > (1ll << 27)) { ctl[CTL_BAR_ERR] = 1; break; }
            }
        }
        __threadfence();
    }
    __syncthreads();
}

struct CgFused {
    int M, block, nblocks, max_iter;
    AmatParts parts;
    const int32_t *order;
    const double *inv;
    double *p, *Ap, *x, *r, *z, *scal, *part1, *part2;
    int *ctl;
    double tol;
};

__global__ void __launch_bounds__(DOT_THREADS) cg_fused_rbj_kernel(CgFused a) {
    extern __shared__ double s_dyn[];       // [max(block, 0) + DOT_THREADS]
    __shared__ double s_bc[3];
    int *ctl = a.ctl;
    if (*((volatile int *)&ctl[CTL_STOP])) return;
    const unsigned G = gridDim.x;
    const int M = a.M, tid = threadIdx.x;
    const int iters0 = *((volatile int *)&ctl[CTL_ITERS]);
    const double rz_old = a.scal[0];
    // ---- phase 1
    const int ntask1 = (M + 31) / 32;
    for (int task = blockIdx.x; task < ntask1; task += G) {
        const double t = amat_row_sum_block(a.parts, M, task * 32, s_dyn);
        const int k = task * 32 + tid;
        if (tid < 32) {
            double dot = 0.0;
            if (k < M) { a.Ap[k] = t; dot = a.p[k] * t; }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) dot += __shfl_down_sync(0xffffffffu, dot, o);
            if (tid == 0) a.part1[task] = dot;
        }
        __syncthreads();
    }
    grid_sync(ctl, G);
    {
        const double pAp = ordered_sum(a.part1, ntask1);
        if (tid == 0) s_bc[0] = pAp;
        __syncthreads();
    }
    const double pAp = s_bc[0];
    const double alpha = rz_old / pAp;
    // ---- phase 2: the body of cg_update_rbj_kernel, one RBJ block per pass
    const int block = a.block;
    double *s_r = s_dyn, *s_part = s_dyn + block;
    for (int b = blockIdx.x; b < a.nblocks; b += G) {
        const long long start = (long long)b * block;
        const int n = (int)min((long long)block, (long long)M - start);
        const double *am = a.inv + (size_t)b * block * block;
        const int32_t *idx = a.order + start;
        double rr = 0.0, rz = 0.0;
        for (int j = tid; j < n; j += DOT_THREADS) {
            const int i = idx[j];
            a.x[i] = fma(alpha, a.p[i], a.x[i]);
            const double ri = fma(-alpha, a.Ap[i], a.r[i]);
            a.r[i] = ri;
            s_r[j] = ri;
            rr = fma(ri, ri, rr);
        }
        __syncthreads();
        const int np = n >= DOT_THREADS ? 1 : DOT_THREADS / n;
        const int rpp = DOT_THREADS / np;
        const int part = tid / rpp, il = tid - part * rpp;
        for (int i0 = 0; i0 < n; i0 += rpp) {
            const int i = i0 + il;
            double sacc = 0.0;
            if (i < n && part < np) {
                // eight loads in flight (the inverse block comes from L2), same summation order
                int j = part;
                for (; j + 7 * np < n; j += 8 * np) {
                    double v[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) v[u] = __ldg(am + (size_t)(j + u * np) * n + i);
#pragma unroll
                    for (int u = 0; u < 8; ++u) sacc = fma(v[u], s_r[j + u * np], sacc);
                }
                for (; j < n; j += np) sacc = fma(__ldg(am + (size_t)j * n + i), s_r[j], sacc);
            }
            s_part[tid] = sacc;
            __syncthreads();
            if (part == 0 && i < n) {
                double t = 0.0;
                for (int q = 0; q < np; ++q) t += s_part[q * rpp + il];
                a.z[idx[i]] = t;
                rz = fma(s_r[i], t, rz);
            }
            __syncthreads();
        }
        rr = block_sum(rr);
        rz = block_sum(rz);
        if (tid == 0) { a.part2[b] = rr; a.part2[a.nblocks + b] = rz; }
        __syncthreads();
    }
    grid_sync(ctl, G);
    {
        const double srr = ordered_sum(a.part2, a.nblocks);
        const double srz = ordered_sum(a.part2 + a.nblocks, a.nblocks);
        if (tid == 0) { s_bc[1] = srr; s_bc[2] = srz; }
        __syncthreads();
    }
    const double srr = s_bc[1], srz = s_bc[2];
    const double beta = srz / rz_old;
    const bool stop = !(sqrt(srr) > a.tol) || iters0 + 1 >= a.max_iter;
    if (blockIdx.x == 0 && tid == 0) {
        a.scal[1] = pAp;
        a.scal[5] = beta;
        a.scal[0] = srz;
        a.scal[2] = srr;
        ctl[CTL_ITERS] = iters0 + 1;
        if (stop) ctl[CTL_STOP] = 1;
    }
    // ---- phase 3 (a converged solve keeps p, as cg_direction_kernel does)
    if (!stop)
        for (int i = blockIdx.x * DOT_THREADS + tid; i < M; i += (int)G * DOT_THREADS) a.p[i] = fma(beta, a.p[i], a.z[i]);
}

// Jacobi (C = diag(A)^-1) or no preconditioner (diag == nullptr)
__global__ void __launch_bounds__(DOT_THREADS) cg_update_diag_kernel(int M, const double *__restrict__ diag,
                                                                     const double *__restrict__ p, const double *__restrict__ Ap,
                                                                     double *__restrict__ x, double *__restrict__ r,
                                                                     double *__restrict__ z, double *__restrict__ scal,
                                                                     double *__restrict__ partial, int *__restrict__ ctl,
                                                                     double tol, int max_iter, int init) {
    if (*((volatile int *)&ctl[CTL_STOP])) return;
    const double alpha = init ? 0.0 : scal[0] / scal[1];
    double rr = 0.0, rz = 0.0;
    for (int i = blockIdx.x * DOT_THREADS + threadIdx.x; i < M; i += DOT_BLOCKS * DOT_THREADS) {
        double ri = r[i];
        if (!init) {
            x[i] = fma(alpha, p[i], x[i]);
            ri = fma(-alpha, Ap[i], ri);
            r[i] = ri;
        }
        const double zi = diag ? ri / diag[i] : ri;
        z[i] = zi;
        rr = fma(ri, ri, rr);
        rz = fma(ri, zi, rz);
    }
    rr = block_sum(rr);
    rz = block_sum(rz);
    if (threadIdx.x == 0) { partial[blockIdx.x] = rr; partial[DOT_BLOCKS + blockIdx.x] = rz; }
    if (last_block(ctl)) {
        const double srr = ordered_sum(partial, DOT_BLOCKS);
        const double srz = ordered_sum(partial + DOT_BLOCKS, DOT_BLOCKS);
        cg_finish(srr, srz, scal, ctl, tol, max_iter, init);
    }
}

// p = z + beta p  (init: p = z)
__global__ void cg_direction_kernel(int M, const double *__restrict__ scal, const double *__restrict__ z, double *__restrict__ p,
                                    const int *__restrict__ ctl, int init) {
    if (!init && *((volatile const int *)&ctl[CTL_STOP])) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    p[i] = init ? z[i] : fma(scal[5], p[i], z[i]);
}
__global__ void residual_kernel(int M, const double *__restrict__ b, const double *__restrict__ Ax, double *__restrict__ r) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) r[i] = b[i] - Ax[i];
}
// scal[o] = a.a  (single CTA per DOT_BLOCKS slice, then last-CTA sum)
__global__ void __launch_bounds__(DOT_THREADS) norm2_kernel(int M, const double *__restrict__ a, double *__restrict__ scal, int o,
                                                            double *__restrict__ partial, int *__restrict__ ctl) {
    double s = 0.0;
    for (int i = blockIdx.x * DOT_THREADS + threadIdx.x; i < M; i += DOT_BLOCKS * DOT_THREADS) s = fma(a[i], a[i], s);
    s = block_sum(s);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
    if (last_block(ctl)) {
        const double t = ordered_sum(partial, DOT_BLOCKS);
        if (threadIdx.x == 0) { scal[o] = t; ctl[CTL_TICKET] = 0; }
    }
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
// The rest of a C-PCM step (Eq. 1, 4, 13): u = B z, b = -f (u - v), Delta G_els.
// ---------------------------------------------------------------------------------------------
// u_k = sum_J z_J erf(zeta_k r_kJ)/r_kJ (Eq. 4): thread = point (sorted order), nuclei staged in shared memory and
// summed in the caller's order; far field (zeta_k^2 r^2 >= 38: erf = 1) is z/r, otherwise (2 zeta/sqrt pi) F_0(zeta^2 r^2).
__global__ void __launch_bounds__(128) nuclear_potential_kernel(const double4 *__restrict__ pt, int M, const double4 *__restrict__ atoms,
                                                                int natom, const int32_t *__restrict__ s2c,
                                                                const double *__restrict__ boys0, double *__restrict__ u) {
    __shared__ double4 s_at[256];
    const int k = blockIdx.x * 128 + threadIdx.x;
    const double4 a = pt[min(k, M - 1)];
    const double thr = TFAR_AMAT * a.w;   // zeta_k^2 r^2 >= 38  <=>  r^2 >= 38/zeta_k^2
    const double zk = rsqrt_fast(a.w);
    double sum = 0.0;
    for (int base = 0; base < natom; base += 256) {
        const int cnt = min(256, natom - base);
        __syncthreads();
        for (int t = threadIdx.x; t < cnt; t += 128) s_at[t] = atoms[base + t];
        __syncthreads();
        for (int t = 0; t < cnt; ++t) {
            const double4 b = s_at[t];
            const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            double ev;
            if (r2 >= thr) {
                ev = rsqrt_fast(r2);
            } else {
                const double T = r2 * zk * zk;
                const int i = __double2int_rn(T * 16.0);
                const double d = T - (double)i * 0.0625;
                const double *row = boys0 + (size_t)i * BOYS_STRIDE;
                double f = __ldg(row + BOYS_TERMS - 1);
#pragma unroll
                for (int n = BOYS_TERMS - 2; n >= 0; --n) f = fma(f, d, __ldg(row + n));
                ev = 1.1283791670955125739 * zk * f;  // 2/sqrt(pi)
            }
            sum = fma(b.w, ev, sum);
        }
    }
    if (k < M) u[s2c[k]] = sum;
}

__global__ void rhs_kernel(int M, const double *__restrict__ u, const double *__restrict__ v, double f, double *__restrict__ b) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) b[i] = -f * (u[i] - v[i]);
}

// scal[12..14] = u.q, -v.q, q.Aq  (per-CTA partials, then the last CTA sums them in index order)
constexpr int ENERGY_BLOCKS = 128;
__global__ void __launch_bounds__(DOT_THREADS) energy_kernel(int M, const double *__restrict__ u, const double *__restrict__ v,
                                                             const double *__restrict__ q, const double *__restrict__ Aq,
                                                             double *__restrict__ scal, double *__restrict__ partial,
                                                             int *__restrict__ ctl) {
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int i = blockIdx.x * DOT_THREADS + threadIdx.x; i < M; i += ENERGY_BLOCKS * DOT_THREADS) {
        const double qi = q[i];
        s0 = fma(u[i], qi, s0);
        s1 = fma(-v[i], qi, s1);
        s2 = fma(qi, Aq[i], s2);
    }
    s0 = block_sum(s0);
    s1 = block_sum(s1);
    s2 = block_sum(s2);
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = s0;
        partial[ENERGY_BLOCKS + blockIdx.x] = s1;
        partial[2 * ENERGY_BLOCKS + blockIdx.x] = s2;
    }
    if (last_block(ctl)) {
        const double t0 = ordered_sum(partial, ENERGY_BLOCKS);
        const double t1 = ordered_sum(partial + ENERGY_BLOCKS, ENERGY_BLOCKS);
        const double t2 = ordered_sum(partial + 2 * ENERGY_BLOCKS, ENERGY_BLOCKS);
        if (threadIdx.x == 0) { scal[12] = t0; scal[13] = t1; scal[14] = t2; ctl[CTL_TICKET] = 0; }
    }
}

int launch_nuclear_potential(pcm_ctx *ctx, double *u, cudaStream_t s) {
    const int M = (int)ctx->M;
    if (M == 0) return PCM_OK;
    nuclear_potential_kernel<<<(unsigned)cdiv(M, 128), 128, 0, s>>>(ctx->pt, M, ctx->atoms, (int)ctx->natom, ctx->s2c, ctx->boys, u);
    ctx->launch_total += 1;
    PCM_CUDA(ctx, cudaGetLastError());
    return PCM_OK;
}

int launch_rhs(pcm_ctx *ctx, const double *u, const double *v, double f, double *b, cudaStream_t s) {
    const int M = (int)ctx->M;
    if (M == 0) return PCM_OK;
    rhs_kernel<<<(unsigned)cdiv(M, 256), 256, 0, s>>>(M, u, v, f, b);
    ctx->launch_total += 1;
    PCM_CUDA(ctx, cudaGetLastError());
    return PCM_OK;
}

int energy_terms(pcm_ctx *ctx, const double *u, const double *v, const double *q, double f, double *terms, cudaStream_t s) {
    const int M = (int)ctx->M;
    terms[0] = terms[1] = terms[2] = terms[3] = 0.0;
    if (M == 0) return PCM_OK;
    double *Aq = ctx->cg_vec;   // scratch (caller order)
    double *scal = ctx->cg_scal;
    int *ctl = reinterpret_cast<int *>(scal + 8);
    const int saved_timing = ctx->timing;
    ctx->timing = 0;
    int rc = launch_amatvec(ctx, q, Aq, s);
    ctx->timing = saved_timing;
    if (rc) return rc;
    energy_kernel<<<ENERGY_BLOCKS, DOT_THREADS, 0, s>>>(M, u, v, q, Aq, scal, scal + 16, ctl);
    ctx->launch_total += 1;
    PCM_CUDA(ctx, cudaGetLastError());
    double *h = ctx->cg_scal_host;
    PCM_CUDA(ctx, cudaMemcpyAsync(h, scal, 16 * sizeof(double), cudaMemcpyDeviceToHost, s));
    PCM_CUDA(ctx, cudaStreamSynchronize(s));
    terms[0] = h[12];
    terms[1] = h[13];
    terms[2] = h[14] / (2.0 * f);
    terms[3] = terms[0] + terms[1] + terms[2];
    return PCM_OK;
}

// ---------------------------------------------------------------------------------------------
// host drivers
// ---------------------------------------------------------------------------------------------
// Completes an asynchronous build: orders `s` after it, reads its status and, in the (capacity) case the neighbourhood
// selection gave up, repeats the build synchronously with the global row scan.
int rbj_finish(pcm_ctx *ctx, cudaStream_t s) {
    if (!ctx->rbj_pending) return PCM_OK;
    ctx->rbj_pending = false;
    PCM_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_rbj, 0));
    PCM_CUDA(ctx, cudaEventSynchronize(ctx->ev_rbj));
    const int h_err = *reinterpret_cast<const int *>(ctx->cg_scal_host + 32);
    if (h_err == 3) {
        std::vector<int64_t> perm = ctx->rbj_last_perm;
        return rbj_build(ctx, (int)ctx->rbj_block, ctx->rbj_last_seed, perm.empty() ? nullptr : perm.data(), s, false, true);
    }
    if (h_err) {
        ctx->rbj_block = 0; ctx->rbj_nblocks = 0; ctx->info.rbj_block = 0; ctx->info.rbj_nblocks = 0;
        if (h_err == 1 || h_err == 2) return set_error(ctx, PCM_ERR_STATE, "pcm_rbj_build: block selection did not cover all points");
        return set_error(ctx, PCM_ERR_NUMERIC, "pcm_rbj_build: a diagonal block of A is not positive definite");
    }
    return PCM_OK;
}

// async: everything is queued on s and the call returns; rbj_finish (pcm_cg_solve, pcm_rbj_get, the next build) completes it.
int rbj_build(pcm_ctx *ctx, int block, uint64_t seed, const int64_t *pivot_order_host, cudaStream_t s, bool async, bool force_global) {
    const int64_t M = ctx->M;
    if (block < 1) return set_error(ctx, PCM_ERR_ARG, "pcm_rbj_build: block < 1");
    {   // a build still in flight owns the arena
        int rcf = rbj_finish(ctx, s);
        if (rcf) return rcf;
    }
    if (M == 0) { ctx->rbj_block = block; ctx->rbj_nblocks = 0; return PCM_OK; }
    const bool verbose = getenv("PCM_VERBOSE") != nullptr;
    auto now = []() { return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count(); };
    const double t0 = now();
    if ((int64_t)block > M) block = (int)M;
    // the CG update kernels keep a block's residual in shared memory: (block + 256) doubles must fit
    if (((size_t)block + 256) * 8 > 200 * 1024) return set_error(ctx, PCM_ERR_ARG, "pcm_rbj_build: block size above 25 000 is not supported");
    std::vector<int32_t> &perm = ctx->rbj_perm_sorted;  // pivot order in the library's sorted point numbering
    if (pivot_order_host) {
        std::vector<char> seen((size_t)M, 0);
        for (int64_t i = 0; i < M; ++i) {
            const int64_t v = pivot_order_host[i];
            if (v < 0 || v >= M || seen[v]) return set_error(ctx, PCM_ERR_ARG, "pcm_rbj_build: pivot order is not a permutation");
            seen[v] = 1;
        }
        if (pivot_order_host != ctx->rbj_last_perm.data()) ctx->rbj_last_perm.assign(pivot_order_host, pivot_order_host + M);
        perm.resize((size_t)M);
        for (int64_t i = 0; i < M; ++i) perm[i] = ctx->c2s_host[(size_t)pivot_order_host[i]];
        ctx->rbj_perm_seeded = false;
    } else if (!(ctx->rbj_perm_seeded && ctx->rbj_last_seed == seed && (int64_t)perm.size() == M)) {
        // the seeded order is a pure function of (seed, M): kept for the next build with the same seed
        std::vector<int64_t> perm64((size_t)M);
        pivot_order(seed, M, perm64.data());
        perm.resize((size_t)M);
        for (int64_t i = 0; i < M; ++i) perm[i] = ctx->c2s_host[(size_t)perm64[i]];
        ctx->rbj_last_perm.clear();
        ctx->rbj_perm_seeded = true;
    }
    ctx->rbj_last_seed = seed;

    const int64_t nb = cdiv(M, block);
    // RBJ storage and build scratch live in one grow-only device arena (no allocation when a build is repeated)
    auto al = [](size_t b) { return (b + 255) / 256 * 256; };
    const size_t blk2 = (size_t)nb * block * block * 8;
    const size_t need = al((size_t)M * 4) + al(blk2) + al((size_t)2 * nb * 8) + al(blk2) + al((size_t)M * 4) + al((size_t)M) +
                        al((size_t)M * 8) + al((size_t)2 * M * 8) + al((size_t)2 * M * 4) + al(3 * RBJ_BINS * 4) + al(64);
    int rc;
    ctx->rbj_block = 0; ctx->rbj_nblocks = 0;
    if (need > ctx->rbj_arena_bytes) {
        if (ctx->rbj_arena) {
            auto it = std::find(ctx->allocs.begin(), ctx->allocs.end(), (void *)ctx->rbj_arena);
            if (it != ctx->allocs.end()) ctx->allocs.erase(it);
            cudaFree(ctx->rbj_arena);
            ctx->device_bytes -= (int64_t)ctx->rbj_arena_bytes;
            ctx->rbj_arena = nullptr; ctx->rbj_arena_bytes = 0;
        }
        if ((rc = dev_alloc(ctx, (void **)&ctx->rbj_arena, need))) return rc;
        ctx->rbj_arena_bytes = need;
    }
    char *cur = ctx->rbj_arena;
    auto take = [&](size_t b) { char *p = cur; cur += al(b); return (void *)p; };
    ctx->rbj_order = (int32_t *)take((size_t)M * 4);
    ctx->rbj_inv = (double *)take(blk2);
    ctx->rbj_partial = (double *)take((size_t)2 * nb * 8);
    double *d_work = (double *)take(blk2);
    int32_t *d_perm = (int32_t *)take((size_t)M * 4);
    RbjWork w{};
    w.assigned = (unsigned char *)take((size_t)M);
    w.keys = (double *)take((size_t)M * 8);
    w.cand_key = (double *)take((size_t)2 * M * 8);
    w.cand_idx = (int *)take((size_t)2 * M * 4);
    w.hist = (int *)take(3 * RBJ_BINS * 4);
    char *small = (char *)take(64);
    w.cand_count = (int *)small;
    w.err = (int *)(small + 16);
    w.bar = (unsigned long long *)(small + 32);
    auto cleanup = [&]() {};
#define RBJ_TRY(call)                                                                                     \
    do {                                                                                                  \
        cudaError_t e__ = (call);                                                                         \
        if (e__ != cudaSuccess) { cleanup(); return set_error(ctx, PCM_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__)); } \
    } while (0)
    RBJ_TRY(cudaMemcpyAsync(d_perm, perm.data(), (size_t)M * 4, cudaMemcpyHostToDevice, s));
    RBJ_TRY(cudaMemsetAsync(w.assigned, 0, (size_t)M, s));
    RBJ_TRY(cudaMemsetAsync(w.hist, 0, 3 * RBJ_BINS * 4, s));
    RBJ_TRY(cudaMemsetAsync(small, 0, 64, s));
    int *d_err = w.err;

    double t1 = 0, t2 = 0;
    if (verbose) { cudaStreamSynchronize(s); t1 = now(); }
    // block sizes up to 256: the single-CTA neighbourhood selection; it reports err = 3 (capacity) to fall back
    bool local_done = false, fell_back = force_global;
    // (measured: 0.8 vs 1.6 ms at M = 8 930, 6.1 vs 9.6 ms at 50k, 86 vs 78 ms at 200k, where scanning 6 250 group boxes per
    // block with one CTA costs more than the two grid barriers of the global scan)
    if (block <= 256 && M <= RBJ_LOCAL_MAX && !force_global && !ctx->opt.rbj_global_scan) {
        const int ng = (int)cdiv(M, 32);
        int *d_gcount = (int *)w.cand_idx, *d_glist = d_gcount + ng;   // scratch of the global path, 2 M ints
        const size_t base_smem = (sizeof(RblShared) + 15) / 16 * 16;
        const size_t cache_smem = base_smem + (size_t)ng * 6 * 8 + (size_t)ng * 4 + (size_t)M + 16;
        const int cache = cache_smem <= 200 * 1024;
        const size_t smem = cache ? cache_smem : base_smem;
        RBJ_TRY(cudaFuncSetAttribute(rbj_select_local_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        rbj_select_local_kernel<<<1, RBL_THREADS, smem, s>>>(ctx->pt, (int)M, block, d_perm, ctx->s2c, ctx->rbj_order, w.assigned,
                                                              ctx->pt_boxes, ng, d_gcount, d_glist, d_err, ctx->boys, cache);
        RBJ_TRY(cudaGetLastError());
        ctx->launch_total += 1;
        int h_e = 0;
        if (async) {   // the status is read by rbj_finish; the inversion below is a no-op on a failed selection
            local_done = true;
        } else {
        RBJ_TRY(cudaMemcpyAsync(&h_e, d_err, 4, cudaMemcpyDeviceToHost, s));
        RBJ_TRY(cudaStreamSynchronize(s));
        if (verbose) {
            int h4[4];
            cudaMemcpy(h4, d_err, 16, cudaMemcpyDeviceToHost);
            fprintf(stderr, "[pcm] rbj local: retries %d, ranked candidates %d, raw candidates %d over %lld blocks\n", h4[1], h4[2], h4[3], (long long)nb);
        }
        if (h_e == 0) local_done = true;
        else if (h_e == 3) {   // start over with the global row scan
            fell_back = true;
            RBJ_TRY(cudaMemsetAsync(w.assigned, 0, (size_t)M, s));
            RBJ_TRY(cudaMemsetAsync(small, 0, 64, s));
        }
        }
    }
    ctx->info.rbj_selection = local_done ? 1 : fell_back ? 3 : 2;
    // one cooperative launch: all CTAs must be co-resident for the grid barrier
    if (!local_done) {
        int per_sm = 0;
        RBJ_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, rbj_select_kernel, RBJ_THREADS, 0));
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(cdiv(M, RBJ_THREADS), (int64_t)std::max(per_sm, 1) * ctx->sm_count));
        int Mi = (int)M;
        const double4 *pt = ctx->pt;
        const double *diag = ctx->pt_diag, *boys = ctx->boys;
        const int32_t *permc = d_perm, *s2c = ctx->s2c;
        int32_t *order = ctx->rbj_order;
        void *args[] = {&pt, &diag, &Mi, &block, &permc, &s2c, &order, &w, &boys};
        RBJ_TRY(cudaLaunchCooperativeKernel((const void *)rbj_select_kernel, dim3(grid), dim3(RBJ_THREADS), args, 0, s));
        ctx->launch_total += 1;
    }
    ctx->launch_total += 1;
    RBJ_TRY(cudaGetLastError());
    if (verbose) { cudaStreamSynchronize(s); t2 = now(); }
    {
        const size_t inv_smem = (size_t)2 * block * block * 8;
        const int use_smem = inv_smem <= 160 * 1024;
        if (use_smem) RBJ_TRY(cudaFuncSetAttribute(rbj_invert_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)inv_smem));
        rbj_invert_kernel<<<(unsigned)nb, 256, use_smem ? inv_smem : 0, s>>>(ctx->pt, ctx->pt_diag, (int)M, block, ctx->rbj_order, ctx->rbj_inv,
                                                                            d_work, d_err, ctx->boys, use_smem);
    }
    RBJ_TRY(cudaGetLastError());
    if (async) {
        RBJ_TRY(cudaMemcpyAsync(ctx->cg_scal_host + 32, d_err, 16, cudaMemcpyDeviceToHost, s));
        RBJ_TRY(cudaEventRecord(ctx->ev_rbj, s));
        ctx->rbj_pending = true;
        ctx->rbj_block = block; ctx->rbj_nblocks = nb;
        ctx->info.rbj_block = block; ctx->info.rbj_nblocks = nb;
        return PCM_OK;
    }
    int h_err = 0;
    RBJ_TRY(cudaMemcpyAsync(&h_err, d_err, 4, cudaMemcpyDeviceToHost, s));
    RBJ_TRY(cudaStreamSynchronize(s));
    if (verbose) fprintf(stderr, "[pcm] rbj_build M=%lld l=%d: host prep %.3f ms, select %.3f ms, invert %.3f ms\n", (long long)M, block,
                         t1 - t0, t2 - t1, now() - t2);
    cleanup();
#undef RBJ_TRY
    if (h_err == 1 || h_err == 2) return set_error(ctx, PCM_ERR_STATE, "pcm_rbj_build: block selection did not cover all points");
    if (h_err) return set_error(ctx, PCM_ERR_NUMERIC, "pcm_rbj_build: a diagonal block of A is not positive definite");
    ctx->rbj_block = block;
    ctx->rbj_nblocks = nb;
    ctx->info.rbj_block = block;
    ctx->info.rbj_nblocks = nb;
    return PCM_OK;
}

int cg_solve(pcm_ctx *ctx, const double *b_caller, double *x_caller, double tol, int max_iter, int precond, int use_x0,
             int *iters, double *resid, cudaStream_t s) {
    const int M = (int)ctx->M;
    if (precond < 0 || precond > 2) return set_error(ctx, PCM_ERR_ARG, "pcm_cg_solve: precond must be 0, 1 or 2");
    if (precond == 2) {
        int rcf = rbj_finish(ctx, s);
        if (rcf) return rcf;
    }
    if (precond == 2 && ctx->rbj_block == 0) return set_error(ctx, PCM_ERR_STATE, "pcm_cg_solve: RBJ requested before pcm_rbj_build");
    if (M == 0) { if (iters) *iters = 0; if (resid) resid[0] = resid[1] = 0.0; return PCM_OK; }
    // all solver vectors live in the library's sorted point order; b is gathered on entry, x scattered on exit
    double *r = ctx->cg_vec, *z = r + M, *p = z + M, *Ap = p + M, *x = Ap + M, *b = x + M;
    double *scal = ctx->cg_scal, *partial = precond == 2 ? ctx->rbj_partial : scal + 16;
    int *ctl = reinterpret_cast<int *>(scal + 8);
    double *h = ctx->cg_scal_host;   // pinned: scal[0..8) then ctl
    int rc;
    const int saved_timing = ctx->timing;
    ctx->timing = 0;
    ctx->cg_ev_n = 0;
    const unsigned gb = (unsigned)cdiv(M, 256);
#define CG_TRY(expr) do { rc = (expr); if (rc) { ctx->timing = saved_timing; return rc; } } while (0)
#define CG_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { ctx->timing = saved_timing; \
        return set_error(ctx, PCM_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__)); } } while (0)
    auto update = [&](int init) -> int {
        if (precond == 2) {
            const int block = (int)ctx->rbj_block;
            if (((size_t)block + DOT_THREADS) * 8 > 48 * 1024)    // large blocks: opt in to more dynamic shared memory
                cudaFuncSetAttribute(cg_update_rbj_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(((size_t)block + DOT_THREADS) * 8));
            cg_update_rbj_kernel<<<(unsigned)ctx->rbj_nblocks, DOT_THREADS, ((size_t)block + DOT_THREADS) * 8, s>>>(
                M, block, ctx->rbj_order, ctx->rbj_inv, p, Ap, x, r, z, scal, partial, ctl, tol, max_iter, init);
        } else {
            cg_update_diag_kernel<<<DOT_BLOCKS, DOT_THREADS, 0, s>>>(M, precond == 1 ? ctx->pt_diag : nullptr, p, Ap, x, r, z, scal,
                                                                      scal + 16, ctl, tol, max_iter, init);
        }
        cg_direction_kernel<<<gb, 256, 0, s>>>(M, scal, z, p, ctl, init);
        ctx->launch_total += 2;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return set_error(ctx, PCM_ERR_CUDA, std::string("CG kernel launch: ") + cudaGetErrorString(e));
        return PCM_OK;
    };
    CG_CUDA(cudaMemsetAsync(scal, 0, 16 * sizeof(double), s));
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
    int it = 0;
    double rr = 0.0;
    // below AMAT_PERSIST_MAX points: every iteration inside one persistent cooperative kernel (pcm_cgp.cu)
    const bool persistent = ctx->opt.cg_path != 1 && ctx->opt.cg_path != 3 && cgp_can_solve(ctx, precond);
    if (persistent) {
        CG_TRY(cgp_solve(ctx, r, z, p, Ap, x, tol, max_iter, precond, s));
        CG_CUDA(cudaMemcpyAsync(h, scal, 16 * sizeof(double), cudaMemcpyDeviceToHost, s));
        CG_CUDA(cudaStreamSynchronize(s));
        const int *hc = reinterpret_cast<const int *>(h + 8);
        it = hc[CTL_ITERS];
        rr = h[2];
        if (hc[CTL_BAR_ERR]) { ctx->timing = saved_timing; return set_error(ctx, PCM_ERR_STATE, "pcm_cg_solve: grid barrier timed out"); }
    } else {
    CG_TRY(update(1));  // z = C r, p = z, rz, rr; raises STOP if already converged (or max_iter == 0)
    // RBJ: everything after the sweep in one cooperative kernel (cg_fused_rbj_kernel)
    bool fused = precond == 2 && ctx->opt.cg_path != 3;
    CgFused fa{};
    int fgrid = 0;
    size_t fsmem = 0;
    if (fused) {
        const int block = (int)ctx->rbj_block;
        fsmem = ((size_t)block + DOT_THREADS) * 8;
        int per_sm = 0;
        if (fsmem > 48 * 1024 ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, cg_fused_rbj_kernel, DOT_THREADS, fsmem) != cudaSuccess || per_sm < 1) {
            fused = false;
            (void)cudaGetLastError();
        } else {
            const int64_t want = std::max<int64_t>(cdiv(M, 32), ctx->rbj_nblocks);
            fgrid = (int)std::max<int64_t>(1, std::min<int64_t>(want, (int64_t)per_sm * ctx->sm_count));
            fa.M = M; fa.block = block; fa.nblocks = (int)ctx->rbj_nblocks; fa.max_iter = max_iter;
            fa.parts = amat_parts(ctx);
            fa.order = ctx->rbj_order; fa.inv = ctx->rbj_inv;
            fa.p = p; fa.Ap = Ap; fa.x = x; fa.r = r; fa.z = z; fa.scal = scal; fa.part1 = ctx->cg_part; fa.part2 = ctx->rbj_partial;
            fa.ctl = ctl; fa.tol = tol;
        }
    }
    const int batch = 8;   // iterations queued per read-back of the device-side convergence flag
    while (true) {
        CG_CUDA(cudaMemcpyAsync(h, scal, 16 * sizeof(double), cudaMemcpyDeviceToHost, s));
        CG_CUDA(cudaStreamSynchronize(s));
        const int *hc = reinterpret_cast<const int *>(h + 8);
        it = hc[CTL_ITERS];
        rr = h[2];
        if (hc[CTL_BAR_ERR]) { ctx->timing = saved_timing; return set_error(ctx, PCM_ERR_STATE, "pcm_cg_solve: grid barrier timed out"); }
        if (hc[CTL_STOP]) break;
        for (int k = 0; k < batch; ++k) {
            const bool ev = saved_timing && ctx->cg_ev_n < pcm_ctx::CG_EV;
            if (ev) CG_CUDA(cudaEventRecord(ctx->cg_ev[2 * ctx->cg_ev_n], s));
            CG_TRY(launch_amatvec_partials(ctx, p, ctl, s));
            if (ev) { CG_CUDA(cudaEventRecord(ctx->cg_ev[2 * ctx->cg_ev_n + 1], s)); ctx->cg_ev_n++; }
            if (fused) {
                void *args[] = {&fa};
                CG_CUDA(cudaLaunchCooperativeKernel((const void *)cg_fused_rbj_kernel, dim3((unsigned)fgrid), dim3(DOT_THREADS), args, fsmem, s));
                ctx->launch_total += 1;
            } else {
                cg_matvec_reduce_kernel<<<(unsigned)cdiv(M, 32), DOT_THREADS, 0, s>>>(M, amat_parts(ctx), p, Ap, scal, ctx->cg_part, ctl);
                ctx->launch_total += 1;
                CG_TRY(update(0));
            }
        }
    }
    }
    const double rn = std::sqrt(rr);
    // true residual
    CG_TRY(launch_amatvec_sorted(ctx, x, Ap, s));
    residual_kernel<<<gb, 256, 0, s>>>(M, b, Ap, z);
    norm2_kernel<<<DOT_BLOCKS, DOT_THREADS, 0, s>>>(M, z, scal, 4, scal + 16, ctl);
    scatter_kernel<<<gb, 256, 0, s>>>(M, ctx->s2c, x, x_caller);
    ctx->launch_total += 3;
    CG_CUDA(cudaGetLastError());
    CG_CUDA(cudaMemcpyAsync(h, scal, 16 * sizeof(double), cudaMemcpyDeviceToHost, s));
    CG_CUDA(cudaStreamSynchronize(s));
#undef CG_TRY
#undef CG_CUDA
    ctx->timing = saved_timing;
    if (iters) *iters = it;
    if (resid) { resid[0] = rn; resid[1] = std::sqrt(h[4]); }
    if (!std::isfinite(rn) || !std::isfinite(h[4]))
        return set_error(ctx, PCM_ERR_NUMERIC, "pcm_cg_solve: the residual is not finite (non-finite right-hand side, or p.Ap = 0)");
    return rn > tol ? PCM_NOT_CONVERGED : PCM_OK;
}

}  // namespace pcm
