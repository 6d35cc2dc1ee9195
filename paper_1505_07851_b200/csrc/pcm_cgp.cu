// pcm_cgp.cu -- the whole preconditioned CG solve as ONE persistent cooperative kernel, and the
// warp-granular symmetric A q sweep it is built on, for cavities below AMAT_PERSIST_MAX points (where an iteration is tens of
// microseconds and launches, tails and partial-sum round trips cost as much as the arithmetic).
//
// Work partition (plan_sweep, fixed at pcm_setup).  Rows are cut into blocks of 4 row groups (128 points); a "strip" is
// one row block against one column group of 32 points with at least one far patch, (rb, cg >= 4 rb); strips inside the
// row block's own columns (cg < 4 rb + 4) are swept for the rows only, the others once for both triangles (A_ij = A_ji), as
// amatvec_kernel does.  The strips, row block after row block, are cut into one contiguous segment per WARP of the
// cooperative grid (148 CTAs x 16 warps), of equal cost -- far patches count 1, the stored near patches a warp takes first
// count CGP_NEAR_COST each.  A warp stages its 32 columns itself (no CTA barrier anywhere in the sweep), keeps 4 rows per
// lane in registers, and leaves row sums in yslot[(segment, row block) run][128] and column sums in colpart[rb][j].
//
// One PCG iteration inside the kernel (three grid barriers, no host involvement until the solve stops):
//   S  sweep with p_j = z_j + beta p_old,j formed while staging           -- barrier --
//   R  Ap_k = fixed-order sum of the partial sums of row k; p_k stored; per-task p.Ap           -- barrier --
//   U  alpha (every CTA adds the per-task partials itself, in index order); x += alpha p, r -= alpha Ap, z = C r
//      (RBJ block inverse, Jacobi or none), per-block r.r and r.z          -- barrier --
//      beta and the convergence test, identically in every CTA.
// Every sum has a fixed order, so a solve is bit-reproducible run to run.  The separate-launch path of pcm_solver.cu
// (pcm_options.cg_path = 1) stays as the reference: same recurrences, another summation order of the A q partial sums.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "pcm_device.cuh"

namespace pcm {

constexpr int CGP_THREADS = 512;
constexpr int CGP_WARPS = CGP_THREADS / 32;
constexpr int CGP_R = 4;                          // row groups per warp
constexpr int CGP_ROWS = CGP_R * 32;              // rows of a row block
constexpr int CGP_C = 2;
constexpr int CGP_MIN_PAIRS = 4;                 // column pairs per warp below which the persistent grid shrinks (plan_sweep)
constexpr double CGP_FAR_AWAY = 1.0715086071862673e301;     // 2^1000: the r^2 of a row that is to contribute nothing
enum { CGP_CTL_STOP = 0, CGP_CTL_ITERS = 1, CGP_CTL_BAR_COUNT = 3, CGP_CTL_BAR_GEN = 4, CGP_CTL_BAR_ERR = 5 };

// What a warp needs to start its share of the sweep, in one 64-byte load (instead of three dependent ones through seg_start,
// strip and the near-piece tables: after an L2 flush each of those is a trip to HBM with nothing to overlap it).
struct alignas(16) CgpWarpInit {
    int64_t hb, he;            // its column pairs (pair h belongs to strip h >> 4)
    int2 strip0, strip1;       // descriptors of its first two strips
    int64_t ne, ne_end;        // list entries of its first near piece (piece = warp index)
    int32_t slot0, ncg0;       // first row-sum slot; column group of entry ne
    int32_t pad[2];
};
static_assert(sizeof(CgpWarpInit) == 64, "CgpWarpInit is one 64-byte record");

struct CgpArgs {
    int M, ng, nrb, nwarp;
    const CgpWarpInit *winit;
    const double4 *pt, *colloc, *org;
    const int2 *strip;
    const int64_t *seg_start;
    const int32_t *seg_slot0, *rb_slot_start;
    double *yslot, *colpart;
    double *afar;              // stored far field: [half strip][16 columns][4 row groups][32 lanes] values of 1/r (~2^-500 where near), or nullptr
    // stored near patches (PatchMap of A): pieces of <= NEAR_PIECE patches of one row group
    const double *nblk;
    const int64_t *nstart, *npstart;
    const int32_t *nlist, *npiece_rg;
    int64_t npiece;
    double *near;
    // matvec form: y[qidx ? qidx[k] : k] = (A q)_k, q in sorted order
    const double *q;
    const int32_t *qidx;
    double *y;
    // PCG
    int precond, block, nblocks, max_iter;
    double tol;
    const double *diag;
    const int32_t *order;
    const double *inv;
    double *r, *z, *p0, *p1, *Ap, *x, *part1, *part2, *scal;
    int *ctl;
    int phase;                 // cgp_matvec_kernel: 0 = sweep, grid barrier, row sums (cooperative launch); 1 = sweep only; 2 = row sums only
    unsigned long long *dbg;   // PCM_VERBOSE: %globaltimer of CTA 0 at the phase boundaries of the first iterations
};
constexpr int CGP_DBG_ITERS = 8;
__device__ __forceinline__ void cgp_stamp(const CgpArgs &a, int iter, int phase) {
    if (a.dbg && blockIdx.x == 0 && threadIdx.x == 0 && iter < CGP_DBG_ITERS) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        a.dbg[iter * 8 + phase] = t;
    }
}

__device__ __forceinline__ void cgp_grid_sync(int *ctl, unsigned G) {
    __syncthreads();
    if (threadIdx.x == 0) {
        volatile int *gen = ctl + CGP_CTL_BAR_GEN;
        const int g = *gen;
        __threadfence();
        if (atomicAdd(ctl + CGP_CTL_BAR_COUNT, 1) == (int)G - 1) {
            ctl[CGP_CTL_BAR_COUNT] = 0;
            __threadfence();
            atomicAdd(ctl + CGP_CTL_BAR_GEN, 1);
        } else {
            long long spins = 0;
            while (*gen == g) {
                if (++spins > (1ll << 28)) { ctl[CGP_CTL_BAR_ERR] = 1; break; }
            }
        }
        __threadfence();
    }
    __syncthreads();
}

// fixed-order sum over the CTA; the result is returned to every thread
__device__ __forceinline__ double cgp_block_sum(double v, double *s_w, double *s_bc) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        double t = threadIdx.x < CGP_WARPS ? s_w[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = CGP_WARPS / 2; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
        if (threadIdx.x == 0) *s_bc = t;
    }
    __syncthreads();
    return *s_bc;
}
__device__ __forceinline__ double cgp_ordered_sum(const double *partial, int n, double *s_w, double *s_bc) {
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += CGP_THREADS) s += __ldcg(partial + i);
    return cgp_block_sum(s, s_w, s_bc);
}
// two sums at once: the same additions in the same order as two calls of the functions above, one round of barriers instead
// of two (s_w: 2 x CGP_WARPS doubles, s_bc: 2)
__device__ __forceinline__ void cgp_block_sum2(double &a, double &b, double *s_w, double *s_bc) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
    }
    __syncthreads();
    if ((threadIdx.x & 31) == 0) { s_w[threadIdx.x >> 5] = a; s_w[CGP_WARPS + (threadIdx.x >> 5)] = b; }
    __syncthreads();
    if (threadIdx.x < 32) {
        double ta = threadIdx.x < CGP_WARPS ? s_w[threadIdx.x] : 0.0, tb = threadIdx.x < CGP_WARPS ? s_w[CGP_WARPS + threadIdx.x] : 0.0;
#pragma unroll
        for (int o = CGP_WARPS / 2; o > 0; o >>= 1) {
            ta += __shfl_down_sync(0xffffffffu, ta, o);
            tb += __shfl_down_sync(0xffffffffu, tb, o);
        }
        if (threadIdx.x == 0) { s_bc[0] = ta; s_bc[1] = tb; }
    }
    __syncthreads();
    a = s_bc[0];
    b = s_bc[1];
}
__device__ __forceinline__ void cgp_ordered_sum2(const double *pa, const double *pb, int n, double &a, double &b, double *s_w, double *s_bc) {
    a = 0.0; b = 0.0;
    for (int i = threadIdx.x; i < n; i += CGP_THREADS) { a += __ldcg(pa + i); b += __ldcg(pb + i); }
    cgp_block_sum2(a, b, s_w, s_bc);
}

// cp.async (LDGSTS): global -> shared without registers; src_bytes < size zero-fills the rest (padding columns)
__device__ __forceinline__ void cgp_cp16(void *dst, const void *src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cgp_cp8(void *dst, const void *src, int src_bytes) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cgp_cp_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Per-warp shared memory (doubles): two staging buffers {columns (-2 (b - o), |b - o|^2) [32] double4, origin double4,
// A-values [32], B-values [32]} (the charge of column t is fma(beta, B_t, A_t): CG direction z + beta p_old, or the caller's q
// with beta = 0), the charges [32], the column-sum transpose [16][33], one half of a stored near patch [16][32] with the
// A / B values of its 32 columns and the charges formed from them.
constexpr int CGP_STG = 128 + 4 + 32 + 32;             // one staging buffer
constexpr int CGP_OFF_Q = 2 * CGP_STG;                 // charges
constexpr int CGP_OFF_SC = CGP_OFF_Q + 32;             // transpose
constexpr int CGP_OFF_NB = CGP_OFF_SC + 16 * 33;       // near half patch
constexpr int CGP_OFF_NA = CGP_OFF_NB + 16 * 32;       // near A / B values
constexpr int CGP_OFF_NQ = CGP_OFF_NA + 64;            // charges of the near patch's 32 columns
constexpr int CGP_WSMEM2 = CGP_OFF_NQ + 32;

// where the vector the sweep multiplies comes from: value_j = fma(beta, B[j], A[j]), all in sorted order (a caller-order q is
// gathered first, cgp_gather_kernel: an index load in front of every staged column would sit on the sweep's critical path)
struct PSrc {
    const double *A, *B;         // CG: z, p_old; matvec: q (sorted), nullptr
    double beta;
    __device__ __forceinline__ double operator()(int j) const {
        const double av = __ldcg(A + j);
        return B ? fma(beta, __ldcg(B + j), av) : av;
    }
};

// The warp's share of the sweep: its segment of far half-strips, with the stored near patches of its near pieces streamed
// through shared memory underneath (one half patch per half strip, copied asynchronously while the previous half strip
// computes), and the columns of the next strip prefetched the same way.
// MODE 0: 1/r evaluated on the fly; MODE 1: evaluated and written to a.afar (pcm_setup, no sums needed); MODE 2: read from a.afar
// (the stored-A variant of the paper, PAPER.md:106 -- same FMAs in the same order, so the result equals MODE 0 bit for bit).
template <int MODE>
__device__ __forceinline__ void cgp_sweep(const CgpArgs &a, const PSrc &pv, int gw, int lane, double *wsm) {
    constexpr int R = CGP_R, C = CGP_C;
    const int M = a.M;
    double *s_q = wsm + CGP_OFF_Q, *sc = wsm + CGP_OFF_SC, *s_nb = wsm + CGP_OFF_NB, *s_na = wsm + CGP_OFF_NA, *s_nq = wsm + CGP_OFF_NQ;
    // ---- near pieces of this warp: piece gw, gw + nwarp, ...; state = (entry e, half) of the half patch in flight
    int64_t piece = gw, ne = 0, ne_end = 0;
    int nhalf = 0, ncg = 0, ncg_next = 0;     // column group of patch ne, and of patch ne + 1 (loaded one half strip ahead)
    double ynear = 0.0;
    bool near_inflight = false;
    auto near_open = [&]() {          // bounds of the current piece (or none left)
        if (piece < a.npiece) {
            const int64_t rg = a.npiece_rg[piece];
            ne = a.nstart[rg] + (piece - a.npstart[rg]) * NEAR_PIECE;
            ne_end = min(a.nstart[rg + 1], ne + NEAR_PIECE);
            nhalf = 0;
            ynear = 0.0;
            ncg = a.nlist[ne];
        }
    };
    auto near_issue = [&]() {         // copy half `nhalf` of patch `ne` and the A / B values of its columns
        if (piece >= a.npiece) { near_inflight = false; return; }
        const double *blk = a.nblk + (size_t)ne * 1024 + (size_t)nhalf * 512;
#pragma unroll
        for (int k = 0; k < 8; ++k) cgp_cp16(s_nb + (k * 32 + lane) * 2, blk + (k * 32 + lane) * 2, 16);
        const int j = ncg * 32 + lane;
        cgp_cp8(s_na + lane, pv.A + min(j, M - 1), j < M ? 8 : 0);
        cgp_cp8(s_na + 32 + lane, pv.B ? pv.B + min(j, M - 1) : pv.A, (pv.B && j < M) ? 8 : 0);
        if (nhalf == 0 && ne + 1 < ne_end) ncg_next = a.nlist[ne + 1];      // used a half strip from now: no wait on this load
        near_inflight = true;
    };
    auto near_consume = [&]() {       // after cp_wait_all + __syncwarp: add the half patch, advance, store a finished piece
        if (!near_inflight) return;
        // the charges go through shared memory and come back as broadcast loads, two per instruction (a shuffle of a double
        // by a run-time lane costs ~20 instructions here; this loop was 500 of them per half patch)
        s_nq[lane] = fma(pv.beta, s_na[32 + lane], s_na[lane]);
        __syncwarp();
        const double *col = s_nb + lane;
        const double2 *qq = reinterpret_cast<const double2 *>(s_nq + nhalf * 16);
#pragma unroll
        for (int t = 0; t < 16; t += 2) {
            const double2 q2 = qq[t >> 1];
            ynear = fma(q2.x, col[t * 32], ynear);
            ynear = fma(q2.y, col[(t + 1) * 32], ynear);
        }
        if (++nhalf == 2) {
            nhalf = 0;
            ncg = ncg_next;
            if (++ne == ne_end) {
                a.near[piece * 32 + lane] = ynear;
                piece += a.nwarp;
                near_open();
            }
        }
        near_inflight = false;
        __syncwarp();                 // every lane has read its column before the next copy may overwrite the buffer
    };
    CgpWarpInit wi;
    {
        const int4 *src = reinterpret_cast<const int4 *>(a.winit + gw);
        int4 *dst = reinterpret_cast<int4 *>(&wi);
#pragma unroll
        for (int k = 0; k < 4; ++k) dst[k] = __ldg(src + k);
    }
    if (piece < a.npiece) { ne = wi.ne; ne_end = wi.ne_end; ncg = wi.ncg0; }
    near_issue();
    // ---- far column pairs [hb, he): pair h is columns 2 (h & 7), 2 (h & 7) + 1 of half (h >> 3) & 1 of strip h >> 4
    const int hb = (int)wi.hb, he = (int)wi.he;
    int slot = wi.slot0;
    int cur_rb = -1, buf = 0;
    double qa[R], y[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { qa[r] = y[r] = 0.0; }
    auto stage_issue = [&](int2 st, int b) {     // columns of strip st into staging buffer b
        double *sb = wsm + b * CGP_STG;
        const int cg = st.y & 0xffffff, j = cg * 32 + lane;
        const double4 *src = a.colloc + min(j, M - 1);
        cgp_cp16(sb + 4 * lane, src, j < M ? 16 : 0);
        cgp_cp16(sb + 4 * lane + 2, reinterpret_cast<const double *>(src) + 2, j < M ? 16 : 0);
        if (lane < 2) cgp_cp16(sb + 128 + 2 * lane, reinterpret_cast<const double *>(a.org + cg) + 2 * lane, 16);
        cgp_cp8(sb + 132 + lane, pv.A + min(j, M - 1), j < M ? 8 : 0);
        cgp_cp8(sb + 164 + lane, pv.B ? pv.B + min(j, M - 1) : pv.A, (pv.B && j < M) ? 8 : 0);
    };
    // d_next: the strip whose columns are in flight into buffer nbuf; d_next2: the one after it (descriptor only)
    const int last_s = (he - 1) >> 4;
    int2 d_next = make_int2(0, 0), d_next2 = make_int2(0, 0);
    int nbuf = 0;
    // The rows' coordinates are NOT kept in registers across strips: they are read again (4 x 32 bytes per lane, L1 hits)
    // whenever a strip starts and turned into the strip's local coordinates at once -- 24 registers less in the inner loop.
    auto load_rows = [&](int rb_) {      // charges of the 4 x 32 rows of row block rb_
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int ii = (rb_ * R + r) * 32 + lane;
            qa[r] = ii < M ? pv(ii) : 0.0;              // padding rows: zero charge, their sums are not used
            y[r] = 0.0;
        }
    };
    if (hb < he) {
        d_next = wi.strip0;
        d_next2 = wi.strip1;
        stage_issue(d_next, 0);
        cur_rb = d_next.x;        // the first row block's rows are loaded here, beside the copies, not after waiting for them
        load_rows(cur_rb);
    }
    int cur_s = -1;
    double alx[R], aly[R], alz[R], a2[R];
    unsigned m = 0;
    bool sym = false;
    int rb = 0, cg = 0;
    for (int h = hb; h < he;) {
        // one pass = the columns [tb, te) of one half strip: all 16 except at the two ends of the segment, which may lie
        // anywhere (a column, with all 128 rows, still belongs to one warp, so the sums keep their fixed order)
        const int sidx = h >> 4;
        const int half = (h >> 3) & 1;
        const int tb = 2 * (h & 7), te = min(16, tb + 2 * (he - h));
        cgp_cp_wait_all();
        __syncwarp();
        near_consume();
        if (sidx != cur_s) {                     // a new strip: its columns have landed in staging buffer nbuf
            const int2 st = d_next;
            buf = nbuf;
            cur_s = sidx;
            rb = st.x; cg = st.y & 0xffffff; m = (unsigned)st.y >> 24;
            if (rb != cur_rb) {
                if (cur_rb >= 0) {
#pragma unroll
                    for (int r = 0; r < R; ++r) a.yslot[(size_t)slot * CGP_ROWS + r * 32 + lane] = y[r];
                    ++slot;
                }
                cur_rb = rb;
                load_rows(rb);
            }
            sym = cg >= rb * R + R;
            const double *sb = wsm + buf * CGP_STG;
            s_q[lane] = fma(pv.beta, sb[164 + lane], sb[132 + lane]);
            const double4 o = *reinterpret_cast<const double4 *>(sb + 128);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int ii = (rb * R + r) * 32 + lane;
                const double4 p = a.pt[min(ii, M - 1)];
                alx[r] = (ii < M ? p.x : p.x + 3e8) - o.x; aly[r] = p.y - o.y; alz[r] = p.z - o.z;   // padding rows: far away
                a2[r] = fma(alz[r], alz[r], fma(aly[r], aly[r], alx[r] * alx[r]));
                // Row groups whose patch against this column group is near (stored, added by the near pieces) are moved out
                // of reach instead of being selected away per evaluation: r^2 = 2^1000 whatever the column, 1/r ~ 2^-500, and
                // a charge times that is absorbed without a trace by the first genuine term of any sum it enters.
                if (!((m >> r) & 1u)) a2[r] = CGP_FAR_AWAY;
            }
            // prefetch the next strip of this segment into the other buffer, and the descriptor of the one after it
            if (sidx + 1 <= last_s) {
                d_next = d_next2;
                nbuf = buf ^ 1;
                stage_issue(d_next, nbuf);
                if (sidx + 2 <= last_s) d_next2 = a.strip[sidx + 2];
            }
            __syncwarp();
        }
        near_issue();
        const double4 *sp = reinterpret_cast<const double4 *>(wsm + buf * CGP_STG) + half * 16 + tb;
        const double *sq = s_q + half * 16 + tb;
        // Strips with a near patch among the 4 row groups run the same blocked loop (the near rows sit at r^2 = 2^1000, see
        // above): three rows of wasted arithmetic at worst, but no slow path whose cost the partition would have to know
        // (near patches cluster at the start of a row block's strips), and no select in the loop.
        double *ah = MODE ? a.afar + (size_t)(h >> 3) * (16 * R * 32) + lane : nullptr;
        double *scp = sc + lane + tb * 33;
#pragma unroll 1
        for (int t = tb; t < te; t += C, sp += C, sq += C, scp += C * 33) {
            double4 b[C];
            double qb[C], r2[C][R], cc[C];
#pragma unroll
            for (int c = 0; c < C; ++c) { b[c] = sp[c]; qb[c] = sq[c]; }
            if (MODE == 2) {
#pragma unroll
                for (int c = 0; c < C; ++c)
#pragma unroll
                    for (int r = 0; r < R; ++r) r2[c][r] = __ldg(ah + ((t + c) * R + r) * 32);     // the stored 1/r itself
            } else {
#pragma unroll
                for (int c = 0; c < C; ++c)
#pragma unroll
                    for (int r = 0; r < R; ++r) r2[c][r] = fma(alx[r], b[c].x, fma(aly[r], b[c].y, fma(alz[r], b[c].z, a2[r] + b[c].w)));
            }
#pragma unroll
            for (int c = 0; c < C; ++c) {
                cc[c] = 0.0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    double rs;
                    if (MODE == 2) {
                        rs = r2[c][r];
                    } else {
                        rs = rsqrt_fast(r2[c][r]);
                        if (MODE == 1) ah[((t + c) * R + r) * 32] = rs;
                    }
                    y[r] = fma(qb[c], rs, y[r]);
                    cc[c] = fma(qa[r], rs, cc[c]);
                }
                if (sym) scp[c * 33] = cc[c];
            }
        }
        if (sym) {
            __syncwarp();
            // lane l sums column (l & 15) over the lanes [16 (l >> 4), 16 (l >> 4) + 16), fixed order
            const double *col = sc + (lane & 15) * 33 + (lane >> 4) * 16;
            double t = col[0];
#pragma unroll
            for (int k = 1; k < 16; ++k) t += col[k];
            const double o2 = __shfl_xor_sync(0xffffffffu, t, 16);
            const int j = cg * 32 + half * 16 + lane;
            if (lane >= tb && lane < te && j < M) a.colpart[(size_t)rb * M + j] = t + o2;
        }
        h += (te - tb) >> 1;
    }
    if (cur_rb >= 0) {
#pragma unroll
        for (int r = 0; r < R; ++r) a.yslot[(size_t)slot * CGP_ROWS + r * 32 + lane] = y[r];
    }
    // near half patches the far segment was too short to carry
    while (near_inflight) {
        cgp_cp_wait_all();
        __syncwarp();
        near_consume();
        __syncwarp();
        near_issue();
    }
}

// Sum of the partial sums of the rows of row group g, in a fixed order.  The CTA works as CGP_TEAMS teams of CGP_TW warps,
// one row group per team: warp `part` of the team adds every CGP_TW-th term of the three lists (row slots of the row block,
// column sums of the earlier row blocks, near pieces; eight loads in flight), the team's first warp adds the CGP_TW partial
// sums.  Valid in the team's first warp (0.0 for rows >= M or g >= ng); s_tmp: CGP_WARPS x 32 doubles; all threads call.
constexpr int CGP_TW = 4, CGP_TEAMS = CGP_WARPS / CGP_TW;
template <class F>
__device__ __forceinline__ double cgp_strided_sum(int first, int end, F load) {
    double s = 0.0;
    int c = first;
    for (; c + 7 * CGP_TW < end; c += 8 * CGP_TW) {
        double v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = load(c + u * CGP_TW);
#pragma unroll
        for (int u = 0; u < 8; ++u) s += v[u];
    }
    for (; c < end; c += CGP_TW) s += load(c);
    return s;
}
__device__ __forceinline__ double cgp_row_sum(const CgpArgs &a, int g, double *s_tmp) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, part = warp % CGP_TW;
    const int k = g * 32 + lane, M = a.M;
    double s = 0.0;
    if (g < a.ng && k < M) {
        const int rb = g / CGP_R, sub = g - rb * CGP_R;
        const double *ys = a.yslot + (size_t)sub * 32 + lane;
        s += cgp_strided_sum(a.rb_slot_start[rb] + part, a.rb_slot_start[rb + 1], [&](int c) { return __ldcg(ys + (size_t)c * CGP_ROWS); });
        s += cgp_strided_sum(part, rb, [&](int c) { return __ldcg(a.colpart + (size_t)c * M + k); });
        s += cgp_strided_sum((int)a.npstart[g] + part, (int)a.npstart[g + 1], [&](int c) { return __ldcg(a.near + (size_t)c * 32 + lane); });
    }
    s_tmp[warp * 32 + lane] = s;
    __syncthreads();
    double t = 0.0;
    if (part == 0) {
#pragma unroll
        for (int q = 0; q < CGP_TW; ++q) t += s_tmp[(warp + q) * 32 + lane];
    }
    return t;
}

// x += alpha p, r -= alpha Ap, z = C r and the per-block r.r, r.z (init: r is given, no update).  part2[0..nU) and
// part2[nU..2 nU) receive the partial sums, nU = nblocks (RBJ) or gridDim.x (Jacobi, none).
__device__ __forceinline__ void cgp_update(const CgpArgs &a, const double *p, double alpha, bool init, double *dyn, double *s_w, double *s_bc) {
    const int M = a.M, tid = threadIdx.x;
    const unsigned G = gridDim.x;
    if (a.precond == 2) {
        // two teams of 256 threads, one RBJ block each (named barriers: the teams' trip counts may differ)
        constexpr int TT = CGP_THREADS / 2;
        const int team = tid / TT, tt = tid - team * TT;
        const int block = a.block;
        double *s_r = dyn + (size_t)team * (block + TT), *s_part = s_r + block;
        auto team_sync = [&]() { asm volatile("bar.sync %0, %1;" ::"r"(1 + team), "r"(TT) : "memory"); };
        auto team_sum = [&](double v) {      // fixed-order sum over the team, valid in its thread 0
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
            team_sync();
            if ((tt & 31) == 0) s_part[tt >> 5] = v;
            team_sync();
            double t = 0.0;
            if (tt < 32) {
                t = tt < TT / 32 ? s_part[tt] : 0.0;
#pragma unroll
                for (int o = TT / 64; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
            }
            team_sync();
            return t;
        };
        for (int b = blockIdx.x * 2 + team; b < a.nblocks; b += (int)G * 2) {
            const long long start = (long long)b * block;
            const int n = (int)min((long long)block, (long long)M - start);
            const double *am = a.inv + (size_t)b * block * block;
            const int32_t *idx = a.order + start;
            double rr = 0.0, rz = 0.0;
            for (int j = tt; j < n; j += TT) {
                const int i = idx[j];
                double ri = __ldcg(a.r + i);
                if (!init) {
                    a.x[i] = fma(alpha, __ldcg(p + i), __ldcg(a.x + i));
                    ri = fma(-alpha, __ldcg(a.Ap + i), ri);
                    a.r[i] = ri;
                }
                s_r[j] = ri;
                rr = fma(ri, ri, rr);
            }
            team_sync();
            // z = M_b^-1 r: np threads per row, each over every np-th column (the inverse is symmetric: the column read is
            // coalesced across the rows), the np partial sums added in order through shared memory
            const int np = n >= TT ? 1 : TT / n;
            const int rpp = TT / np;
            const int part = tt / rpp, il = tt - part * rpp;
            for (int i0 = 0; i0 < n; i0 += rpp) {
                const int i = i0 + il;
                double sacc = 0.0;
                if (i < n && part < np) {
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
                s_part[tt] = sacc;
                team_sync();
                if (part == 0 && i < n) {
                    double t = 0.0;
                    for (int q = 0; q < np; ++q) t += s_part[q * rpp + il];
                    a.z[idx[i]] = t;
                    rz = fma(s_r[i], t, rz);
                }
                team_sync();
            }
            {   // both sums in one round of team barriers (the additions and their order are those of team_sum)
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    rr += __shfl_down_sync(0xffffffffu, rr, o);
                    rz += __shfl_down_sync(0xffffffffu, rz, o);
                }
                team_sync();
                if ((tt & 31) == 0) { s_part[tt >> 5] = rr; s_part[TT / 32 + (tt >> 5)] = rz; }
                team_sync();
                if (tt < 32) {
                    rr = tt < TT / 32 ? s_part[tt] : 0.0;
                    rz = tt < TT / 32 ? s_part[TT / 32 + tt] : 0.0;
#pragma unroll
                    for (int o = TT / 64; o > 0; o >>= 1) {
                        rr += __shfl_down_sync(0xffffffffu, rr, o);
                        rz += __shfl_down_sync(0xffffffffu, rz, o);
                    }
                }
                team_sync();
            }
            if (tt == 0) { a.part2[b] = rr; a.part2[a.nblocks + b] = rz; }
        }
        __syncthreads();
    } else {
        double rr = 0.0, rz = 0.0;
        for (int i = blockIdx.x * CGP_THREADS + tid; i < M; i += (int)G * CGP_THREADS) {
            double ri = __ldcg(a.r + i);
            if (!init) {
                a.x[i] = fma(alpha, __ldcg(p + i), __ldcg(a.x + i));
                ri = fma(-alpha, __ldcg(a.Ap + i), ri);
                a.r[i] = ri;
            }
            const double zi = a.precond == 1 ? ri / a.diag[i] : ri;
            a.z[i] = zi;
            rr = fma(ri, ri, rr);
            rz = fma(ri, zi, rz);
        }
        cgp_block_sum2(rr, rz, s_w, s_bc);
        if (tid == 0) { a.part2[blockIdx.x] = rr; a.part2[G + blockIdx.x] = rz; }
    }
}

template <int MODE>
__global__ void __launch_bounds__(CGP_THREADS, 1) cgp_solve_kernel(CgpArgs a) {
    extern __shared__ double dyn[];
    __shared__ double s_w[2 * CGP_WARPS];
    __shared__ double s_bc2[2];
    double &s_bc = s_bc2[0];
    const unsigned G = gridDim.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int gw = blockIdx.x * CGP_WARPS + warp;
    const int nU = a.precond == 2 ? a.nblocks : (int)G;
    double *wsm = dyn + warp * CGP_WSMEM2;
    // z = C r, r.r, r.z of the initial residual
    cgp_update(a, nullptr, 0.0, true, dyn, s_w, s_bc2);
    cgp_grid_sync(a.ctl, G);
    double srr, rz_old;
    cgp_ordered_sum2(a.part2, a.part2 + nU, nU, srr, rz_old, s_w, s_bc2);
    double beta = 0.0, pAp = 0.0;
    int iters = 0, cur = 0;
    bool stop = !(sqrt(srr) > a.tol) || a.max_iter <= 0;
    while (!stop) {
        const double *pold = cur ? a.p1 : a.p0;
        double *pnew = cur ? a.p0 : a.p1;
        PSrc pv{a.z, pold, beta};
        cgp_stamp(a, iters, 0);
        unsigned long long t0 = 0;
        if (a.dbg && iters == 1 && tid == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
        unsigned long long w0 = 0;
        if (a.dbg && iters == 1) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(w0));
        cgp_sweep<MODE>(a, pv, gw, lane, wsm);
        if (a.dbg && iters == 1 && lane == 0) {      // this warp's own sweep time (calibrates the cost model of plan_sweep)
            unsigned long long w1;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(w1));
            a.dbg[CGP_DBG_ITERS * 8 + 1024 + gw] = w1 - w0;
        }
        if (a.dbg && iters == 1) {
            __syncthreads();
            if (tid == 0) { unsigned long long t1; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1)); a.dbg[CGP_DBG_ITERS * 8 + blockIdx.x] = t1 - t0; }
        }
        cgp_stamp(a, iters, 1);
        cgp_grid_sync(a.ctl, G);
        cgp_stamp(a, iters, 2);
        for (int g0 = blockIdx.x * CGP_TEAMS; g0 < a.ng; g0 += (int)G * CGP_TEAMS) {
            const int g = g0 + warp / CGP_TW;
            const double t = cgp_row_sum(a, g, dyn);
            if (warp % CGP_TW == 0 && g < a.ng) {
                const int k = g * 32 + lane;
                double dot = 0.0;
                if (k < a.M) {
                    const double pk = pv(k);
                    a.Ap[k] = t;
                    pnew[k] = pk;
                    dot = pk * t;
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) dot += __shfl_down_sync(0xffffffffu, dot, o);
                if (lane == 0) a.part1[g] = dot;
            }
            __syncthreads();
        }
        cgp_stamp(a, iters, 3);
        cgp_grid_sync(a.ctl, G);
        cgp_stamp(a, iters, 4);
        pAp = cgp_ordered_sum(a.part1, a.ng, s_w, &s_bc);
        const double alpha = rz_old / pAp;
        cgp_update(a, pnew, alpha, false, dyn, s_w, s_bc2);
        cgp_stamp(a, iters, 5);
        cgp_grid_sync(a.ctl, G);
        cgp_stamp(a, iters, 6);
        double srz;
        cgp_ordered_sum2(a.part2, a.part2 + nU, nU, srr, srz, s_w, s_bc2);
        beta = srz / rz_old;
        rz_old = srz;
        ++iters;
        cur ^= 1;
        stop = !(sqrt(srr) > a.tol) || iters >= a.max_iter || *((volatile int *)&a.ctl[CGP_CTL_BAR_ERR]) != 0;
    }
    if (blockIdx.x == 0 && tid == 0) {
        a.scal[0] = rz_old; a.scal[1] = pAp; a.scal[2] = srr; a.scal[5] = beta;
        a.ctl[CGP_CTL_ITERS] = iters;
        a.ctl[CGP_CTL_STOP] = 1;
    }
}

// The three launches of a single A q (gather, sweep, row sums) form a chain of programmatic dependent launches: a kernel lets
// its successor be scheduled at once and the successor waits for it (completion and visibility) before it touches memory, so
// the launch latencies overlap the kernel before.  Without the launch attribute both instructions do nothing.
__device__ __forceinline__ void cgp_pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void cgp_pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// q in the caller's order -> sorted order
__global__ void cgp_gather_kernel(const double *__restrict__ q, const int32_t *__restrict__ idx, double *__restrict__ qs, int M) {
    cgp_pdl_launch_dependents();
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < M) qs[k] = q[idx[k]];
}

// y = A q with the same sweep and row sums: one launch, one grid barrier
template <int MODE>
__global__ void __launch_bounds__(CGP_THREADS, 1) cgp_matvec_kernel(CgpArgs a) {
    extern __shared__ double dyn[];
    const unsigned G = gridDim.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    PSrc pv{a.q, nullptr, 0.0};
    cgp_pdl_launch_dependents();
    cgp_pdl_wait();
    if (a.phase != 2) cgp_sweep<MODE>(a, pv, blockIdx.x * CGP_WARPS + warp, lane, dyn + warp * CGP_WSMEM2);
    if (MODE == 1 || a.phase == 1) return;      // filling the store, or the sweep half of a two-launch product
    if (a.phase == 0) cgp_grid_sync(a.ctl, G);
    for (int g0 = blockIdx.x * CGP_TEAMS; g0 < a.ng; g0 += (int)G * CGP_TEAMS) {
        const int g = g0 + warp / CGP_TW;
        const double t = cgp_row_sum(a, g, dyn);
        const int k = g * 32 + lane;
        if (warp % CGP_TW == 0 && g < a.ng && k < a.M) a.y[a.qidx ? a.qidx[k] : k] = t;
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// host: the partition and the launches
// ---------------------------------------------------------------------------------------------
static int64_t cdiv2(int64_t a, int64_t b) { return (a + b - 1) / b; }

template <class T>
static int upload2(pcm_ctx *ctx, T **dst, const std::vector<T> &src) {
    int rc = dev_alloc_t(ctx, dst, std::max<size_t>(src.size(), 1));
    if (rc) return rc;
    if (!src.empty()) PCM_CUDA(ctx, cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return PCM_OK;
}

static CgpArgs cgp_args(pcm_ctx *ctx);

// Builds the warp-granular partition for contexts whose A q sweep is latency-dominated (M < AMAT_PERSIST_MAX) and whose
// near patches are stored.  Leaves ctx->cgp.ready = false otherwise (the separate-launch path is used).
int plan_sweep(pcm_ctx *ctx) {
    SweepPlan &sp = ctx->cgp;
    sp.ready = false;
    const int64_t M = ctx->M;
    const PatchMap &pm = ctx->amat_map;
    if (M == 0 || ctx->opt.cg_path == 1 || ctx->opt.cg_path == 3) return PCM_OK;
    if (ctx->opt.cg_path == 0 && M >= AMAT_PERSIST_MAX) return PCM_OK;
    if (pm.npiece > 0 && ctx->amat_blocks == nullptr) return PCM_OK;      // near patches not stored: classic path
    if (pm.far_host.empty()) return PCM_OK;
    int per_sm = 0;
    const size_t smem = (size_t)CGP_WARPS * CGP_WSMEM2 * 8;
    if (cudaFuncSetAttribute(cgp_solve_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess ||
        cudaFuncSetAttribute(cgp_solve_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess ||
        cudaFuncSetAttribute(cgp_matvec_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess ||
        cudaFuncSetAttribute(cgp_matvec_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess ||
        cudaFuncSetAttribute(cgp_matvec_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, cgp_solve_kernel<0>, CGP_THREADS, smem) != cudaSuccess || per_sm < 1) {
        (void)cudaGetLastError();
        return PCM_OK;
    }
    int coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device);
    if (!coop) return PCM_OK;
    const int64_t ng = pm.nrg, nrb = cdiv2(ng, CGP_R), nbyte = pm.nbyte;
    sp.ng = (int)ng; sp.nrb = (int)nrb;
    // strips with at least one far patch
    std::vector<int2> strip;
    std::vector<float> cost;
    for (int64_t rb = 0; rb < nrb; ++rb)
        for (int64_t cg = rb * CGP_R; cg < ng; ++cg) {
            unsigned m = 0;
            for (int r = 0; r < CGP_R; ++r) {
                const int64_t rg = rb * CGP_R + r;
                if (rg < ng && ((pm.far_host[(size_t)rg * nbyte + cg / 8] >> (cg & 7)) & 1)) m |= 1u << r;
            }
            if (!m) continue;
            strip.push_back(make_int2((int)rb, (int)(cg | ((int64_t)m << 24))));
            cost.push_back((float)CGP_R);      // a strip costs its 4 patches whatever the mask (the near rows are computed and discarded)
        }
    // One CTA of 16 warps per SM -- fewer for small cavities, where an iteration is barrier and load latency rather than sweep:
    // a warp then gets at least CGP_MIN_PAIRS column pairs and the grid barriers have fewer arrivals (M = 247: 12 CTAs, 30.8 ->
    // 26.9 us per PCG iteration; M = 1 000: 50 CTAs, 33.8 -> 29.7; from 2 500 points on all SMs; 16 pairs per warp measured slower
    // at 2 500 points: 34.2 against 29.3 us).
    {
        const int64_t want = cdiv2(16 * (int64_t)strip.size(), (int64_t)CGP_WARPS * CGP_MIN_PAIRS);
        sp.grid = (int)std::min<int64_t>(ctx->sm_count, std::max<int64_t>(want, std::min<int64_t>(8, ctx->sm_count)));
        sp.nwarp = sp.grid * CGP_WARPS;
    }
    // near pieces go round-robin to the warps (piece q to warp q mod nwarp), before the far segment; their cost shortens it
    const double near_cost = 0.5;    // a stored near patch against a far patch, in warp time (PCM_VERBOSE prints the mean sweep
                                     // time of warps with / without a near piece: 0.3 left the near CTAs 1.8 us behind at M = 10k)
    std::vector<double> wnear((size_t)sp.nwarp, 0.0);
    for (int64_t q = 0; q < pm.npiece; ++q) {
        const int64_t rg = pm.piece_rg_host[q];
        const int64_t ebeg = pm.start_host[rg] + (q - pm.pstart_host[rg]) * NEAR_PIECE, eend = std::min(pm.start_host[rg + 1], ebeg + NEAR_PIECE);
        wnear[(size_t)(q % sp.nwarp)] += near_cost * (double)(eend - ebeg);
    }
    double total = 0.0;
    for (float c : cost) total += c;
    for (double c : wnear) total += c;
    const double target = total / sp.nwarp;
    // Segments in column PAIRS (2 columns against the 4 row groups, cost CGP_R / 16; pair h belongs to strip h >> 4): what one
    // pass of the sweep's inner loop does, so every warp gets its share to within one pass.  (Half strips as the unit left
    // warps with 10 or 11 of them at M = 10k, and the CTAs with the 11s finished 3 us after the others.)
    const int64_t nhalf = 2 * (int64_t)strip.size(), npair = 16 * (int64_t)strip.size();
    if (npair >= (int64_t)1 << 30) return PCM_OK;      // the sweep indexes pairs with 32-bit integers: the classic path takes over
    std::vector<int64_t> seg_start((size_t)sp.nwarp + 1, 0);
    {
        int64_t h = 0;
        double boundary = 0.0;
        const double pc = CGP_R / 16.0;
        for (int w = 0; w < sp.nwarp; ++w) {
            seg_start[w] = h;
            boundary += target - wnear[w];
            const int64_t to = w == sp.nwarp - 1 ? npair : std::min<int64_t>(npair, (int64_t)std::llround(boundary / pc));
            h = std::max(h, to);
        }
        seg_start[sp.nwarp] = npair;
    }
    // row-sum slots: one per (segment, row block) run, numbered in order (the slots of a row block are consecutive)
    std::vector<int32_t> seg_slot0((size_t)sp.nwarp + 1, 0), rb_slot_start((size_t)nrb + 1, 0);
    int32_t nslot = 0;
    {
        std::vector<int32_t> cnt((size_t)nrb, 0);
        for (int w = 0; w < sp.nwarp; ++w) {
            seg_slot0[w] = nslot;
            int last = -1;
            if (seg_start[w] < seg_start[w + 1])
                for (int64_t si = seg_start[w] >> 4; si <= (seg_start[w + 1] - 1) >> 4; ++si)
                    if (strip[(size_t)si].x != last) { last = strip[(size_t)si].x; ++nslot; ++cnt[last]; }
        }
        seg_slot0[sp.nwarp] = nslot;
        for (int64_t rb = 0; rb < nrb; ++rb) rb_slot_start[rb + 1] = rb_slot_start[rb] + cnt[rb];
    }
    sp.nslot = nslot;
    sp.nstrip = (int64_t)strip.size();
    // columns in the local coordinates of their group: (-2 (b - o), |b - o|^2), o = the group's first point
    std::vector<double4> pt((size_t)M), colloc((size_t)M), org((size_t)ng);
    PCM_CUDA(ctx, cudaMemcpy(pt.data(), ctx->pt, (size_t)M * sizeof(double4), cudaMemcpyDeviceToHost));
    for (int64_t j = 0; j < M; ++j) {
        const double4 o = pt[(size_t)(j & ~31LL)];
        if ((j & 31) == 0) org[(size_t)(j >> 5)] = o;
        const double x = pt[j].x - o.x, y = pt[j].y - o.y, z = pt[j].z - o.z;
        colloc[j] = make_double4(-2.0 * x, -2.0 * y, -2.0 * z, std::fma(z, z, std::fma(y, y, x * x)));
    }
    std::vector<CgpWarpInit> winit((size_t)sp.nwarp);
    {
        std::vector<int32_t> list_host((size_t)std::max<int64_t>(pm.nnear, 1), 0);
        if (pm.nnear > 0) PCM_CUDA(ctx, cudaMemcpy(list_host.data(), pm.list, (size_t)pm.nnear * sizeof(int32_t), cudaMemcpyDeviceToHost));
        for (int w = 0; w < sp.nwarp; ++w) {
            CgpWarpInit &wi = winit[(size_t)w];
            wi = CgpWarpInit{};
            wi.hb = seg_start[w]; wi.he = seg_start[w + 1];
            wi.slot0 = seg_slot0[w];
            if (wi.hb < wi.he) {
                const int64_t s0 = wi.hb >> 4, last = (wi.he - 1) >> 4;
                wi.strip0 = strip[(size_t)s0];
                wi.strip1 = s0 + 1 <= last ? strip[(size_t)s0 + 1] : make_int2(0, 0);
            }
            if (w < pm.npiece) {
                const int64_t rg = pm.piece_rg_host[(size_t)w];
                wi.ne = pm.start_host[rg] + (w - pm.pstart_host[rg]) * NEAR_PIECE;
                wi.ne_end = std::min(pm.start_host[rg + 1], wi.ne + NEAR_PIECE);
                wi.ncg0 = list_host[(size_t)wi.ne];
            }
        }
    }
    int rc;
    if ((rc = upload2(ctx, &sp.winit, winit))) return rc;
    if ((rc = upload2(ctx, &sp.strip, strip))) return rc;
    if ((rc = upload2(ctx, &sp.seg_start, seg_start))) return rc;
    if ((rc = upload2(ctx, &sp.seg_slot0, seg_slot0))) return rc;
    if ((rc = upload2(ctx, &sp.rb_slot_start, rb_slot_start))) return rc;
    if ((rc = upload2(ctx, &sp.colloc, colloc))) return rc;
    if ((rc = upload2(ctx, &sp.org, org))) return rc;
    if ((rc = dev_alloc_t(ctx, &sp.yslot, (size_t)std::max<int32_t>(nslot, 1) * CGP_ROWS))) return rc;
    if ((rc = dev_alloc_t(ctx, &sp.colpart, (size_t)nrb * (size_t)M))) return rc;
    if ((rc = dev_alloc_t(ctx, &sp.pbuf, (size_t)M))) return rc;
    // column sums of strips nobody sweeps (no far patch) are never written: they must read as zero
    PCM_CUDA(ctx, cudaMemset(sp.colpart, 0, (size_t)nrb * (size_t)M * 8));
    PCM_CUDA(ctx, cudaMemset(sp.yslot, 0, (size_t)std::max<int32_t>(nslot, 1) * CGP_ROWS * 8));
    sp.smem = smem;
    sp.ready = true;
    // The stored-A variant (PAPER.md:106 stores all of A): the far field kept as the sweep consumes it, 16 KB per half strip,
    // M^2/2 values in all.  It replaces ~9 FP64 instructions and a MUFU per pair by an 8-byte load, i.e. it trades the FP64 pipe
    // for memory bandwidth: from HBM that is a tie at best (4 M^2 bytes per product: 400 MB at M = 10k = 61 us at 6.5 TB/s
    // against ~59 us of arithmetic), from L2 it wins.  Rule (store_far = 0): store when the far field and the stored near
    // patches together stay resident in L2; store_far = 1 stores whenever memory allows (measurements), -1 never.
    {
        const double far_bytes = (double)nhalf * 16.0 * CGP_R * 32.0 * 8.0;
        const double near_bytes = ctx->amat_blocks ? (double)pm.nnear * 1024.0 * 8.0 : 0.0;
        const double l2_budget = 96e6;     // of the 126 MB L2: the vectors, partial sums and inverse blocks need room too
        size_t free_b = 0, total_b = 0;
        cudaMemGetInfo(&free_b, &total_b);
        const bool fits_mem = far_bytes < 0.5 * (double)free_b;
        const bool want = ctx->opt.store_far == 1 ? fits_mem : (ctx->opt.store_far == 0 && far_bytes + near_bytes <= l2_budget && fits_mem);
        sp.far_bytes = 0;
        if (want && nhalf > 0) {
            if ((rc = dev_alloc_t(ctx, &sp.afar, (size_t)nhalf * 16 * CGP_R * 32))) return rc;
            CgpArgs a = cgp_args(ctx);
            a.afar = sp.afar;
            a.q = sp.pbuf; a.qidx = nullptr; a.y = nullptr;     // any finite vector: only the 1/r values are kept
            PCM_CUDA(ctx, cudaMemset(sp.pbuf, 0, (size_t)M * 8));
            void *args[] = {&a};
            PCM_CUDA(ctx, cudaLaunchCooperativeKernel((const void *)cgp_matvec_kernel<1>, dim3((unsigned)sp.grid), dim3(CGP_THREADS), args, smem, 0));
            PCM_CUDA(ctx, cudaDeviceSynchronize());
            sp.far_bytes = (int64_t)far_bytes;
        }
    }
    if (getenv("PCM_VERBOSE")) {
        double mx = 0.0;
        for (int w = 0; w < sp.nwarp; ++w) {
            const double c = wnear[w] + CGP_R / 16.0 * (double)(seg_start[w + 1] - seg_start[w]);
            mx = std::max(mx, c);
        }
        int64_t partial = 0, pfar = 0, ffar = 0;
        for (size_t i = 0; i < strip.size(); ++i) {
            const unsigned m = (unsigned)strip[i].y >> 24;
            if (m != 15) { ++partial; pfar += __builtin_popcount(m); } else ffar += 4;
        }
        fprintf(stderr, "[pcm] sweep plan: %lld strips (%lld partial with %lld far patches, %lld far patches in full strips), %d warps, %d row slots, "
                "cost per warp %.2f (max %.2f), near pieces %lld\n", (long long)sp.nstrip, (long long)partial, (long long)pfar, (long long)ffar,
                sp.nwarp, nslot, target, mx, (long long)pm.npiece);
    }
    return PCM_OK;
}

static CgpArgs cgp_args(pcm_ctx *ctx) {
    const SweepPlan &sp = ctx->cgp;
    const PatchMap &pm = ctx->amat_map;
    CgpArgs a{};
    a.M = (int)ctx->M; a.ng = sp.ng; a.nrb = sp.nrb; a.nwarp = sp.nwarp;
    a.winit = sp.winit;
    a.pt = ctx->pt; a.colloc = sp.colloc; a.org = sp.org;
    a.strip = sp.strip; a.seg_start = sp.seg_start; a.seg_slot0 = sp.seg_slot0; a.rb_slot_start = sp.rb_slot_start;
    a.yslot = sp.yslot; a.colpart = sp.colpart;
    a.afar = sp.afar;
    a.nblk = ctx->amat_blocks; a.nstart = pm.start; a.npstart = pm.pstart; a.nlist = pm.list; a.npiece_rg = pm.piece_rg;
    a.npiece = pm.npiece; a.near = ctx->near_amat;
    a.diag = ctx->pt_diag;
    a.scal = ctx->cg_scal;
    a.ctl = reinterpret_cast<int *>(ctx->cg_scal + 8);
    return a;
}

// y = A q in one cooperative launch (q, y in the caller's order through idx, or sorted when idx == nullptr)
int cgp_matvec(pcm_ctx *ctx, const double *q, const int32_t *idx, double *y, cudaStream_t s) {
    CgpArgs a = cgp_args(ctx);
    a.q = q; a.qidx = idx; a.y = y;
    if (idx) {      // (pbuf is the solve's second direction vector: free between solves, calls on a context are stream-ordered)
        cgp_gather_kernel<<<(unsigned)cdiv2(a.M, 256), 256, 0, s>>>(q, idx, ctx->cgp.pbuf, a.M);
        a.q = ctx->cgp.pbuf;
        ctx->launch_total += 1;
    }
    // Two ordinary launches (sweep; row sums) instead of one cooperative launch with a grid barrier: a cooperative launch costs
    // ~20 us more between the events around it than its kernel runs (measured at M = 10k: 94 us against 72 us under ncu), which a
    // single A q does not win back; inside a solve the launch happens once, so pcm_cg_solve keeps the cooperative kernel.
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3(CGP_THREADS);
    cfg.stream = s;
    cfg.attrs = at;
    a.phase = 1;
    cfg.gridDim = dim3((unsigned)ctx->cgp.grid);
    cfg.dynamicSmemBytes = ctx->cgp.smem;
    cfg.numAttrs = idx ? 1 : 0;          // chained to the gather kernel, if there is one
    PCM_CUDA(ctx, cudaLaunchKernelEx(&cfg, a.afar ? cgp_matvec_kernel<2> : cgp_matvec_kernel<0>, a));
    a.phase = 2;
    cfg.gridDim = dim3((unsigned)std::max<int64_t>(1, std::min<int64_t>(cdiv2(a.ng, CGP_TEAMS), 4 * (int64_t)ctx->cgp.grid)));
    cfg.dynamicSmemBytes = CGP_WARPS * 32 * 8;
    cfg.numAttrs = 1;
    PCM_CUDA(ctx, cudaLaunchKernelEx(&cfg, cgp_matvec_kernel<0>, a));
    PCM_CUDA(ctx, cudaGetLastError());
    ctx->launch_total += 2;
    return PCM_OK;
}

// the iterations of a PCG solve: r (the initial residual), x, b are set by the caller (pcm_solver.cu); on return x is the
// solution, scal / ctl hold r.z, p.Ap, r.r, beta, the iteration count
int cgp_solve(pcm_ctx *ctx, double *r, double *z, double *p, double *Ap, double *x, double tol, int max_iter, int precond, cudaStream_t s) {
    CgpArgs a = cgp_args(ctx);
    a.precond = precond; a.max_iter = max_iter; a.tol = tol;
    a.block = (int)ctx->rbj_block; a.nblocks = (int)ctx->rbj_nblocks;
    a.order = ctx->rbj_order; a.inv = ctx->rbj_inv;
    a.r = r; a.z = z; a.p0 = p; a.p1 = ctx->cgp.pbuf; a.Ap = Ap; a.x = x;
    a.part1 = ctx->cg_part;
    a.part2 = precond == 2 ? ctx->rbj_partial : ctx->cg_scal + 16;
    size_t smem = ctx->cgp.smem;
    if (precond == 2) smem = std::max(smem, 2 * ((size_t)a.block + CGP_THREADS / 2) * 8);
    PCM_CUDA(ctx, cudaMemsetAsync(p, 0, (size_t)ctx->M * 8, s));                // beta = 0 on the first iteration: p = z + 0 * 0
    const bool verbose = getenv("PCM_VERBOSE") != nullptr;
    if (verbose) {
        PCM_CUDA(ctx, cudaMalloc(&a.dbg, (CGP_DBG_ITERS * 8 + 1024 + (size_t)a.nwarp) * 8));
        PCM_CUDA(ctx, cudaMemsetAsync(a.dbg, 0, (CGP_DBG_ITERS * 8 + 1024 + (size_t)a.nwarp) * 8, s));
    }
    void *args[] = {&a};
    const void *k = a.afar ? (const void *)cgp_solve_kernel<2> : (const void *)cgp_solve_kernel<0>;
    PCM_CUDA(ctx, cudaLaunchCooperativeKernel(k, dim3((unsigned)ctx->cgp.grid), dim3(CGP_THREADS), args, smem, s));
    ctx->launch_total += 1;
    if (verbose) {   // CTA 0's view of the phases: sweep, wait, row sums, wait, update, wait (microseconds)
        std::vector<unsigned long long> hv(CGP_DBG_ITERS * 8 + 1024 + (size_t)a.nwarp);
        unsigned long long *h = hv.data();
        PCM_CUDA(ctx, cudaMemcpyAsync(h, a.dbg, hv.size() * 8, cudaMemcpyDeviceToHost, s));
        PCM_CUDA(ctx, cudaStreamSynchronize(s));
        cudaFree(a.dbg);
        {
            double sn = 0.0, sf = 0.0, mx = 0.0;
            int64_t nn = 0, nf = 0;
            for (int w = 0; w < a.nwarp; ++w) {
                const double t = h[CGP_DBG_ITERS * 8 + 1024 + w] * 1e-3;
                mx = std::max(mx, t);
                if (w < a.npiece) { sn += t; ++nn; } else { sf += t; ++nf; }
            }
            fprintf(stderr, "[pcm] sweep time per warp (us): %lld warps with a near piece, mean %.1f; %lld without, mean %.1f; max %.1f\n", (long long)nn,
                    nn ? sn / nn : 0.0, (long long)nf, nf ? sf / nf : 0.0, mx);
        }
        {
            std::vector<double> t;
            for (int c = 0; c < ctx->cgp.grid && c < 1024; ++c) t.push_back(h[CGP_DBG_ITERS * 8 + c] * 1e-3);
            if (getenv("PCM_CTADUMP")) { for (size_t c = 0; c < t.size(); ++c) fprintf(stderr, "[cta] %zu %.2f\n", c, t[c]); }
            std::sort(t.begin(), t.end());
            if (!t.empty()) fprintf(stderr, "[pcm] sweep time per CTA (us): min %.1f p25 %.1f median %.1f p75 %.1f max %.1f\n", t.front(), t[t.size() / 4],
                                    t[t.size() / 2], t[3 * t.size() / 4], t.back());
        }
        for (int it = 1; it < CGP_DBG_ITERS && h[it * 8 + 6]; it += 3)
            fprintf(stderr, "[pcm] cg iteration %d (CTA 0, us): sweep %.1f wait %.1f rowsum %.1f wait %.1f update %.1f wait %.1f | total %.1f\n", it,
                    (h[it * 8 + 1] - h[it * 8]) * 1e-3, (h[it * 8 + 2] - h[it * 8 + 1]) * 1e-3, (h[it * 8 + 3] - h[it * 8 + 2]) * 1e-3,
                    (h[it * 8 + 4] - h[it * 8 + 3]) * 1e-3, (h[it * 8 + 5] - h[it * 8 + 4]) * 1e-3, (h[it * 8 + 6] - h[it * 8 + 5]) * 1e-3,
                    (h[it * 8] - h[(it - 1) * 8]) * 1e-3);
    }
    return PCM_OK;
}

bool cgp_can_solve(const pcm_ctx *ctx, int precond) {
    if (!ctx->cgp.ready) return false;
    if (precond == 2 && 2 * ((size_t)ctx->rbj_block + CGP_THREADS / 2) * 8 > 190 * 1024) return false;
    return true;
}

}  // namespace pcm
