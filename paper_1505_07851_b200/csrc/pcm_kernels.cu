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
#include <cstdlib>

#include "pcm_device.cuh"

namespace pcm {

constexpr int TPB = 128;   // threads per block of the hot kernels ("1 x 128", still a good size)
constexpr int SUB = 32;    // rows / columns per classified group
constexpr int PT_TILE = 256;  // surface points staged per shared-memory tile (Fock, A q): 8 groups = one byte of the far map

// ---------------------------------------------------------------------------------------------
// Blocking.  Every hot kernel is a "rows x columns" sweep: a thread keeps R row objects in registers (points for
// A q and the potential, Hermite products for Fock) and the column objects stream through shared memory, C per
// inner step, so that R*C independent evaluations are in flight per thread (instruction-level parallelism is what
// keeps the FP64 pipe busy; profiles/).  Rows and columns are sorted in space and cut into groups of 32; pcm_setup
// classified every (row group, column group) patch from the groups' bounding boxes (PatchMap).  The *main* kernels
// below run the far patches only, branch-free (derivatives of 1/R, no table, no exp); the *near* kernels further
// down run the remaining patches with the per-evaluation far/near switch.  Lane = row inside a group, so a warp
// holds R whole row groups and every skip/run decision is warp-uniform.
// ---------------------------------------------------------------------------------------------
struct Blocking { int R, C; };
// A q blocking (plan_all): R = 4 / tile 256 from AMAT_R4_MIN points on, R = 2 / tile 64 below
constexpr int AMAT_C = 2;
constexpr int64_t AMAT_R4_MIN = 20000;
__host__ __device__ constexpr Blocking fock_blocking(int L) {
    return L == 0 ? Blocking{4, 2} : L == 1 ? Blocking{2, 2} : L == 2 ? Blocking{1, 4} : Blocking{1, 2};
}
__host__ __device__ constexpr Blocking pot_blocking(int L) {
    return L == 0 ? Blocking{4, 2} : L == 1 ? Blocking{4, 1} : L == 2 ? Blocking{2, 2} : L == 3 ? Blocking{2, 2} : Blocking{1, 1};
}
// Large cavities (POT_BIG_MIN points and more) take twice the points per thread for L >= 2: the product record (14, 27, 39 doubles)
// is then read from shared memory once per 4 (2) evaluations instead of 2 (1) -- every load is an issue slot the FP64 pipe does
// not get -- at the price of half as many point blocks, which small cavities cannot afford (configs[1], L = 2: 0.186 -> 0.223 ms;
// configs[3]: 24.3 -> 23.6, 11.2 -> 11.05, 4.51 -> 4.43 ms for L = 2, 3, 4).
constexpr int64_t POT_BIG_MIN = 40000;
__host__ __device__ constexpr Blocking pot_blocking_big(int L) {
    return L <= 1 ? pot_blocking(L) : L <= 3 ? Blocking{4, 1} : Blocking{2, 1};
}
__host__ __device__ constexpr int pot_tile(int L) { return L <= 2 ? 256 : 64; }  // products staged per tile (8 or 2 groups)

// ---- programmatic dependent launch (PTX griddepcontrol, sm_90+) -----------------------------------------------------------
// The class kernels of one call are independent of one another, but each is only a few waves long at small and medium sizes
// and its last wave leaves most of the SMs idle (PAPER.md:160 launches its per-class kernels one after the other).  A class
// kernel therefore signals at its very start that the next launch of the stream may be scheduled, and a kernel launched with
// the programmatic-serialization attribute (launch_class below) begins as soon as every CTA of its predecessor has started,
// i.e. it fills the SM slots the predecessor's last wave leaves free.  Before it exits, each of its CTAs waits for the
// predecessor to have completed, so that completion stays in launch order and the ordinary launch that follows the chain
// (the reduction) sees all of it.  Both instructions do nothing in a kernel launched the ordinary way.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait_predecessor() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// far bits of the R row groups of this warp for the NS column groups starting at column group cg0 (cg0 % NS == 0,
// NS = 8 or 2): bit (r * 8 + s) = patch (row group rg0 + r, column group cg0 + s) is far.  Warp-uniform result.
template <int R, int NS>
__device__ __forceinline__ unsigned far_bits(const uint8_t *__restrict__ farmap, int64_t nbyte, int64_t rg0, int64_t nrg,
                                             int64_t cg0, int lane) {
    unsigned mine = 0;
    if (lane < R && rg0 + lane < nrg) mine = farmap[(rg0 + lane) * nbyte + (cg0 >> 3)];
    mine = (mine >> (cg0 & 7)) & ((1u << NS) - 1u);
    unsigned bits = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) bits |= __shfl_sync(0xffffffffu, mine, r) << (8 * r);
    return bits;
}
// rows of the warp that are far from column group s: bit r
template <int R>
__device__ __forceinline__ unsigned row_mask(unsigned bits, int s) {
    unsigned m = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) m |= ((bits >> (8 * r + s)) & 1u) << r;
    return m;
}

// ---------------------------------------------------------------------------------------------
// a4: y = A q on the fly (Eq. 2, 3, 8).  Rows = points i (registers), columns = points j (shared memory).
//   far (zeta'^2 r^2 >= 38, erf = 1 to fp64):  A_ij = 1/r                       -- 12 FP64 instructions + MUFU
//   general:  A_ij = (2 zeta'/sqrt pi) F_0(zeta'^2 r^2), zeta'^2 = 1/(1/zeta_i^2 + 1/zeta_j^2); A_ii from pt_diag
// q is read through qidx (sorted -> caller index) when qidx != nullptr; the partial sums are in sorted order.
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

// stages the points [base, base + nst*32) of the chunk ending at jend as (x, y, z, charge)
__device__ __forceinline__ void stage_points(const double4 *__restrict__ pt, const double *__restrict__ q,
                                             const int32_t *__restrict__ qidx, int base, int jend, int nst, double4 *s_pt) {
    for (int t = threadIdx.x; t < nst * SUB; t += TPB) {
        const int j = base + t;
        if (j < jend) {
            const double4 b = pt[j];
            s_pt[t] = make_double4(b.x, b.y, b.z, q[qidx ? qidx[j] : j]);
        } else {  // padding: far from everything, zero charge (its patch bit is never set anyway)
            s_pt[t] = make_double4(3e8, 3e8, 3e8, 0.0);
        }
    }
}

// The stored near patches (amat_near_fill_kernel below) as the main kernel sees them: when `blocks` is set, the grid of
// amatvec_kernel is extended by rows of CTAs (blockIdx.y >= chunks) that do the near pieces, four per CTA, so that one
// launch does the whole product and the light, memory-bound near work fills the tail of the sweep.
struct NearStored {
    const double *blocks;        // [nnear][32][32], nullptr: the near pieces are done by a separate kernel
    const int64_t *start, *pstart;
    const int32_t *list, *piece_rg;
    int64_t npiece;
    double *near;                // [npiece][32]
};
// near[piece][lane] = sum over the piece's patches (list order) of sum_t A(lane, t) q_t (t ascending)
__device__ __forceinline__ void amat_near_stored_piece(const NearStored &ns, const double *__restrict__ q,
                                                       const int32_t *__restrict__ qidx, int M, int64_t piece, int lane) {
    const int64_t rg = ns.piece_rg[piece];
    const int64_t ebeg = ns.start[rg] + (piece - ns.pstart[rg]) * NEAR_PIECE, eend = min(ns.start[rg + 1], ebeg + NEAR_PIECE);
    double y = 0.0;
    for (int64_t e = ebeg; e < eend; ++e) {
        const int j = ns.list[e] * SUB + lane;
        const double qj = j < M ? q[qidx ? qidx[j] : j] : 0.0;
        const double *blk = ns.blocks + (size_t)e * (SUB * SUB) + lane;
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            double a[16];
#pragma unroll
            for (int t = 0; t < 16; ++t) a[t] = __ldg(blk + (half * 16 + t) * SUB);
#pragma unroll
            for (int t = 0; t < 16; ++t) y = fma(__shfl_sync(0xffffffffu, qj, half * 16 + t), a[t], y);
        }
    }
    ns.near[piece * SUB + lane] = y;
}

// Symmetric sweep: A_ij = A_ji, so an evaluation 1/r_ij serves row i (y_i += q_j/r) and column j (y_j += q_i/r).
// Block (rb, chunk) owns the rows [rb RB, (rb+1) RB), RB = TPB R, and the column tiles of its chunk that do not lie
// before its rows:  tiles inside the row range (the diagonal band) are swept for the rows only; tiles beyond it are
// swept once for both triangles.  Row sums go to out[chunk][i] (only chunks that reach the row's block are written),
// column sums to colpart[rb][j] (only the row blocks before the tile of j); amat_row_sum_block adds them in a fixed order.
// Column sums: a lane adds its R rows in registers, the 32 lanes are then summed through a [16][33] shared-memory
// transpose per warp (one DADD per column and lane), the 4 warps at the end of the tile.
//
// Geometry in local coordinates: the 32 columns of a group are staged relative to their first point o as
// (-2 (b - o), |b - o|^2), a row is shifted once per group (a - o, |a - o|^2: 6 instructions per 32 evaluations),
// and r^2 = |a - o|^2 + |b - o|^2 - 2 (a - o).(b - o) costs 1 DADD + 3 DFMA instead of 3 DADD + DMUL + 2 DFMA.  |b - o| is
// the extent of 32 neighbouring points and far patches are further apart than that, so the cancellation costs a few ulp
// of r^2 (<= 20 eps for a gap of 2 bohr and an extent of 3.5).  Per evaluation 11.4 FP64 instructions (R = 4) for two
// entries of A: geometry 4 + 3/16, rsqrt 5, two FMAs, 1/R DADD of the column reduction.
__device__ __forceinline__ double r2_local(double alx, double aly, double alz, double a2, const double4 &b) {
    return fma(alx, b.x, fma(aly, b.y, fma(alz, b.z, a2 + b.w)));
}

// stages the columns [base, base + nst*32) of the chunk ending at jend: s_pt = (-2 (b - o), |b - o|^2), s_q = charge,
// s_org[g] = origin o of column group g (its first point).
// Padding columns sit on the origin with zero charge.
__device__ __forceinline__ void stage_points_local(const double4 *__restrict__ pt, const double *__restrict__ q,
                                                   const int32_t *__restrict__ qidx, int base, int jend, int nst, double4 *s_pt,
                                                   double *s_q, double4 *s_org) {
    for (int t = threadIdx.x; t < nst * SUB; t += TPB) {
        const int j = base + t, jo = min(base + (t & ~31), jend - 1);
        const double4 o = pt[jo];
        if ((t & 31) == 0) s_org[t >> 5] = o;
        if (j < jend) {
            const double4 b = pt[j];
            const double x = b.x - o.x, y = b.y - o.y, z = b.z - o.z;
            s_pt[t] = make_double4(-2.0 * x, -2.0 * y, -2.0 * z, fma(z, z, fma(y, y, x * x)));
            s_q[t] = q[qidx ? qidx[j] : j];
        } else {
            s_pt[t] = make_double4(0.0, 0.0, 0.0, 0.0);
            s_q[t] = 0.0;
        }
    }
}

template <int R, int C, int TILE>
__global__ void __launch_bounds__(TPB) amatvec_kernel(const double4 *__restrict__ pt, const double *__restrict__ q,
                                                      const int32_t *__restrict__ qidx, int M, int chunk_len,
                                                      double *__restrict__ out, double *__restrict__ colpart,
                                                      const uint8_t *__restrict__ farmap, int64_t nbyte, int64_t nrg,
                                                      const int *__restrict__ stop, int chunks, NearStored ns) {
    constexpr int NS = TILE / SUB;
    constexpr int RB = TPB * R;
    constexpr int NW = TPB / 32;
    static_assert(RB % TILE == 0, "row blocks must be whole column tiles");
    if ((int)blockIdx.y >= chunks) {   // the extra rows of the grid: stored near pieces, one per warp
        if (stop && *stop) return;
        const int64_t piece = ((int64_t)(blockIdx.y - chunks) * gridDim.x + blockIdx.x) * NW + (threadIdx.x >> 5);
        if (piece < ns.npiece) amat_near_stored_piece(ns, q, qidx, M, piece, threadIdx.x & 31);
        return;
    }
    __shared__ double4 s_pt[TILE];          // -2 (b - o), |b - o|^2
    __shared__ double s_q[TILE];            // column charges
    __shared__ double4 s_org[TILE / 32];    // origin of every column group
    __shared__ double s_c[NW][16 * 33];     // per warp: [column of the half group][lane]
    __shared__ double s_cs[NW][TILE];       // per warp: column sums of the tile
    if (stop && *stop) return;  // a converged CG solve: the iterations queued behind it are no-ops
    const int r0 = blockIdx.x * RB;
    const int jbeg = blockIdx.y * chunk_len, jend = min(M, jbeg + chunk_len);
    if (jend <= r0) return;     // the chunk lies before the rows: the blocks of those rows cover it
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t rg0 = ((int64_t)blockIdx.x * NW + warp) * R;
    double qa[R], y[R], ax[R], ay[R], az[R];
    int ii[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        ii[r] = (int)(rg0 + r) * SUB + lane;
        qa[r] = ii[r] < M ? q[qidx ? qidx[ii[r]] : ii[r]] : 0.0;   // padding rows: zero charge, their sums are not stored
        const double4 a = pt[min(ii[r], M - 1)];
        ax[r] = ii[r] < M ? a.x : a.x + 3e8; ay[r] = a.y; az[r] = a.z;   // padding rows: far away
        y[r] = 0.0;
    }
    double *sc = s_c[warp];
    for (int base = max(jbeg, r0); base < jend; base += TILE) {
        const int nst = (min(TILE, jend - base) + SUB - 1) / SUB;
        const bool sym = base >= r0 + RB;
        const unsigned bits = far_bits<R, NS>(farmap, nbyte, rg0, nrg, base / SUB, lane);
        __syncthreads();
        stage_points_local(pt, q, qidx, base, jend, nst, s_pt, s_q, s_org);
        __syncthreads();
        for (int st = 0; st < nst; ++st) {
            const unsigned m = row_mask<R>(bits, st);
            if (m == 0) {
                if (sym) s_cs[warp][st * SUB + lane] = 0.0;
                continue;
            }
            // the rows of this thread relative to the column group's origin
            const double4 o = s_org[st];
            double alx[R], aly[R], alz[R], a2[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                alx[r] = ax[r] - o.x; aly[r] = ay[r] - o.y; alz[r] = az[r] - o.z;
                a2[r] = fma(alz[r], alz[r], fma(aly[r], aly[r], alx[r] * alx[r]));
            }
#pragma unroll 1
            for (int half = 0; half < 2; ++half) {
                const double4 *sp = s_pt + st * SUB + half * 16;
                const double *sq = s_q + st * SUB + half * 16;
                if (m == (1u << R) - 1u) {
#pragma unroll 1
                    for (int t = 0; t < 16; t += C) {
                        double4 b[C];
                        double qb[C], r2[C][R], cc[C];
#pragma unroll
                        for (int c = 0; c < C; ++c) { b[c] = sp[t + c]; qb[c] = sq[t + c]; }
#pragma unroll
                        for (int c = 0; c < C; ++c)
#pragma unroll
                            for (int r = 0; r < R; ++r) r2[c][r] = r2_local(alx[r], aly[r], alz[r], a2[r], b[c]);
#pragma unroll
                        for (int c = 0; c < C; ++c) {
                            cc[c] = 0.0;
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                const double rs = rsqrt_fast(r2[c][r]);
                                y[r] = fma(qb[c], rs, y[r]);
                                cc[c] = fma(qa[r], rs, cc[c]);
                            }
                            if (sym) sc[(t + c) * 33 + lane] = cc[c];
                        }
                    }
                } else {
#pragma unroll 1
                    for (int t = 0; t < 16; ++t) {
                        const double4 b = sp[t];
                        const double qb = sq[t];
                        double cc = 0.0;
#pragma unroll
                        for (int r = 0; r < R; ++r)
                            if ((m >> r) & 1u) {
                                const double rs = rsqrt_fast(r2_local(alx[r], aly[r], alz[r], a2[r], b));
                                y[r] = fma(qb, rs, y[r]);
                                cc = fma(qa[r], rs, cc);
                            }
                        if (sym) sc[t * 33 + lane] = cc;
                    }
                }
                if (sym) {
                    __syncwarp();
                    // lane l sums column (l & 15) over the lanes [16 (l >> 4), 16 (l >> 4) + 16), fixed order
                    const double *col = sc + (lane & 15) * 33 + (lane >> 4) * 16;
                    double s = col[0];
#pragma unroll
                    for (int k = 1; k < 16; ++k) s += col[k];
                    const double o2 = __shfl_xor_sync(0xffffffffu, s, 16);
                    if (lane < 16) s_cs[warp][st * SUB + half * 16 + lane] = s + o2;
                    __syncwarp();
                }
            }
        }
        if (sym) {
            __syncthreads();
            for (int t = threadIdx.x; t < nst * SUB; t += TPB) {
                const int j = base + t;
                double s = s_cs[0][t];
#pragma unroll
                for (int w2 = 1; w2 < NW; ++w2) s += s_cs[w2][t];
                if (j < M) colpart[(size_t)blockIdx.x * M + j] = s;
            }
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r)
        if (ii[r] < M) out[(size_t)blockIdx.y * M + ii[r]] = y[r];
}

// near patches of A q: one warp per piece (<= NEAR_PIECE listed patches of one row group); lane = row; the 32 columns
// of a listed group are staged in the warp's own shared memory.  Writes near[piece][lane].
__global__ void __launch_bounds__(TPB) amat_near_kernel(const double4 *__restrict__ pt, const double *__restrict__ diag,
                                                        const double *__restrict__ q, const int32_t *__restrict__ qidx, int M,
                                                        const int64_t *__restrict__ start, const int32_t *__restrict__ list,
                                                        const int64_t *__restrict__ pstart, const int32_t *__restrict__ piece_rg,
                                                        int64_t npiece, double *__restrict__ near,
                                                        const double *__restrict__ boys0, double thr,
                                                        const int *__restrict__ stop) {
    __shared__ double4 s_pt[TPB / 32][SUB];
    __shared__ double s_iz[TPB / 32][SUB];
    if (stop && *stop) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t piece = (int64_t)blockIdx.x * (TPB / 32) + warp;
    if (piece >= npiece) return;
    const int64_t rg = piece_rg[piece];
    const int i = (int)rg * SUB + lane;
    const double4 a = pt[min(i, M - 1)];
    const int thr_hi = hi32(thr);
    const int64_t ebeg = start[rg] + (piece - pstart[rg]) * NEAR_PIECE, eend = min(start[rg + 1], ebeg + NEAR_PIECE);
    double y = 0.0;
    for (int64_t e = ebeg; e < eend; ++e) {
        const int j0 = list[e] * SUB, j = j0 + lane;
        __syncwarp();
        if (j < M) {
            const double4 b = pt[j];
            s_pt[warp][lane] = make_double4(b.x, b.y, b.z, q[qidx ? qidx[j] : j]);
            s_iz[warp][lane] = b.w;
        } else {
            s_pt[warp][lane] = make_double4(3e8, 3e8, 3e8, 0.0);
            s_iz[warp][lane] = 1.0;
        }
        __syncwarp();
#pragma unroll 2
        for (int t = 0; t < SUB; ++t) {
            const double4 b = s_pt[warp][t];
            const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            double ev;
            if (hi32(r2) > thr_hi) ev = rsqrt_fast(r2);
            else ev = (j0 + t == i) ? diag[i] : amat_general(r2, a.w, s_iz[warp][t], boys0);
            y = fma(b.w, ev, y);
        }
    }
    near[piece * SUB + lane] = y;
}

// Stored near field (the paper stores all of A; here only the patches that are not far are kept, which is
// what fits and what pays: they are the entries that need erf).  A depends on the geometry only, so pcm_setup evaluates
// every listed patch once -- with the same arithmetic as amat_near_kernel -- into blocks[e][t][lane] = A(row lane of the
// row group, column t of column group list[e]); entries of rows or columns beyond M are 0.
__global__ void __launch_bounds__(TPB) amat_near_fill_kernel(const double4 *__restrict__ pt, const double *__restrict__ diag, int M,
                                                             const int64_t *__restrict__ start, const int32_t *__restrict__ list,
                                                             const int64_t *__restrict__ pstart, const int32_t *__restrict__ piece_rg,
                                                             int64_t npiece, double *__restrict__ blocks,
                                                             const double *__restrict__ boys0, double thr) {
    __shared__ double4 s_pt[TPB / 32][SUB];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t piece = (int64_t)blockIdx.x * (TPB / 32) + warp;
    if (piece >= npiece) return;
    const int64_t rg = piece_rg[piece];
    const int i = (int)rg * SUB + lane;
    const double4 a = pt[min(i, M - 1)];
    const int thr_hi = hi32(thr);
    const int64_t ebeg = start[rg] + (piece - pstart[rg]) * NEAR_PIECE, eend = min(start[rg + 1], ebeg + NEAR_PIECE);
    for (int64_t e = ebeg; e < eend; ++e) {
        const int j0 = list[e] * SUB, j = j0 + lane;
        __syncwarp();
        s_pt[warp][lane] = pt[min(j, M - 1)];
        __syncwarp();
        double *blk = blocks + (size_t)e * (SUB * SUB);
        for (int t = 0; t < SUB; ++t) {
            const double4 b = s_pt[warp][t];
            const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            double ev;
            if (i >= M || j0 + t >= M) ev = 0.0;
            else if (hi32(r2) > thr_hi) ev = rsqrt_fast(r2);
            else ev = (j0 + t == i) ? diag[i] : amat_general(r2, a.w, b.w, boys0);
            blk[t * SUB + lane] = ev;
        }
    }
}

// sums of the near pieces, per class: near[c][piece][lane], pieces of row group rg = pstart[c][rg] .. pstart[c][rg+1]
struct NearRefs {
    const double *near[MAXL + 1];
    const int64_t *pstart[MAXL + 1];
    int count;
};
// out[idx ? idx[k] : k] = sum_slots part[slot][k] + sum of the near pieces of row k.  A 256-thread block sums 32 rows:
// warp w adds every 8th slot (and every 8th near piece of every class) for row lane, coalesced across the lanes; the
// eight partial sums are then added in order.  Fixed order, so the result is bit-reproducible.
__global__ void __launch_bounds__(256) reduce_slots_kernel(const double *__restrict__ part, int64_t n, int slots,
                                                           double *__restrict__ out, const int32_t *__restrict__ idx, NearRefs nr) {
    __shared__ double s_tmp[8 * 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t k = (int64_t)blockIdx.x * 32 + lane;
    double s = 0.0;
    if (k < n) {
        for (int c = w; c < slots; c += 8) s += part[(size_t)c * n + k];
        const int64_t rg = k / SUB;
        for (int c = 0; c < nr.count; ++c)
            for (int64_t q = nr.pstart[c][rg] + w; q < nr.pstart[c][rg + 1]; q += 8) s += nr.near[c][q * SUB + lane];
    }
    s_tmp[w * 32 + lane] = s;
    __syncthreads();
    if (w == 0 && k < n) {
        double t = 0.0;
#pragma unroll
        for (int q = 0; q < 8; ++q) t += s_tmp[q * 32 + lane];
        out[idx ? idx[k] : k] = t;
    }
}

// y[idx ? idx[k] : k] = the partial sums of row k of the symmetric A q sweep, in amat_row_sum's fixed order
__global__ void __launch_bounds__(256) amat_reduce_kernel(AmatParts parts, int M, double *__restrict__ out, const int32_t *__restrict__ idx) {
    __shared__ double s_tmp[AMAT_RED_PARTS * 32];
    const double t = amat_row_sum_block(parts, M, blockIdx.x * 32, s_tmp);
    const int k = blockIdx.x * 32 + threadIdx.x;
    if (threadIdx.x < 32 && k < M) out[idx ? idx[k] : k] = t;
}
AmatParts amat_parts(const pcm_ctx *ctx) {
    AmatParts a;
    a.ypart = ctx->ypart; a.colpart = ctx->colpart; a.near = ctx->near_amat; a.pstart = ctx->amat_map.pstart;
    a.slots = (int)ctx->plan_amat.chunks; a.chunk_len = (int)ctx->plan_amat.chunk_len; a.RB = TPB * ctx->amat_R; a.tile = ctx->amat_tile;
    return a;
}

// ---------------------------------------------------------------------------------------------
// a3 main kernel: H_h(product) = sum_k q_k Rt_h(P - C_k).  Rows = R products per thread (R NHERM(L) register
// accumulators), columns = surface points (shared memory), C points per step.
// ---------------------------------------------------------------------------------------------
template <int L>
struct FockSink {
    static constexpr bool kSplit = false;
    __device__ __forceinline__ void lower(int, double) {}
    double acc[nherm(L)];
    __device__ __forceinline__ void value(int h, int, int, int, double v) { acc[h] += v; }
    __device__ __forceinline__ void product(int h, int, int, int, double a, double b) { acc[h] = fma(a, b, acc[h]); }
};

// The main Fock sweep accumulates the order-0 integrals in two parts: R_h = c R^1_h1 + (pw - 1) R^1_h2 (the last recursion step,
// pw = the power being lowered).  acc_h takes the first term by FMA; the second terms of all components are multiples of the
// few R^1_h2 with degree(h2) <= L - 2 (g_1 alone for L = 2; g_1, x g_2, y g_2, z g_2 for L = 3), which are summed once per
// evaluation into accL and added to the components at the end of the kernel (hermite_fixup): 3 -> 1 additions per evaluation
// at L = 2, 12 -> 4 at L = 3.  Another (still fixed) summation order than FockSink's.
constexpr int FOCK_SPLIT_MAXL = 4;      // L = 5 (gradient of the dd class): 216 registers with it
template <int L>
struct FockSinkSplit {
    static constexpr bool kSplit = (L >= 2 && L <= FOCK_SPLIT_MAXL);
    double acc[nherm(L)];
    double accL[nherm(L >= 2 ? L - 2 : 0)];
    __device__ __forceinline__ void value(int h, int, int, int, double v) { acc[h] += v; }
    __device__ __forceinline__ void product(int h, int, int, int, double a, double b) { acc[h] = fma(a, b, acc[h]); }
    __device__ __forceinline__ void lower(int h2, double v) { accL[h2] += v; }
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int h = 0; h < nherm(L); ++h) acc[h] = 0.0;
#pragma unroll
        for (int h = 0; h < nherm(L >= 2 ? L - 2 : 0); ++h) accL[h] = 0.0;
    }
    __device__ __forceinline__ void finish() {
        if (kSplit) hermite_fixup<L>(acc, accL);
    }
};

template <int L, class Sink>
__device__ __forceinline__ void fock_far_unit(const double4 &A, const double4 &pc, Sink &sink) {
    const double x = A.x - pc.x, y = A.y - pc.y, z = A.z - pc.z;
    double g[L + 1];
    seeds_far_scaled<L>(fma(z, z, fma(y, y, x * x)), pc.w, g);
    hermite_R<L>(x, y, z, g, sink);
}

template <int L, int R, int C>
__global__ void __launch_bounds__(TPB) fock_kernel(const double4 *__restrict__ prodA, int64_t npad,
                                                   const double4 *__restrict__ pt, const double *__restrict__ q,
                                                   const int32_t *__restrict__ qidx, int M, int chunk_len,
                                                   double *__restrict__ herm, const uint8_t *__restrict__ farmap,
                                                   int64_t nbyte, int64_t nrg) {
    constexpr int NH = nherm(L);
    constexpr int NS = PT_TILE / SUB;
    __shared__ double4 s_pt[PT_TILE];  // x, y, z, q
    pdl_launch_dependents();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t rg0 = ((int64_t)blockIdx.x * (TPB / 32) + warp) * R;
    double4 A[R];
    FockSinkSplit<L> sink[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        A[r] = prodA[min((rg0 + r) * SUB + lane, npad - 1)];
        sink[r].clear();
    }
    const int kbeg = blockIdx.y * chunk_len, kend = min(M, kbeg + chunk_len);
    for (int base = kbeg; base < kend; base += PT_TILE) {
        const int nst = (min(PT_TILE, kend - base) + SUB - 1) / SUB;
        const unsigned bits = far_bits<R, NS>(farmap, nbyte, rg0, nrg, base / SUB, lane);
        __syncthreads();
        stage_points(pt, q, qidx, base, kend, nst, s_pt);
        __syncthreads();
        for (int st = 0; st < nst; ++st) {
            const double4 *sp = s_pt + st * SUB;
            const unsigned m = row_mask<R>(bits, st);
            if (m == (1u << R) - 1u) {
#pragma unroll 1
                for (int t = 0; t < SUB; t += C) {
#pragma unroll
                    for (int c = 0; c < C; ++c) {
                        const double4 pc = sp[t + c];
#pragma unroll
                        for (int r = 0; r < R; ++r) fock_far_unit<L>(A[r], pc, sink[r]);
                    }
                }
            } else if (R > 1 && m) {
#pragma unroll 1
                for (int t = 0; t < SUB; ++t) {
                    const double4 pc = sp[t];
#pragma unroll
                    for (int r = 0; r < R; ++r)
                        if ((m >> r) & 1u) fock_far_unit<L>(A[r], pc, sink[r]);
                }
            }
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        sink[r].finish();
        const int64_t ip = (rg0 + r) * SUB + lane;
        if (ip < npad) {
            double *out = herm + (size_t)blockIdx.y * NH * npad + ip;
#pragma unroll
            for (int h = 0; h < NH; ++h) out[(size_t)h * npad] = sink[r].acc[h];
        }
    }
    pdl_wait_predecessor();
}

// ---- the same sweep with the point tiles brought in by the TMA unit (cp.async.bulk, 1-D) --------------------------------
// north_star: "surface-point tiles staged in shared memory (TMA where tiles are regular)".  The tiles become regular once
// the charges are gathered into the library's sorted point order and packed with the coordinates, ptq[k] = (x, y, z, q_k)
// (pack_points_kernel, M x 32 B per call): a tile is then 256 x 32 B = 8 KB of contiguous memory.  One elected thread issues
// the bulk copy of tile i + 1 into the other buffer while the CTA computes on tile i; completion is an mbarrier transaction
// count, so the two __syncthreads() per tile of fock_kernel become one (the buffer hand-back) plus the mbarrier wait.
// Selected by pcm_options.tma_tiles (measured against fock_kernel: DESIGN.md "Tried").
__global__ void pack_points_kernel(const double4 *__restrict__ pt, const double *__restrict__ q, const int32_t *__restrict__ qidx, int M,
                                   double4 *__restrict__ ptq) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= M) return;
    const double4 p = pt[k];
    ptq[k] = make_double4(p.x, p.y, p.z, q[qidx ? qidx[k] : k]);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void tma_load_1d(void *dst, const void *src, unsigned bytes, uint64_t *bar) {
    const unsigned b = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     (unsigned)__cvta_generic_to_shared(dst)),
                 "l"(src), "r"(bytes), "r"(b)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
    const unsigned b = (unsigned)__cvta_generic_to_shared(bar);
    unsigned done = 0;
    while (!done) {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done) : "r"(b), "r"(parity) : "memory");
    }
}

template <int L, int R, int C>
__global__ void __launch_bounds__(TPB) fock_tma_kernel(const double4 *__restrict__ prodA, int64_t npad, const double4 *__restrict__ ptq, int M,
                                                       int chunk_len, double *__restrict__ herm, const uint8_t *__restrict__ farmap,
                                                       int64_t nbyte, int64_t nrg) {
    constexpr int NH = nherm(L);
    constexpr int NS = PT_TILE / SUB;
    __shared__ __align__(128) double4 s_pt[2][PT_TILE];  // x, y, z, q
    __shared__ __align__(8) uint64_t s_bar[2];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t rg0 = ((int64_t)blockIdx.x * (TPB / 32) + warp) * R;
    double4 A[R];
    FockSinkSplit<L> sink[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        A[r] = prodA[min((rg0 + r) * SUB + lane, npad - 1)];
        sink[r].clear();
    }
    const int kbeg = blockIdx.y * chunk_len, kend = min(M, kbeg + chunk_len);
    if (threadIdx.x == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0 && kbeg < kend) tma_load_1d(s_pt[0], ptq + kbeg, (unsigned)min(PT_TILE, kend - kbeg) * 32u, &s_bar[0]);
    int it = 0;
    for (int base = kbeg; base < kend; base += PT_TILE, ++it) {
        const int buf = it & 1;
        const int cnt = min(PT_TILE, kend - base), nst = (cnt + SUB - 1) / SUB;
        const unsigned bits = far_bits<R, NS>(farmap, nbyte, rg0, nrg, base / SUB, lane);
        // the next tile into the other buffer (every thread left it at the __syncthreads() that closed the previous tile)
        if (threadIdx.x == 0 && base + PT_TILE < kend)
            tma_load_1d(s_pt[buf ^ 1], ptq + base + PT_TILE, (unsigned)min(PT_TILE, kend - base - PT_TILE) * 32u, &s_bar[buf ^ 1]);
        mbar_wait(&s_bar[buf], (unsigned)(it >> 1) & 1u);
        if (cnt < nst * SUB) {     // ragged last group: padding points far from everything, zero charge
            for (int t = cnt + threadIdx.x; t < nst * SUB; t += TPB) s_pt[buf][t] = make_double4(3e8, 3e8, 3e8, 0.0);
            __syncthreads();
        }
        for (int st = 0; st < nst; ++st) {
            const double4 *sp = s_pt[buf] + st * SUB;
            const unsigned m = row_mask<R>(bits, st);
            if (m == (1u << R) - 1u) {
#pragma unroll 1
                for (int t = 0; t < SUB; t += C) {
#pragma unroll
                    for (int c = 0; c < C; ++c) {
                        const double4 pc = sp[t + c];
#pragma unroll
                        for (int r = 0; r < R; ++r) fock_far_unit<L>(A[r], pc, sink[r]);
                    }
                }
            } else if (R > 1 && m) {
#pragma unroll 1
                for (int t = 0; t < SUB; ++t) {
                    const double4 pc = sp[t];
#pragma unroll
                    for (int r = 0; r < R; ++r)
                        if ((m >> r) & 1u) fock_far_unit<L>(A[r], pc, sink[r]);
                }
            }
        }
        __syncthreads();           // this buffer may be refilled from now on
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        sink[r].finish();
        const int64_t ip = (rg0 + r) * SUB + lane;
        if (ip < npad) {
            double *out = herm + (size_t)blockIdx.y * NH * npad + ip;
#pragma unroll
            for (int h = 0; h < NH; ++h) out[(size_t)h * npad] = sink[r].acc[h];
        }
    }
}

// near patches of the Fock sweep: one CTA per piece (<= NEAR_PIECE listed point groups of one product group); lane = product;
// warp w takes the points [8 w, 8 w + 8) of every listed group, so a piece is four chains of <= 32 evaluations instead of one
// of <= 128 (the kernel is latency-bound: at 300 atoms its grid was one wave of warps that each ran 128 evaluations in series,
// 17 - 47 % of the warp slots occupied).  The four partial sums are added in warp order.  Writes near[piece][h][lane].
constexpr int NEAR_WARPS = TPB / 32;                 // warps that share a piece
constexpr int NEAR_PER = SUB / NEAR_WARPS;           // listed entries of a patch per warp
static_assert(NEAR_PIECE * NEAR_PER <= SUB, "a warp stages its share of a piece in one pass, one record per lane");
template <int L>
__global__ void __launch_bounds__(TPB) fock_near_kernel(const double4 *__restrict__ prodA, const double2 *__restrict__ prodB,
                                                        int64_t npad, const double4 *__restrict__ pt, const double *__restrict__ q,
                                                        const int32_t *__restrict__ qidx, int M, const int64_t *__restrict__ start,
                                                        const int32_t *__restrict__ list, const int64_t *__restrict__ pstart,
                                                        const int32_t *__restrict__ piece_rg, int64_t npiece,
                                                        double *__restrict__ near, const double *__restrict__ boysL) {
    constexpr int NH = nherm(L);
    __shared__ double4 s_pt[NEAR_WARPS][SUB];
    __shared__ double s_iz[NEAR_WARPS][SUB];
    __shared__ double s_sum[NEAR_WARPS - 1][NH * SUB];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t piece = blockIdx.x;
    const int64_t rg = piece_rg[piece];
    const int64_t ip = rg * SUB + lane;  // < npad (npad is a multiple of 32)
    const double4 A = prodA[ip];
    const double2 B = prodB[ip];
    const int thr_hi = hi32(A.w);
    FockSink<L> sink;
#pragma unroll
    for (int h = 0; h < NH; ++h) sink.acc[h] = 0.0;
    const int64_t ebeg = start[rg] + (piece - pstart[rg]) * NEAR_PIECE, eend = min(start[rg + 1], ebeg + NEAR_PIECE);
    const int np = (int)(eend - ebeg);
    {   // lane -> point (lane & 7) of this warp's share of listed group lane >> 3
        const int pe = lane / NEAR_PER;
        const int k = pe < np ? list[ebeg + pe] * SUB + warp * NEAR_PER + (lane % NEAR_PER) : M;
        if (k < M) {
            const double4 c = pt[k];
            s_pt[warp][lane] = make_double4(c.x, c.y, c.z, q[qidx ? qidx[k] : k]);
            s_iz[warp][lane] = c.w;
        } else {
            s_pt[warp][lane] = make_double4(-3e8, -3e8, -3e8, 0.0);
            s_iz[warp][lane] = 1.0;
        }
    }
    __syncwarp();
    const int nev = np * NEAR_PER;
#pragma unroll 1
    for (int t = 0; t < nev; t += 2) {
        const double4 c0 = s_pt[warp][t], c1 = s_pt[warp][t + 1];
        const double x0 = A.x - c0.x, y0 = A.y - c0.y, z0 = A.z - c0.z;
        const double x1 = A.x - c1.x, y1 = A.y - c1.y, z1 = A.z - c1.z;
        const double r20 = fma(z0, z0, fma(y0, y0, x0 * x0));
        const double r21 = fma(z1, z1, fma(y1, y1, x1 * x1));
        double g0[L + 1], g1[L + 1];
        if (min(hi32(r20), hi32(r21)) > thr_hi) {
            seeds_far<L>(r20, g0);
            seeds_far<L>(r21, g1);
        } else {
            seeds_general<L>(r20, B.x, B.y, s_iz[warp][t], boysL, g0);
            seeds_general<L>(r21, B.x, B.y, s_iz[warp][t + 1], boysL, g1);
        }
#pragma unroll
        for (int n2 = 0; n2 <= L; ++n2) { g0[n2] *= c0.w; g1[n2] *= c1.w; }
        hermite_R<L>(x0, y0, z0, g0, sink);
        hermite_R<L>(x1, y1, z1, g1, sink);
    }
    if (warp > 0) {
#pragma unroll
        for (int h = 0; h < NH; ++h) s_sum[warp - 1][h * SUB + lane] = sink.acc[h];
    }
    __syncthreads();
    if (warp == 0) {
        double *out = near + (size_t)piece * NH * SUB + lane;
#pragma unroll
        for (int h = 0; h < NH; ++h) {
            double v = sink.acc[h];
#pragma unroll
            for (int w = 0; w < NEAR_WARPS - 1; ++w) v += s_sum[w][h * SUB + lane];
            out[h * SUB] = v;
        }
    }
}

// herm[0][h][i] = sum_c herm[c][h][i] + sum of the near pieces of product i; plane = nh * npad.  As reduce_slots_kernel:
// a 256-thread block sums 32 consecutive elements, warp w taking every 8th chunk and every 8th near piece (fixed order).
__global__ void __launch_bounds__(256) reduce_herm_kernel(double *__restrict__ herm, int64_t plane, int chunks, int64_t npad, int nh,
                                                          const double *__restrict__ near, const int64_t *__restrict__ pstart) {
    __shared__ double s_tmp[8 * 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t k = (int64_t)blockIdx.x * 32 + lane;   // npad is a multiple of 32: the 32 elements share h and the row group
    double s = 0.0;
    pdl_launch_dependents();
    if (k < plane) {
        for (int c = w; c < chunks; c += 8) s += herm[(size_t)c * plane + k];
        const int64_t h = k / npad, i = k - h * npad, rg = i / SUB;
        for (int64_t q = pstart[rg] + w; q < pstart[rg + 1]; q += 8) s += near[((size_t)q * nh + h) * SUB + lane];
    }
    s_tmp[w * 32 + lane] = s;
    __syncthreads();
    if (w == 0 && k < plane) {
        double t = 0.0;
#pragma unroll
        for (int q = 0; q < 8; ++q) t += s_tmp[q * 32 + lane];
        herm[k] = t;
    }
    pdl_wait_predecessor();
}

// ---------------------------------------------------------------------------------------------
// a2 main kernel: v_k = sum_products sum_h D_h Rt_h(P - C_k).  Rows = R points per thread (register accumulators),
// columns = products (centre, Hermite density) staged in shared memory, C per step.
// ---------------------------------------------------------------------------------------------
template <int L>
struct PotSink {
    static constexpr bool kSplit = false;
    __device__ __forceinline__ void lower(int, double) {}
    const double *D;
    double v;
    __device__ __forceinline__ void value(int h, int, int, int, double x) { v = fma(D[h], x, v); }
    __device__ __forceinline__ void product(int h, int, int, int, double a, double b) { v = fma(D[h], a * b, v); }
};

template <int L>
__host__ __device__ constexpr int pot_rec() { return (4 + nherm(L) + 1) / 2 * 2; }      // main kernel: centre, pad, D_h
// potential_kernel's own record: for L = 3 four more slots (the first-order coefficients of the third-order block)
template <int L>
__host__ __device__ constexpr int pot_rec_main() { return pot_rec<L>() + (L == 3 ? 4 : 0) + (L == 1 ? 2 : 0); }
// L = 0, 1: the main kernel works in the local coordinates of its row block (pot_local_unit below)
__host__ __device__ constexpr bool pot_local(int L) { return L <= 1; }
template <int L>
__host__ __device__ constexpr int pot_rec_near() { return (4 + nherm(L) + 2 + 1) / 2 * 2; }  // + (p, 1/kappa)

template <int L>
__device__ __forceinline__ void pot_far_unit(const double *rec, const double4 &c, double &v) {
    const double2 h01 = *reinterpret_cast<const double2 *>(rec);
    const double x = h01.x - c.x, y = h01.y - c.y, z = rec[2] - c.z;
    double g[L + 1];
    seeds_far<L>(fma(z, z, fma(y, y, x * x)), g);
    PotSink<L> sink{rec + 4, v};
    hermite_R<L>(x, y, z, g, sink);
    v = sink.v;
}

// L = 1 contracted before the seeds are formed: D.R = g0 [D_0 - u (D_x x + D_y y + D_z z)], u = 1/R^2 -- 17 FP64 instructions
// per evaluation instead of the 19.5 of the generic recursion (x g1 products and a separate g1)
template <>
__device__ __forceinline__ void pot_far_unit<1>(const double *rec, const double4 &c, double &v) {
    const double2 h01 = *reinterpret_cast<const double2 *>(rec);
    const double x = h01.x - c.x, y = h01.y - c.y, z = rec[2] - c.z;
    const double ri = rsqrt_fast(fma(z, z, fma(y, y, x * x)));
    const double u = ri * ri;
    const double s = fma(rec[5], x, fma(rec[6], y, rec[7] * z));   // hidx(1,0,0) = 1, (0,1,0) = 2, (0,0,1) = 3
    v = fma(ri, fma(-u, s, rec[4]), v);
}

// L = 2 contracted the same way: with g1 = -u g0, g2 = 3 u^2 g0 and R_200 = g1 + x^2 g2, R_110 = x y g2, ...
//   D.R = g0 [ D_000 - u (D_1 . r + tr) + 3 u^2 (r^T D_2 r) ],  tr = D_200 + D_020 + D_002 (staged in the record's pad slot),
// 28 FP64 instructions per evaluation instead of the ~36 of the generic recursion followed by the contraction.
template <>
__device__ __forceinline__ void pot_far_unit<2>(const double *rec, const double4 &c, double &v) {
    const double2 h01 = *reinterpret_cast<const double2 *>(rec);
    const double2 h23 = *reinterpret_cast<const double2 *>(rec + 2);
    const double x = h01.x - c.x, y = h01.y - c.y, z = h23.x - c.z;
    const double ri = rsqrt_fast(fma(z, z, fma(y, y, x * x)));
    const double u = ri * ri;
    // components: 4 = (2,0,0), 5 = (1,1,0), 6 = (1,0,1), 7 = (0,2,0), 8 = (0,1,1), 9 = (0,0,2)
    const double q2 = fma(x, fma(rec[8], x, fma(rec[9], y, rec[10] * z)), fma(y, fma(rec[11], y, rec[12] * z), z * (rec[13] * z)));
    const double lin = fma(rec[5], x, fma(rec[6], y, fma(rec[7], z, h23.y)));
    const double e1 = fma(u, q2, -lin);          // the record carries 3 D_2 (pot_scale_record)
    v = fma(ri, fma(u, e1, rec[4]), v);
}

// L = 3: R_300 = 3 x g2 + x^3 g3, R_210 = y g2 + x^2 y g3, R_111 = x y z g3, ... and g3 = -15 u^3 g0, so
//   D.R = g0 [ D_000 - u (D_1 . r + tr) + 3 u^2 (r^T D_2 r + l . r) - 15 u^3 C_3(r) ],
// C_3 the cubic form of the third-order block, l = (3 D_300 + D_120 + D_102, 3 D_030 + D_210 + D_012, 3 D_003 + D_201 + D_021)
// staged behind the record (slots 24..26) and tr in the pad slot.  51 FP64 instructions per evaluation.
template <>
__device__ __forceinline__ void pot_far_unit<3>(const double *rec, const double4 &c, double &v) {
    const double2 h01 = *reinterpret_cast<const double2 *>(rec);
    const double2 h23 = *reinterpret_cast<const double2 *>(rec + 2);
    const double x = h01.x - c.x, y = h01.y - c.y, z = h23.x - c.z;
    const double ri = rsqrt_fast(fma(z, z, fma(y, y, x * x)));
    const double u = ri * ri;
    const double *D = rec + 4;
    // third order: 10 = (3,0,0), 11 = (2,1,0), 12 = (2,0,1), 13 = (1,2,0), 14 = (1,1,1), 15 = (1,0,2), 16 = (0,3,0),
    // 17 = (0,2,1), 18 = (0,1,2), 19 = (0,0,3)
    const double A = fma(D[10], x, fma(D[11], y, D[12] * z));
    const double B = fma(y, fma(D[13], y, D[14] * z), (D[15] * z) * z);
    const double Cc = fma(y * y, fma(D[16], y, D[17] * z), (z * z) * fma(D[18], y, D[19] * z));
    const double c3 = fma(x, fma(x, A, B), Cc);
    double q2 = fma(x, fma(D[4], x, fma(D[5], y, D[6] * z)), fma(y, fma(D[7], y, D[8] * z), z * (D[9] * z)));
    q2 = fma(rec[24], x, fma(rec[25], y, fma(rec[26], z, q2)));
    const double lin = fma(D[1], x, fma(D[2], y, fma(D[3], z, h23.y)));
    const double e2 = fma(u, c3, q2);            // the record carries 3 D_2, 3 l and -15 D_3 (pot_scale_record)
    const double e1 = fma(u, e2, -lin);
    v = fma(ri, fma(u, e1, D[0]), v);
}

// L = 0, 1 in local coordinates, as the A q sweep: with o the first point of the CTA's row block, a = C - o (the point, in
// registers with |a|^2) and the record staged as (-2 (P - o), |P - o|^2, D_h[, D_1 . (P - o)]),
//   R^2 = |a|^2 + |P - o|^2 - 2 a . (P - o)                      1 DADD + 3 DFMA instead of 3 DADD + DMUL + 2 DFMA,
//   D_1 . (P - C) = D_1 . (P - o) - D_1 . a                      3 DFMA instead of 3 DADD + DMUL + 2 DFMA (x, y, z are never formed):
// 10 and 15 FP64 instructions per evaluation instead of 12 and 17.  The cancellation costs (|a| + |P - o|)^2 / R^2 ulps of R^2
// (|a| <= the extent of the 512 points of a row block; a few tens of ulps for the closest far products, as in amatvec_kernel).
template <int L>
__device__ __forceinline__ void pot_local_unit(const double *rec, const double4 &a, double &v) {
    const double2 h01 = *reinterpret_cast<const double2 *>(rec);
    const double2 h23 = *reinterpret_cast<const double2 *>(rec + 2);
    const double ri = rsqrt_fast(fma(a.x, h01.x, fma(a.y, h01.y, fma(a.z, h23.x, a.w + h23.y))));
    if (L == 0) {
        v = fma(rec[4], ri, v);
    } else {
        const double u = ri * ri;
        const double ms = fma(rec[5], a.x, fma(rec[6], a.y, fma(rec[7], a.z, -rec[8])));     // -(D_1 . (P - C))
        v = fma(ri, fma(u, ms, rec[4]), v);
    }
}

// (forcing the old occupancy back with a minimum-blocks launch bound -- 64 / 72 instead of 72 / 80 registers -- measured slower
// for L = 0 and no different for L = 1)
// Derived slots of a staged record r = (centre, pad, D_h ...): the trace of D_2 in the pad slot (L = 2, 3), the first-order
// coefficients l of the third-order block behind the record (L = 3); then the constants of the Horner form are folded into the
// coefficients -- D_2 <- 3 D_2 (L = 2, 3), l <- 3 l and D_3 <- -15 D_3 (L = 3) -- so that pot_far_unit multiplies by u only
// (one FP64 instruction less per evaluation at L = 2, two at L = 3).
template <int L>
__device__ __forceinline__ void pot_scale_record(double *r) {
    if (L == 2 || L == 3) {
        r[3] = r[4 + 4] + r[4 + 7] + r[4 + 9];
        if (L == 3) {
            r[24] = 3.0 * fma(3.0, r[4 + 10], r[4 + 13] + r[4 + 15]);
            r[25] = 3.0 * fma(3.0, r[4 + 16], r[4 + 11] + r[4 + 18]);
            r[26] = 3.0 * fma(3.0, r[4 + 19], r[4 + 12] + r[4 + 17]);
#pragma unroll
            for (int h = 10; h < 20; ++h) r[4 + h] *= -15.0;
        }
#pragma unroll
        for (int h = 4; h < 10; ++h) r[4 + h] *= 3.0;
    }
}

template <int L, int R, int C>
__global__ void __launch_bounds__(TPB) potential_kernel(const double4 *__restrict__ prodA, const double *__restrict__ herm,
                                                        int64_t npad, int chunk_len, const double4 *__restrict__ pt, int M,
                                                        double *__restrict__ vpart, const uint8_t *__restrict__ farmap,
                                                        int64_t nbyte, int64_t nrg) {
    constexpr int NH = nherm(L);
    constexpr int REC = pot_rec_main<L>();
    constexpr int TILE = pot_tile(L), NS = TILE / SUB;
    __shared__ __align__(16) double s_rec[TILE * REC];
    pdl_launch_dependents();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t rg0 = ((int64_t)blockIdx.x * (TPB / 32) + warp) * R;
    double4 c[R];
    int kk[R];
    double v[R];
    double4 org = make_double4(0.0, 0.0, 0.0, 0.0);
    if (pot_local(L)) org = pt[min((int)blockIdx.x * (TPB * R), M - 1)];      // origin of the row block's local coordinates
#pragma unroll
    for (int r = 0; r < R; ++r) {
        kk[r] = (int)(rg0 + r) * SUB + lane;
        c[r] = pt[min(kk[r], M - 1)];
        if (pot_local(L)) {       // (a, |a|^2), a = C - o
            c[r].x -= org.x; c[r].y -= org.y; c[r].z -= org.z;
            c[r].w = fma(c[r].z, c[r].z, fma(c[r].y, c[r].y, c[r].x * c[r].x));
        }
        v[r] = 0.0;
    }
    // products [pbeg, pend): pend <= npad, both multiples of 32 (the padding carries zero density)
    const int64_t pbeg = (int64_t)blockIdx.y * chunk_len, pend = min(npad, pbeg + (int64_t)chunk_len);
    for (int64_t base = pbeg; base < pend; base += TILE) {
        const int cnt = (int)min((int64_t)TILE, pend - base), nst = cnt / SUB;
        const unsigned bits = far_bits<R, NS>(farmap, nbyte, rg0, nrg, base / SUB, lane);
        __syncthreads();
        for (int t = threadIdx.x; t < cnt; t += TPB) {
            const double4 a = prodA[base + t];
            double *r = s_rec + t * REC;
            if (pot_local(L)) {
                const double x = a.x - org.x, y = a.y - org.y, z = a.z - org.z;
                r[0] = -2.0 * x; r[1] = -2.0 * y; r[2] = -2.0 * z; r[3] = fma(z, z, fma(y, y, x * x));
            } else {
                r[0] = a.x; r[1] = a.y; r[2] = a.z; r[3] = 0.0;
            }
        }
        for (int t = threadIdx.x; t < cnt * NH; t += TPB) {
            const int h = t / cnt, i = t - h * cnt;  // consecutive threads read consecutive products of one component
            s_rec[i * REC + 4 + h] = herm[(size_t)h * npad + base + i];
        }
        if (L == 1) {             // pot_local_unit<1> wants D_1 . (P - o) behind the record
            __syncthreads();
            for (int t = threadIdx.x; t < cnt; t += TPB) {
                double *r = s_rec + t * REC;
                r[8] = -0.5 * fma(r[5], r[0], fma(r[6], r[1], r[7] * r[2]));
            }
        }
        if (L == 2 || L == 3) {   // pot_far_unit<2>, <3> want the trace of the second-order block in the pad slot
            __syncthreads();
            for (int t = threadIdx.x; t < cnt; t += TPB) pot_scale_record<L>(s_rec + t * REC);
        }
        __syncthreads();
        for (int st = 0; st < nst; ++st) {
            const double *sr = s_rec + st * SUB * REC;
            const unsigned m = row_mask<R>(bits, st);
            if (m == (1u << R) - 1u) {
#pragma unroll 1
                for (int t = 0; t < SUB; t += C) {
#pragma unroll
                    for (int cc = 0; cc < C; ++cc)
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            if (pot_local(L)) pot_local_unit<L>(sr + (t + cc) * REC, c[r], v[r]);
                            else pot_far_unit<L>(sr + (t + cc) * REC, c[r], v[r]);
                        }
                }
            } else if (R > 1 && m) {
#pragma unroll 1
                for (int t = 0; t < SUB; ++t) {
#pragma unroll
                    for (int r = 0; r < R; ++r)
                        if ((m >> r) & 1u) {
                            if (pot_local(L)) pot_local_unit<L>(sr + t * REC, c[r], v[r]);
                            else pot_far_unit<L>(sr + t * REC, c[r], v[r]);
                        }
                }
            }
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r)
        if (kk[r] < M) vpart[(size_t)blockIdx.y * M + kk[r]] = v[r];
    pdl_wait_predecessor();
}

// ---- the potential in the Fock layout ("product in registers", pcm_options.potential_pr) -------------------------------
// north_star describes the P-contraction as "warp-shuffle reductions": thread = one Hermite product with its centre and
// D_h in REGISTERS, the points of the CTA's point block (PR_PTS of them) staged once in shared memory, and the 32 products
// of a warp summed per point by a fixed-order shuffle butterfly -- NB point values per lane are reduced together, halving
// the live values at every step (NB/2 + NB/4 + ... + 1 + log2(32/NB) exchanges for NB points: ~1 SHFL.64 + 1 DADD per
// evaluation), after which lane pair (2j, 2j+1) holds the warp's sum for point j.  Per-warp point accumulators in shared
// memory, added over the warps at the end -> vpart[product chunk][point].  Against potential_kernel this trades the
// broadcast reads of the product record (27 doubles per evaluation at L = 3) for one shuffle-add per evaluation.
// Far patches come from the class's Fock map (rows = product groups, columns = point groups: the same boxes and the same
// symmetric criterion as the potential map, so the near kernel's complement is unchanged).
constexpr int PR_PTS = 512;
template <int L, int NB>
__global__ void __launch_bounds__(TPB) potential_pr_kernel(const double4 *__restrict__ prodA, const double *__restrict__ herm,
                                                           int64_t npad, int pchunk, const double4 *__restrict__ pt, int M,
                                                           double *__restrict__ vpart, const uint8_t *__restrict__ farmap,
                                                           int64_t nbyte) {
    constexpr int NH = nherm(L);
    constexpr int REC = pot_rec<L>() + (L == 3 ? 4 : 0);
    __shared__ double4 s_pt[PR_PTS];                 // x, y, z of the point block (padding: far away)
    __shared__ double s_acc[TPB / 32][PR_PTS];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int k0 = blockIdx.x * PR_PTS, npts = min(PR_PTS, M - k0), ngrp = (npts + 31) / 32;
    for (int t = threadIdx.x; t < PR_PTS; t += TPB) {
        s_pt[t] = (t < npts) ? pt[k0 + t] : make_double4(3e8, 3e8, 3e8, 1.0);
#pragma unroll
        for (int w = 0; w < TPB / 32; ++w) s_acc[w][t] = 0.0;
    }
    __syncthreads();
    const int64_t pbeg = (int64_t)blockIdx.y * pchunk, pend = min(npad, pbeg + (int64_t)pchunk);
    for (int64_t pb = pbeg; pb < pend; pb += TPB) {
        const int64_t ip = pb + threadIdx.x;       // < npad: npad and pchunk are multiples of TPB
        double rec[REC];
        {
            const double4 a = prodA[ip];
            rec[0] = a.x; rec[1] = a.y; rec[2] = a.z; rec[3] = 0.0;
#pragma unroll
            for (int h = 0; h < NH; ++h) rec[4 + h] = herm[(size_t)h * npad + ip];
            pot_scale_record<L>(rec);
        }
        const uint8_t *frow = farmap + (size_t)(ip >> 5) * nbyte;     // the warp's product group (warp-uniform)
        for (int g = 0; g < ngrp; ++g) {
            const int cg = (k0 >> 5) + g;
            if (!((frow[cg >> 3] >> (cg & 7)) & 1)) continue;
#pragma unroll 1
            for (int t0 = 0; t0 < 32; t0 += NB) {
                double val[NB];
#pragma unroll
                for (int j = 0; j < NB; ++j) {
                    val[j] = 0.0;
                    pot_far_unit<L>(rec, s_pt[g * 32 + t0 + j], val[j]);
                }
                // butterfly: after the step with lane mask `off` a lane keeps the half of its values its bit selects
                int nv = NB;
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) {
                    if (nv > 1) {
                        nv >>= 1;
                        const bool up = (lane & off) != 0;
#pragma unroll
                        for (int j = 0; j < NB / 2; ++j) {
                            if (j < nv) {
                                const double keep = up ? val[j + nv] : val[j], send = up ? val[j] : val[j + nv];
                                val[j] = keep + __shfl_xor_sync(0xffffffffu, send, off);
                            }
                        }
                    } else {
                        val[0] += __shfl_xor_sync(0xffffffffu, val[0], off);
                    }
                }
                // lane bits (from 16 down) selected the upper halves in turn: the point index is their bit pattern
                constexpr int LOG_NB = NB == 16 ? 4 : NB == 8 ? 3 : NB == 4 ? 2 : 1;
                const int j = (lane >> (5 - LOG_NB)) & (NB - 1);
                if ((lane & ((1 << (5 - LOG_NB)) - 1)) == 0) s_acc[warp][g * 32 + t0 + j] += val[0];
            }
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < npts; t += TPB) {
        double v = s_acc[0][t];
#pragma unroll
        for (int w = 1; w < TPB / 32; ++w) v += s_acc[w][t];
        vpart[(size_t)blockIdx.y * M + k0 + t] = v;
    }
}

// near patches of the potential sweep: one CTA per piece; lane = point; warp w takes the products [8 w, 8 w + 8) of every listed
// product group (see fock_near_kernel) and stages their records -- one per lane, the whole piece in one pass -- in its own
// shared memory.  The four partial sums are added in warp order.  Writes near[piece][lane].
template <int L>
__global__ void __launch_bounds__(TPB) potential_near_kernel(const double4 *__restrict__ prodA, const double2 *__restrict__ prodB,
                                                             const double *__restrict__ herm, int64_t npad,
                                                             const double4 *__restrict__ pt, int M,
                                                             const int64_t *__restrict__ start, const int32_t *__restrict__ list,
                                                             const int64_t *__restrict__ pstart, const int32_t *__restrict__ piece_rg,
                                                             int64_t npiece, double *__restrict__ near,
                                                             const double *__restrict__ boysL) {
    constexpr int NH = nherm(L);
    constexpr int REC = pot_rec_near<L>();
    __shared__ __align__(16) double s_rec[NEAR_WARPS][SUB * REC];
    __shared__ double s_sum[NEAR_WARPS][SUB];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t piece = blockIdx.x;
    const int64_t rg = piece_rg[piece];
    const int k = (int)rg * SUB + lane;
    const double4 c = pt[min(k, M - 1)];
    double v = 0.0;
    const int64_t ebeg = start[rg] + (piece - pstart[rg]) * NEAR_PIECE, eend = min(start[rg + 1], ebeg + NEAR_PIECE);
    const int np = (int)(eend - ebeg);
    double *mine = s_rec[warp];
    if (lane / NEAR_PER < np) {     // lane -> product (lane & 7) of this warp's share of listed group lane >> 3
        const int64_t i = (int64_t)list[ebeg + lane / NEAR_PER] * SUB + warp * NEAR_PER + (lane % NEAR_PER);
        const double4 a = prodA[i];
        const double2 b = prodB[i];
        double *r = mine + lane * REC;
        r[0] = a.x; r[1] = a.y; r[2] = a.z; r[3] = a.w;
        r[4 + NH] = b.x; r[5 + NH] = b.y;
#pragma unroll
        for (int h = 0; h < NH; ++h) r[4 + h] = herm[(size_t)h * npad + i];
    }
    __syncwarp();
    const int nev = np * NEAR_PER;
#pragma unroll 1
    for (int t = 0; t < nev; ++t) {
        const double *rec = mine + t * REC;
        const double2 h01 = *reinterpret_cast<const double2 *>(rec);
        const double2 h23 = *reinterpret_cast<const double2 *>(rec + 2);
        const double x = h01.x - c.x, y = h01.y - c.y, z = h23.x - c.z;
        const double r2 = fma(z, z, fma(y, y, x * x));
        double g[L + 1];
        if (hi32(r2) > hi32(h23.y)) seeds_far<L>(r2, g);
        else seeds_general<L>(r2, rec[4 + NH], rec[5 + NH], c.w, boysL, g);
        PotSink<L> sink{rec + 4, v};
        hermite_R<L>(x, y, z, g, sink);
        v = sink.v;
    }
    s_sum[warp][lane] = v;
    __syncthreads();
    if (warp == 0) {
        double t = s_sum[0][lane];
#pragma unroll
        for (int w = 1; w < NEAR_WARPS; ++w) t += s_sum[w][lane];
        near[piece * SUB + lane] = t;
    }
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
    pdl_launch_dependents();
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
    pdl_wait_predecessor();
}

// The same transform with one warp per product (used for L >= 2, where a product has several members of up to 25
// components each): lane = component (a, b) of the member, members in order, then a fixed-order butterfly over the lanes.
template <int L>
__global__ void __launch_bounds__(128) density_to_hermite_warp_kernel(int64_t n, int64_t first, int64_t npad,
                                                                      const int64_t *__restrict__ pm_start,
                                                                      const int32_t *__restrict__ pm_list, const int32_t *__restrict__ m_sp,
                                                                      const int32_t *__restrict__ m_cls, const int64_t *__restrict__ m_goff,
                                                                      const double *__restrict__ G, const int32_t *__restrict__ sp_i0,
                                                                      const int32_t *__restrict__ sp_j0, const int32_t *__restrict__ sp_dims,
                                                                      const double *__restrict__ P, int64_t ldp, double *__restrict__ herm) {
    constexpr int NH = nherm(L);
    const int lane = threadIdx.x & 31;
    const int64_t i = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
    pdl_launch_dependents();
    if (i >= npad) { pdl_wait_predecessor(); return; }
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
            for (int ab = lane; ab < na * nb; ab += 32) {
                const int a = ab / nb, b = ab - a * nb;
                double pw = P[(size_t)(i0 + a) * ldp + j0 + b];
                if (!diag) pw += P[(size_t)(j0 + b) * ldp + i0 + a];
                const double *row = gm + (size_t)ab * nhm;
#pragma unroll
                for (int h = 0; h < NH; ++h)
                    if (h < nhm) D[h] = fma(row[h], pw, D[h]);
            }
        }
    }
#pragma unroll
    for (int h = 0; h < NH; ++h) {
        double v = D[h];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) herm[(size_t)h * npad + i] = v;
    }
    pdl_wait_predecessor();
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
// work partition (fixed by the sizes, the SM count and the kernels' occupancy only -> results are reproducible)
// ---------------------------------------------------------------------------------------------
static int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

// rows: register-resident objects, rows_per_block of them per block; cols: streamed objects, cut into chunks of whole
// tiles.  The grid (xb x chunks) is cut into about four waves of `wave` co-resident blocks when the sizes allow (the
// hardware block scheduler then evens out what the skipped near patches unbalance): the smallest chunk count >= 4
// waves whose last wave is at least 90 % full, or the best available.
static Plan make_plan(int64_t rows, int rows_per_block, int64_t cols, int tile, int64_t wave, double fill = 1.0, double waves = 4.0) {
    Plan p;
    p.xb = ceil_div(std::max<int64_t>(rows, 1), rows_per_block);
    const int64_t tiles = ceil_div(std::max<int64_t>(cols, 1), tile);
    const int64_t maxc = std::min<int64_t>(tiles, 512);
    int64_t best = 1;
    double best_score = 0.0;
    for (int64_t c = 1; c <= maxc; ++c) {
        const int64_t len = ceil_div(tiles, c);            // tiles per chunk
        const int64_t cc = ceil_div(tiles, len);           // chunks actually needed
        const double t = std::max(1.0, (double)p.xb * (double)cc * fill);   // blocks that have work (fill < 1: triangular sweep)
        const double eff = t / ((double)ceil_div((int64_t)t, wave) * (double)wave);
        const double score = eff * std::min(1.0, 0.55 + 0.45 * t / (waves * (double)wave));  // prefer >= `waves` waves
        if (score > best_score + 1e-9) { best_score = score; best = cc; }
        if (t >= waves * (double)wave && eff >= 0.9) break;
    }
    const int64_t len = ceil_div(tiles, best);
    p.chunk_len = len * tile;
    p.chunks = ceil_div(tiles, len);
    return p;
}

template <class K>
static int64_t wave_of(const pcm_ctx *ctx, K kernel) {
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel, TPB, 0) != cudaSuccess || nb < 1) nb = 1;
    return (int64_t)nb * ctx->sm_count;
}

template <int L>
static void plan_class(pcm_ctx *ctx) {
    constexpr Blocking fb = fock_blocking(L), pb = pot_blocking(L);
    const ClassData &c = ctx->cls[L];
    const double iw = 4.0;   // wave target of the work partition (more waves measured no different on configs[1])
    ctx->plan_fock[L] = make_plan(c.npad, TPB * fb.R, ctx->M, PT_TILE, wave_of(ctx, fock_kernel<L, fb.R, fb.C>), 1.0, iw);
    ctx->plan_pot[L] = make_plan(ctx->M, TPB * pb.R, c.npad, pot_tile(L), wave_of(ctx, potential_kernel<L, pb.R, pb.C>), 1.0, iw);
    constexpr Blocking pbb = pot_blocking_big(L);
    if (ctx->M >= POT_BIG_MIN && (pbb.R != pb.R || pbb.C != pb.C))
        ctx->plan_pot[L] = make_plan(ctx->M, TPB * pbb.R, c.npad, pot_tile(L), wave_of(ctx, potential_kernel<L, pbb.R, pbb.C>), 1.0, iw);
    if ((ctx->opt.potential_pr >> L) & 1)    // product-in-registers layout: rows = point blocks of PR_PTS, chunks of whole product blocks
        ctx->plan_pot[L] = make_plan(ctx->M, PR_PTS, c.npad, TPB, wave_of(ctx, potential_pr_kernel<L, (L <= 3 ? 16 : 8)>), 1.0, iw);
}

int plan_all(pcm_ctx *ctx) {
    // symmetric sweep: about half of the (row block, chunk) grid has work.  From AMAT_R4_MIN points on: row blocks of 512
    // (R = 4) and column tiles of 256; below: row blocks of 256 (R = 2) and tiles of 64, i.e. 16 times as many, smaller
    // work items, so that a 9k-point sweep still loads 148 SMs evenly (R = 1 / tile 128 and R = 2 / tile 32 or 128 measured slower).
    ctx->amat_R = ctx->M >= AMAT_R4_MIN ? 4 : 2;
    ctx->amat_tile = ctx->amat_R == 4 ? 256 : 64;
    const double aw = 8.0;
    ctx->plan_amat = ctx->amat_R == 4       ? make_plan(ctx->M, TPB * 4, ctx->M, 256, wave_of(ctx, amatvec_kernel<4, AMAT_C, 256>), 0.5, aw)
                     : ctx->amat_tile == 64  ? make_plan(ctx->M, TPB * 2, ctx->M, 64, wave_of(ctx, amatvec_kernel<2, AMAT_C, 64>), 0.5, aw)
                     : ctx->amat_tile == 128 ? make_plan(ctx->M, TPB * 2, ctx->M, 128, wave_of(ctx, amatvec_kernel<2, AMAT_C, 128>), 0.5, aw)
                                             : make_plan(ctx->M, TPB * 2, ctx->M, 256, wave_of(ctx, amatvec_kernel<2, AMAT_C, 256>), 0.5, aw);
    if (getenv("PCM_VERBOSE")) fprintf(stderr, "[pcm] amat plan: R %d xb %lld chunks %lld chunk_len %lld\n", ctx->amat_R,
                                       (long long)ctx->plan_amat.xb, (long long)ctx->plan_amat.chunks, (long long)ctx->plan_amat.chunk_len);
    plan_class<0>(ctx); plan_class<1>(ctx); plan_class<2>(ctx); plan_class<3>(ctx); plan_class<4>(ctx);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_error(ctx, PCM_ERR_CUDA, std::string("plan_all: ") + cudaGetErrorString(e));
    return PCM_OK;
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

// Partial sums of y = A q: near pieces into near_amat (near stream, forked from and joined back into s), main kernel
// slots into ypart.  idx: sorted -> caller index of q (nullptr: q is in sorted order).  stop: see cg_solve.
static int launch_amatvec_kernels(pcm_ctx *ctx, const double *q, const int32_t *idx, const int *stop, cudaStream_t s) {
    const int M = (int)ctx->M;
    const Plan &pl = ctx->plan_amat;
    const PatchMap &pm = ctx->amat_map;
    const double thr = TFAR_AMAT * 2.0 / (ctx->zeta_min * ctx->zeta_min);
    const bool stored = ctx->amat_blocks != nullptr && pm.npiece > 0;
    NearStored ns{};
    int64_t extra = 0;
    if (stored) {   // one launch: the near pieces ride in extra rows of the main kernel's grid
        ns.blocks = ctx->amat_blocks; ns.start = pm.start; ns.pstart = pm.pstart; ns.list = pm.list; ns.piece_rg = pm.piece_rg;
        ns.npiece = pm.npiece; ns.near = ctx->near_amat;
        extra = ceil_div(ceil_div(pm.npiece, TPB / 32), pl.xb);
    }
    dim3 grid((unsigned)pl.xb, (unsigned)(pl.chunks + extra));
    const bool fork = !stored && pm.npiece > 0;
    if (fork) {     // near patches evaluated on the fly: their own kernel on the near stream
        PCM_CUDA(ctx, cudaEventRecord(ctx->ev_fork, s));
        PCM_CUDA(ctx, cudaStreamWaitEvent(ctx->near_stream, ctx->ev_fork, 0));
        amat_near_kernel<<<(unsigned)ceil_div(pm.npiece, TPB / 32), TPB, 0, ctx->near_stream>>>(
            ctx->pt, ctx->pt_diag, q, idx, M, pm.start, pm.list, pm.pstart, pm.piece_rg, pm.npiece, ctx->near_amat, ctx->boys, thr, stop);
        PCM_LAUNCH_CHECK(ctx);
        PCM_CUDA(ctx, cudaEventRecord(ctx->ev_join, ctx->near_stream));
        { ctx->launches[2]++; ctx->launch_total++; }
    }
    const int ch = (int)pl.chunks;
#define PCM_AMAT_LAUNCH(R_, T_)                                                                                                   \
    amatvec_kernel<R_, AMAT_C, T_><<<grid, TPB, 0, s>>>(ctx->pt, q, idx, M, (int)pl.chunk_len, ctx->ypart, ctx->colpart, pm.far, \
                                                        pm.nbyte, pm.nrg, stop, ch, ns)
    if (ctx->amat_R == 4) PCM_AMAT_LAUNCH(4, 256);
    else if (ctx->amat_tile == 64) PCM_AMAT_LAUNCH(2, 64);
    else if (ctx->amat_tile == 128) PCM_AMAT_LAUNCH(2, 128);
    else PCM_AMAT_LAUNCH(2, 256);
#undef PCM_AMAT_LAUNCH
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[2]++; ctx->launch_total++; }
    if (fork) PCM_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_join, 0));
    return PCM_OK;
}
// evaluates the near patches of A once (pcm_setup), if they fit the budget
int fill_amat_blocks(pcm_ctx *ctx) {
    const PatchMap &pm = ctx->amat_map;
    ctx->amat_blocks = nullptr;
    const double budget_gb = 16.0;
    const double need = (double)pm.nnear * SUB * SUB * 8.0;
    if (ctx->opt.store_near == 0 || pm.npiece == 0 || need > budget_gb * 1e9) return PCM_OK;
    int rc = dev_alloc_t(ctx, &ctx->amat_blocks, (size_t)pm.nnear * SUB * SUB);
    if (rc) return rc;
    const double thr = TFAR_AMAT * 2.0 / (ctx->zeta_min * ctx->zeta_min);
    amat_near_fill_kernel<<<(unsigned)ceil_div(pm.npiece, TPB / 32), TPB>>>(ctx->pt, ctx->pt_diag, (int)ctx->M, pm.start, pm.list, pm.pstart,
                                                                           pm.piece_rg, pm.npiece, ctx->amat_blocks, ctx->boys, thr);
    PCM_LAUNCH_CHECK(ctx);
    return PCM_OK;
}
int launch_amatvec_partials(pcm_ctx *ctx, const double *q_sorted, const int *stop, cudaStream_t s) {
    return launch_amatvec_kernels(ctx, q_sorted, nullptr, stop, s);
}

// y = A q.  caller_order: q and y are indexed by the caller's point order (gather/scatter through s2c);
// otherwise both are in the library's sorted order (the CG solver's internal vectors).
static int launch_amatvec_impl(pcm_ctx *ctx, const double *q, double *y, bool caller_order, cudaStream_t s) {
    ctx->cur_op = 2;
    ctx->launches[2] = 0;
    ctx->timed[2] = ctx->timing != 0;
    const int M = (int)ctx->M;
    if (M == 0) return PCM_OK;
    const int32_t *idx = caller_order ? ctx->s2c : nullptr;
    int rc;
    // timing: one event before and one after (each event record is a command of its own on the stream, ~1 us: eight of them
    // would be a tenth of a 10k-point product)
    if ((rc = mark(ctx, 0, s))) return rc;
    if (ctx->cgp.ready) {   // small cavities: the warp-granular sweep of pcm_cgp.cu and its row sums, two launches
        if ((rc = cgp_matvec(ctx, q, idx, y, s))) return rc;
        ctx->launches[2] += 2;
        return mark(ctx, 7, s);
    }
    if ((rc = launch_amatvec_kernels(ctx, q, idx, nullptr, s))) return rc;
    amat_reduce_kernel<<<(unsigned)ceil_div(M, 32), 256, 0, s>>>(amat_parts(ctx), M, y, idx);
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    return mark(ctx, 7, s);
}
int launch_amatvec(pcm_ctx *ctx, const double *q, double *y, cudaStream_t s) { return launch_amatvec_impl(ctx, q, y, true, s); }
int launch_amatvec_sorted(pcm_ctx *ctx, const double *q, double *y, cudaStream_t s) { return launch_amatvec_impl(ctx, q, y, false, s); }

// One class kernel; chained: with the programmatic-serialization attribute, i.e. it may start while the last wave of the launch
// before it on s is still running (see pdl_launch_dependents above; both kernels must be class kernels of the same call).
constexpr int64_t PDL_DENSITY_MAX = 16384;    // products up to which the density transforms of a call are chained
template <class... KArgs, class... Args>
static cudaError_t launch_class_b(void (*kernel)(KArgs...), dim3 grid, int block, cudaStream_t s, bool chained, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = chained ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
template <class... KArgs, class... Args>
static cudaError_t launch_class(void (*kernel)(KArgs...), dim3 grid, cudaStream_t s, bool chained, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(TPB);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = chained ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

template <int L>
static int launch_fock_near(pcm_ctx *ctx, const double *q, cudaStream_t s) {
    ClassData &c = ctx->cls[L];
    const PatchMap &pm = c.fock_map;
    if (c.n == 0 || pm.npiece == 0) return PCM_OK;
    fock_near_kernel<L><<<(unsigned)pm.npiece, TPB, 0, s>>>(
        c.prodA, c.prodB, c.npad, ctx->pt, q, ctx->s2c, (int)ctx->M, pm.start, pm.list, pm.pstart, pm.piece_rg, pm.npiece,
        c.near_fock, ctx->boys + (size_t)L * BOYS_ROWS * BOYS_STRIDE);
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    return PCM_OK;
}

template <int L>
static int launch_fock_class(pcm_ctx *ctx, const double *q, cudaStream_t s, bool chained = false) {
    constexpr Blocking fb = fock_blocking(L);
    ClassData &c = ctx->cls[L];
    if (c.n == 0) return PCM_OK;
    const Plan &pl = ctx->plan_fock[L];
    const PatchMap &pm = c.fock_map;
    dim3 grid((unsigned)pl.xb, (unsigned)pl.chunks);
    if (ctx->opt.tma_tiles && ctx->ptq)
        fock_tma_kernel<L, fb.R, fb.C><<<grid, TPB, 0, s>>>(c.prodA, c.npad, ctx->ptq, (int)ctx->M, (int)pl.chunk_len, c.herm, pm.far, pm.nbyte,
                                                            pm.nrg);
    else
        PCM_CUDA(ctx, launch_class(fock_kernel<L, fb.R, fb.C>, grid, s, chained, c.prodA, c.npad, ctx->pt, q, ctx->s2c, (int)ctx->M,
                                   (int)pl.chunk_len, c.herm, pm.far, pm.nbyte, pm.nrg));
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    return PCM_OK;
}

template <int L>
static int reduce_fock_class(pcm_ctx *ctx, cudaStream_t s, bool chained = false) {
    ClassData &c = ctx->cls[L];
    const int64_t chunks = ctx->plan_fock[L].chunks;
    if (c.n == 0) return PCM_OK;
    const int64_t plane = (int64_t)nherm(L) * c.npad;
    PCM_CUDA(ctx, launch_class_b(reduce_herm_kernel, dim3((unsigned)ceil_div(plane, 32)), 256, s, chained, c.herm, plane, (int)chunks, c.npad,
                                 nherm(L), (const double *)c.near_fock, (const int64_t *)c.fock_map.pstart));
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
        if (ctx->opt.tma_tiles && ctx->ptq) {   // (x, y, z, q) in sorted order: the regular tiles the bulk copies want
            pack_points_kernel<<<(unsigned)ceil_div(ctx->M, 256), 256, 0, s>>>(ctx->pt, q, ctx->s2c, (int)ctx->M, ctx->ptq);
            PCM_LAUNCH_CHECK(ctx);
            { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
        }
        // near kernels of all classes on the near stream, concurrently with the main kernels on s
        PCM_CUDA(ctx, cudaEventRecord(ctx->ev_fork, s));
        PCM_CUDA(ctx, cudaStreamWaitEvent(ctx->near_stream, ctx->ev_fork, 0));
        if ((rc = launch_fock_near<0>(ctx, q, ctx->near_stream))) return rc;
        if ((rc = launch_fock_near<1>(ctx, q, ctx->near_stream))) return rc;
        if ((rc = launch_fock_near<2>(ctx, q, ctx->near_stream))) return rc;
        if ((rc = launch_fock_near<3>(ctx, q, ctx->near_stream))) return rc;
        if ((rc = launch_fock_near<4>(ctx, q, ctx->near_stream))) return rc;
        PCM_CUDA(ctx, cudaEventRecord(ctx->ev_join, ctx->near_stream));
        if (ctx->timing || ctx->opt.serial_classes || (ctx->opt.tma_tiles && ctx->ptq)) {   // ordinary launches, per-class events
            if ((rc = launch_fock_class<0>(ctx, q, s)) || (rc = mark(ctx, 2, s))) return rc;
            if ((rc = launch_fock_class<1>(ctx, q, s)) || (rc = mark(ctx, 3, s))) return rc;
            if ((rc = launch_fock_class<2>(ctx, q, s)) || (rc = mark(ctx, 4, s))) return rc;
            if ((rc = launch_fock_class<3>(ctx, q, s)) || (rc = mark(ctx, 5, s))) return rc;
            if ((rc = launch_fock_class<4>(ctx, q, s)) || (rc = mark(ctx, 6, s))) return rc;
        } else {   // a chain of programmatic dependent launches, as in launch_potential
            bool ch = false;
            if ((rc = launch_fock_class<1>(ctx, q, s, ch))) return rc;
            ch = ch || ctx->cls[1].n > 0;
            if ((rc = launch_fock_class<0>(ctx, q, s, ch))) return rc;
            ch = ch || ctx->cls[0].n > 0;
            if ((rc = launch_fock_class<2>(ctx, q, s, ch))) return rc;
            ch = ch || ctx->cls[2].n > 0;
            if ((rc = launch_fock_class<3>(ctx, q, s, ch))) return rc;
            ch = ch || ctx->cls[3].n > 0;
            if ((rc = launch_fock_class<4>(ctx, q, s, ch))) return rc;
        }
        PCM_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_join, 0));
    } else {
        for (int i = 2; i <= 6; ++i)
            if ((rc = mark(ctx, i, s))) return rc;
    }
    if (!accumulate && ctx->nbf > 0)
        PCM_CUDA(ctx, cudaMemset2DAsync(F, (size_t)ldf * 8, 0, (size_t)ctx->nbf * 8, (size_t)ctx->nbf, s));
    if (ctx->M > 0 && ctx->ncomp > 0) {
        // the per-class reductions are independent of one another: a chain of programmatic dependent launches (each starts
        // as soon as the one before it is resident and waits for it before it exits), the pair transform after them an ordinary one
        const bool chain = !ctx->opt.serial_classes;      // serial_classes: ordinary launches throughout (the reference of the tests)
        bool ch = false;
        if ((rc = reduce_fock_class<0>(ctx, s, ch))) return rc;
        ch = chain && (ch || ctx->cls[0].n > 0);
        if ((rc = reduce_fock_class<1>(ctx, s, ch))) return rc;
        ch = chain && (ch || ctx->cls[1].n > 0);
        if ((rc = reduce_fock_class<2>(ctx, s, ch))) return rc;
        ch = chain && (ch || ctx->cls[2].n > 0);
        if ((rc = reduce_fock_class<3>(ctx, s, ch))) return rc;
        ch = chain && (ch || ctx->cls[3].n > 0);
        if ((rc = reduce_fock_class<4>(ctx, s, ch))) return rc;
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
static int launch_density_class(pcm_ctx *ctx, const double *P, int64_t ldp, cudaStream_t s, bool chained = false) {
    ClassData &c = ctx->cls[L];
    if (c.n == 0) return PCM_OK;
    if (L >= 2)
        PCM_CUDA(ctx, launch_class_b(density_to_hermite_warp_kernel<L>, dim3((unsigned)(c.npad / 4)), 128, s, chained, c.n, c.first, c.npad,
                                     (const int64_t *)ctx->pm_start, (const int32_t *)ctx->pm_list, (const int32_t *)ctx->m_sp,
                                     (const int32_t *)ctx->m_cls, (const int64_t *)ctx->m_goff, (const double *)ctx->G,
                                     (const int32_t *)ctx->sp_i0, (const int32_t *)ctx->sp_j0, (const int32_t *)ctx->sp_dims, P, ldp, c.herm));
    else
        PCM_CUDA(ctx, launch_class_b(density_to_hermite_kernel<L>, dim3((unsigned)(c.npad / 128)), 128, s, chained, c.n, c.first, c.npad,
                                     (const int64_t *)ctx->pm_start, (const int32_t *)ctx->pm_list, (const int32_t *)ctx->m_sp,
                                     (const int32_t *)ctx->m_cls, (const int64_t *)ctx->m_goff, (const double *)ctx->G,
                                     (const int32_t *)ctx->sp_i0, (const int32_t *)ctx->sp_j0, (const int32_t *)ctx->sp_dims, P, ldp, c.herm));
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    return PCM_OK;
}

template <int L>
static int launch_potential_near(pcm_ctx *ctx, cudaStream_t s) {
    ClassData &c = ctx->cls[L];
    const PatchMap &pm = c.pot_map;
    if (c.n == 0 || pm.npiece == 0) return PCM_OK;
    potential_near_kernel<L><<<(unsigned)pm.npiece, TPB, 0, s>>>(
        c.prodA, c.prodB, c.herm, c.npad, ctx->pt, (int)ctx->M, pm.start, pm.list, pm.pstart, pm.piece_rg, pm.npiece,
        c.near_pot, ctx->boys + (size_t)L * BOYS_ROWS * BOYS_STRIDE);
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    return PCM_OK;
}

// slot: first partial-sum slot of the class (fixed by the class order, whatever the launch order)
template <int L>
static int launch_potential_class(pcm_ctx *ctx, int64_t slot, cudaStream_t s, bool chained = false) {
    constexpr Blocking pb = pot_blocking(L);
    ClassData &c = ctx->cls[L];
    if (c.n == 0) return PCM_OK;
    const Plan &pl = ctx->plan_pot[L];
    const PatchMap &pm = c.pot_map;
    dim3 grid((unsigned)pl.xb, (unsigned)pl.chunks);
    if ((ctx->opt.potential_pr >> L) & 1) {
        potential_pr_kernel<L, (L <= 3 ? 16 : 8)><<<grid, TPB, 0, s>>>(c.prodA, c.herm, c.npad, (int)pl.chunk_len, ctx->pt, (int)ctx->M,
                                                                    ctx->vpart + (size_t)slot * ctx->M, c.fock_map.far, c.fock_map.nbyte);
        PCM_LAUNCH_CHECK(ctx);
        { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
        return PCM_OK;
    }
    constexpr Blocking pbb = pot_blocking_big(L);
    if (ctx->M >= POT_BIG_MIN && (pbb.R != pb.R || pbb.C != pb.C))
        PCM_CUDA(ctx, launch_class(potential_kernel<L, pbb.R, pbb.C>, grid, s, chained, c.prodA, c.herm, c.npad, (int)pl.chunk_len, ctx->pt,
                                   (int)ctx->M, ctx->vpart + (size_t)slot * ctx->M, pm.far, pm.nbyte, pm.nrg));
    else
        PCM_CUDA(ctx, launch_class(potential_kernel<L, pb.R, pb.C>, grid, s, chained, c.prodA, c.herm, c.npad, (int)pl.chunk_len, ctx->pt,
                                   (int)ctx->M, ctx->vpart + (size_t)slot * ctx->M, pm.far, pm.nbyte, pm.nrg));
    PCM_LAUNCH_CHECK(ctx);
    { ctx->launches[ctx->cur_op]++; ctx->launch_total++; }
    return PCM_OK;
}

int launch_potential(pcm_ctx *ctx, const double *P, int64_t ldp, double *v, cudaStream_t s) {
    ctx->cur_op = 0;
    ctx->launches[0] = 0;
    ctx->timed[0] = ctx->timing != 0;
    int rc;
    if (ctx->M == 0) return PCM_OK;
    if ((rc = mark(ctx, 0, s))) return rc;
    {   // The per-class transforms are independent of one another.  For small solutes, where a call is a string of launch
        // latencies, they form a chain of programmatic dependent launches (configs[0]: pcm_potential 96 -> 79 us); at 300 atoms
        // the chain measured 3 - 6 % slower for the whole call than three ordinary launches, so it stops at PDL_DENSITY_MAX products.
        const bool chain = ctx->nprod <= PDL_DENSITY_MAX && !ctx->opt.serial_classes;
        bool ch = false;
        if ((rc = launch_density_class<0>(ctx, P, ldp, s, ch))) return rc;
        ch = chain && (ch || ctx->cls[0].n > 0);
        if ((rc = launch_density_class<1>(ctx, P, ldp, s, ch))) return rc;
        ch = chain && (ch || ctx->cls[1].n > 0);
        if ((rc = launch_density_class<2>(ctx, P, ldp, s, ch))) return rc;
        ch = chain && (ch || ctx->cls[2].n > 0);
        if ((rc = launch_density_class<3>(ctx, P, ldp, s, ch))) return rc;
        ch = chain && (ch || ctx->cls[3].n > 0);
        if ((rc = launch_density_class<4>(ctx, P, ldp, s, ch))) return rc;
    }
    if ((rc = mark(ctx, 1, s))) return rc;
    // near kernels of all classes on the near stream (they need the Hermite densities), concurrently with the main kernels on s
    PCM_CUDA(ctx, cudaEventRecord(ctx->ev_fork, s));
    PCM_CUDA(ctx, cudaStreamWaitEvent(ctx->near_stream, ctx->ev_fork, 0));
    if ((rc = launch_potential_near<0>(ctx, ctx->near_stream))) return rc;
    if ((rc = launch_potential_near<1>(ctx, ctx->near_stream))) return rc;
    if ((rc = launch_potential_near<2>(ctx, ctx->near_stream))) return rc;
    if ((rc = launch_potential_near<3>(ctx, ctx->near_stream))) return rc;
    if ((rc = launch_potential_near<4>(ctx, ctx->near_stream))) return rc;
    PCM_CUDA(ctx, cudaEventRecord(ctx->ev_join, ctx->near_stream));
    int64_t base[MAXL + 2] = {0};
    for (int L = 0; L <= MAXL; ++L) base[L + 1] = base[L] + (ctx->cls[L].n > 0 ? ctx->plan_pot[L].chunks : 0);
    const int64_t slot = base[MAXL + 1];
    if (ctx->timing || ctx->opt.serial_classes || ctx->opt.potential_pr) {   // ordinary launches, one after the other, per-class events
        if ((rc = launch_potential_class<0>(ctx, base[0], s)) || (rc = mark(ctx, 2, s))) return rc;
        if ((rc = launch_potential_class<1>(ctx, base[1], s)) || (rc = mark(ctx, 3, s))) return rc;
        if ((rc = launch_potential_class<2>(ctx, base[2], s)) || (rc = mark(ctx, 4, s))) return rc;
        if ((rc = launch_potential_class<3>(ctx, base[3], s)) || (rc = mark(ctx, 5, s))) return rc;
        if ((rc = launch_potential_class<4>(ctx, base[4], s)) || (rc = mark(ctx, 6, s))) return rc;
    } else {
        // A chain of programmatic dependent launches on s (pdl_launch_dependents above): every class kernel after the first may
        // start while the last wave of the one before it is still running, so the tail of one class overlaps the body of the
        // next (PAPER.md:160 launches its per-class kernels sequentially).  The classes with the most work go first, the
        // shortest last: its tail is the only one left.  The partial-sum slots are fixed by the class order, not the launch order.
        bool ch = false;
        if ((rc = launch_potential_class<1>(ctx, base[1], s, ch))) return rc;
        ch = ch || ctx->cls[1].n > 0;
        if ((rc = launch_potential_class<0>(ctx, base[0], s, ch))) return rc;
        ch = ch || ctx->cls[0].n > 0;
        if ((rc = launch_potential_class<2>(ctx, base[2], s, ch))) return rc;
        ch = ch || ctx->cls[2].n > 0;
        if ((rc = launch_potential_class<3>(ctx, base[3], s, ch))) return rc;
        ch = ch || ctx->cls[3].n > 0;
        if ((rc = launch_potential_class<4>(ctx, base[4], s, ch))) return rc;
    }
    PCM_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_join, 0));
    if (slot == 0) {
        PCM_CUDA(ctx, cudaMemsetAsync(v, 0, (size_t)ctx->M * 8, s));
    } else {
        NearRefs nr;
        nr.count = 0;
        for (int L = 0; L <= MAXL; ++L)
            if (ctx->cls[L].n > 0) { nr.near[nr.count] = ctx->cls[L].near_pot; nr.pstart[nr.count] = ctx->cls[L].pot_map.pstart; nr.count++; }
        reduce_slots_kernel<<<(unsigned)ceil_div(ctx->M, 32), 256, 0, s>>>(ctx->vpart, ctx->M, (int)slot, v, ctx->s2c, nr);
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

#include "pcm_gradient.inl"

}  // namespace pcm
