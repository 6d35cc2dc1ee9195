// pcm_device.cuh -- device arithmetic shared by the three hot kernels: fp64 reciprocal square root,
// tabulated Boys function, and the Hermite Coulomb recursion R_tuv (McMurchie-Davidson) with the
// effective exponent rho = p zeta^2/(p + zeta^2) of the smeared-charge operator (Eq. 6).
#pragma once

#include "pcm_internal.h"

namespace pcm {

__device__ __forceinline__ int hi32(double x) { return __double2hiint(x); }

// 1/sqrt(x), x > 0 normal.  MUFU.RSQ64H seed (2^-22.9 relative) + one third-order step:
// y <- y (1 + e/2 + 3 e^2/8), e = 1 - x y^2; remaining error 5 e^3/16 ~ 2^-70, i.e. rounding only.
__device__ __forceinline__ double rsqrt_fast(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double h = x * y;
    const double e = fma(-h, y, 1.0);
    const double t = fma(e, 0.375, 0.5);
    const double ye = y * e;
    return fma(ye, t, y);
}

// Partial sums of y = A q as the symmetric sweep leaves them (pcm_kernels.cu, amatvec_kernel): row slots
// ypart[chunk][k] for the chunks that reach the row block of k, column sums colpart[rb][k] of the row blocks lying
// wholly before the tile of k, and the near pieces of k's row group.  Summed in this fixed order.
struct AmatParts {
    const double *ypart, *colpart, *near;
    const int64_t *pstart;
    int slots, chunk_len, RB, tile;
};
// A 256-thread block sums the rows k0 .. k0+31: warp `part` (0..7) of the block adds, for row k0 + lane, every 8th term
// of each of the three lists (coalesced across the lanes), the eight partial sums are then added in order by warp 0.
// Returns the row sum in the threads of warp 0 (0.0 for rows >= M); s_tmp: shared, 8 * 32 doubles; all 256 threads call.
constexpr int AMAT_RED_PARTS = 8;
__device__ __forceinline__ double amat_row_sum_block(const AmatParts &a, int M, int k0, double *s_tmp) {
    const int lane = threadIdx.x & 31, part = threadIdx.x >> 5;
    const int k = k0 + lane;
    double s = 0.0;
    if (k < M) {
        const int r0 = k / a.RB * a.RB;
        // four loads in flight per loop (the partial sums come from L2), same summation order
        int c = r0 / a.chunk_len + part;
        for (; c + 3 * AMAT_RED_PARTS < a.slots; c += 4 * AMAT_RED_PARTS) {
            const double v0 = a.ypart[(size_t)c * M + k], v1 = a.ypart[(size_t)(c + AMAT_RED_PARTS) * M + k],
                         v2 = a.ypart[(size_t)(c + 2 * AMAT_RED_PARTS) * M + k], v3 = a.ypart[(size_t)(c + 3 * AMAT_RED_PARTS) * M + k];
            s += v0; s += v1; s += v2; s += v3;
        }
        for (; c < a.slots; c += AMAT_RED_PARTS) s += a.ypart[(size_t)c * M + k];
        const int nsym = (k / a.tile * a.tile) / a.RB;
        int rb = part;
        for (; rb + 3 * AMAT_RED_PARTS < nsym; rb += 4 * AMAT_RED_PARTS) {
            const double v0 = a.colpart[(size_t)rb * M + k], v1 = a.colpart[(size_t)(rb + AMAT_RED_PARTS) * M + k],
                         v2 = a.colpart[(size_t)(rb + 2 * AMAT_RED_PARTS) * M + k], v3 = a.colpart[(size_t)(rb + 3 * AMAT_RED_PARTS) * M + k];
            s += v0; s += v1; s += v2; s += v3;
        }
        for (; rb < nsym; rb += AMAT_RED_PARTS) s += a.colpart[(size_t)rb * M + k];
        const int64_t rg = k / 32;
        for (int64_t e = a.pstart[rg] + part; e < a.pstart[rg + 1]; e += AMAT_RED_PARTS) s += a.near[e * 32 + lane];
    }
    s_tmp[part * 32 + lane] = s;
    __syncthreads();
    double t = 0.0;
    if (part == 0) {
#pragma unroll
        for (int q = 0; q < AMAT_RED_PARTS; ++q) t += s_tmp[q * 32 + lane];
    }
    return t;
}

AmatParts amat_parts(const pcm_ctx *ctx);  // pcm_kernels.cu

// Far-field Hermite seeds, normalised so that g_n = (-1)^n (2n-1)!! / R^(2n+1)  (derivatives of 1/R):
// for T >= TFAR(L) the smeared charge is a point charge to fp64 and
//   (2 pi/p) sqrt(rho/p) (-2 rho)^n F_n(T) = (pi/p)^{3/2} K^-1 ... = [ (2 pi/p) kappa ] g_n,  kappa = sqrt(pi/p)/2.
template <int L>
__device__ __forceinline__ void seeds_far(double R2, double (&g)[L + 1]) {
    const double ri = rsqrt_fast(R2);
    g[0] = ri;
    if (L > 0) {
        const double u = ri * ri;
#pragma unroll
        for (int n = 1; n <= L; ++n) g[n] = g[n - 1] * (u * (double)(-(2 * n - 1)));
    }
}
// the same seeds times a common factor w (the point's charge in the Fock sweep): one multiplication instead of L + 1
template <int L>
__device__ __forceinline__ void seeds_far_scaled(double R2, double w, double (&g)[L + 1]) {
    const double ri = rsqrt_fast(R2);
    g[0] = ri * w;
    if (L > 0) {
        const double u = ri * ri;
#pragma unroll
        for (int n = 1; n <= L; ++n) g[n] = g[n - 1] * (u * (double)(-(2 * n - 1)));
    }
}

// General seeds: g_n = (w/kappa) (-2 rho)^n F_n(rho R2), w = sqrt(rho/p) = 1/sqrt(1 + p/zeta^2).
// F_L by an 8-term Taylor expansion about the nearest table row, lower orders by downward recursion
// F_{n-1} = (2T F_n + exp(-T))/(2n-1); beyond the switch the far-field form.
template <int L>
__device__ __forceinline__ void seeds_general(double R2, double p, double invk, double iz2,
                                               const double *__restrict__ boysL, double (&g)[L + 1]) {
    const double w = rsqrt_fast(fma(p, iz2, 1.0));
    const double rho = p * w * w;
    const double T = rho * R2;
    if (T >= tfar(L)) {
        seeds_far<L>(R2, g);
        return;
    }
    const int i = __double2int_rn(T * 16.0);
    const double d = T - (double)i * 0.0625;
    const double *row = boysL + (size_t)i * BOYS_STRIDE;
    double f = __ldg(row + BOYS_TERMS - 1);
#pragma unroll
    for (int k = BOYS_TERMS - 2; k >= 0; --k) f = fma(f, d, __ldg(row + k));
    double F[L + 1];
    F[L] = f;
    if (L > 0) {
        // exp(-T) = exp(-T_i) exp(-d), |d| <= 1/32: degree-8 Taylor polynomial (next term 8e-20)
        double e = 1.0 / 40320.0;
        e = fma(e, -d, 1.0 / 5040.0);
        e = fma(e, -d, 1.0 / 720.0);
        e = fma(e, -d, 1.0 / 120.0);
        e = fma(e, -d, 1.0 / 24.0);
        e = fma(e, -d, 1.0 / 6.0);
        e = fma(e, -d, 0.5);
        e = fma(e, -d, 1.0);
        e = fma(e, -d, 1.0);
        e *= __ldg(row + BOYS_TERMS);
        const double T2 = T + T;
#pragma unroll
        for (int n = L; n >= 1; --n) F[n - 1] = fma(T2, F[n], e) * (1.0 / (double)(2 * n - 1));
    }
    double s = w * invk;
    const double m2r = -2.0 * rho;
#pragma unroll
    for (int n = 0; n <= L; ++n) {
        g[n] = s * F[n];
        s *= m2r;
    }
}

// ---------------------------------------------------------------------------------------------
// Hermite Coulomb integrals from the seeds:  R^n_000 = g_n,
//   R^n_{t+1,u,v} = t R^{n+1}_{t-1,u,v} + x R^{n+1}_{t,u,v}   (and likewise for u, v), (x,y,z) = P - C.
// All loops have compile-time bounds: after unrolling every index is a constant and the arrays live in
// registers.  The direction lowered is the one with the smallest non-zero power (a power of 1 or 2
// costs one instruction, 3 or 4 costs two).
// The order-0 integrals are handed to `sink` once per component h = hidx(t,u,v): sink.value(h, t, u, v, R) or, when R
// is a single product a*b, sink.product(h, t, u, v, a, b) so that the consumer can fuse it into an FMA.
// ---------------------------------------------------------------------------------------------
__host__ __device__ constexpr int pick_dir(int t, int u, int v) {
    int best = -1, bp = 99;
    if (t > 0 && t < bp) { best = 0; bp = t; }
    if (u > 0 && u < bp) { best = 1; bp = u; }
    if (v > 0 && v < bp) { best = 2; bp = v; }
    return best;
}

template <int L, class Sink>
__device__ __forceinline__ void hermite_R(double x, double y, double z, const double (&g)[L + 1], Sink &sink) {
    constexpr int NH = nherm(L);
    double R[L + 1][NH];  // R[n][h] for degree(h) <= L - n; unused entries are never materialised
#pragma unroll
    for (int n = 0; n <= L; ++n) R[n][0] = g[n];
    sink.value(0, 0, 0, 0, R[0][0]);
#pragma unroll
    for (int d = 1; d <= L; ++d) {
#pragma unroll
        for (int n = L - d; n >= 0; --n) {
#pragma unroll
            for (int t = d; t >= 0; --t) {
#pragma unroll
                for (int u = d - t; u >= 0; --u) {
                    const int v = d - t - u;
                    const int dir = pick_dir(t, u, v);
                    const int pw = dir == 0 ? t : (dir == 1 ? u : v);          // power being lowered
                    const double c = dir == 0 ? x : (dir == 1 ? y : z);
                    const int h1 = dir == 0 ? hidx(t - 1, u, v) : (dir == 1 ? hidx(t, u - 1, v) : hidx(t, u, v - 1));
                    const int h2 = pw < 2 ? 0 : (dir == 0 ? hidx(t - 2, u, v) : (dir == 1 ? hidx(t, u - 2, v) : hidx(t, u, v - 2)));
                    const int h = hidx(t, u, v);
                    if (pw == 1) {
                        if (n == 0) sink.product(h, t, u, v, c, R[n + 1][h1]);
                        else R[n][h] = c * R[n + 1][h1];
                    } else if (n == 0 && Sink::kSplit) {
                        // a sink that accumulates: acc_h += c R1_h1 now, and (pw - 1) x [sum over evaluations of R1_h2] at the end
                        // (hermite_lower / hermite_fixup) -- the "lower" terms of many components are the same few values
                        sink.product(h, t, u, v, c, R[n + 1][h1]);
                    } else {
                        const double lower = (pw == 2) ? R[n + 1][h2] : (double)(pw - 1) * R[n + 1][h2];
                        const double val = fma(c, R[n + 1][h1], lower);
                        if (n == 0) sink.value(h, t, u, v, val);
                        else R[n][h] = val;
                    }
                }
            }
        }
    }
    if (Sink::kSplit && L >= 2) {   // the lower terms of the order-0 integrals: R^1_h2 for every h2 of degree <= L - 2, once each
#pragma unroll
        for (int h2 = 0; h2 < nherm(L >= 2 ? L - 2 : 0); ++h2) sink.lower(h2, R[1][h2]);
    }
}

// For a split sink: acc[h] += (pw - 1) x accL[h2] for every component whose lowered power pw is >= 2 (the same pick_dir walk)
template <int L>
__device__ __forceinline__ void hermite_fixup(double (&acc)[nherm(L)], const double (&accL)[nherm(L >= 2 ? L - 2 : 0)]) {
#pragma unroll
    for (int d = 2; d <= L; ++d)
#pragma unroll
        for (int t = d; t >= 0; --t)
#pragma unroll
            for (int u = d - t; u >= 0; --u) {
                const int v = d - t - u;
                const int dir = pick_dir(t, u, v);
                const int pw = dir == 0 ? t : (dir == 1 ? u : v);
                if (pw >= 2) {
                    const int h2 = dir == 0 ? hidx(t - 2, u, v) : (dir == 1 ? hidx(t, u - 2, v) : hidx(t, u, v - 2));
                    acc[hidx(t, u, v)] = fma((double)(pw - 1), accL[h2], acc[hidx(t, u, v)]);
                }
            }
}

}  // namespace pcm
