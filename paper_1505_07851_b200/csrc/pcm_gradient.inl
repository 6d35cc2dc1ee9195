// pcm_gradient.inl -- pcm_gradient: the one-electron PCM gradient term (grad* c^T) q of Eq. 14 / Eq. 22
// (PAPER.md:88, 202-218), included at the end of pcm_kernels.cu (inside namespace pcm; it reuses that file's kernels).
//
// In the Hermite formulation E = v.q = sum_k q_k sum_products sum_h D_h Rt_h(P - C_k), and
// d/dx Rt_tuv = Rt_{t+1,u,v}.  With H'_h(product) = sum_k q_k Rt_h(P - C_k) for h up to degree L + 1:
//   point k      (gc of Eq. 22):  dE/dC_k,x = -q_k sum_products sum_h D_h Rt_{h+1x}(P - C_k)      -- grad_point_kernel<L>
//   bra centre A (ga):  dE/dA_x = sum_ab Pw_ab [ (alpha/p) sum_h G[ab][h] H'_{h+1x} + sum_h dG[ab][x][h] H'_h ]
//   ket centre B (gb):  dE/dB_x = sum_ab Pw_ab [ (beta/p)  sum_h G[ab][h] H'_{h+1x} - sum_h dG[ab][x][h] H'_h ]
// because P = (alpha A + beta B)/p moves with weight alpha/p and the expansion coefficients depend on A - B only
// (dG = dG/dX_AB at fixed P, built by pcm_setup from the differentiated E recursion).  H' is the Fock kernel of
// pcm_kernels.cu run one order higher (fock_kernel<L + 1> on the class-L products), so the paper's "hybrid of the
// pair-driven and the point-driven kernels" is here two sweeps that share nothing but q and D.
// Every reduction has a fixed order (slots, pieces, components, shell pairs): the result is bit-reproducible.

// ---------------------------------------------------------------------------------------------
// point side: three accumulators per point, Hermite integrals to order L + 1 contracted with D shifted by one
// ---------------------------------------------------------------------------------------------
template <int L>
struct PotGradSink {
    static constexpr bool kSplit = false;
    __device__ __forceinline__ void lower(int, double) {}
    const double *D;   // D_h of the product, h < nherm(L)
    double gx, gy, gz;
    __device__ __forceinline__ void value(int, int t, int u, int v, double x) {
        if (t > 0) gx = fma(D[hidx(t > 0 ? t - 1 : 0, u, v)], x, gx);
        if (u > 0) gy = fma(D[hidx(t, u > 0 ? u - 1 : 0, v)], x, gy);
        if (v > 0) gz = fma(D[hidx(t, u, v > 0 ? v - 1 : 0)], x, gz);
    }
    __device__ __forceinline__ void product(int h, int t, int u, int v, double a, double b) { value(h, t, u, v, a * b); }
};

__host__ __device__ constexpr Blocking gpoint_blocking(int L) {
    return L == 0 ? Blocking{4, 1} : L == 1 ? Blocking{2, 1} : L == 2 ? Blocking{1, 2} : Blocking{1, 1};
}

template <int L>
__device__ __forceinline__ void pot_grad_far_unit(const double *rec, const double4 &c, double (&g)[3]) {
    const double2 h01 = *reinterpret_cast<const double2 *>(rec);
    const double x = h01.x - c.x, y = h01.y - c.y, z = rec[2] - c.z;
    double s[L + 2];
    seeds_far<L + 1>(fma(z, z, fma(y, y, x * x)), s);
    PotGradSink<L> sink{rec + 4, g[0], g[1], g[2]};
    hermite_R<L + 1>(x, y, z, s, sink);
    g[0] = sink.gx; g[1] = sink.gy; g[2] = sink.gz;
}

// Classes L = 0, 1, 2 (all of an s/p basis) without the Hermite recursion: the far unit of the potential is g0 F(u, r),
// g0 = 1/R, u = 1/R^2, F = D_0 - u (D_1.r + tr) + 3 u^2 Q_2(r) (pot_far_unit<1>, <2>), and with dg0/dr = -u g0 r, du/dr = -2 u^2 r
//   sum_h D_h Rt_{h+1_d} = d/dr_d [g0 F] = g0 u [ -r_d (D_0 - 3 u (D_1.r + tr) + 15 u^2 Q_2) - D_1,d + 3 u dQ_2/dr_d ]
// (the odd double factorials 1, 3, 15 again).  17 / 24 / 45 FP64 instructions instead of 21 / 40 / 75.
template <>
__device__ __forceinline__ void pot_grad_far_unit<0>(const double *rec, const double4 &c, double (&g)[3]) {
    const double2 h01 = *reinterpret_cast<const double2 *>(rec);
    const double x = h01.x - c.x, y = h01.y - c.y, z = rec[2] - c.z;
    const double ri = rsqrt_fast(fma(z, z, fma(y, y, x * x)));
    const double t = -(ri * ri) * (ri * rec[4]);
    g[0] = fma(t, x, g[0]); g[1] = fma(t, y, g[1]); g[2] = fma(t, z, g[2]);
}
template <>
__device__ __forceinline__ void pot_grad_far_unit<1>(const double *rec, const double4 &c, double (&g)[3]) {
    const double2 h01 = *reinterpret_cast<const double2 *>(rec);
    const double x = h01.x - c.x, y = h01.y - c.y, z = rec[2] - c.z;
    const double ri = rsqrt_fast(fma(z, z, fma(y, y, x * x)));
    const double u = ri * ri;
    const double s = fma(rec[5], x, fma(rec[6], y, rec[7] * z));
    const double a = fma(u * -3.0, s, rec[4]);           // D_0 - 3 u D_1.r
    const double mc = -(ri * u);                         // -g0 u
    g[0] = fma(mc, fma(x, a, rec[5]), g[0]);
    g[1] = fma(mc, fma(y, a, rec[6]), g[1]);
    g[2] = fma(mc, fma(z, a, rec[7]), g[2]);
}
template <>
__device__ __forceinline__ void pot_grad_far_unit<2>(const double *rec, const double4 &c, double (&g)[3]) {
    const double2 h01 = *reinterpret_cast<const double2 *>(rec);
    const double x = h01.x - c.x, y = h01.y - c.y, z = rec[2] - c.z;
    const double ri = rsqrt_fast(fma(z, z, fma(y, y, x * x)));
    const double u = ri * ri;
    const double *D = rec + 4;   // 4 = (2,0,0), 5 = (1,1,0), 6 = (1,0,1), 7 = (0,2,0), 8 = (0,1,1), 9 = (0,0,2)
    const double qx = fma(D[4] + D[4], x, fma(D[5], y, D[6] * z));   // dQ_2/dx
    const double qy = fma(D[5], x, fma(D[7] + D[7], y, D[8] * z));
    const double qz = fma(D[6], x, fma(D[8], y, (D[9] + D[9]) * z));
    const double q2 = 0.5 * fma(x, qx, fma(y, qy, z * qz));          // Euler: r.dQ_2/dr = 2 Q_2
    const double lin = fma(D[1], x, fma(D[2], y, fma(D[3], z, (D[4] + D[7]) + D[9])));
    const double a = fma(u, fma(u * 15.0, q2, -3.0 * lin), D[0]);    // D_0 - 3 u lin + 15 u^2 Q_2
    const double u3 = u * 3.0, mc = -(ri * u);
    g[0] = fma(mc, fma(x, a, fma(-u3, qx, D[1])), g[0]);
    g[1] = fma(mc, fma(y, a, fma(-u3, qy, D[2])), g[1]);
    g[2] = fma(mc, fma(z, a, fma(-u3, qz, D[3])), g[2]);
}

// far patches: rows = R points per thread, columns = products of class L staged in shared memory (as potential_kernel)
template <int L, int R, int C>
__global__ void __launch_bounds__(TPB) grad_point_kernel(const double4 *__restrict__ prodA, const double *__restrict__ herm,
                                                         int64_t npad, int chunk_len, const double4 *__restrict__ pt, int M,
                                                         double *__restrict__ gpart, const uint8_t *__restrict__ farmap,
                                                         int64_t nbyte, int64_t nrg) {
    constexpr int NH = nherm(L);
    constexpr int REC = pot_rec<L>();
    constexpr int TILE = pot_tile(L), NS = TILE / SUB;
    __shared__ __align__(16) double s_rec[TILE * REC];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t rg0 = ((int64_t)blockIdx.x * (TPB / 32) + warp) * R;
    double4 c[R];
    int kk[R];
    double g[R][3];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        kk[r] = (int)(rg0 + r) * SUB + lane;
        c[r] = pt[min(kk[r], M - 1)];
        g[r][0] = g[r][1] = g[r][2] = 0.0;
    }
    const int64_t pbeg = (int64_t)blockIdx.y * chunk_len, pend = min(npad, pbeg + (int64_t)chunk_len);
    for (int64_t base = pbeg; base < pend; base += TILE) {
        const int cnt = (int)min((int64_t)TILE, pend - base), nst = cnt / SUB;
        const unsigned bits = far_bits<R, NS>(farmap, nbyte, rg0, nrg, base / SUB, lane);
        __syncthreads();
        for (int t = threadIdx.x; t < cnt; t += TPB) {
            const double4 a = prodA[base + t];
            double *r = s_rec + t * REC;
            r[0] = a.x; r[1] = a.y; r[2] = a.z; r[3] = 0.0;
        }
        for (int t = threadIdx.x; t < cnt * NH; t += TPB) {
            const int h = t / cnt, i = t - h * cnt;
            s_rec[i * REC + 4 + h] = herm[(size_t)h * npad + base + i];
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
                        for (int r = 0; r < R; ++r) pot_grad_far_unit<L>(sr + (t + cc) * REC, c[r], g[r]);
                }
            } else if (R > 1 && m) {
#pragma unroll 1
                for (int t = 0; t < SUB; ++t) {
#pragma unroll
                    for (int r = 0; r < R; ++r)
                        if ((m >> r) & 1u) pot_grad_far_unit<L>(sr + t * REC, c[r], g[r]);
                }
            }
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r)
        if (kk[r] < M) {
#pragma unroll
            for (int d = 0; d < 3; ++d) gpart[((size_t)blockIdx.y * 3 + d) * M + kk[r]] = g[r][d];
        }
}

// near patches: one warp per piece of the class's potential patch map; lane = point.  Writes near[piece][3][lane].
template <int L>
__global__ void __launch_bounds__(TPB) grad_point_near_kernel(const double4 *__restrict__ prodA, const double2 *__restrict__ prodB,
                                                              const double *__restrict__ herm, int64_t npad,
                                                              const double4 *__restrict__ pt, int M,
                                                              const int64_t *__restrict__ start, const int32_t *__restrict__ list,
                                                              const int64_t *__restrict__ pstart, const int32_t *__restrict__ piece_rg,
                                                              int64_t npiece, double *__restrict__ near,
                                                              const double *__restrict__ boysL1) {
    constexpr int NH = nherm(L);
    constexpr int REC = pot_rec_near<L>();
    __shared__ __align__(16) double s_rec[TPB / 32][SUB * REC];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t piece = (int64_t)blockIdx.x * (TPB / 32) + warp;
    if (piece >= npiece) return;
    const int64_t rg = piece_rg[piece];
    const int k = (int)rg * SUB + lane;
    const double4 c = pt[min(k, M - 1)];
    double g[3] = {0.0, 0.0, 0.0};
    const int64_t ebeg = start[rg] + (piece - pstart[rg]) * NEAR_PIECE, eend = min(start[rg + 1], ebeg + NEAR_PIECE);
    double *mine = s_rec[warp];
    for (int64_t e = ebeg; e < eend; ++e) {
        const int64_t i0 = (int64_t)list[e] * SUB;
        __syncwarp();
        {
            const double4 a = prodA[i0 + lane];
            const double2 b = prodB[i0 + lane];
            double *r = mine + lane * REC;
            r[0] = a.x; r[1] = a.y; r[2] = a.z; r[3] = a.w;
            r[4 + NH] = b.x; r[5 + NH] = b.y;
#pragma unroll
            for (int h = 0; h < NH; ++h) r[4 + h] = herm[(size_t)h * npad + i0 + lane];
        }
        __syncwarp();
#pragma unroll 1
        for (int t = 0; t < SUB; ++t) {
            const double *rec = mine + t * REC;
            const double2 h01 = *reinterpret_cast<const double2 *>(rec);
            const double2 h23 = *reinterpret_cast<const double2 *>(rec + 2);
            const double x = h01.x - c.x, y = h01.y - c.y, z = h23.x - c.z;
            const double r2 = fma(z, z, fma(y, y, x * x));
            double s[L + 2];
            if (hi32(r2) > hi32(h23.y)) seeds_far<L + 1>(r2, s);
            else seeds_general<L + 1>(r2, rec[4 + NH], rec[5 + NH], c.w, boysL1, s);
            PotGradSink<L> sink{rec + 4, g[0], g[1], g[2]};
            hermite_R<L + 1>(x, y, z, s, sink);
            g[0] = sink.gx; g[1] = sink.gy; g[2] = sink.gz;
        }
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) near[((size_t)piece * 3 + d) * SUB + lane] = g[d];
}

// g_point[3 s2c[k] + d] = -q_k (sum of the slots + the near pieces of point k); q in the caller's order.  A 256-thread
// block sums 32 points: warp w adds every 8th slot and every 8th near piece, the eight partial sums are added in order.
__global__ void __launch_bounds__(256) grad_point_reduce_kernel(const double *__restrict__ gpart, int64_t M, int slots,
                                                                const double *__restrict__ q, const int32_t *__restrict__ s2c,
                                                                NearRefs nr, double *__restrict__ g_point) {
    __shared__ double s_tmp[3][8 * 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t k = (int64_t)blockIdx.x * 32 + lane;
    double s[3] = {0.0, 0.0, 0.0};
    if (k < M) {
        const int64_t rg = k / SUB;
        for (int d = 0; d < 3; ++d) {
            for (int c = w; c < slots; c += 8) s[d] += gpart[((size_t)c * 3 + d) * M + k];
            for (int c = 0; c < nr.count; ++c)
                for (int64_t e = nr.pstart[c][rg] + w; e < nr.pstart[c][rg + 1]; e += 8) s[d] += nr.near[c][((size_t)e * 3 + d) * SUB + lane];
        }
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) s_tmp[d][w * 32 + lane] = s[d];
    __syncthreads();
    if (w == 0 && k < M) {
        const int32_t kc = s2c[k];
        const double mq = -q[kc];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double t = 0.0;
#pragma unroll
            for (int p = 0; p < 8; ++p) t += s_tmp[d][p * 32 + lane];
            g_point[(size_t)kc * 3 + d] = mq * t;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// pair side: from H' (order L + 1) to the shell centres
// ---------------------------------------------------------------------------------------------
// thread = one component (a, b) of one shell pair: gcomp[c][0..2] = dE/dA, [3..5] = dE/dB contributed by P_ab (+ P_ba)
__global__ void grad_pair_kernel(int64_t ncomp, const int32_t *__restrict__ c_sp, const int32_t *__restrict__ c_ab,
                                 const int64_t *__restrict__ sp_mstart, const int32_t *__restrict__ m_prod,
                                 const int32_t *__restrict__ m_cls, const int64_t *__restrict__ m_goff,
                                 const double *__restrict__ m_ap, const double *__restrict__ G, const double *__restrict__ dG,
                                 const int32_t *__restrict__ sp_i0, const int32_t *__restrict__ sp_j0,
                                 const int32_t *__restrict__ sp_dims, const int32_t *__restrict__ hshift, ClassPtrs cp,
                                 const double *__restrict__ P, int64_t ldp, double *__restrict__ gcomp) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncomp) return;
    constexpr int NHM = nherm(MAXL);
    const int sp = c_sp[c], ab = c_ab[c];
    const int dims = sp_dims[sp], nb = (dims >> 8) & 0xff, diag = dims >> 16;
    const int a = ab / nb, b = ab - a * nb;
    const size_t mu = (size_t)sp_i0[sp] + a, nu = (size_t)sp_j0[sp] + b;
    double pw = P[mu * ldp + nu];
    if (!diag) pw += P[nu * ldp + mu];
    double gA[3] = {0.0, 0.0, 0.0}, gB[3] = {0.0, 0.0, 0.0};
    for (int64_t m = sp_mstart[sp]; m < sp_mstart[sp + 1]; ++m) {
        const int cl = m_cls[m], Lm = cl & 0xff, Lp = cl >> 8;
        const int nhm = (Lm + 1) * (Lm + 2) * (Lm + 3) / 6;
        const double *row = G + m_goff[m] + (size_t)ab * nhm;
        const double *drow = dG + 3 * m_goff[m] + (size_t)ab * 3 * nhm;
        const double *H = cp.herm[Lp] + (m_prod[m] - cp.first[Lp]);
        const int64_t np = cp.npad[Lp];
        const double ap = m_ap[m];
        for (int d = 0; d < 3; ++d) {
            double S = 0.0, T = 0.0;
            for (int h = 0; h < nhm; ++h) {
                S = fma(row[h], H[(size_t)hshift[d * NHM + h] * np], S);
                T = fma(drow[d * nhm + h], H[(size_t)h * np], T);
            }
            gA[d] += fma(ap, S, T);
            gB[d] += fma(1.0 - ap, S, -T);
        }
    }
    double *out = gcomp + (size_t)c * 6;
#pragma unroll
    for (int d = 0; d < 3; ++d) { out[d] = pw * gA[d]; out[3 + d] = pw * gB[d]; }
}

// gsp[sp][e] = sum over the components of shell pair sp, in component order
__global__ void grad_sp_reduce_kernel(int64_t nsp, const int64_t *__restrict__ sp_cstart, const double *__restrict__ gcomp,
                                      double *__restrict__ gsp) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nsp * 6) return;
    const int64_t sp = i / 6, e = i - sp * 6;
    double s = 0.0;
    for (int64_t c = sp_cstart[sp]; c < sp_cstart[sp + 1]; ++c) s += gcomp[(size_t)c * 6 + e];
    gsp[i] = s;
}

// g_shell[S][d] = sum over the shell pairs containing S (bra side: dE/dA, ket side: dE/dB), in list order
__global__ void grad_shell_reduce_kernel(int64_t nshell, const int64_t *__restrict__ sh_start, const int32_t *__restrict__ sh_list,
                                         const double *__restrict__ gsp, double *__restrict__ g_shell) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nshell * 3) return;
    const int64_t S = i / 3, d = i - S * 3;
    double s = 0.0;
    for (int64_t e = sh_start[S]; e < sh_start[S + 1]; ++e) {
        const int32_t v = sh_list[e];
        s += gsp[(size_t)(v >> 1) * 6 + (v & 1) * 3 + d];
    }
    g_shell[i] = s;
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
template <int L>
static void grad_plan_class(pcm_ctx *ctx) {
    constexpr Blocking fb = fock_blocking(L + 1), pb = gpoint_blocking(L);
    const ClassData &c = ctx->cls[L];
    ctx->plan_gfock[L] = make_plan(c.npad, TPB * fb.R, ctx->M, PT_TILE, wave_of(ctx, fock_kernel<L + 1, fb.R, fb.C>));
    ctx->plan_gpoint[L] = make_plan(ctx->M, TPB * pb.R, c.npad, pot_tile(L), wave_of(ctx, grad_point_kernel<L, pb.R, pb.C>));
}

// plans and scratch of pcm_gradient, once per context (at its first call)
static int grad_prepare(pcm_ctx *ctx) {
    if (ctx->grad_ready) return PCM_OK;
    grad_plan_class<0>(ctx); grad_plan_class<1>(ctx); grad_plan_class<2>(ctx); grad_plan_class<3>(ctx); grad_plan_class<4>(ctx);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_error(ctx, PCM_ERR_CUDA, std::string("grad_prepare: ") + cudaGetErrorString(e));
    int rc;
    const int64_t M = std::max<int64_t>(ctx->M, 1);
    ctx->gpart_slots = 0;
    for (int L = 0; L <= MAXL; ++L) {
        ClassData &c = ctx->cls[L];
        if (c.n == 0) continue;
        const size_t nh1 = (size_t)nherm(L + 1);
        if ((rc = dev_alloc_t(ctx, &c.gherm, (size_t)ctx->plan_gfock[L].chunks * nh1 * c.npad))) return rc;
        if ((rc = dev_alloc_t(ctx, &c.near_gfock, (size_t)c.fock_map.npiece * nh1 * 32))) return rc;
        if ((rc = dev_alloc_t(ctx, &c.near_gpoint, (size_t)c.pot_map.npiece * 3 * 32))) return rc;
        ctx->gpart_slots += ctx->plan_gpoint[L].chunks;
    }
    if ((rc = dev_alloc_t(ctx, &ctx->gpart, (size_t)std::max<int64_t>(ctx->gpart_slots, 1) * 3 * M))) return rc;
    if ((rc = dev_alloc_t(ctx, &ctx->gcomp, (size_t)std::max<int64_t>(ctx->ncomp, 1) * 6))) return rc;
    if ((rc = dev_alloc_t(ctx, &ctx->gsp, (size_t)std::max<int64_t>(ctx->nsp, 1) * 6))) return rc;
    ctx->info.device_bytes = ctx->device_bytes;
    ctx->grad_ready = true;
    return PCM_OK;
}

template <int L>
static int grad_launch_near(pcm_ctx *ctx, const double *q, cudaStream_t s) {
    ClassData &c = ctx->cls[L];
    if (c.n == 0) return PCM_OK;
    const double *boysL1 = ctx->boys + (size_t)(L + 1) * BOYS_ROWS * BOYS_STRIDE;
    if (c.pot_map.npiece > 0) {
        const PatchMap &pm = c.pot_map;
        grad_point_near_kernel<L><<<(unsigned)ceil_div(pm.npiece, TPB / 32), TPB, 0, s>>>(
            c.prodA, c.prodB, c.herm, c.npad, ctx->pt, (int)ctx->M, pm.start, pm.list, pm.pstart, pm.piece_rg, pm.npiece,
            c.near_gpoint, boysL1);
        PCM_LAUNCH_CHECK(ctx);
        ctx->launch_total++;
    }
    if (c.fock_map.npiece > 0) {
        const PatchMap &pm = c.fock_map;
        fock_near_kernel<L + 1><<<(unsigned)pm.npiece, TPB, 0, s>>>(
            c.prodA, c.prodB, c.npad, ctx->pt, q, ctx->s2c, (int)ctx->M, pm.start, pm.list, pm.pstart, pm.piece_rg, pm.npiece,
            c.near_gfock, boysL1);
        PCM_LAUNCH_CHECK(ctx);
        ctx->launch_total++;
    }
    return PCM_OK;
}

template <int L>
static int grad_launch_main(pcm_ctx *ctx, const double *q, int64_t &slot, cudaStream_t s) {
    constexpr Blocking fb = fock_blocking(L + 1), pb = gpoint_blocking(L);
    ClassData &c = ctx->cls[L];
    if (c.n == 0) return PCM_OK;
    {
        const Plan &pl = ctx->plan_gpoint[L];
        const PatchMap &pm = c.pot_map;
        dim3 grid((unsigned)pl.xb, (unsigned)pl.chunks);
        grad_point_kernel<L, pb.R, pb.C><<<grid, TPB, 0, s>>>(c.prodA, c.herm, c.npad, (int)pl.chunk_len, ctx->pt, (int)ctx->M,
                                                              ctx->gpart + (size_t)slot * 3 * ctx->M, pm.far, pm.nbyte, pm.nrg);
        PCM_LAUNCH_CHECK(ctx);
        slot += pl.chunks;
        ctx->launch_total++;
    }
    {
        const Plan &pl = ctx->plan_gfock[L];
        const PatchMap &pm = c.fock_map;
        dim3 grid((unsigned)pl.xb, (unsigned)pl.chunks);
        fock_kernel<L + 1, fb.R, fb.C><<<grid, TPB, 0, s>>>(c.prodA, c.npad, ctx->pt, q, ctx->s2c, (int)ctx->M, (int)pl.chunk_len,
                                                            c.gherm, pm.far, pm.nbyte, pm.nrg);
        PCM_LAUNCH_CHECK(ctx);
        ctx->launch_total++;
    }
    return PCM_OK;
}

template <int L>
static int grad_reduce_herm(pcm_ctx *ctx, cudaStream_t s) {
    ClassData &c = ctx->cls[L];
    if (c.n == 0) return PCM_OK;
    const int64_t plane = (int64_t)nherm(L + 1) * c.npad;
    reduce_herm_kernel<<<(unsigned)ceil_div(plane, 32), 256, 0, s>>>(c.gherm, plane, (int)ctx->plan_gfock[L].chunks, c.npad,
                                                                      nherm(L + 1), c.near_gfock, c.fock_map.pstart);
    PCM_LAUNCH_CHECK(ctx);
    ctx->launch_total++;
    return PCM_OK;
}

int launch_gradient(pcm_ctx *ctx, const double *P, int64_t ldp, const double *q, double *g_shell, double *g_point, cudaStream_t s) {
    int rc;
    if ((rc = grad_prepare(ctx))) return rc;
    const int64_t M = ctx->M;
    if (M == 0 || ctx->nprod == 0) {
        if (g_shell && ctx->nshell > 0) PCM_CUDA(ctx, cudaMemsetAsync(g_shell, 0, (size_t)ctx->nshell * 24, s));
        if (g_point && M > 0) PCM_CUDA(ctx, cudaMemsetAsync(g_point, 0, (size_t)M * 24, s));
        return PCM_OK;
    }
    const int saved_timing = ctx->timing;
    ctx->timing = 0;
    ctx->cur_op = 0;
    // D_h of every product (into cls[L].herm, as pcm_potential)
    if ((rc = launch_density_class<0>(ctx, P, ldp, s)) || (rc = launch_density_class<1>(ctx, P, ldp, s)) ||
        (rc = launch_density_class<2>(ctx, P, ldp, s)) || (rc = launch_density_class<3>(ctx, P, ldp, s)) ||
        (rc = launch_density_class<4>(ctx, P, ldp, s))) { ctx->timing = saved_timing; return rc; }
    ctx->timing = saved_timing;
    // near kernels on the near stream, concurrently with the main kernels
    PCM_CUDA(ctx, cudaEventRecord(ctx->ev_fork, s));
    PCM_CUDA(ctx, cudaStreamWaitEvent(ctx->near_stream, ctx->ev_fork, 0));
    if ((rc = grad_launch_near<0>(ctx, q, ctx->near_stream)) || (rc = grad_launch_near<1>(ctx, q, ctx->near_stream)) ||
        (rc = grad_launch_near<2>(ctx, q, ctx->near_stream)) || (rc = grad_launch_near<3>(ctx, q, ctx->near_stream)) ||
        (rc = grad_launch_near<4>(ctx, q, ctx->near_stream))) return rc;
    PCM_CUDA(ctx, cudaEventRecord(ctx->ev_join, ctx->near_stream));
    int64_t slot = 0;
    if ((rc = grad_launch_main<0>(ctx, q, slot, s)) || (rc = grad_launch_main<1>(ctx, q, slot, s)) ||
        (rc = grad_launch_main<2>(ctx, q, slot, s)) || (rc = grad_launch_main<3>(ctx, q, slot, s)) ||
        (rc = grad_launch_main<4>(ctx, q, slot, s))) return rc;
    PCM_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_join, 0));
    if (g_point) {
        NearRefs nr;
        nr.count = 0;
        for (int L = 0; L <= MAXL; ++L)
            if (ctx->cls[L].n > 0) { nr.near[nr.count] = ctx->cls[L].near_gpoint; nr.pstart[nr.count] = ctx->cls[L].pot_map.pstart; nr.count++; }
        grad_point_reduce_kernel<<<(unsigned)ceil_div(M, 32), 256, 0, s>>>(ctx->gpart, M, (int)slot, q, ctx->s2c, nr, g_point);
        PCM_LAUNCH_CHECK(ctx);
        ctx->launch_total++;
    }
    if (g_shell) {
        if ((rc = grad_reduce_herm<0>(ctx, s)) || (rc = grad_reduce_herm<1>(ctx, s)) || (rc = grad_reduce_herm<2>(ctx, s)) ||
            (rc = grad_reduce_herm<3>(ctx, s)) || (rc = grad_reduce_herm<4>(ctx, s))) return rc;
        ClassPtrs cp;
        for (int L = 0; L <= MAXL; ++L) { cp.herm[L] = ctx->cls[L].gherm; cp.npad[L] = ctx->cls[L].npad; cp.first[L] = ctx->cls[L].first; }
        grad_pair_kernel<<<(unsigned)ceil_div(ctx->ncomp, 128), 128, 0, s>>>(
            ctx->ncomp, ctx->c_sp, ctx->c_ab, ctx->sp_mstart, ctx->m_prod, ctx->m_cls, ctx->m_goff, ctx->m_ap, ctx->G, ctx->dG,
            ctx->sp_i0, ctx->sp_j0, ctx->sp_dims, ctx->hshift, cp, P, ldp, ctx->gcomp);
        PCM_LAUNCH_CHECK(ctx);
        grad_sp_reduce_kernel<<<(unsigned)ceil_div(ctx->nsp * 6, 256), 256, 0, s>>>(ctx->nsp, ctx->sp_cstart, ctx->gcomp, ctx->gsp);
        PCM_LAUNCH_CHECK(ctx);
        grad_shell_reduce_kernel<<<(unsigned)ceil_div(ctx->nshell * 3, 256), 256, 0, s>>>(ctx->nshell, ctx->sh_start, ctx->sh_list,
                                                                                         ctx->gsp, g_shell);
        PCM_LAUNCH_CHECK(ctx);
        ctx->launch_total += 3;
    }
    return PCM_OK;
}
