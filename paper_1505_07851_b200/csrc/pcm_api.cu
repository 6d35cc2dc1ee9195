// pcm_api.cu -- the C ABI of include/pcm.h: argument checks, context life cycle, host-buffer forms.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "pcm_internal.h"

namespace pcm {
int build_context(pcm_ctx *ctx, int nshell, const int *shell_l, const double *shell_xyz, const int *shell_nprim,
                  const double *prim_exp, const double *prim_coef, int64_t npoint, const double *pt_xyz,
                  const double *pt_zeta, const double *pt_switch);
const char *setup_error_text();
void setup_stage(const char *name);
void pivot_order(uint64_t seed, int64_t M, int64_t *perm);
int cg_solve(pcm_ctx *ctx, const double *b, double *x, double tol, int max_iter, int precond, int use_x0, int *iters,
             double *resid, cudaStream_t s);
}  // namespace pcm

using namespace pcm;

// One call replayed from its CUDA graph when pcm_options.graph_calls allows: captured on ctx->graph_stream the first time and
// whenever the key (p0, p1, ld, flag) changes, launched into the caller's stream s.  Falls back to plain launches on s when
// graphs are off, per-kernel timing is on, s is itself being captured, or anything about the capture fails.
template <class F>
static int graphed_call(pcm_ctx *ctx, CallGraph &cg, const void *p0, const void *p1, int64_t ld, int flag, int op, cudaStream_t s, F &&launch) {
    if (!ctx->graph_ok || ctx->timing) return launch(s);
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s, &st) != cudaSuccess || st != cudaStreamCaptureStatusNone) {
        (void)cudaGetLastError();
        return launch(s);
    }
    if (cg.exec && cg.p0 == p0 && cg.p1 == p1 && cg.ld == ld && cg.flag == flag) {
        PCM_CUDA(ctx, cudaGraphLaunch(cg.exec, s));
        ctx->launches[op] = cg.nlaunch;
        ctx->launch_total += cg.nlaunch;
        return PCM_OK;
    }
    if (cg.exec) { cudaGraphExecDestroy(cg.exec); cg.exec = nullptr; }
    cudaStream_t cs = ctx->graph_stream;
    if (cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        (void)cudaGetLastError();
        ctx->graph_ok = false;
        return launch(s);
    }
    const int64_t before = ctx->launch_total;
    const int rc = launch(cs);
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(cs, &g);
    if (rc == PCM_OK && e == cudaSuccess && g) e = cudaGraphInstantiate(&cg.exec, g, 0);
    if (g) cudaGraphDestroy(g);
    if (rc != PCM_OK) return rc;
    if (e != cudaSuccess || !cg.exec) {       // no graph on this system: plain launches from now on
        (void)cudaGetLastError();
        cg.exec = nullptr;
        ctx->graph_ok = false;
        ctx->launch_total = before;
        return launch(s);
    }
    cg.p0 = p0; cg.p1 = p1; cg.ld = ld; cg.flag = flag;
    cg.nlaunch = (int)(ctx->launch_total - before);
    PCM_CUDA(ctx, cudaGraphLaunch(cg.exec, s));
    return PCM_OK;
}

extern "C" {

void pcm_options_default(pcm_options *opt) {
    if (!opt) return;
    std::memset(opt, 0, sizeof(*opt));
    opt->screen_eps = 1e-12;
    opt->d_pure = 1;
    opt->device = -1;
    opt->merge_products = 1;
    opt->gradient = 0;
    opt->store_near = 1;
}

static void free_ctx(pcm_ctx *ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    for (void *p : ctx->allocs) cudaFree(p);
    if (ctx->cg_scal_host) cudaFreeHost(ctx->cg_scal_host);
    if (ctx->io_pin) cudaFreeHost(ctx->io_pin);
    if (ctx->io_c) cudaFree(ctx->io_c);
    if (ctx->io_a) cudaFree(ctx->io_a);
    if (ctx->io_b) cudaFree(ctx->io_b);
    for (auto &e : ctx->ev) if (e) cudaEventDestroy(e);
    for (auto &e : ctx->cg_ev) if (e) cudaEventDestroy(e);
    if (ctx->graph_pot.exec || ctx->graph_fock.exec) cudaDeviceSynchronize();     // a replay may still be running
    if (ctx->graph_pot.exec) cudaGraphExecDestroy(ctx->graph_pot.exec);
    if (ctx->graph_fock.exec) cudaGraphExecDestroy(ctx->graph_fock.exec);
    if (ctx->graph_stream) cudaStreamDestroy(ctx->graph_stream);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    if (ctx->near_stream) cudaStreamDestroy(ctx->near_stream);
    if (ctx->ev_rbj) { if (ctx->rbj_pending) cudaEventSynchronize(ctx->ev_rbj); cudaEventDestroy(ctx->ev_rbj); }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    delete[] ctx->rbj_bstart_host;
    delete ctx;
}

int pcm_setup(pcm_ctx **out, int nshell, const int *shell_l, const double *shell_xyz, const int *shell_nprim,
              const double *prim_exp, const double *prim_coef, int64_t npoint, const double *pt_xyz,
              const double *pt_zeta, const double *pt_switch, const pcm_options *opt) {
    if (!out) return set_error(nullptr, PCM_ERR_ARG, "pcm_setup: out is NULL");
    *out = nullptr;
    if (nshell < 0 || npoint < 0 || npoint > 0x7fffffff) return set_error(nullptr, PCM_ERR_ARG, "pcm_setup: negative or too large size");
    if (nshell > 0 && (!shell_l || !shell_xyz || !shell_nprim || !prim_exp || !prim_coef))
        return set_error(nullptr, PCM_ERR_ARG, "pcm_setup: NULL shell array");
    if (npoint > 0 && (!pt_xyz || !pt_zeta)) return set_error(nullptr, PCM_ERR_ARG, "pcm_setup: NULL point array");
    int64_t np = 0;
    for (int s = 0; s < nshell; ++s) {
        if (shell_l[s] < 0 || shell_l[s] > 2) return set_error(nullptr, PCM_ERR_ARG, "pcm_setup: shell_l must be 0, 1 or 2");
        if (shell_nprim[s] < 1) return set_error(nullptr, PCM_ERR_ARG, "pcm_setup: shell_nprim must be >= 1");
        np += shell_nprim[s];
    }
    for (int64_t i = 0; i < np; ++i)
        if (!(prim_exp[i] > 0.0) || !std::isfinite(prim_exp[i]) || !std::isfinite(prim_coef[i]))
            return set_error(nullptr, PCM_ERR_ARG, "pcm_setup: exponents must be positive and finite, coefficients finite");
    for (int64_t k = 0; k < npoint; ++k)
        if (!(pt_zeta[k] > 0.0) || !std::isfinite(pt_zeta[k]) || (pt_switch && !(pt_switch[k] > 0.0)))
            return set_error(nullptr, PCM_ERR_ARG, "pcm_setup: pt_zeta and pt_switch must be positive");

    pcm_ctx *ctx = new (std::nothrow) pcm_ctx();
    if (!ctx) return set_error(nullptr, PCM_ERR_ALLOC, "pcm_setup: out of host memory");
    if (opt) ctx->opt = *opt; else pcm_options_default(&ctx->opt);
    if (!(ctx->opt.screen_eps >= 0.0)) { delete ctx; return set_error(nullptr, PCM_ERR_ARG, "pcm_setup: screen_eps < 0"); }

    auto fail = [&](int rc) {
        set_error(nullptr, rc, ctx->err.empty() ? std::string("pcm_setup failed") : ctx->err);
        free_ctx(ctx);
        return rc;
    };
    cudaError_t e;
    int dev = ctx->opt.device;
    if (dev < 0) {
        e = cudaGetDevice(&dev);
        if (e != cudaSuccess) { ctx->err = std::string("cudaGetDevice: ") + cudaGetErrorString(e); return fail(PCM_ERR_CUDA); }
    }
    e = cudaSetDevice(dev);
    if (e != cudaSuccess) { ctx->err = std::string("cudaSetDevice: ") + cudaGetErrorString(e); return fail(PCM_ERR_CUDA); }
    ctx->device = dev;
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) { ctx->err = std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e); return fail(PCM_ERR_CUDA); }
    ctx->sm_count = prop.multiProcessorCount;
    e = cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) {
        int prio_lo = 0, prio_hi = 0;
        cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
        // low priority: the near kernels (branchy, ~40 % of the FP64 pipe) then fill the tails of the main kernels instead
        // of displacing them (measured 2-3 % on pcm_potential / pcm_fock against a high-priority stream)
        (void)prio_hi;
        e = cudaStreamCreateWithPriority(&ctx->near_stream, cudaStreamNonBlocking, prio_lo);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_rbj, cudaEventDisableTiming);
    if (e != cudaSuccess) { ctx->err = std::string("cudaStreamCreate: ") + cudaGetErrorString(e); return fail(PCM_ERR_CUDA); }
    for (auto &ev : ctx->ev) {
        e = cudaEventCreate(&ev);
        if (e != cudaSuccess) { ctx->err = std::string("cudaEventCreate: ") + cudaGetErrorString(e); return fail(PCM_ERR_CUDA); }
    }

    for (auto &ev : ctx->cg_ev) {
        e = cudaEventCreate(&ev);
        if (e != cudaSuccess) { ctx->err = std::string("cudaEventCreate: ") + cudaGetErrorString(e); return fail(PCM_ERR_CUDA); }
    }

    int rc = build_context(ctx, nshell, shell_l, shell_xyz, shell_nprim, prim_exp, prim_coef, npoint, pt_xyz, pt_zeta, pt_switch);
    if (rc) return fail(rc);

    // scratch sized from the fixed work partition
    const int64_t M = ctx->M;
    setup_stage("gradient tables");
    if ((rc = plan_all(ctx))) return fail(rc);
    for (int L = 0; L <= MAXL; ++L) {
        ClassData &c = ctx->cls[L];
        c.herm_slots = ctx->plan_fock[L].chunks;
        if ((rc = dev_alloc_t(ctx, &c.near_fock, (size_t)c.fock_map.npiece * nherm(L) * 32))) return fail(rc);
        if ((rc = dev_alloc_t(ctx, &c.near_pot, (size_t)c.pot_map.npiece * 32))) return fail(rc);
        if ((rc = dev_alloc_t(ctx, &c.herm, (size_t)c.herm_slots * nherm(L) * std::max<int64_t>(c.npad, 1)))) return fail(rc);
        ctx->vpart_slots += (c.n > 0) ? ctx->plan_pot[L].chunks : 0;
    }
    ctx->ypart_slots = ctx->plan_amat.chunks;
    if (ctx->opt.tma_tiles && (rc = dev_alloc_t(ctx, &ctx->ptq, (size_t)std::max<int64_t>(M, 1)))) return fail(rc);
    if ((rc = dev_alloc_t(ctx, &ctx->near_amat, (size_t)ctx->amat_map.npiece * 32))) return fail(rc);
    setup_stage("work partition, scratch");
    if ((rc = fill_amat_blocks(ctx))) return fail(rc);
    if (getenv("PCM_VERBOSE")) cudaDeviceSynchronize();
    setup_stage("stored near patches of A");
    if ((rc = plan_sweep(ctx))) return fail(rc);
    setup_stage("persistent sweep plan");
    if ((rc = dev_alloc_t(ctx, &ctx->vpart, (size_t)std::max<int64_t>(ctx->vpart_slots, 1) * std::max<int64_t>(M, 1)))) return fail(rc);
    if ((rc = dev_alloc_t(ctx, &ctx->ypart, (size_t)ctx->ypart_slots * std::max<int64_t>(M, 1)))) return fail(rc);
    if ((rc = dev_alloc_t(ctx, &ctx->colpart, (size_t)std::max<int64_t>(ctx->plan_amat.xb, 1) * std::max<int64_t>(M, 1)))) return fail(rc);
    if ((rc = dev_alloc_t(ctx, &ctx->cg_vec, (size_t)6 * std::max<int64_t>(M, 1)))) return fail(rc);
    if ((rc = dev_alloc_t(ctx, &ctx->cg_part, (size_t)(M / 32 + 2)))) return fail(rc);
    if ((rc = dev_alloc_t(ctx, &ctx->cg_scal, (size_t)1024))) return fail(rc);
    e = cudaMemset(ctx->cg_scal, 0, 1024 * 8);
    if (e == cudaSuccess) e = cudaMallocHost(&ctx->cg_scal_host, 64 * sizeof(double));
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { ctx->err = std::string("pcm_setup: ") + cudaGetErrorString(e); return fail(PCM_ERR_CUDA); }
    setup_stage("solver scratch");
    // small solutes: a call is a string of launch latencies -> replay it from a CUDA graph (pcm_options.graph_calls)
    ctx->graph_ok = ctx->opt.graph_calls > 0 || (ctx->opt.graph_calls == 0 && ctx->info.product_points < 5e7);
    if (ctx->graph_ok && cudaStreamCreateWithFlags(&ctx->graph_stream, cudaStreamNonBlocking) != cudaSuccess) {
        (void)cudaGetLastError();
        ctx->graph_ok = false;
    }
    ctx->info.device_bytes = ctx->device_bytes;
    ctx->info.amat_near_patches = ctx->amat_map.nnear;
    ctx->info.amat_stored_bytes = ctx->amat_blocks ? ctx->amat_map.nnear * 32 * 32 * 8 : 0;
    ctx->info.amat_far_stored_bytes = ctx->cgp.far_bytes;
    ctx->info.amat_persistent = ctx->cgp.ready ? 1 : 0;
    ctx->info.components = ctx->ncomp;
    *out = ctx;
    return PCM_OK;
}

#define PCM_CHECK_CTX(ctx) \
    if (!(ctx)) return PCM_ERR_ARG

int pcm_potential(pcm_ctx *ctx, const double *P_dev, int64_t ldp, double *v_dev, void *stream) {
    PCM_CHECK_CTX(ctx);
    if (ctx->M == 0) return PCM_OK;
    if (!v_dev || (ctx->nbf > 0 && (!P_dev || ldp < ctx->nbf))) return set_error(ctx, PCM_ERR_ARG, "pcm_potential: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return graphed_call(ctx, ctx->graph_pot, P_dev, v_dev, ldp, 0, 0, (cudaStream_t)stream,
                        [&](cudaStream_t s) { return launch_potential(ctx, P_dev, ldp, v_dev, s); });
}

int pcm_fock(pcm_ctx *ctx, const double *q_dev, double *F_dev, int64_t ldf, int accumulate, void *stream) {
    PCM_CHECK_CTX(ctx);
    if (ctx->nbf == 0) return PCM_OK;
    if (!F_dev || ldf < ctx->nbf || (ctx->M > 0 && !q_dev)) return set_error(ctx, PCM_ERR_ARG, "pcm_fock: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return graphed_call(ctx, ctx->graph_fock, q_dev, F_dev, ldf, accumulate ? 1 : 0, 1, (cudaStream_t)stream,
                        [&](cudaStream_t s) { return launch_fock(ctx, q_dev, F_dev, ldf, accumulate, s); });
}

int pcm_amatvec(pcm_ctx *ctx, const double *q_dev, double *y_dev, void *stream) {
    PCM_CHECK_CTX(ctx);
    if (ctx->M == 0) return PCM_OK;
    if (!q_dev || !y_dev || q_dev == y_dev) return set_error(ctx, PCM_ERR_ARG, "pcm_amatvec: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_amatvec(ctx, q_dev, y_dev, (cudaStream_t)stream);
}

int pcm_set_nuclei(pcm_ctx *ctx, int natom, const double *atom_xyz_host, const double *z_host) {
    PCM_CHECK_CTX(ctx);
    if (natom < 0 || (natom > 0 && (!atom_xyz_host || !z_host))) return set_error(ctx, PCM_ERR_ARG, "pcm_set_nuclei: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    std::vector<double4> at((size_t)std::max(natom, 1));
    for (int j = 0; j < natom; ++j) at[j] = make_double4(atom_xyz_host[3 * j], atom_xyz_host[3 * j + 1], atom_xyz_host[3 * j + 2], z_host[j]);
    if (ctx->atoms == nullptr || natom > ctx->natom) {   // grow-only; the old buffer stays on the context's free list
        int rc = dev_alloc_t(ctx, &ctx->atoms, at.size());
        if (rc) return rc;
    }
    PCM_CUDA(ctx, cudaMemcpy(ctx->atoms, at.data(), at.size() * sizeof(double4), cudaMemcpyHostToDevice));
    ctx->natom = natom;
    ctx->cavity_set = false;   // radii belong to the atom list
    if (ctx->cav_natom == natom && natom >= 0 && (int64_t)ctx->cav_owner_host.size() == ctx->M)   // context of pcm_setup_cavity
        return pcm_set_cavity(ctx, ctx->cav_radius_host.data(), ctx->cav_owner_host.data());
    return PCM_OK;
}

int pcm_nuclear_potential(pcm_ctx *ctx, double *u_dev, void *stream) {
    PCM_CHECK_CTX(ctx);
    if (ctx->natom < 0) return set_error(ctx, PCM_ERR_STATE, "pcm_nuclear_potential: call pcm_set_nuclei first");
    if (ctx->M == 0) return PCM_OK;
    if (!u_dev) return set_error(ctx, PCM_ERR_ARG, "pcm_nuclear_potential: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_nuclear_potential(ctx, u_dev, (cudaStream_t)stream);
}

int pcm_rhs(pcm_ctx *ctx, const double *u_dev, const double *v_dev, double f, double *b_dev, void *stream) {
    PCM_CHECK_CTX(ctx);
    if (ctx->M == 0) return PCM_OK;
    if (!u_dev || !v_dev || !b_dev) return set_error(ctx, PCM_ERR_ARG, "pcm_rhs: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_rhs(ctx, u_dev, v_dev, f, b_dev, (cudaStream_t)stream);
}

int pcm_energy(pcm_ctx *ctx, const double *u_dev, const double *v_dev, const double *q_dev, double f, double *terms_host,
               void *stream) {
    PCM_CHECK_CTX(ctx);
    if (!terms_host || !(f != 0.0) || (ctx->M > 0 && (!u_dev || !v_dev || !q_dev)))
        return set_error(ctx, PCM_ERR_ARG, "pcm_energy: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return energy_terms(ctx, u_dev, v_dev, q_dev, f, terms_host, (cudaStream_t)stream);
}

int pcm_gradient(pcm_ctx *ctx, const double *P_dev, int64_t ldp, const double *q_dev, double *g_shell_dev, double *g_point_dev,
                 void *stream) {
    PCM_CHECK_CTX(ctx);
    if (!ctx->opt.gradient) return set_error(ctx, PCM_ERR_STATE, "pcm_gradient: pcm_setup was called without pcm_options.gradient");
    if ((ctx->nbf > 0 && !P_dev) || (ctx->M > 0 && !q_dev) || ldp < ctx->nbf) return set_error(ctx, PCM_ERR_ARG, "pcm_gradient: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_gradient(ctx, P_dev, ldp, q_dev, g_shell_dev, g_point_dev, (cudaStream_t)stream);
}

int pcm_switching(int64_t npoint, const double *pt_xyz_host, const double *pt_zeta_host, const int32_t *pt_atom_host, int natom,
                  const double *atom_xyz_host, const double *atom_radius_host, double *S_host, int device) {
    if (npoint < 0 || natom < 0 || (npoint > 0 && (!pt_xyz_host || !pt_zeta_host || !pt_atom_host || !S_host)) ||
        (natom > 0 && (!atom_xyz_host || !atom_radius_host)))
        return set_error(nullptr, PCM_ERR_ARG, "pcm_switching: bad argument");
    if (device >= 0) {
        cudaError_t e = cudaSetDevice(device);
        if (e != cudaSuccess) return set_error(nullptr, PCM_ERR_CUDA, std::string("pcm_switching: ") + cudaGetErrorString(e));
    }
    return switching_host(npoint, pt_xyz_host, pt_zeta_host, pt_atom_host, natom, atom_xyz_host, atom_radius_host, S_host);
}

int pcm_set_cavity(pcm_ctx *ctx, const double *atom_radius_host, const int32_t *pt_atom_host) {
    PCM_CHECK_CTX(ctx);
    if (ctx->natom < 0) return set_error(ctx, PCM_ERR_STATE, "pcm_set_cavity: call pcm_set_nuclei first");
    if ((ctx->natom > 0 && !atom_radius_host) || (ctx->M > 0 && !pt_atom_host)) return set_error(ctx, PCM_ERR_ARG, "pcm_set_cavity: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    std::vector<int32_t> own((size_t)std::max<int64_t>(ctx->M, 1), -1);
    for (int64_t s = 0; s < ctx->M; ++s) {
        const int32_t a = pt_atom_host[ctx->s2c_host[(size_t)s]];
        if (a < -1 || a >= ctx->natom) return set_error(ctx, PCM_ERR_ARG, "pcm_set_cavity: owner index out of range");
        own[(size_t)s] = a;
    }
    int rc;
    if ((rc = dev_alloc_t(ctx, &ctx->atom_radius, (size_t)std::max<int64_t>(ctx->natom, 1)))) return rc;
    if ((rc = dev_alloc_t(ctx, &ctx->pt_owner, own.size()))) return rc;
    if (ctx->natom > 0) PCM_CUDA(ctx, cudaMemcpy(ctx->atom_radius, atom_radius_host, (size_t)ctx->natom * 8, cudaMemcpyHostToDevice));
    PCM_CUDA(ctx, cudaMemcpy(ctx->pt_owner, own.data(), own.size() * 4, cudaMemcpyHostToDevice));
    ctx->cavity_set = true;
    return PCM_OK;
}

int pcm_surface_gradient(pcm_ctx *ctx, const double *q_dev, double f, double *g_point_dev, double *g_atom_dev, void *stream) {
    PCM_CHECK_CTX(ctx);
    if (!ctx->cavity_set) return set_error(ctx, PCM_ERR_STATE, "pcm_surface_gradient: call pcm_set_nuclei and pcm_set_cavity first");
    if ((ctx->M > 0 && !q_dev) || !(f != 0.0)) return set_error(ctx, PCM_ERR_ARG, "pcm_surface_gradient: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_surface_gradient(ctx, q_dev, f, g_point_dev, g_atom_dev, (cudaStream_t)stream);
}

int pcm_cg_threshold(double diis_prev, double delta_min, double *delta_out) {
    if (!delta_out) return PCM_ERR_ARG;
    double delta = 1.0;   // first SCF iteration: no previous DIIS error
    if (diis_prev > 0.0) delta = std::exp(std::log(0.1 * diis_prev) / 1.07);   // 0.01 delta^1.07 = 1e-3 diis_prev
    *delta_out = std::min(1.0, std::max(delta_min, delta));
    return PCM_OK;
}

int pcm_pivot_order(uint64_t seed, int64_t M, int64_t *perm_host) {
    if (M < 0 || (M > 0 && !perm_host)) return PCM_ERR_ARG;
    pivot_order(seed, M, perm_host);
    return PCM_OK;
}

int pcm_rbj_build(pcm_ctx *ctx, int block, uint64_t seed, const int64_t *pivot_order_host, void *stream) {
    PCM_CHECK_CTX(ctx);
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return rbj_build(ctx, block, seed, pivot_order_host, (cudaStream_t)stream, false, false);
}

int pcm_rbj_build_async(pcm_ctx *ctx, int block, uint64_t seed, const int64_t *pivot_order_host, void *stream) {
    PCM_CHECK_CTX(ctx);
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return rbj_build(ctx, block, seed, pivot_order_host, (cudaStream_t)stream, true, false);
}

int pcm_rbj_get(pcm_ctx *ctx, int64_t *order_host, int64_t *bstart_host, double *inv_host) {
    PCM_CHECK_CTX(ctx);
    {
        int rcf = rbj_finish(ctx, ctx->own_stream);
        if (rcf) return rcf;
    }
    if (ctx->rbj_block == 0) return set_error(ctx, PCM_ERR_STATE, "pcm_rbj_get: no RBJ preconditioner built");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    const int64_t M = ctx->M, l = ctx->rbj_block, nb = ctx->rbj_nblocks;
    if (order_host && M > 0) {
        std::vector<int32_t> o((size_t)M);
        PCM_CUDA(ctx, cudaMemcpy(o.data(), ctx->rbj_order, (size_t)M * 4, cudaMemcpyDeviceToHost));
        for (int64_t i = 0; i < M; ++i) order_host[i] = ctx->s2c_host[(size_t)o[i]];  // sorted -> caller numbering
    }
    if (bstart_host)
        for (int64_t b = 0; b <= nb; ++b) bstart_host[b] = std::min(b * l, M);
    if (inv_host) {
        // device layout: block b at b*l*l with its own leading dimension n_b; host layout: back to back
        size_t off = 0;
        for (int64_t b = 0; b < nb; ++b) {
            const int64_t n = std::min(l, M - b * l);
            PCM_CUDA(ctx, cudaMemcpy(inv_host + off, ctx->rbj_inv + (size_t)b * l * l, (size_t)n * n * 8, cudaMemcpyDeviceToHost));
            off += (size_t)n * n;
        }
    }
    return PCM_OK;
}

int pcm_cg_solve(pcm_ctx *ctx, const double *b_dev, double *x_dev, double tol, int max_iter, int precond, int use_x0,
                 int *iters, double *resid, void *stream) {
    PCM_CHECK_CTX(ctx);
    if (ctx->M > 0 && (!b_dev || !x_dev)) return set_error(ctx, PCM_ERR_ARG, "pcm_cg_solve: NULL vector");
    if (max_iter < 0 || !(tol >= 0.0)) return set_error(ctx, PCM_ERR_ARG, "pcm_cg_solve: bad tol or max_iter");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return cg_solve(ctx, b_dev, x_dev, tol, max_iter, precond, use_x0, iters, resid, (cudaStream_t)stream);
}

// ---- host-buffer forms ------------------------------------------------------------------------
// P and F are dense nbf x nbf on the host, but the path reads / writes only the elements of surviving shell pairs (a few
// per cent at configs[3]: 2 GB of matrix, some tens of MB of components).  The host-buffer calls therefore gather those
// elements into a pinned compact buffer (OpenMP), copy that, and scatter on the other side; the device kernels keep working
// on a dense device image whose other elements are never read.
namespace pcm {
__global__ void scatter_components_kernel(int64_t nc, const int32_t *__restrict__ mu, const int32_t *__restrict__ nu,
                                          const uint8_t *__restrict__ diag, const double *__restrict__ comp, double *__restrict__ D, int64_t ld) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nc) return;
    D[(size_t)mu[c] * ld + nu[c]] = comp[2 * c];
    if (!diag[c]) D[(size_t)nu[c] * ld + mu[c]] = comp[2 * c + 1];
}
__global__ void gather_components_kernel(int64_t nc, const int32_t *__restrict__ mu, const int32_t *__restrict__ nu,
                                         const uint8_t *__restrict__ diag, const double *__restrict__ D, int64_t ld, double *__restrict__ comp) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nc) return;
    comp[2 * c] = D[(size_t)mu[c] * ld + nu[c]];
    comp[2 * c + 1] = diag[c] ? 0.0 : D[(size_t)nu[c] * ld + mu[c]];
}
}  // namespace pcm

static int ensure_compact_io(pcm_ctx *ctx) {
    if (ctx->io_pin && ctx->io_c) return PCM_OK;
    const size_t bytes = std::max<size_t>((size_t)ctx->ncomp * 16, 16);
    if (!ctx->io_pin && cudaMallocHost((void **)&ctx->io_pin, bytes) != cudaSuccess)
        return set_error(ctx, PCM_ERR_ALLOC, "cudaMallocHost (component staging) failed");
    if (!ctx->io_c && cudaMalloc((void **)&ctx->io_c, bytes) != cudaSuccess)
        return set_error(ctx, PCM_ERR_ALLOC, "cudaMalloc (component staging) failed");
    return PCM_OK;
}

static int ensure_io(pcm_ctx *ctx, double **buf, size_t *have, size_t bytes) {
    if (*have >= bytes && *buf) return PCM_OK;
    if (*buf) cudaFree(*buf);
    *buf = nullptr;
    *have = 0;
    cudaError_t e = cudaMalloc((void **)buf, std::max<size_t>(bytes, 8));
    if (e != cudaSuccess) return set_error(ctx, PCM_ERR_ALLOC, std::string("cudaMalloc (staging): ") + cudaGetErrorString(e));
    *have = bytes;
    return PCM_OK;
}

int pcm_potential_host(pcm_ctx *ctx, const double *P_host, int64_t ldp, double *v_host) {
    PCM_CHECK_CTX(ctx);
    if (ctx->M == 0) return PCM_OK;
    if (!v_host || (ctx->nbf > 0 && (!P_host || ldp < ctx->nbf))) return set_error(ctx, PCM_ERR_ARG, "pcm_potential_host: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t nb = (size_t)ctx->nbf;
    const int64_t nc = ctx->ncomp;
    int rc;
    if ((rc = ensure_io(ctx, &ctx->io_a, &ctx->io_a_bytes, nb * nb * 8))) return rc;
    if ((rc = ensure_io(ctx, &ctx->io_b, &ctx->io_b_bytes, (size_t)ctx->M * 8))) return rc;
    if ((rc = ensure_compact_io(ctx))) return rc;
    cudaStream_t s = ctx->own_stream;
    if (nc > 0) {
        const int32_t *mu = ctx->comp_mu_host.data(), *nu = ctx->comp_nu_host.data();
        double *pin = ctx->io_pin;
#pragma omp parallel for schedule(static)
        for (int64_t c = 0; c < nc; ++c) {
            pin[2 * c] = P_host[(size_t)mu[c] * ldp + nu[c]];
            pin[2 * c + 1] = P_host[(size_t)nu[c] * ldp + mu[c]];
        }
        PCM_CUDA(ctx, cudaMemcpyAsync(ctx->io_c, pin, (size_t)nc * 16, cudaMemcpyHostToDevice, s));
        scatter_components_kernel<<<(unsigned)((nc + 255) / 256), 256, 0, s>>>(nc, ctx->comp_mu, ctx->comp_nu, ctx->comp_diag, ctx->io_c, ctx->io_a,
                                                                             (int64_t)nb);
        PCM_CUDA(ctx, cudaGetLastError());
        ctx->launch_total += 1;
    }
    if ((rc = launch_potential(ctx, ctx->io_a, (int64_t)nb, ctx->io_b, s))) return rc;
    PCM_CUDA(ctx, cudaMemcpyAsync(v_host, ctx->io_b, (size_t)ctx->M * 8, cudaMemcpyDeviceToHost, s));
    PCM_CUDA(ctx, cudaStreamSynchronize(s));
    return PCM_OK;
}

int pcm_fock_host(pcm_ctx *ctx, const double *q_host, double *F_host, int64_t ldf, int accumulate) {
    PCM_CHECK_CTX(ctx);
    if (ctx->nbf == 0) return PCM_OK;
    if (!F_host || ldf < ctx->nbf || (ctx->M > 0 && !q_host)) return set_error(ctx, PCM_ERR_ARG, "pcm_fock_host: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t nb = (size_t)ctx->nbf;
    const int64_t nc = ctx->ncomp;
    int rc;
    if ((rc = ensure_io(ctx, &ctx->io_a, &ctx->io_a_bytes, nb * nb * 8))) return rc;
    if ((rc = ensure_io(ctx, &ctx->io_b, &ctx->io_b_bytes, (size_t)ctx->M * 8))) return rc;
    if ((rc = ensure_compact_io(ctx))) return rc;
    cudaStream_t s = ctx->own_stream;
    if (ctx->M) PCM_CUDA(ctx, cudaMemcpyAsync(ctx->io_b, q_host, (size_t)ctx->M * 8, cudaMemcpyHostToDevice, s));
    // the device image is built from zero (only its component elements come back); accumulate is applied on the host
    if ((rc = launch_fock(ctx, ctx->io_b, ctx->io_a, (int64_t)nb, 0, s))) return rc;
    if (nc > 0) {
        gather_components_kernel<<<(unsigned)((nc + 255) / 256), 256, 0, s>>>(nc, ctx->comp_mu, ctx->comp_nu, ctx->comp_diag, ctx->io_a, (int64_t)nb,
                                                                            ctx->io_c);
        PCM_CUDA(ctx, cudaGetLastError());
        ctx->launch_total += 1;
        PCM_CUDA(ctx, cudaMemcpyAsync(ctx->io_pin, ctx->io_c, (size_t)nc * 16, cudaMemcpyDeviceToHost, s));
    }
    if (!accumulate) {     // zero-fill on the host while the device works
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < (int64_t)nb; ++i) std::memset(F_host + (size_t)i * ldf, 0, nb * 8);
    }
    PCM_CUDA(ctx, cudaStreamSynchronize(s));
    if (nc > 0) {
        const int32_t *mu = ctx->comp_mu_host.data(), *nu = ctx->comp_nu_host.data();
        const uint8_t *dg = ctx->comp_diag_host.data();
        const double *pin = ctx->io_pin;
        // every (mu, nu) is written by exactly one component, so the loop is race-free
#pragma omp parallel for schedule(static)
        for (int64_t c = 0; c < nc; ++c) {
            F_host[(size_t)mu[c] * ldf + nu[c]] += pin[2 * c];
            if (!dg[c]) F_host[(size_t)nu[c] * ldf + mu[c]] += pin[2 * c + 1];
        }
    }
    return PCM_OK;
}

int pcm_amatvec_host(pcm_ctx *ctx, const double *q_host, double *y_host) {
    PCM_CHECK_CTX(ctx);
    if (ctx->M == 0) return PCM_OK;
    if (!q_host || !y_host) return set_error(ctx, PCM_ERR_ARG, "pcm_amatvec_host: bad argument");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    int rc;
    const size_t bytes = (size_t)ctx->M * 8;
    if ((rc = ensure_io(ctx, &ctx->io_a, &ctx->io_a_bytes, bytes))) return rc;
    if ((rc = ensure_io(ctx, &ctx->io_b, &ctx->io_b_bytes, bytes))) return rc;
    cudaStream_t s = ctx->own_stream;
    PCM_CUDA(ctx, cudaMemcpyAsync(ctx->io_a, q_host, bytes, cudaMemcpyHostToDevice, s));
    if ((rc = launch_amatvec(ctx, ctx->io_a, ctx->io_b, s))) return rc;
    PCM_CUDA(ctx, cudaMemcpyAsync(y_host, ctx->io_b, bytes, cudaMemcpyDeviceToHost, s));
    PCM_CUDA(ctx, cudaStreamSynchronize(s));
    return PCM_OK;
}

int pcm_cg_solve_host(pcm_ctx *ctx, const double *b_host, double *x_host, double tol, int max_iter, int precond,
                      int use_x0, int *iters, double *resid) {
    PCM_CHECK_CTX(ctx);
    if (ctx->M > 0 && (!b_host || !x_host)) return set_error(ctx, PCM_ERR_ARG, "pcm_cg_solve_host: NULL vector");
    if (max_iter < 0 || !(tol >= 0.0)) return set_error(ctx, PCM_ERR_ARG, "pcm_cg_solve_host: bad tol or max_iter");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    int rc;
    const size_t bytes = (size_t)ctx->M * 8;
    if ((rc = ensure_io(ctx, &ctx->io_a, &ctx->io_a_bytes, bytes))) return rc;
    if ((rc = ensure_io(ctx, &ctx->io_b, &ctx->io_b_bytes, bytes))) return rc;
    cudaStream_t s = ctx->own_stream;
    if (bytes) PCM_CUDA(ctx, cudaMemcpyAsync(ctx->io_a, b_host, bytes, cudaMemcpyHostToDevice, s));
    if (bytes && use_x0) PCM_CUDA(ctx, cudaMemcpyAsync(ctx->io_b, x_host, bytes, cudaMemcpyHostToDevice, s));
    const int status = cg_solve(ctx, ctx->io_a, ctx->io_b, tol, max_iter, precond, use_x0, iters, resid, s);
    if (status < 0) return status;
    if (bytes) PCM_CUDA(ctx, cudaMemcpyAsync(x_host, ctx->io_b, bytes, cudaMemcpyDeviceToHost, s));
    PCM_CUDA(ctx, cudaStreamSynchronize(s));
    return status;
}

int pcm_get_info(pcm_ctx *ctx, pcm_info *out) {
    PCM_CHECK_CTX(ctx);
    if (!out) return set_error(ctx, PCM_ERR_ARG, "pcm_get_info: out is NULL");
    ctx->info.device_bytes = ctx->device_bytes;
    *out = ctx->info;
    return PCM_OK;
}

int pcm_set_timing(pcm_ctx *ctx, int enable) {
    PCM_CHECK_CTX(ctx);
    ctx->timing = enable ? 1 : 0;
    return PCM_OK;
}

int pcm_last_kernel_ms(pcm_ctx *ctx, int op, double ms[2], int *n_launch) {
    PCM_CHECK_CTX(ctx);
    if (op < 0 || op > 2) return set_error(ctx, PCM_ERR_ARG, "pcm_last_kernel_ms: op must be 0, 1 or 2");
    if (n_launch) *n_launch = ctx->launches[op];
    if (!ms) return PCM_OK;
    ms[0] = ms[1] = 0.0;
    if (!ctx->timed[op]) return set_error(ctx, PCM_ERR_STATE, "pcm_last_kernel_ms: the last call of this op was not timed (pcm_set_timing)");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaEvent_t *ev = ctx->ev + 8 * op;
    PCM_CUDA(ctx, cudaEventSynchronize(ev[7]));
    float a = 0, b = 0, c = 0;
    if (op == 2) {   // pcm_amatvec records one event before and one after its launches
        PCM_CUDA(ctx, cudaEventElapsedTime(&b, ev[0], ev[7]));
        ms[0] = b;
        return PCM_OK;
    }
    PCM_CUDA(ctx, cudaEventElapsedTime(&a, ev[0], ev[1]));
    PCM_CUDA(ctx, cudaEventElapsedTime(&b, ev[1], ev[6]));
    PCM_CUDA(ctx, cudaEventElapsedTime(&c, ev[6], ev[7]));
    ms[0] = b;
    ms[1] = (double)a + c;
    return PCM_OK;
}

int pcm_last_class_ms(pcm_ctx *ctx, int op, double ms[PCM_NL]) {
    PCM_CHECK_CTX(ctx);
    if (op < 0 || op > 2 || !ms) return set_error(ctx, PCM_ERR_ARG, "pcm_last_class_ms: bad argument");
    if (!ctx->timed[op]) return set_error(ctx, PCM_ERR_STATE, "pcm_last_class_ms: the last call of this op was not timed (pcm_set_timing)");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaEvent_t *ev = ctx->ev + 8 * op;
    PCM_CUDA(ctx, cudaEventSynchronize(ev[7]));
    if (op == 2) {
        float t = 0;
        PCM_CUDA(ctx, cudaEventElapsedTime(&t, ev[0], ev[7]));
        ms[0] = t;
        for (int L = 1; L < PCM_NL; ++L) ms[L] = 0.0;
        return PCM_OK;
    }
    for (int L = 0; L < PCM_NL; ++L) {
        float t = 0;
        PCM_CUDA(ctx, cudaEventElapsedTime(&t, ev[1 + L], ev[2 + L]));
        ms[L] = t;
    }
    return PCM_OK;
}

int pcm_last_cg_matvec_ms(pcm_ctx *ctx, double *avg_ms, int *n) {
    PCM_CHECK_CTX(ctx);
    if (!avg_ms) return set_error(ctx, PCM_ERR_ARG, "pcm_last_cg_matvec_ms: avg_ms is NULL");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    double sum = 0.0;
    for (int i = 0; i < ctx->cg_ev_n; ++i) {
        float t = 0;
        PCM_CUDA(ctx, cudaEventSynchronize(ctx->cg_ev[2 * i + 1]));
        PCM_CUDA(ctx, cudaEventElapsedTime(&t, ctx->cg_ev[2 * i], ctx->cg_ev[2 * i + 1]));
        sum += t;
    }
    *avg_ms = ctx->cg_ev_n ? sum / ctx->cg_ev_n : 0.0;
    if (n) *n = ctx->cg_ev_n;
    return PCM_OK;
}

int pcm_launch_count(pcm_ctx *ctx, int64_t *total) {
    PCM_CHECK_CTX(ctx);
    if (!total) return set_error(ctx, PCM_ERR_ARG, "pcm_launch_count: total is NULL");
    *total = ctx->launch_total;
    return PCM_OK;
}

int pcm_fp64_peak(pcm_ctx *ctx, int reps, double *tflops) {
    PCM_CHECK_CTX(ctx);
    if (!tflops) return set_error(ctx, PCM_ERR_ARG, "pcm_fp64_peak: tflops is NULL");
    PCM_CUDA(ctx, cudaSetDevice(ctx->device));
    return fp64_peak(ctx, reps, tflops);
}

int pcm_schwarz_bound(int la, double alpha, const double *A, int lb, double beta, const double *B, double *out) {
    if (la < 0 || la > 2 || lb < 0 || lb > 2 || !A || !B || !out || !(alpha > 0.0) || !(beta > 0.0)) return PCM_ERR_ARG;
    *out = schwarz_bound(la, alpha, A, lb, beta, B);
    return PCM_OK;
}

const char *pcm_last_error(pcm_ctx *ctx) { return ctx ? ctx->err.c_str() : setup_error_text(); }

int pcm_destroy(pcm_ctx *ctx) {
    free_ctx(ctx);
    return PCM_OK;
}

}  // extern "C"
