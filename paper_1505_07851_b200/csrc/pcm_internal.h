// pcm_internal.h -- context layout and shared host/device constants of libpcm_b200.
// Product code: shares nothing with oracle/ (see DESIGN.md "Independence").
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/pcm.h"

namespace pcm {

// ---------------------------------------------------------------------------------------------
// Hermite index space.  A Hermite Gaussian product of total angular momentum L carries
// NHERM(L) = (L+1)(L+2)(L+3)/6 components Lambda_tuv, t+u+v <= L, ordered by degree d = t+u+v
// first so that the components of a lower L are a prefix of those of a higher L:
//   index(t,u,v) = d(d+1)(d+2)/6 + (d-t)(d-t+1)/2 + (d-t-u)
// ---------------------------------------------------------------------------------------------
__host__ __device__ constexpr int nherm(int L) { return (L + 1) * (L + 2) * (L + 3) / 6; }
__host__ __device__ constexpr int hidx(int t, int u, int v) {
    return (t + u + v) * (t + u + v + 1) * (t + u + v + 2) / 6 + (u + v) * (u + v + 1) / 2 + v;
}

// Far-field switch: for T = rho |P-C|^2 >= TFAR(L) the Boys functions F_0..F_L equal
// their asymptotic forms to better than 2e-17 relative (the neglected tail is exp(-T) T^{n-1/2}/Gamma(n+1/2)).
__host__ __device__ constexpr double tfar(int L) { return 38.0 + 3.0 * L; }
constexpr double TFAR_AMAT = 38.0;  // erfc(sqrt(38)) = 3e-18

// Boys table: rows T_i = i/16, i = 0..BOYS_ROWS-1 (covers [0, 54] >= tfar(MAXLG)); per L a table of rows
// {c_0..c_7, exp(-T_i), 0} with c_k = (-1)^k F_{L+k}(T_i)/k!  so that F_L(T_i + d) = sum_k c_k d^k.
constexpr int BOYS_ROWS = 54 * 16 + 1;
constexpr int BOYS_STRIDE = 10;
constexpr int BOYS_TERMS = 8;

constexpr int MAXL = 4;
constexpr int MAXLG = MAXL + 1;  // the gradient kernels evaluate Hermite integrals one order higher (Boys tables 0..MAXLG)

struct DeviceBuf {  // owning device allocation
    void *p = nullptr;
    size_t bytes = 0;
};

// Far/near classification of the (32 rows) x (32 columns) patches of a hot kernel's sweep, fixed at setup from the
// bounding boxes of the groups: a patch is "far" when its boxes are further apart than the far-field radius of every
// evaluation in it.  The main kernels run the far patches branch-free and skip the others, which the near kernels
// pick up from the per-row-group lists.
struct PatchMap {
    int64_t nrg = 0;            // row groups
    int64_t ncg = 0;            // column groups
    int64_t nbyte = 0;          // bytes per row of `far` = ceil(ncg / 8)
    uint8_t *far = nullptr;     // [nrg][nbyte]: bit s of byte b = patch (row group, column group 8 b + s) is far
    int64_t *start = nullptr;   // [nrg + 1] CSR into list
    int32_t *list = nullptr;    // column groups of the patches that are not far, row group after row group
    int64_t nnear = 0;          // entries of list
    // near-kernel work items ("pieces"): piece q belongs to row group piece_rg[q] and covers entries
    // start[rg] + NEAR_PIECE (q - pstart[rg]) ... of that group's list; pieces of one group are consecutive.
    int64_t npiece = 0;
    int64_t *pstart = nullptr;  // [nrg + 1] CSR: pieces of each row group
    int32_t *piece_rg = nullptr;  // [npiece]
    // host copies, kept for the A q map only (plan_sweep partitions the sweep from them)
    std::vector<uint8_t> far_host;
    std::vector<int64_t> start_host, pstart_host;
    std::vector<int32_t> piece_rg_host;
};
constexpr int NEAR_PIECE = 4;

// Warp-granular partition of the symmetric A q sweep and the buffers of the persistent PCG kernel (pcm_cgp.cu); built by
// plan_sweep at pcm_setup for cavities below AMAT_PERSIST_MAX points whose near patches are stored.
constexpr int64_t AMAT_PERSIST_MAX = 26000;     // measured crossover with the R = 4 kernel: one A q 24k points, a PCG iteration 28 - 30k
struct SweepPlan {
    bool ready = false;
    int grid = 0, nwarp = 0, ng = 0, nrb = 0, nslot = 0;
    int64_t nstrip = 0;
    size_t smem = 0;
    struct CgpWarpInit *winit = nullptr;   // [nwarp] start-up record of every warp (pcm_cgp.cu)
    int2 *strip = nullptr;            // [nstrip] (row block, column group | far mask of the 4 row groups << 24)
    int64_t *seg_start = nullptr;     // [nwarp + 1] column pairs of every warp (pair h belongs to strip h >> 4)
    int32_t *seg_slot0 = nullptr;     // [nwarp + 1] first row-sum slot of every warp
    int32_t *rb_slot_start = nullptr; // [nrb + 1] slots of every row block (consecutive)
    double4 *colloc = nullptr;        // [M] (-2 (b - o), |b - o|^2), o = first point of the column's group
    double4 *org = nullptr;           // [ng] o
    double *yslot = nullptr;          // [nslot][128] row sums of a (segment, row block) run
    double *colpart = nullptr;        // [nrb][M] column sums of a row block
    double *pbuf = nullptr;           // [M] second buffer of the CG direction
    double *afar = nullptr;           // stored far field [2 nstrip][16][4][32] (nullptr: evaluated on the fly)
    int64_t far_bytes = 0;
};

struct ClassData {        // products of one total angular momentum L, padded to a multiple of 128
    int64_t n = 0;        // products
    int64_t npad = 0;     // padded count (SoA leading dimension); the padding repeats the last product
    int64_t first = 0;    // global index of the first product of this class
    double4 *prodA = nullptr;  // (Px, Py, Pz, thr): hi word of thr is the far-field threshold on |P-C|^2
    double2 *prodB = nullptr;  // (p, 1/kappa) with kappa = sqrt(pi/p)/2
    PatchMap pot_map;          // rows = groups of 32 points, columns = groups of 32 products of this class
    PatchMap fock_map;         // rows = groups of 32 products of this class, columns = groups of 32 points
    double *herm = nullptr;    // [chunks][nherm(L)][npad] Hermite vectors (density D or potential sums H)
    int64_t herm_slots = 0;    // chunks the herm buffer holds
    double *near_fock = nullptr;  // [fock_map.npiece][nherm(L)][32] sums of the near pieces
    double *near_pot = nullptr;   // [pot_map.npiece][32]
    // pcm_gradient scratch (allocated by its first call): Hermite potential sums one order higher
    double *gherm = nullptr;       // [plan_gfock.chunks][nherm(L+1)][npad]
    double *near_gfock = nullptr;  // [fock_map.npiece][nherm(L+1)][32]
    double *near_gpoint = nullptr; // [pot_map.npiece][3][32]
};

struct Plan {             // work partition of one hot kernel launch: grid = (xb, chunks)
    int64_t xb = 0;        // blocks along the register-resident ("row") dimension
    int64_t chunks = 1;    // pieces the streamed ("column") dimension is cut into; each writes its own partial-sum slot
    int64_t chunk_len = 0; // columns per chunk (a multiple of the tile)
};

}  // namespace pcm

// One pcm_potential / pcm_fock call as an instantiated CUDA graph (pcm_options.graph_calls); the key is what the captured
// kernels were given: two pointers, a leading dimension, a flag.
struct CallGraph {
    cudaGraphExec_t exec = nullptr;
    const void *p0 = nullptr, *p1 = nullptr;
    int64_t ld = 0;
    int flag = 0;
    int nlaunch = 0;
};

struct pcm_ctx {
    int device = 0;
    CallGraph graph_pot, graph_fock;
    cudaStream_t graph_stream = nullptr;     // the calls are captured here and replayed into the caller's stream
    bool graph_ok = false;
    int sm_count = 148;
    pcm_options opt{};
    pcm_info info{};
    std::string err;

    // points
    int64_t M = 0;
    // points, stored in Morton order ("sorted index" s); the caller's index of sorted point s is s2c[s].
    // Vectors crossing the C ABI (v, q, y, b, x) are in the caller's order; the kernels gather/scatter through s2c.
    double4 *pt = nullptr;      // (x, y, z, 1/zeta^2)
    double4 *ptq = nullptr;     // (x, y, z, q_k) in sorted order, packed per pcm_fock call (pcm_options.tma_tiles)
    double *pt_diag = nullptr;  // A_kk = zeta_k sqrt(2/pi)/S_k
    double *pt_boxes = nullptr; // [ceil(M/32)][6] bounding boxes of the groups of 32 sorted points
    pcm::PatchMap amat_map;     // rows and columns = groups of 32 sorted points
    int32_t *s2c = nullptr;     // [M] device
    std::vector<int32_t> s2c_host, c2s_host;
    double zeta_min = 0, zeta_max = 0;

    // basis / pairs
    int64_t nbf = 0;
    int64_t nprod = 0;   // all products
    int64_t nmember = 0; // surviving primitive pairs (diagonal shell pairs: i <= j)
    int64_t nsp = 0;     // surviving shell pairs
    int64_t ncomp = 0;   // sum over shell pairs of na*nb
    pcm::ClassData cls[pcm::MAXL + 1];

    // members (sorted by shell pair)
    int32_t *m_prod = nullptr;   // global product index
    int32_t *m_sp = nullptr;     // shell pair of the member
    int32_t *m_cls = nullptr;    // packed: L_member | (L_product << 8)
    int64_t *m_goff = nullptr;   // offset of the member's G matrix [na*nb][nherm(L_member)]
    double *G = nullptr;
    // product -> members CSR (global product order)
    int64_t *pm_start = nullptr;
    int32_t *pm_list = nullptr;
    // shell pairs
    int64_t *sp_mstart = nullptr;  // [nsp+1] member range
    int32_t *sp_i0 = nullptr, *sp_j0 = nullptr;  // basis-function offsets
    int32_t *sp_dims = nullptr;    // na | nb<<8 | diag<<16
    // component -> (shell pair, ab)
    int32_t *c_sp = nullptr;
    int32_t *c_ab = nullptr;

    // nuclei (pcm_set_nuclei): (x, y, z, charge)
    int64_t natom = -1;
    double4 *atoms = nullptr;
    // cavity (pcm_set_cavity): radius of every atom's sphere, owning atom of every point (sorted point order)
    double *atom_radius = nullptr;
    int32_t *pt_owner = nullptr;
    bool cavity_set = false;
    // a context made by pcm_setup_cavity remembers the cavity's atoms: pcm_set_nuclei with as many atoms re-registers them
    int cav_natom = -1;
    std::vector<double> cav_radius_host;
    std::vector<int32_t> cav_owner_host;   // caller (= cavity) point order
    double *surf_scratch = nullptr;   // pcm_surface_gradient partial sums (grow-only)
    size_t surf_scratch_n = 0;

    // pcm_gradient (pcm_options.gradient): derivative tables and the shell bookkeeping of the pair transform
    int64_t nshell = 0;
    double *dG = nullptr;        // per member [na*nb][3][nherm(L_member)] = dG/dX_AB at fixed P, at 3 * m_goff[m]
    double *m_ap = nullptr;      // per member alpha/p (weight of the bra centre in P)
    int32_t *sp_shI = nullptr, *sp_shJ = nullptr;  // shells of a shell pair
    int64_t *sp_cstart = nullptr;  // [nsp+1] first component of a shell pair (components are grouped by shell pair)
    int64_t *sh_start = nullptr;   // [nshell+1] CSR: shell -> entries 2 * sp + side (0: bra, 1: ket)
    int32_t *sh_list = nullptr;
    int32_t *hshift = nullptr;     // [3][nherm(MAXL)]: index of (t,u,v) + 1_x
    double *gcomp = nullptr;       // [ncomp][6] per component: dE/dA xyz, dE/dB xyz
    double *gsp = nullptr;         // [nsp][6]
    double *gpart = nullptr;       // [slots][3][M] partial sums of the point gradient
    int64_t gpart_slots = 0;
    bool grad_ready = false;
    pcm::Plan plan_gfock[pcm::MAXL + 1], plan_gpoint[pcm::MAXL + 1];

    double *boys = nullptr;  // [MAXLG+1][BOYS_ROWS][BOYS_STRIDE]

    // fixed work partitions (sizes and SM count only; set once in pcm_setup by plan_all)
    pcm::Plan plan_pot[pcm::MAXL + 1], plan_fock[pcm::MAXL + 1], plan_amat;
    pcm::SweepPlan cgp;

    // scratch
    double *vpart = nullptr;    // potential partial sums [slots][M]
    int64_t vpart_slots = 0;
    double *near_amat = nullptr;  // [amat_map.npiece][32] sums of the near pieces
    double *amat_blocks = nullptr;  // [amat_map.nnear][32][32] stored near patches of A (nullptr: evaluated on the fly)
    double *ypart = nullptr;    // amatvec row partial sums [slots][M]
    int64_t ypart_slots = 0;
    double *colpart = nullptr;  // amatvec column partial sums of the symmetric sweep [plan_amat.xb][M]
    int amat_tile = 256;        // column tile of the A q kernel (128 for small M)
    int amat_R = 4;             // row groups per warp of the A q kernel (row block = 128 amat_R points)
    double *cg_vec = nullptr;   // 6 M doubles: r, z, p, Ap, x, b (sorted point order)
    double *cg_part = nullptr;  // [ceil(M/32)] per-CTA partial dot products of cg_matvec_reduce_kernel
    double *cg_scal = nullptr;  // device scalars
    double *cg_scal_host = nullptr;  // pinned
    // host-buffer calls: only the elements of P / F that belong to a surviving shell pair cross PCIe.  Per component c of the
    // component table: its element (mu, nu) and whether the shell pair is diagonal (then (nu, mu) is a component of its own).
    std::vector<int32_t> comp_mu_host, comp_nu_host;
    std::vector<uint8_t> comp_diag_host;
    int32_t *comp_mu = nullptr, *comp_nu = nullptr;   // device copies
    uint8_t *comp_diag = nullptr;
    double *io_pin = nullptr;                         // pinned staging, 2 ncomp doubles: (mu, nu) and (nu, mu) of every component
    double *io_c = nullptr;                           // its device image
    double *io_a = nullptr, *io_b = nullptr;  // staging for the *_host calls
    size_t io_a_bytes = 0, io_b_bytes = 0;

    // RBJ
    int64_t rbj_block = 0, rbj_nblocks = 0;
    int32_t *rbj_order = nullptr;    // [M] point indices block after block
    int64_t *rbj_bstart_host = nullptr;
    double *rbj_inv = nullptr;       // inverse blocks back to back (block b at b*l*l)
    double *rbj_partial = nullptr;   // [2][rbj_nblocks] per-block r.r and r.z of the CG update kernel
    // asynchronous build (pcm_rbj_build_async): status in cg_scal_host[32..], completed by rbj_finish
    bool rbj_pending = false;
    cudaEvent_t ev_rbj = nullptr;
    uint64_t rbj_last_seed = 0;
    bool rbj_perm_seeded = false;
    std::vector<int32_t> rbj_perm_sorted;   // pivot order of the last build, sorted point numbering
    std::vector<int64_t> rbj_last_perm;     // caller-given pivot order of the last build (empty: seeded)
    char *rbj_arena = nullptr;       // grow-only allocation holding the three arrays above and the build scratch
    size_t rbj_arena_bytes = 0;

    cudaStream_t own_stream = nullptr;
    // the near kernels run on near_stream (low priority), forked from and joined back into the caller's stream around the
    // main kernels of the same call, so that their latency-bound work fills what the FP64-bound main kernels leave idle
    cudaStream_t near_stream = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    // the class kernels of one call run concurrently on these (forked from / joined into the caller's stream), unless timing is on
    // events: 0 start, 1 after the pre-transform, 2+L after the class-L main kernel, 7 end, 8 CG residual read-back
    cudaEvent_t ev[28] = {};   // ev[8*op + i], op = 0 potential, 1 fock, 2 amatvec; 24 CG; 25, 26 peak benchmark
    // CG: events around the A q launches (main + near kernels) of the first CG_EV iterations of the last timed solve
    static constexpr int CG_EV = 16;
    cudaEvent_t cg_ev[2 * CG_EV] = {};
    int cg_ev_n = 0;
    int timing = 0;
    int cur_op = 0;
    int launches[3] = {0, 0, 0};   // kernels launched by the last call of each op
    int64_t launch_total = 0;   // kernels launched by this context since pcm_setup
    bool timed[3] = {false, false, false};

    std::vector<void *> allocs;  // everything cudaMalloc'ed, freed in pcm_destroy
    int64_t device_bytes = 0;
};

// ---- internal entry points (pcm_setup.cu, pcm_kernels.cu, pcm_solver.cu) ----
namespace pcm {
int set_error(pcm_ctx *ctx, int code, const std::string &msg);
int dev_alloc(pcm_ctx *ctx, void **p, size_t bytes);
template <class T>
inline int dev_alloc_t(pcm_ctx *ctx, T **p, size_t count) {
    return dev_alloc(ctx, reinterpret_cast<void **>(p), count * sizeof(T));
}
int launch_potential(pcm_ctx *ctx, const double *P, int64_t ldp, double *v, cudaStream_t s);
int launch_fock(pcm_ctx *ctx, const double *q, double *F, int64_t ldf, int accumulate, cudaStream_t s);
int launch_amatvec(pcm_ctx *ctx, const double *q, double *y, cudaStream_t s);
int launch_amatvec_sorted(pcm_ctx *ctx, const double *q_sorted, double *y_sorted, cudaStream_t s);  // both in sorted order
int launch_amatvec_partials(pcm_ctx *ctx, const double *q_sorted, const int *stop, cudaStream_t s);  // ypart slots + near_amat only
int launch_nuclear_potential(pcm_ctx *ctx, double *u, cudaStream_t s);
int launch_rhs(pcm_ctx *ctx, const double *u, const double *v, double f, double *b, cudaStream_t s);
int energy_terms(pcm_ctx *ctx, const double *u, const double *v, const double *q, double f, double *terms_host, cudaStream_t s);
int launch_gradient(pcm_ctx *ctx, const double *P, int64_t ldp, const double *q, double *g_shell, double *g_point, cudaStream_t s);
int rbj_build(pcm_ctx *ctx, int block, uint64_t seed, const int64_t *pivot_order_host, cudaStream_t s, bool async, bool force_global);
int rbj_finish(pcm_ctx *ctx, cudaStream_t s);
int launch_surface_gradient(pcm_ctx *ctx, const double *q, double f, double *g_point, double *g_atom, cudaStream_t s);
int switching_host(int64_t M, const double *xyz, const double *zeta, const int32_t *owner, int natom, const double *atom_xyz,
                   const double *atom_radius, double *S);
int plan_all(pcm_ctx *ctx);
int plan_sweep(pcm_ctx *ctx);
int cgp_matvec(pcm_ctx *ctx, const double *q, const int32_t *idx, double *y, cudaStream_t s);
int cgp_solve(pcm_ctx *ctx, double *r, double *z, double *p, double *Ap, double *x, double tol, int max_iter, int precond, cudaStream_t s);
bool cgp_can_solve(const pcm_ctx *ctx, int precond);
int fill_amat_blocks(pcm_ctx *ctx);
int fp64_peak(pcm_ctx *ctx, int reps, double *tflops);
void build_boys_tables(std::vector<double> &tab);
double schwarz_bound(int la, double alpha, const double *A, int lb, double beta, const double *B);
}  // namespace pcm

#define PCM_CUDA(ctx, call)                                                                               \
    do {                                                                                                  \
        cudaError_t e__ = (call);                                                                         \
        if (e__ != cudaSuccess)                                                                           \
            return pcm::set_error(ctx, PCM_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__)); \
    } while (0)
