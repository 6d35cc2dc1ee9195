/*
 * pcm.h -- C ABI of libpcm_b200: the data-parallel hot path of GPU C-PCM with
 * switching/Gaussian surface discretization (arxiv 1505.07851; citations are PAPER.md lines).
 *
 * What the library computes (all fp64, atomic units: bohr, hartree):
 *   J_k(r)  = erf(zeta_k |r - r_k|) / |r - r_k|                                  Eq. 6
 *   v_k     = sum_{mu,nu} P_mu,nu (mu|J_k|nu)      -- pcm_potential               Eq. 5
 *   F_mu,nu = sum_k q_k (mu|J_k|nu)                -- pcm_fock                    Eq. 10
 *   (mu|J_k|nu) = sum_ij c_mu,i c_nu,j [chi_i|J_k|chi_j]                          Eq. 11-12
 *   A_kl    = erf(zeta'_kl r_kl)/r_kl, zeta'_kl = zeta_k zeta_l/sqrt(zeta_k^2+zeta_l^2),
 *   A_kk    = zeta_k sqrt(2/pi) / S_k              -- pcm_amatvec (y = A q)       Eq. 2, 3, 8
 *   A x = b by preconditioned CG with the Jacobi or the randomized block-Jacobi
 *   preconditioner                                  -- pcm_rbj_build, pcm_cg_solve section 4b
 *
 * Sign convention: the paper's L^k_mu,nu = -(mu|J_k|nu) carries the electron's charge, so
 * its c = -v and Delta F^S = -F.  This library returns the unsigned v and F.  Eq. 3 is printed with
 * zeta/sqrt(2 pi); the Gaussian self-energy is zeta sqrt(2/pi), which is what is used (R1).
 *
 * Conventions
 *   - every call returns int: 0 = PCM_OK, < 0 = error (pcm_last_error gives text), > 0 = a
 *     documented non-error status (PCM_NOT_CONVERGED).  No exception crosses the ABI.
 *   - "host" / "device" is stated for every pointer.  Device pointers must be valid on the
 *     context's device until the given stream has passed the call.
 *   - the context owns COPIES of everything given to pcm_setup; the caller owns P, q, b, v, F, y, x.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Hot calls
 *     are asynchronous with respect to the host unless stated otherwise.
 *   - a context must not be used from two host threads at once, and calls on one context must be stream-ordered (it owns
 *     scratch buffers, internal streams and events); the one exception is pcm_rbj_build_async, made to overlap another call.
 *   - there is no CPU fallback: every call fails with PCM_ERR_CUDA if the device is unusable.
 */
#ifndef PCM_B200_H
#define PCM_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PCM_OK 0
#define PCM_NOT_CONVERGED 1    /* pcm_cg_solve hit max_iter; x, iters and resid are still valid */
#define PCM_ERR_ARG (-1)       /* bad argument (NULL, negative size, l > 2, nprim < 1, ...) */
#define PCM_ERR_CUDA (-2)      /* a CUDA call failed (text in pcm_last_error) */
#define PCM_ERR_ALLOC (-3)     /* host or device allocation failed */
#define PCM_ERR_STATE (-4)     /* call needs something not built (e.g. RBJ before pcm_rbj_build) */
#define PCM_ERR_NUMERIC (-5)   /* a diagonal block of A was not positive definite */

#define PCM_NCLASS 6           /* shell-pair classes in the paper's order ss, sp, pp, sd, pd, dd */
#define PCM_NL 5               /* total angular momentum L = l_a + l_b = 0..4 */

typedef struct pcm_ctx pcm_ctx;

typedef struct pcm_options {
    double screen_eps;     /* primitive-pair Schwarz-like cutoff of Eq. 15; default 1e-12 */
    int d_pure;            /* 1 (default): 5 real solid harmonics per d shell; 0: 6 Cartesian components */
    int device;            /* CUDA device ordinal; -1 (default) = the calling thread's current device */
    int merge_products;    /* 1 (default): primitive pairs with identical (A, alpha, B, beta) -- e.g. the s and p
                              parts of an sp shell -- share one Hermite Gaussian product in the kernels (exact) */
    int gradient;          /* 1: also build what pcm_gradient needs (derivative tables, 3x the G matrices); default 0 */
    int store_near;        /* 1 (default): the patches of A that are not in the far field (the entries that need erf) are
                              evaluated once at pcm_setup and kept on the device (8 KB per 32 x 32 patch, up to 16 GB; beyond
                              that, or with 0, they are re-evaluated in every pcm_amatvec).  Same values either way. */
    int cg_path;           /* pcm_cg_solve / pcm_amatvec: 0 (default) = one persistent cooperative kernel per solve and one launch per
                              A q below 26 000 points, separate kernel launches above; 1 = always separate launches (the
                              reference path); 2 = the persistent kernel at any size its buffers allow; 3 = separate launches with
                              every CG vector operation in a kernel of its own (no fused update kernel: the bit-exactness
                              reference of path 1).  Same recurrences; paths 0/2 and 1/3 add the partial sums of A q in different
                              (each fixed) orders */
    int store_far;         /* the stored-A variant (PAPER.md:106 stores all of A) for the far field of the persistent path: 0 (default) =
                              keep the far-field 1/r values too (4 M^2 bytes) when they and the stored near patches stay resident
                              in L2 (<= 96 MB: about M <= 4 500); 1 = whenever device memory allows; -1 = never.  Same values,
                              same summation order: the result does not depend on it */
    int serial_classes;    /* 1: pcm_potential / pcm_fock launch their per-class kernels the ordinary way, each after the one before
                              it has finished (as with pcm_set_timing on); 0 (default): as a chain of programmatic dependent
                              launches on the caller's stream, so that a class kernel starts while the last wave of the one before
                              it is still running.  Same results bit for bit */
    int tma_tiles;         /* 1: pcm_fock brings its surface-point tiles into shared memory with TMA bulk copies (cp.async.bulk +
                              mbarrier, double-buffered) from a per-call packed (x, y, z, q) array instead of per-thread loads;
                              0 (default).  Same results bit for bit */
    int rbj_global_scan;   /* 1: pcm_rbj_build selects every block with the cooperative global row scan instead of the one-CTA
                              neighbourhood search (same blocks; the default uses the scan only above 150 000 points or l > 256) */
    int potential_pr;      /* bit L set: pcm_potential sweeps the products of total angular momentum L in the Fock layout (product
                              in registers, warp-shuffle reduction over the 32 products of a warp per point) instead of the
                              point-in-registers layout.  Same values up to the summation order.  Default 0 (measured: DESIGN.md) */
    int graph_calls;       /* pcm_potential / pcm_fock replayed from a CUDA graph: the ~10 launches of a call are captured once
                              (on an internal stream) and the instantiated graph is launched into the caller's stream for as
                              long as the call's pointer arguments, leading dimension and flags stay the same (they are the key;
                              any change re-captures).  0 (default) = for small solutes only, where a call is a string of launch
                              latencies (products x points < 5e7); 1 = always; -1 = never.  Not used while pcm_set_timing is on
                              or while the caller's stream is itself being captured (the launches then go into that capture).
                              Same kernels, same results bit for bit */
} pcm_options;

typedef struct pcm_info {
    int64_t nbf;                       /* basis functions */
    int64_t nshell;
    int64_t npoint;                    /* M, surface points */
    int64_t shell_pairs[PCM_NCLASS];   /* unordered shell pairs (I <= J) with at least one surviving primitive pair */
    int64_t prim_pairs[PCM_NCLASS];    /* surviving primitive pairs per class, counted as the paper does: every
                                          (i in I, j in J) of an unordered shell pair I <= J, both orders of a
                                          diagonal shell pair (I == J, i != j) counted once */
    int64_t prim_pairs_total;
    int64_t prim_pairs_unscreened;     /* before Eq. 15 */
    int64_t products[PCM_NL];          /* distinct Hermite Gaussian products per L after merging */
    int64_t products_total;
    double prim_pair_points;           /* prim_pairs_total * npoint: the work unit count of one potential or Fock call */
    double product_points;             /* products_total * npoint: kernel evaluations actually performed */
    double zeta_min, zeta_max;
    int64_t rbj_block;                 /* 0 until pcm_rbj_build */
    int64_t rbj_nblocks;
    int64_t device_bytes;              /* device memory held by the context */
    int64_t amat_near_patches;         /* 32 x 32 patches of A that are not far field (evaluated with erf) */
    int64_t amat_stored_bytes;         /* bytes of those patches kept on the device (0: re-evaluated in every A q) */
    int64_t amat_far_stored_bytes;     /* bytes of the stored far field (pcm_options.store_far; 0: evaluated on the fly) */
    int64_t amat_persistent;           /* 1: pcm_cg_solve / pcm_amatvec use the persistent-kernel path (pcm_options.cg_path) */
    int64_t components;                /* elements (mu, nu) of P / F in blocks of surviving shell pairs I <= J: what pcm_potential reads
                                          and pcm_fock writes (times two for the transposes of off-diagonal shell pairs) */
    int64_t rbj_selection;             /* how the last pcm_rbj_build chose its blocks: 1 = one-CTA neighbourhood selection, 2 = global row
                                          scan, 3 = global row scan after the neighbourhood selection reported "capacity" (an asynchronous
                                          build shows 1 until the call that completes it has seen the report); same blocks in every case */
} pcm_info;

/* Fills *opt with the defaults listed above. */
void pcm_options_default(pcm_options *opt);

/*
 * pcm_setup -- step a1: enumerate shell pairs I <= J, screen primitive pairs with
 *   |c_i c_j| max_components [chi_a chi_b|chi_a chi_b]^{1/2} >= screen_eps   (Eq. 15),
 * sort by class and total angular momentum, pack the SoA pair / point arrays and upload them.
 * All pointers are HOST pointers and are copied.
 *   nshell, shell_l[nshell] in {0,1,2}, shell_xyz[3*nshell] (bohr), shell_nprim[nshell] >= 1,
 *   prim_exp / prim_coef[sum nprim]: exponents and contraction coefficients, shell after shell.
 *     prim_coef multiplies the RAW primitive (x-Ax)^i (y-Ay)^j (z-Az)^k exp(-a |r-A|^2) (normalisation
 *     folded in by the caller).  An sp shell is passed as an s shell and a p shell with equal exponents.
 *   basis-function order = shell order; within a shell: s; p = (x,y,z); pure d = (sqrt3 xy, sqrt3 yz,
 *     zz-(xx+yy)/2, sqrt3 xz, (sqrt3/2)(xx-yy)); Cartesian d = (xx,xy,xz,yy,yz,zz).
 *   npoint, pt_xyz[3*npoint] (bohr), pt_zeta[npoint] > 0 (Eq. 7), pt_switch[npoint] > 0 (S_k of Eq. 3/9;
 *     NULL means 1).  npoint == 0 and nshell == 0 are allowed (calls then do nothing / zero-fill).
 *   opt may be NULL (defaults).
 * On success *out is a new context.  Errors: PCM_ERR_ARG, PCM_ERR_ALLOC, PCM_ERR_CUDA (*out = NULL;
 * the text is available from pcm_last_error(NULL)).
 */
int pcm_setup(pcm_ctx **out, int nshell, const int *shell_l, const double *shell_xyz, const int *shell_nprim,
              const double *prim_exp, const double *prim_coef, int64_t npoint, const double *pt_xyz,
              const double *pt_zeta, const double *pt_switch, const pcm_options *opt);

/*
 * pcm_potential -- v_k = sum over the FULL square of P_mu,nu (mu|J_k|nu), k = 0..M-1  (Eq. 5; the paper's
 * "build c", c_k = -v_k).  P_dev: DEVICE, row-major nbf x nbf, leading dimension ldp >= nbf;
 * read only where a shell pair survived screening; (mu,nu) and (nu,mu) are both read, P need not be symmetric.
 * v_dev: DEVICE, M doubles, overwritten.  Asynchronous on `stream`.
 */
int pcm_potential(pcm_ctx *ctx, const double *P_dev, int64_t ldp, double *v_dev, void *stream);

/*
 * pcm_fock -- F_mu,nu (+)= sum_k q_k (mu|J_k|nu)  (Eq. 10; the paper's "build Delta F^S", PAPER.md:126-143,
 * Delta F^S = -F).  q_dev: DEVICE, M doubles.  F_dev: DEVICE, row-major nbf x nbf, leading dimension ldf.
 * accumulate = 0: F is zero-filled first; 1: added to.  Both (mu,nu) and (nu,mu) are written; elements of
 * screened-out shell pairs are left as they are (or zero).  Deterministic (no atomics).  Asynchronous.
 */
int pcm_fock(pcm_ctx *ctx, const double *q_dev, double *F_dev, int64_t ldf, int accumulate, void *stream);

/*
 * pcm_amatvec -- y = A q with A evaluated on the fly (Eq. 2, 3, 8); what pcm_options.store_near / store_far keep of A (the paper
 * stores all of it) is read back instead of re-evaluated, with the same values and summation order.
 * q_dev, y_dev: DEVICE, M doubles, must not alias.  Coincident points i != j (a caller error) are treated as
 * r = 0 -> 2 zeta'/sqrt(pi), never NaN.  Deterministic.  Asynchronous.
 */
int pcm_amatvec(pcm_ctx *ctx, const double *q_dev, double *y_dev, void *stream);

/*
 * pcm_pivot_order -- the seeded pivot order used by pcm_rbj_build: indices 0..M-1 sorted by
 * (splitmix64-finaliser(seed + (i+1)*0x9E3779B97F4A7C15), i).  perm_host: HOST, M int64.  No device work.
 */
int pcm_pivot_order(uint64_t seed, int64_t M, int64_t *perm_host);

/*
 * pcm_rbj_build -- the randomized block-Jacobi preconditioner of PAPER.md:190: take the first still-unassigned
 * index k of the pivot order, evaluate row k of A over the unassigned indices, the block is k plus the
 * block-1 unassigned indices with the largest A_kj (ties -> lower index), repeat; the last block takes the
 * remainder.  Every block of A is then inverted (Cholesky) and the inverses are kept on the device.
 * pivot_order_host: HOST, a permutation of 0..M-1, or NULL to use pcm_pivot_order(seed, M).
 * Synchronises the stream before returning.  Errors: PCM_ERR_ARG (block < 1), PCM_ERR_NUMERIC.
 */
int pcm_rbj_build(pcm_ctx *ctx, int block, uint64_t seed, const int64_t *pivot_order_host, void *stream);

/*
 * pcm_rbj_build_async -- the same build queued on `stream` without synchronising, so that it can overlap other work
 * (A and the preconditioner depend on the geometry only: e.g. queue it on a side stream while pcm_potential runs).
 * The next pcm_cg_solve with precond = 2 (or pcm_rbj_get, or the next build) waits for it, orders its own stream after
 * it and returns the build's error, if any.  Argument errors are still returned at once.
 */
int pcm_rbj_build_async(pcm_ctx *ctx, int block, uint64_t seed, const int64_t *pivot_order_host, void *stream);

/*
 * pcm_rbj_get -- copy the block structure back (for inspection and tests).  Any pointer may be NULL.
 * order_host[M]: indices block after block, pivot first then by descending A_kj; bstart_host[nblocks+1];
 * inv_host: the inverse blocks, row-major, back to back (sum of n_b^2 doubles).  Synchronous.
 */
int pcm_rbj_get(pcm_ctx *ctx, int64_t *order_host, int64_t *bstart_host, double *inv_host);

/*
 * pcm_cg_solve -- preconditioned conjugate gradient on A x = b:
 *   r = b - A x0; z = C r; p = z;  repeat { stop if ||r||_2 <= tol;  alpha = (r.z)/(p.Ap); x += alpha p;
 *   r -= alpha Ap; z = C r; beta = (r.z)'/(r.z); p = z + beta p }.
 * precond: 0 none, 1 Jacobi (C = diag(A)^-1), 2 RBJ (needs pcm_rbj_build; C = P M^-1 P).
 * b_dev: DEVICE M doubles.  x_dev: DEVICE M doubles, in: x0 if use_x0 else ignored; out: the solution.
 * tol is the absolute Euclidean norm of the recurrence residual (the paper's delta).
 * iters (HOST, may be NULL): matrix-vector products after the initial residual.
 * resid (HOST, may be NULL): resid[0] = final recurrence ||r||, resid[1] = true ||b - A x|| recomputed at exit.
 * Synchronous.  Below 26 000 points the iterations run inside one persistent kernel and the host reads the outcome once;
 * above, iterations are queued eight at a time between read-backs of the device-side convergence flag.  Returns PCM_OK,
 * PCM_NOT_CONVERGED, or PCM_ERR_NUMERIC when the residual is not finite (non-finite b, p.Ap = 0).
 * SURVEY.md 8(b) proposed `block` and `seed` as arguments of this call: they are arguments of pcm_rbj_build[_async], because
 * the preconditioner depends on the geometry only and is built once for many solves; precond = 2 uses the last build and
 * fails with PCM_ERR_STATE if there is none.
 */
int pcm_cg_solve(pcm_ctx *ctx, const double *b_dev, double *x_dev, double tol, int max_iter, int precond, int use_x0,
                 int *iters, double *resid, void *stream);

/*
 * The rest of one C-PCM step around the hot path (Eq. 1, 4, 13, 21).
 *
 * pcm_set_nuclei -- the solute's nuclei for B z.  atom_xyz_host: HOST, 3*natom doubles (bohr); z_host: HOST,
 * natom doubles (nuclear charges).  The context keeps a copy; a later call replaces it.  natom = 0 is allowed.
 *
 * pcm_nuclear_potential -- u = B z, u_k = sum_J z_J erf(zeta_k |r_k - R_J|)/|r_k - R_J| (Eq. 4): a
 * nucleus is a point charge, so the exponent is the surface point's own zeta_k; r = 0 -> 2 zeta_k/sqrt(pi).
 * u_dev: DEVICE, M doubles, overwritten.  Asynchronous.  PCM_ERR_STATE before pcm_set_nuclei.
 *
 * pcm_rhs -- b = -f (u - v): the right-hand side of Eq. 1, A q = -f (B z + c), with this library's unsigned
 * v (c = -v, see "Sign convention" above); f = (eps - 1)/(eps + k).  u_dev, v_dev, b_dev: DEVICE,
 * M doubles (b may alias u or v).  Asynchronous.
 *
 * pcm_energy -- Delta G_els = (B z).q + c.q + (1/2f) q.A q (Eq. 13) with c = -v; A q by one
 * pcm_amatvec.  u_dev, v_dev, q_dev: DEVICE, M doubles.  terms_host: HOST, 4 doubles: the three terms and their
 * sum.  Fixed-order sums (bit-reproducible).  Synchronises the stream.
 *
 * pcm_cg_threshold -- the dynamic CG threshold of PAPER.md:182-184: the delta at which Err(delta) = 0.01 delta^1.07
 * (Eq. 21) equals 1e-3 x the DIIS error of the previous SCF iteration, clamped to [delta_min, 1];
 * diis_prev <= 0 means "first SCF iteration" -> delta = 1.  Host arithmetic only.
 */
int pcm_set_nuclei(pcm_ctx *ctx, int natom, const double *atom_xyz_host, const double *z_host);
int pcm_nuclear_potential(pcm_ctx *ctx, double *u_dev, void *stream);
int pcm_rhs(pcm_ctx *ctx, const double *u_dev, const double *v_dev, double f, double *b_dev, void *stream);
int pcm_energy(pcm_ctx *ctx, const double *u_dev, const double *v_dev, const double *q_dev, double f, double *terms_host,
               void *stream);
int pcm_cg_threshold(double diis_prev, double delta_min, double *delta_out);

/*
 * pcm_gradient -- the one-electron PCM gradient term (grad* c^T) q of Eq. 14 (Eq. 22: ga, gb per
 * primitive pair, gc per point), in this library's sign: the gradient of E = v.q = sum_k q_k sum_{mu,nu} P_mu,nu (mu|J_k|nu)
 * at fixed P and q (the paper's c = -v, so its term is -E).
 *   g_shell[3*S + x] = dE/d(x coordinate of the centre of shell S)   (bra and ket derivatives of every pair with S, summed)
 *   g_point[3*k + x] = dE/d(x coordinate of surface point k)         (zeta_k does not move with the point, Eq. 7)
 * The caller adds shell and point rows to the atoms they sit on.  Needs pcm_options.gradient = 1 at pcm_setup.
 * P_dev: DEVICE nbf x nbf (symmetric, as pcm_potential); q_dev: DEVICE M; g_shell_dev: DEVICE 3*nshell doubles;
 * g_point_dev: DEVICE 3*M doubles (either may be NULL).  Overwrites.  Deterministic.  Asynchronous (the first call
 * allocates its scratch and synchronises).
 */
int pcm_gradient(pcm_ctx *ctx, const double *P_dev, int64_t ldp, const double *q_dev, double *g_shell_dev, double *g_point_dev,
                 void *stream);

/*
 * ISWIG cavity quantities (Eq. 9) and the surface terms of the gradient (Eq. 14).
 *
 * pcm_switching -- S_k = prod_{J != owner(k)} S_wf(r_k, R_J), S_wf = 1 - {erf[zeta_k (R_J - d)] + erf[zeta_k (R_J + d)]}/2,
 * d = |r_k - R_J|, R_J = cavity radius of atom J, evaluated on the device.  Standalone (no context: S_k is an input of
 * pcm_setup; the paper drops points with S_k < 1e-8, PAPER.md:106 -- the caller filters).  All arrays HOST: pt_xyz 3*npoint,
 * pt_zeta npoint, pt_atom npoint (owning atom, -1 = none), atom_xyz 3*natom, atom_radius natom, S npoint (out).
 * device: CUDA ordinal, -1 = current.  Synchronous.
 *
 * pcm_set_cavity -- after pcm_set_nuclei: the cavity radius of each of those atoms and the owning atom of every surface
 * point (HOST; caller's point order).  Needed by pcm_surface_gradient only.
 *
 * pcm_surface_gradient -- gradient of E_s = (B z).q + q.A q/(2f) at fixed q (A_kk = zeta_k sqrt(2/pi)/S_k as given to
 * pcm_setup, its derivative through Eq. 9):  g_point[3k + x] = dE_s/d(x of point k) with every atom fixed,
 * g_atom[3J + x] = dE_s/d(x of atom J, as nucleus and as sphere centre) with every point fixed; the caller adds a
 * point's row to the atom it moves with.  Together with pcm_gradient (times -1: c = -v) this is all of
 * Eq. 14.  q_dev: DEVICE M; g_point_dev: DEVICE 3*M; g_atom_dev: DEVICE 3*natom (either may be NULL).  Asynchronous.
 */
int pcm_switching(int64_t npoint, const double *pt_xyz_host, const double *pt_zeta_host, const int32_t *pt_atom_host, int natom,
                  const double *atom_xyz_host, const double *atom_radius_host, double *S_host, int device);
int pcm_set_cavity(pcm_ctx *ctx, const double *atom_radius_host, const int32_t *pt_atom_host);
int pcm_surface_gradient(pcm_ctx *ctx, const double *q_dev, double f, double *g_point_dev, double *g_atom_dev, void *stream);

/*
 * ISWIG cavity construction on the device: the surface points of a molecule from its atoms.
 *
 * pcm_build_cavity -- every atom I (centre R_I, cavity radius rad_I; the paper: 1.2 x Bondi) carries the same unit-sphere
 * quadrature of ngrid nodes u_g (unit vectors) with weights w_g > 0, sum w_g = 4 pi.  The paper uses Lebedev grids; the
 * grid is an INPUT here (any quadrature of the sphere).  For every (I, g):
 *     r_k = R_I + rad_I u_g,   zeta_k = zeta_tab / (rad_I sqrt(w_g))   (Eq. 7; zeta_tab = the tabulated exponent of the
 *     quadrature level),   S_k = prod_{J != I} S_wf(r_k, R_J)   (Eq. 9)
 * and the point is kept iff S_k >= s_min ("MS points with a switching function value less than this threshold are
 * ignored"; the paper's value is 1e-8).  The kept points are in (atom, node) order.  All arrays HOST:
 * atom_xyz 3*natom (bohr), atom_radius natom (> 0), grid_xyz 3*ngrid, grid_weight ngrid.  device: CUDA ordinal, -1 =
 * current.  On success *out owns DEVICE arrays of the kept points (pcm_cavity_device) until pcm_cavity_destroy.
 * Synchronous.  natom = 0 or ngrid = 0 give an empty cavity.  Errors: PCM_ERR_ARG, PCM_ERR_ALLOC, PCM_ERR_CUDA.
 *
 * pcm_cavity_size -- number of kept points.
 * pcm_cavity_get -- copies to HOST arrays (any may be NULL): pt_xyz 3*n, pt_zeta n, pt_switch n (S_k), pt_atom n (owning
 * atom I), pt_node n (grid node g).
 * pcm_cavity_device -- the DEVICE arrays themselves (owned by the cavity; any out pointer may be NULL).
 * pcm_setup_cavity -- pcm_setup with npoint, pt_xyz, pt_zeta and pt_switch taken from the cavity (no caller-side copy of
 * the points); the context also remembers the cavity's radii and owners, so that after pcm_set_nuclei with the same
 * natom atoms pcm_surface_gradient works without pcm_set_cavity.  Point k of the context is point k of the cavity.
 */
typedef struct pcm_cavity pcm_cavity;
int pcm_build_cavity(pcm_cavity **out, int natom, const double *atom_xyz_host, const double *atom_radius_host, int ngrid,
                     const double *grid_xyz_host, const double *grid_weight_host, double zeta_tab, double s_min, int device);
int pcm_cavity_size(const pcm_cavity *cav, int64_t *npoint);
int pcm_cavity_get(const pcm_cavity *cav, double *pt_xyz_host, double *pt_zeta_host, double *pt_switch_host, int32_t *pt_atom_host,
                   int32_t *pt_node_host);
int pcm_cavity_device(const pcm_cavity *cav, const double **xyz_dev, const double **zeta_dev, const double **switch_dev,
                      const int32_t **atom_dev, const int32_t **node_dev);
int pcm_cavity_destroy(pcm_cavity *cav);
int pcm_setup_cavity(pcm_ctx **out, int nshell, const int *shell_l, const double *shell_xyz, const int *shell_nprim,
                     const double *prim_exp, const double *prim_coef, const pcm_cavity *cav, const pcm_options *opt);

/*
 * Host-buffer forms of the four hot calls: same semantics, every array is a HOST pointer; the call
 * copies inputs to the device, runs the device path on the context's own stream, copies the result back
 * and synchronises.  These are what bench.py's end-to-end figure times.  Of P and F only the elements of
 * surviving shell pairs cross PCIe (pcm_info.components x 16 bytes, gathered / scattered on the host with
 * OpenMP through a pinned staging buffer owned by the context): pcm_potential_host reads no other element
 * of P_host; pcm_fock_host zero-fills F_host (accumulate = 0) or leaves the other elements as they are.
 */
int pcm_potential_host(pcm_ctx *ctx, const double *P_host, int64_t ldp, double *v_host);
int pcm_fock_host(pcm_ctx *ctx, const double *q_host, double *F_host, int64_t ldf, int accumulate);
int pcm_amatvec_host(pcm_ctx *ctx, const double *q_host, double *y_host);
int pcm_cg_solve_host(pcm_ctx *ctx, const double *b_host, double *x_host, double tol, int max_iter, int precond,
                      int use_x0, int *iters, double *resid);

/* Counts that define the throughput metric (primitive pair x point per call).  No device work. */
int pcm_get_info(pcm_ctx *ctx, pcm_info *out);

/*
 * Kernel timing.  pcm_set_timing(ctx, 1) makes pcm_potential (op 0), pcm_fock (op 1) and pcm_amatvec (op 2) record
 * CUDA events on the launching stream around their kernels (each op has its own event set).
 * pcm_last_kernel_ms: for the most recent timed call of `op`, ms[0] = the main integral kernels, ms[1] = pre/post transforms
 * and reductions (op 2: ms[0] = the whole product, sweep and row sums, ms[1] = 0); n_launch (may be NULL) = kernels that
 * call launched.
 * pcm_last_class_ms: the same call split by total angular momentum, ms[L] = device time of the main kernel of the
 * products with L = l_a + l_b = 0..4 (op 2: ms[0] is its one kernel).  Both synchronise on the recorded events.
 */
int pcm_set_timing(pcm_ctx *ctx, int enable);
int pcm_last_kernel_ms(pcm_ctx *ctx, int op, double ms[2], int *n_launch);
int pcm_last_class_ms(pcm_ctx *ctx, int op, double ms[PCM_NL]);

/* pcm_last_cg_matvec_ms -- with timing on: mean device time of the A q launches (main + near kernels) of the first
 * 16 iterations of the most recent pcm_cg_solve, and how many were timed (n may be NULL).  Note that queued iterations
 * after convergence are no-ops; only solves of >= 16 iterations give the figure of a working iteration. */
int pcm_last_cg_matvec_ms(pcm_ctx *ctx, double *avg_ms, int *n);

/* pcm_launch_count -- kernels launched by this context since pcm_setup (bench.py's gpu_launches). */
int pcm_launch_count(pcm_ctx *ctx, int64_t *total);

/*
 * pcm_fp64_peak -- a register-resident DFMA-chain microbenchmark on the context's device: the measured
 * FP64 FMA rate in TFLOP/s (2 flop per DFMA), best of `reps`.  The ALU roofline denominator of bench.py.
 */
int pcm_fp64_peak(pcm_ctx *ctx, int reps, double *tflops);

/*
 * pcm_schwarz_bound -- the screening quantity of Eq. 15 for one primitive pair of RAW Cartesian
 * primitives of angular momenta la, lb in {0,1,2}: max over Cartesian components of
 * [chi_a chi_b|chi_a chi_b]^{1/2} (a two-electron self-repulsion integral; contraction coefficients NOT
 * included -- pcm_setup multiplies by |c_i c_j|).  A, B: HOST, 3 doubles.  Host arithmetic only, no device work.
 */
int pcm_schwarz_bound(int la, double alpha, const double *A, int lb, double beta, const double *B, double *out);

/*
 * pcm_amatvec_static -- y = A q (Eq. 2, 3, 8; A_ij = erf(zeta'_ij r_ij)/r_ij,
 * zeta'_ij = zeta_i zeta_j/sqrt(zeta_i^2 + zeta_j^2), A_ii = zeta_i sqrt(2/pi)/S_i) WITHOUT a context and without
 * allocating anything: no cudaMalloc, cudaFree or allocating library routine on this path, so it may be called under
 * CUDA graph capture, from serving loops and from harnesses that forbid allocation.  Its only scratch (16 partial sums
 * per row, added in a fixed order) is a static __device__ array of 16 x PCM_STATIC_MAX_POINTS doubles = 2 MiB that every
 * GPU loading the library holds until the process exits.
 *   npoint: 0 ... PCM_STATIC_MAX_POINTS; more is refused with PCM_ERR_ARG (use pcm_setup + pcm_amatvec, which is also
 *   several times faster: this variant sweeps the full square with erf, no symmetry, no stored near field).
 *   pt_xyz_dev [3 npoint] (x, y, z per point), pt_zeta_dev, pt_switch_dev, q_dev [npoint]: DEVICE, read;
 *   y_dev [npoint]: DEVICE, overwritten; all in the caller's point order; the caller keeps ownership.
 *   stream: cudaStream_t; asynchronous (two launches).  Coincident points give the limit 2 zeta'/sqrt(pi).
 * The scratch array is shared by all calls on a device and keeps the last call's contents; a call writes every slot it
 * reads, so nothing needs clearing, but CALLS THAT OVERLAP ON ONE GPU (two streams, two threads) RACE on it: keep them
 * stream-ordered.  pcm_amatvec_static_init resolves the array's device address for the CURRENT device (once per device;
 * the first use also loads the module): call it at set-up, outside any capture; pcm_amatvec_static does it itself on
 * a device it has not seen.  Errors: PCM_ERR_ARG, PCM_ERR_CUDA (text: pcm_last_error(NULL)).
 */
#define PCM_STATIC_MAX_POINTS 16384
int pcm_amatvec_static_init(void);
int pcm_amatvec_static(int64_t npoint, const double *pt_xyz_dev, const double *pt_zeta_dev, const double *pt_switch_dev,
                       const double *q_dev, double *y_dev, void *stream);

/* Text of the last error on this context (ctx == NULL: of the last failed context-free call on this thread). */
const char *pcm_last_error(pcm_ctx *ctx);

/* Frees device and host state.  NULL is allowed. */
int pcm_destroy(pcm_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* PCM_B200_H */
