/*
 * mop.h -- C-ABI of libmop_b200: the data-parallel hot path of the
 * metadynamics-of-paths (MoP) method, arxiv 2501.11962, for one NVIDIA B200.
 *
 * What the library computes (citations are lines of the paper text PAPER.md):
 *   - the Onsager-Machlup effective potential of an N-bead discretised path,
 *       V_eff = U(R^1) + sum_{n=1}^{N-1} sum_i K_i/2 |R^{n+1}_i - R^n_i - L^n_i|^2     eq. (3)
 *     with K_i = m_i nu / (2 dt) and L^n_i = dt/(m_i nu) F^n_i
 *     (the printed L^n is inverted; reading G1 in DESIGN.md: eqs (5)-(7) need K L/F = 1/2),
 *     F^n = -grad U(R^n);
 *   - its gradient dV_eff/dR^n = -F_eff^n, F_eff^n as in eqs (5),(6),(7), with the
 *     finite-difference bracket [F(R+eps eta)-F(R-eps eta)]/(4 eps) replaced by its eps->0 limit
 *     -(1/2) H(R^n) eta^n, computed analytically (eta^n = R^{n+1}-R^n-L^n);
 *   - velocity-Verlet path MD of the polymer, M d2R^n/dt2 = F_eff^n, eq. (4).
 * U is BASELINE.json's force field: Lennard-Jones 12-6 (optional potential shift) + reaction-field
 * Coulomb with a plain cutoff r_cut, harmonic bonds and harmonic angles, explicit exclusions.
 *
 * Units: nm, ps, u, kJ/mol, e (1 kJ/mol = 1 u nm^2/ps^2).  Coulomb constant 138.935458 kJ mol^-1 nm e^-2.
 *
 * Conventions
 *   - "HOST" / "DEVICE" says where a pointer must live.  Device pointers are plain CUDA device
 *     addresses on `params.device`; the caller (e.g. torch) owns R, V, grad; the library owns
 *     everything else and frees it in mop_destroy.
 *   - All work is enqueued on `params.stream`; a call synchronises the stream only where stated.
 *   - No exceptions or abort() cross the ABI: every call returns a mop_status; CUDA errors are
 *     sticky per context; mop_last_error gives a text.
 *   - Calls on one context are not thread-safe.
 *   - There is no CPU fallback: without a CUDA device mop_create returns MOP_ERR_CUDA.
 */
#ifndef MOP_B200_H
#define MOP_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mop_ctx mop_ctx; /* opaque; one per (device, system) */

typedef enum {
    MOP_OK = 0,
    MOP_ERR_INVALID_ARG = 1,   /* bad size, pointer, index, non-positive mass, asymmetric exclusions */
    MOP_ERR_NO_TOPOLOGY = 2,   /* eval/step before mop_set_topology */
    MOP_ERR_BOX_TOO_SMALL = 3, /* min(box) < 2 (r_cut + r_buf): the in-range periodic image would not be unique */
    MOP_ERR_OOM = 4,           /* device allocation failed, or a pair-list buffer overflowed (not sticky: the buffers
                                  are regrown from the builder's counts and the call can be repeated) */
    MOP_ERR_CUDA = 5,          /* any CUDA runtime error (sticky), or no device */
    MOP_ERR_NONFINITE = 6      /* V_eff came out NaN/Inf (overlapping atoms), or an input coordinate is NaN/Inf or
                                  farther than ~1e6 box lengths from the box (sticky) */
} mop_status;

/* Problem statement of PAPER.md:36-52: Q atoms, N beads at path spacing dt, friction nu.  Copied at create. */
typedef struct {
    int n_atoms;      /* Q >= 1 */
    int n_beads;      /* N >= 1 */
    float box[3];     /* rectangular periodic box (nm) */
    float r_cut;      /* nonbonded cutoff (nm), > 0 */
    float r_buf;      /* Verlet buffer (nm), >= 0.  0: the pair list is rebuilt in every evaluation and the neighbour
                         sets follow the bit-exact predicate of DESIGN.md (reading G8).  > 0: the list is built with
                         r_cut + r_buf and kept while no atom of a force bead has moved farther than r_buf/2 from
                         where it was at the build; a reusing evaluation refreshes the sorted coordinates in the
                         periodic image of that build (wrap(R_ref) + (R - R_ref): the same pairs to FP32 rounding
                         of r^2, not bit for bit) and reads one flag on the host, which synchronises the stream.
                         Results never depend on the list: the r_cut test is applied per atom pair */
    float eps_rf;     /* reaction-field dielectric; <= 0 means infinity (k_rf = 1/(2 r_cut^3)) */
    int lj_shift;     /* 1: potential-shift the LJ energy so that U_LJ(r_cut) = 0 (forces unchanged) */
    double dt_path;   /* path spacing Delta t (ps): enters K_i and L^n only */
    double nu;        /* Smoluchowski friction nu (1/ps): enters K_i and L^n only */
    int device;       /* CUDA ordinal */
    void *stream;     /* cudaStream_t all work is enqueued on (NULL: the legacy default stream) */
} mop_params;

/* HOST pointers; copied to the device inside mop_set_topology; the caller keeps ownership. */
typedef struct {
    const float *mass;   /* [Q] u, > 0 (physical = fictitious masses, reading G4) */
    const float *charge; /* [Q] e */
    const int *type;     /* [Q] in [0, n_types) */
    int n_types;         /* 1..64 */
    const float *c6;     /* [n_types*n_types] symmetric, kJ/mol nm^6 */
    const float *c12;    /* [n_types*n_types] symmetric, kJ/mol nm^12 */
    int n_bonds;
    const int *bond_ij;        /* [n_bonds][2] atom indices */
    const float *bond_b0_kb;   /* [n_bonds][2] = (b0 nm, k_b kJ/mol/nm^2); u = k_b/2 (r-b0)^2 */
    int n_angles;
    const int *angle_ijk;      /* [n_angles][3], j central */
    const float *angle_t0_kt;  /* [n_angles][2] = (theta0 rad, k_theta kJ/mol/rad^2); u = k_t/2 (theta-theta0)^2 */
    const int *excl_start;     /* CSR [Q+1] (may be NULL when there are no exclusions) */
    const int *excl_list;      /* symmetric, sorted; an excluded pair gets NO nonbonded term (no RF correction, G10) */
} mop_topology;

/* Creates a context for (device, Q, N, box, cutoffs); allocates nothing that depends on the topology.
 * Errors: INVALID_ARG, BOX_TOO_SMALL, CUDA, OOM. */
mop_status mop_create(mop_ctx **out, const mop_params *p);

/* Validates and uploads the topology; may be called again to replace it.  Synchronises the stream. */
mop_status mop_set_topology(mop_ctx *c, const mop_topology *t);

/* V_eff (eq. 3) and its gradient (= -F_eff of eqs 5,6,7) for the whole path.
 *   R_dev    DEVICE [N][Q][3] float; beads image-consistent (an atom's coordinate is continuous along the
 *            path; the library wraps only its internal sorted copy).  Read only.
 *   veff_out HOST; non-NULL: the call synchronises the stream and stores V_eff (kJ/mol);
 *            NULL: fully asynchronous, the value stays in the context (mop_get_stats).
 *   grad_dev DEVICE [N][Q][3] float, dV_eff/dR^n_i in kJ/mol/nm, caller-allocated; NULL: not written.
 * Passes: S0 bin+sort, S1 pair list, S2 nonbonded force, S3 bonded force,
 * S4 eta + spring energy, S5 nonbonded H.eta, S6 bonded H.eta, S7 assembly.
 * Errors: NO_TOPOLOGY, INVALID_ARG, OOM (list overflow: flagged on the device by any build, reported at the next
 * synchronising call, after which the regrown buffers let the call be repeated), CUDA, NONFINITE. */
mop_status mop_eval_veff_grad(mop_ctx *c, const float *R_dev, double *veff_out, float *grad_dev);

/* The same evaluation with HOST buffers (the end-to-end form): copies R_host [N][Q][3] to the device on the
 * context stream, evaluates, copies the gradient back to grad_host [N][Q][3] (may be NULL) and V_eff to *veff_out
 * (required).  Pinned host memory makes the copies asynchronous to the host until the final synchronisation;
 * pageable memory works too.  Synchronises.  The device staging buffers belong to the context. */
mop_status mop_eval_veff_grad_host(mop_ctx *c, const float *R_host, double *veff_out, float *grad_host);

/* n_steps velocity-Verlet steps of eq. (4) with F_eff = -grad V_eff and masses m_i, step dt_pmd (ps):
 *   v += dt/2 F_eff/m ; R += dt v ; F_eff(R) ; v += dt/2 F_eff/m.
 * R_dev, V_dev DEVICE [N][Q][3] float, updated in place.  The gradient at the incoming R is evaluated at the
 * start of every call (n_steps + 1 evaluations per call; mop_step_continue skips it).  Only the last evaluation of a
 * call forms U(R^1) (the others need the gradient alone), so mop_get_stats after the call reports V_eff at the final R.
 * Asynchronous. */
mop_status mop_step(mop_ctx *c, float *R_dev, float *V_dev, double dt_pmd, int n_steps);

/* NULL-safe; frees all library-owned memory. */
void mop_destroy(mop_ctx *c);

/* Static or context-owned text for the last non-OK status (c may be NULL: creation errors). */
const char *mop_last_error(const mop_ctx *c);

/* ---- optional, for tests and benches ------------------------------------------------------------- */

/* Synchronises.  out[0]=V_eff, [1]=U(R^1), [2]=E_spring, [3]=U_lj(R^1), [4]=U_coul(R^1), [5]=U_bond(R^1),
 * [6]=U_angle(R^1), [7]=kinetic energy after the last mop_step, [8]=pair-list rebuilds so far,
 * [9]=cluster-pair entries in the current list, [10]=list units, [11]=exclusion masks,
 * [12]=pair slots the list admits per nonbonded pass (sum over entries of popcount(row-pair pattern) * 16), [13]=kernel launches so far,
 * [14]=evaluations that reused a buffered list (r_buf > 0), [15]=pair slots the pair kernels evaluate per pass (64 per row pair
 * of every step's union pattern: [12] plus the steps whose four octets differ in pattern). */
mop_status mop_get_stats(mop_ctx *c, double out[16]);

/* Stage timing with CUDA events on the context stream (the stream the kernels are launched on).  on != 0: every
 * later mop_eval_veff_grad / _host / mop_step evaluation records 9 events around its stages; on or off: the
 * accumulated sums are reset.  Evaluations made through mop_force_hvp are not timed. */
mop_status mop_set_timing(mop_ctx *c, int on);

/* Synchronises with the timed evaluations issued so far.  out[k], k = 0..7: mean milliseconds per evaluation of
 * stage S0 grid build, S1 pair list, S2 nonbonded force kernels, S3 bonded force, S4 eta + spring energy,
 * S5 nonbonded H.eta kernel, S6 bonded H.eta, S7 assembly; out[8] = evaluations averaged; rest 0. */
mop_status mop_get_timing(mop_ctx *c, double out[16]);

/* Copies an internal array of the last evaluation to HOST memory (synchronises).  `what`:
 *   "dims"  int[8]: nx, ny, nz (search grid), slots per bead S (padded, multiple of 32), force beads nf,
 *           cluster size 8, j-clusters per warp step 4, z-bin thickness (float bits)
 *   "cell"  int[nf][Q]   cell id of every atom, cell = (cx*ny+cy)*nz+cz (reading G8)
 *   "perm"  int[nf][S]   original atom index held by each sorted slot, -1 for padding (stable sort, G13)
 *   "xq"    float[nf][S][4] wrapped coordinates + charge in sorted order
 *   "F"     float[nf][Q][3] physical force F^n in ORIGINAL atom order
 *   "eta"   float[nf][Q][3] eta^n in original order;  "Heta" float[nf][Q][3] H^n eta^n likewise
 * bytes must equal the size of the array.  Errors: INVALID_ARG. */
mop_status mop_debug_get(mop_ctx *c, const char *what, void *host_buf, size_t bytes);

/* In-range (r2 < r_cut^2 under the FP32 predicate G8), non-excluded atom pairs of bead `bead` of the last
 * evaluation, found by walking the pair list with the force kernel's own predicate.  Writes up to `cap` pairs
 * (original indices, unordered) to HOST pairs[2*k], pairs[2*k+1] (may be NULL with cap 0) and the total count
 * to *n_pairs.  Synchronises. */
mop_status mop_debug_pairs(mop_ctx *c, int bead, int *pairs, long long cap, long long *n_pairs);

/* Physical force and H.s of ONE configuration treated as bead 1 of a context with n_beads == 1 is what
 * mop_eval_veff_grad already gives (grad = -F).  For a user-supplied direction s:
 *   R_dev, s_dev DEVICE [Q][3]; F_dev, Hs_dev DEVICE [Q][3] outputs (either may be NULL).  Uses bead slot 0.
 * This is the pass-2 kernel with eta := s.  Asynchronous. */
mop_status mop_force_hvp(mop_ctx *c, const float *R_dev, const float *s_dev, float *F_dev, float *Hs_dev);

/* The same V_eff and gradient with the Hessian term of eqs (5),(6) evaluated the way the paper does it
 * (PAPER.md:61-70, 107-110): the central finite difference [F(R^n + eps eta^n) - F(R^n - eps eta^n)] / (4 eps) of two
 * displaced force evaluations (PMD kernels 2, 3) instead of the analytic -1/2 H^n eta^n.  eps > 0 is the paper's
 * dimensionless epsilon, one value for all beads (PAPER.md:64 leaves it open: "small enough"; eps * max|eta| of 1e-5 to
 * 1e-4 nm keeps both the truncation and the FP32 cancellation error small).  Costs three force passes per bead, each
 * displaced configuration with its own cell list and pair list.  With a plain cutoff a pair that crosses r_cut between
 * R + eps eta and R - eps eta contributes its force jump divided by 4 eps (reading G9); the analytic form has no such term.
 * R_dev, grad_dev DEVICE [N][Q][3] (grad_dev required); veff_out HOST or NULL as in mop_eval_veff_grad.  After this
 * call mop_debug_get / mop_debug_pairs describe the last displaced configuration.  Errors: INVALID_ARG, OOM, CUDA. */
mop_status mop_eval_veff_grad_fd(mop_ctx *c, const float *R_dev, double eps, double *veff_out, float *grad_dev);

/* Path MD in the canonical ensemble (the paper's NVT validation and scaling runs: "Langevin thermostat ... damping
 * coefficient 0.25 fs^-1" at 310 K, Fig. 4b).  The paper does not give the discretisation;
 * reading G19: each step is the velocity-Verlet step of mop_step followed by the exact Ornstein-Uhlenbeck
 * velocity update  v <- c v + sqrt((1 - c^2) k_B T / m_i) xi,  c = exp(-gamma dt_pmd),  k_B = 0.0083144626 kJ/mol/K,
 * xi ~ N(0,1) drawn from a counter-based generator keyed by (seed, step0 + step index, index of the coordinate in
 * [N][Q][3]), so a run can be replayed and continued (pass step0 = steps already done).  gamma (1/ps) >= 0; gamma = 0
 * is mop_step.  E_kin in mop_get_stats is taken after the thermostat update of the last step.  Asynchronous. */
mop_status mop_step_langevin(mop_ctx *c, float *R_dev, float *V_dev, double dt_pmd, int n_steps, double gamma,
                             double temperature, unsigned long long seed, unsigned long long step0);

/* Debug: the 64 raw bits of the thermostat's generator for (seed, step, idx), idx = 0..n-1, to HOST memory
 * (compared bit for bit with the oracle's independent implementation).  Synchronises. */
mop_status mop_debug_noise_bits(mop_ctx *c, unsigned long long seed, unsigned long long step, int n,
                                unsigned long long *host_out);

/* Metadynamics of paths: a history-dependent bias V(S) = sum_k height exp(-(S - S_k)^2 / (2 sigma^2))
 * on the end-to-end collective variable S_e2e = s(R^N) - s(R^1) (eq. 8), with s(R) = the distance between the centres of mass
 * of two atom groups ("the center of mass of the ligand and the binding pocket"; minimum image of the COM
 * difference; each group must be whole in the caller's coordinates).  While a bias is set, every evaluation that writes a
 * gradient (mop_eval_veff_grad, _host, mop_step, mop_step_langevin; not mop_eval_veff_grad_fd) adds dV/dR^1 and dV/dR^N to
 * it -- the CV touches the first and last bead only -- and mop_step / mop_step_langevin deposit a hill at the current S_e2e
 * every `pace` steps (PAPER.md:155 deposits one every 500; 0: never).  veff_out stays eq. (3) without V(S).
 * group_a, group_b: HOST index arrays (copied).  n_a = n_b = 0 switches the bias off.  Setting a bias clears the hills.
 * Errors: INVALID_ARG (empty group, index out of range, sigma <= 0, n_beads < 2), OOM, CUDA. */
mop_status mop_set_bias(mop_ctx *c, const int *group_a, int n_a, const int *group_b, int n_b, double sigma, double height,
                        int pace);
/* Deposits one hill centred at s_center by hand (at most 65536 hills; OOM beyond).  Synchronises. */
mop_status mop_add_hill(mop_ctx *c, double s_center);
/* State of the bias at the last evaluation (synchronises): out[0] S_e2e, out[1] s(R^1), out[2] s(R^N), out[3] V(S),
 * out[4] dV/dS, out[5] number of hills; hills_host (may be NULL) receives up to cap hill centres, *n_hills their number. */
mop_status mop_get_bias(mop_ctx *c, double out[8], double *hills_host, int cap, int *n_hills);

/* mop_step / mop_step_langevin without the evaluation at the incoming R: the caller states that R_dev is exactly what the
 * previous mop_step* call on this context left behind (the context still holds the gradient there), so a caller that
 * advances a few steps per call pays n_steps evaluations per call instead of n_steps + 1.  Same results as one longer
 * mop_step call.  Errors: INVALID_ARG when no such gradient is held (first call, or after mop_set_topology,
 * mop_set_bias, mop_add_hill), otherwise as mop_step. */
mop_status mop_step_continue(mop_ctx *c, float *R_dev, float *V_dev, double dt_pmd, int n_steps);
mop_status mop_step_langevin_continue(mop_ctx *c, float *R_dev, float *V_dev, double dt_pmd, int n_steps, double gamma,
                                      double temperature, unsigned long long seed, unsigned long long step0);

/* The production force kernel's OWN in-range decisions over the pair list of the last evaluation: its counting
 * instance (the same code plus a population count of the per-pair results of the predicate G8 and of the exclusion
 * masks) is run once more; HOST *n_inrange receives the count and *pair_hash (may be NULL) an order-independent
 * fingerprint of the decided pair SET: the sum mod 2^64 over the decided pairs of splitmix64(((bead * Q + min(i,j)) * Q +
 * max(i,j)) + 0x9E3779B97F4A7C15) with i, j original atom indices and bead the 0-based force bead.  which = 0: bead 1;
 * 1: the other force beads; 2: all force beads.  This, not the scalar walker of mop_debug_pairs, is what the bit-exact
 * neighbour-set claim of the pair kernels rests on (the tests hold count and fingerprint equal to the oracle's pair list).
 * Synchronises. */
mop_status mop_debug_count_inrange(mop_ctx *c, int which, long long *n_inrange, unsigned long long *pair_hash);

/* Testing aid: replaces the pair-list buffers by ones of the given capacities (work units, octet-pair entries, exclusion-mask
 * rows; 0 keeps one; at least 64 each) and switches off the automatic capacity check of the first evaluation, so that the
 * overflow / regrow path (MOP_ERR_OOM, then a successful repeat) can be driven deterministically.  Synchronises. */
mop_status mop_debug_set_list_capacity(mop_ctx *c, unsigned units, unsigned entries, unsigned masks);

/* ---- bead-block mode -------------------------------------------------------------
 * The paper's parallel layout: the beads of the path are spread over processing elements and only the owners of ADJACENT
 * beads exchange data ("each bead ... a separate processing element"; non-blocking send/recv between
 * neighbouring beads; weak scaling in the number of beads).  Here one context (one GPU, one
 * process) owns the contiguous block of beads [first_bead, first_bead + p->n_beads) of a path of n_beads_path beads.
 * Eqs (3),(5)-(7) couple bead n to beads n-1 and n+1 only, so one evaluation needs two halos, each DEVICE [Q][3] float in
 * original atom order:
 *   from the right neighbour, before pass 1: R_right = its first bead R^{n1} (eta of the block's last bead);
 *   from the left neighbour, before the assembly: K eta^{n0-1}, which that neighbour's mop_block_pass1 writes to its
 *     keta_right_out_dev (the spring term K eta^{n-1} of eqs (5),(7)).
 * The library does no communication: the caller moves the halos (blocks.py: torch.distributed batch_isend_irecv, NCCL point-to-point) and sums
 * the per-block V_eff values (an 8-byte all-reduce).  Call order per evaluation: mop_block_pass1 (S0-S4), mop_block_pass2
 * (S5-S6), mop_block_assemble (S7); the halo for the right neighbour is ready once pass1 has run, so its transfer overlaps
 * pass 2.  Force, eta and H.eta run on every bead of the block except the path's last bead; U(R^1) only in the block with
 * first_bead = 0.  A block that is the whole path (first_bead = 0, n_beads = n_beads_path) also accepts the whole-path calls
 * above; other block contexts refuse them (INVALID_ARG), and none of them takes a bias.  The sum over blocks of
 * veff_local_out is V_eff; the blocks' gradients are the rows of the whole-path gradient.  Path MD on a sharded path: every
 * bead moves with its own gradient, so mop_block_integrate (NVE) and mop_block_thermostat (NVT) need no exchange.
 * Errors: as mop_create / mop_eval_veff_grad; INVALID_ARG for a block outside the path, a missing halo, or calls out of order. */
mop_status mop_create_block(mop_ctx **out, const mop_params *p, int first_bead, int n_beads_path);
mop_status mop_block_pass1(mop_ctx *c, const float *R_dev, const float *R_right_dev, float *keta_right_out_dev);
mop_status mop_block_pass2(mop_ctx *c, const float *R_dev);
/* keta_left_dev: NULL for first_bead = 0.  veff_local_out: HOST, non-NULL synchronises (U(R^1) if the block holds bead 1,
 * plus the spring energy of the block's own eta).  grad_dev DEVICE [n_beads][Q][3]. */
mop_status mop_block_assemble(mop_ctx *c, const float *keta_left_dev, double *veff_local_out, float *grad_dev);
/* One half of a velocity-Verlet step of eq. (4) on the block's beads with a gradient the caller holds (every bead moves
 * with its own gradient, so the integrator needs no exchange): stage 0: v += dt/2 (-grad)/m; R += dt v.  stage 1:
 * v += dt/2 (-grad)/m.  Works on any context. */
mop_status mop_block_integrate(mop_ctx *c, float *R_dev, float *V_dev, const float *grad_dev, double dt_pmd, int stage);
/* The thermostat half of an NVT step on the block's beads -- the configuration of the paper's scaling runs ("for each polymer
 * size, we have performed an NVT simulation"; Langevin, damping 0.25 fs^-1): the exact
 * Ornstein-Uhlenbeck update of mop_step_langevin (reading G19), v <- c v + sqrt((1 - c^2) k_B T / m_i) xi, applied to
 * V_dev DEVICE [n_beads][Q][3] after stage 1 of mop_block_integrate.  The generator is keyed by (seed, step, index of the
 * coordinate in the WHOLE path's [n_beads_path][Q][3] array), so the blocks of a sharded run together draw exactly the numbers
 * one mop_step_langevin call on the whole path draws for PMD step `step` (= its step0 + step index): no exchange is needed
 * and the trajectory does not depend on how the path is cut.  gamma = 0 does nothing.  Works on any context (first bead 0
 * for a whole-path context).  Asynchronous.  Errors: INVALID_ARG. */
mop_status mop_block_thermostat(mop_ctx *c, float *V_dev, double dt_pmd, double gamma, double temperature,
                                unsigned long long seed, unsigned long long step);

/* ---- for callers that must not allocate device memory ------------------------------------------------------------------
 * Everything above works on a context, and a context allocates (mop_create, mop_set_topology, list regrowth).  Some callers
 * cannot accept that: a host program that hands out all device memory from its own pool at start-up and forbids driver
 * allocations afterwards, a process in which another framework has already reserved almost all of HBM, or a stepping loop
 * that cannot afford the device-wide synchronisation of cudaMalloc / cudaFree.  For them, ONE stage of the path is offered
 * as a stateless call that allocates nothing, neither directly nor through a library routine: the displacement and spring-
 * energy stage S4 (the paper's PMD kernels 1 and 7)
 *     eta^n_i = (R^{n+1}_i - R^n_i) - dt/(m_i nu) F^n_i,    E_spring = sum_{n=1}^{N-1} sum_i m_i nu/(4 dt) |eta^n_i|^2
 * (second term of eq. (3); L^n as in reading G1), with the arithmetic of the context path (FP32 eta, FP64 sum).
 *   device, stream   CUDA ordinal and cudaStream_t (NULL: legacy default stream) the work is enqueued on; asynchronous
 *   R_dev            DEVICE [n_beads][n_atoms][3] float, image-consistent beads, n_beads >= 2
 *   F_dev            DEVICE [n_beads-1][n_atoms][3] float, physical forces F^n of beads 1..N-1 (e.g. from the caller's engine)
 *   mass_dev         DEVICE [n_atoms] float, > 0
 *   eta_dev          DEVICE [n_beads-1][n_atoms][3] float, written
 *   e_spring_dev     DEVICE double, written (kJ/mol); summed in a fixed order, so equal inputs give equal bits
 *   err, err_len     HOST buffer for a message on failure (may be NULL / 0)
 * All five device buffers belong to the caller.  The kernel's only working memory (one FP64 partial sum per 256 (atom, bead)
 * pairs and a counter) is a fixed array of MOP_NOALLOC_SCRATCH_BYTES inside the library image; every GPU this process uses
 * the library on holds it until exit.  Consequences the caller must know:
 *   - size limit: n_atoms * (n_beads - 1) <= MOP_NOALLOC_MAX_ATOM_BEADS, otherwise MOP_ERR_INVALID_ARG and nothing is
 *     launched (evaluate a longer path as consecutive bead ranges and add the energies);
 *   - one array per device for all threads and streams: calls that may run on the same GPU at the same time race on it;
 *     keep them on one stream or order them with events.  The call itself resets what has to start at zero, so nothing
 *     carries over from one call to the next;
 *   - the first call on each device looks up the array's device address (with `device` made current for the duration of
 *     the call, restored afterwards); issue that first call outside any stream capture.
 * Errors: INVALID_ARG (sizes, NULL pointers, dt_path or nu <= 0, limit exceeded), CUDA (no device, launch failure). */
#define MOP_NOALLOC_MAX_ATOM_BEADS 33554432              /* 2^25 = 131,072 thread blocks of 256 */
#define MOP_NOALLOC_SCRATCH_BYTES (256 + 131072 * 8)     /* 1,048,832 bytes per GPU */
mop_status mop_eta_spring_noalloc(int device, void *stream, int n_atoms, int n_beads, double dt_path, double nu,
                                  const float *R_dev, const float *F_dev, const float *mass_dev, float *eta_dev,
                                  double *e_spring_dev, char *err, size_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* MOP_B200_H */
