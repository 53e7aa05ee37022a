// mop_api.cu -- the C-ABI of include/mop.h: context, device memory, pass orchestration on one CUDA stream.
// Every step of the hot path runs in the kernels of this directory; there is no CPU fallback.
#include "../../include/mop.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "mop_bias.cuh"
#include "mop_bonded.cuh"
#include "mop_common.cuh"
#include "mop_grid.cuh"
#include "mop_nonbonded.cuh"
#include "mop_nonbonded_packed.cuh"
#include "mop_pairlist.cuh"
#include "mop_path.cuh"

static thread_local char g_create_error[256] = "";

#define MOP_NSTAGE 8  // S0 grid, S1 pair list, S2 nonbonded force, S3 bonded force, S4 eta, S5 nonbonded H.eta, S6 bonded H.eta, S7 assembly
#define MOP_TSETS 64

struct mop_ctx {
    mop_params p;
    int Q, N, nf;              // atoms; beads held by this context; force beads (allocation, >= 1)
    int nfe = 0, nh = 0;       // beads whose force is evaluated (0 for a block that is only the path's last bead); beads with eta and H.eta
    bool has_u1 = true;        // the context's first bead is bead 1 of the path (U(R^1) and the -F^1 term)
    bool blk = false;          // bead-block mode (mop_create_block): beads [blk_n0, blk_n0 + N) of a path of blk_Ntot beads
    int blk_n0 = 0, blk_Ntot = 0;
    int blk_stage = 0;         // 0 idle, 1 after mop_block_pass1, 2 after mop_block_pass2
    cudaStream_t st;
    // library-owned side stream: the bonded kernels (O(Q) terms, latency-bound) run beside the pair kernels of the same pass
    cudaStream_t st2 = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    // copy stream of mop_eval_veff_grad_host: the host->device copy of beads 2..N runs behind the work on bead 1
    cudaStream_t st_copy = nullptr;
    cudaEvent_t ev_copy[4] = {nullptr, nullptr, nullptr, nullptr};
    // CUDA graphs of one evaluation on the context's own staging buffers (d_Rh -> d_Gh), in two parts: A = bead 1 (S0, S1,
    // force + energy kernel), B = everything else.  Captured on st_cap; launched into the caller's stream.
    cudaStream_t st_cap = nullptr;
    cudaGraphExec_t gx[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // A, B, B split in two (host entry point), A without U(R^1)
    bool gx_valid = false;
    double gx_launches[5] = {0, 0, 0, 0, 0};
    MopGrid g;
    float bin_z;
    float rl, rl2, rc2;
    float krf;
    double krf_d, crf_d;
    bool has_topology = false;
    int sticky = MOP_OK;
    std::string err;
    double n_launches = 0, n_rebuilds = 0;
    int sm_count = 148;
    // topology (device)
    int nt = 0, n_bonds = 0, n_angles = 0, max_excl = 0;
    float *d_mass = 0, *d_inv_mass = 0, *d_charge = 0, *d_ai = 0, *d_Ki = 0, *d_tabs = 0;
    float2 *d_tab = 0, *d_bond_par = 0, *d_angle_par = 0;
    int *d_type_row = 0, *d_bond_ij = 0, *d_angle_ijk = 0, *d_excl_start = 0, *d_excl_list = 0;
    // per-bead sorted state
    int *d_cell = 0, *d_cell_count = 0, *d_cell_rel = 0, *d_cell_fill = 0, *d_col_count = 0, *d_col_start = 0;
    int *d_tmp = 0, *d_perm = 0, *d_slot_of = 0, *d_typ = 0;
    float4 *d_xq = 0, *d_et = 0, *d_F4 = 0, *d_H4 = 0, *d_blo = 0, *d_bhi = 0;
    // pair list
    MopUnit *d_units = 0;
    MopEntry *d_entries = 0;
    unsigned long long *d_masks = 0;
    unsigned cap_units = 0, cap_entries = 0, cap_masks = 0;
    MopCounters *d_ctr = 0;
    unsigned long long *d_slots = 0;
    unsigned *d_work = 0;   // [8]
    double *d_energy = 0;   // [8]: U_lj, U_coul, U_bond, U_angle, E_spring, E_kin
    // host mirrors (pinned)
    double *h_energy = 0;
    MopCounters *h_ctr = 0;
    unsigned long long *h_slots = 0;
    // scratch
    float *d_G = 0;     // [N][Q][3] gradient for mop_step
    float *d_dbg = 0;   // [nf][Q][3]
    int nb_blocks_f = 0, nb_blocks_fe = 0, nb_blocks_h = 0, nb_blocks_c = 0;
    bool caps_checked = false;  // the list capacities have been checked against one real build (first evaluation)
    bool g_current = false;     // d_G holds the gradient at the R the last mop_step* call returned (mop_step_continue)
    double last_veff = 0, last_ekin = 0;
    // e2e staging (mop_eval_veff_grad_host)
    float *d_Rh = 0, *d_Gh = 0;
    // reuse of a buffered pair list (r_buf > 0)
    bool list_valid = false;
    float *d_Rref = 0;      // [nf][Q][3] caller coordinates at the last build
    int *d_moved = 0, *h_moved = 0;
    double n_reuses = 0;
    // metadynamics-of-paths bias (mop_set_bias)
    bool bias_on = false;
    int bias_na = 0, bias_nb = 0, bias_pace = 0;
    long long bias_steps = 0;
    double bias_sigma = 0, bias_w = 0;
    int *d_bias_ga = 0, *d_bias_gb = 0, *d_bias_nh = 0;
    double *d_bias_hills = 0, *d_bias_com = 0, *d_bias_state = 0;
    // finite-difference Hessian mode (mop_eval_veff_grad_fd): [nf][Q][3] buffers in original atom order
    float *d_fdR = 0, *d_fdEta = 0, *d_fdF = 0, *d_fdFp = 0, *d_fdFm = 0;
    // stage timing (mop_set_timing): a ring of event sets, one per evaluation
    bool timing = false;
    cudaEvent_t ev[MOP_TSETS][MOP_NSTAGE + 1];
    bool ev_made = false;
    int ev_head = 0, ev_pending = 0;   // sets [head-pending, head) await collection
    double t_sum[MOP_NSTAGE] = {0}, t_cnt = 0;
};

#define FAIL(c, code, ...)                                   \
    do {                                                     \
        char _b[256];                                        \
        snprintf(_b, sizeof _b, __VA_ARGS__);                \
        (c)->err = _b;                                       \
        return (code);                                       \
    } while (0)

#define CK(c, call)                                                                                   \
    do {                                                                                              \
        cudaError_t _e = (call);                                                                      \
        if (_e != cudaSuccess) {                                                                      \
            (c)->sticky = (_e == cudaErrorMemoryAllocation) ? MOP_ERR_OOM : MOP_ERR_CUDA;             \
            char _b[256];                                                                             \
            snprintf(_b, sizeof _b, "%s at %s:%d: %s", #call, __FILE__, __LINE__, cudaGetErrorString(_e)); \
            (c)->err = _b;                                                                            \
            return (mop_status)(c)->sticky;                                                           \
        }                                                                                             \
    } while (0)

#define LAUNCH(c, kernel, grid, block, smem, ...)                 \
    do {                                                          \
        kernel<<<(grid), (block), (smem), (c)->st>>>(__VA_ARGS__); \
        (c)->n_launches += 1;                                     \
    } while (0)

template <typename T>
static cudaError_t dalloc(T **p, size_t n) {
    if (*p) {
        cudaFree(*p);
        *p = nullptr;
    }
    if (n == 0) n = 1;
    return cudaMalloc((void **)p, n * sizeof(T));
}

static inline unsigned cdiv(size_t a, size_t b) { return (unsigned)((a + b - 1) / b); }

typedef void (*nb_kernel_t)(const NbArgs);
// the launched instances of the pair kernel: six resident CTAs per SM (80 registers) for the force passes, five (96)
// for the H.eta pass (measured: profiles/r02_experiments.md)
#ifndef NBP_CTAS_F
#define NBP_CTAS_F 6
#endif
#ifndef NBP_CTAS_H
#define NBP_CTAS_H 5
#endif
#define NBP_CTAS_E 4   // energy variant (bead 1 only): FP64 sums and six more packed accumulators per step
static nb_kernel_t nb_pick(int mode, bool count = false) {
    if (count) return k_nonbonded_p<NB_FORCE, true, NBP_CTAS_F>;
    return mode == NB_FORCE ? k_nonbonded_p<NB_FORCE, false, NBP_CTAS_F>
         : mode == NB_ENERGY ? k_nonbonded_p<NB_ENERGY, false, NBP_CTAS_E> : k_nonbonded_p<NB_HVP, false, NBP_CTAS_H>;
}
static size_t nb_smem(const mop_ctx *c) { return nbp_smem_bytes(c->nt); }

extern "C" const char *mop_last_error(const mop_ctx *c) { return c ? c->err.c_str() : g_create_error; }

static void free_all(mop_ctx *c) {
    void *ptrs[] = {c->d_mass,    c->d_inv_mass, c->d_charge,    c->d_ai,        c->d_Ki,       c->d_tabs,
                    c->d_tab,     c->d_bond_par, c->d_angle_par, c->d_type_row,  c->d_bond_ij,  c->d_angle_ijk,
                    c->d_excl_start, c->d_excl_list, c->d_cell,  c->d_cell_count, c->d_cell_rel, c->d_cell_fill,
                    c->d_col_count, c->d_col_start, c->d_tmp,    c->d_perm,      c->d_slot_of,  c->d_typ,
                    c->d_xq,      c->d_et,       c->d_F4,        c->d_H4,        c->d_blo,      c->d_bhi,
                    c->d_units,   c->d_entries,  c->d_masks,     c->d_ctr,
                    c->d_slots,   c->d_work,     c->d_energy,    c->d_G,         c->d_dbg,       c->d_Rh,
                    c->d_Gh,      c->d_fdR,      c->d_fdEta,     c->d_fdF,       c->d_fdFp,     c->d_fdFm,
                    c->d_Rref,    c->d_moved,
                    c->d_bias_ga, c->d_bias_gb,  c->d_bias_nh,   c->d_bias_hills, c->d_bias_com, c->d_bias_state};
    for (void *p : ptrs)
        if (p) cudaFree(p);
    if (c->h_energy) cudaFreeHost(c->h_energy);
    if (c->h_ctr) cudaFreeHost(c->h_ctr);
    if (c->h_slots) cudaFreeHost(c->h_slots);
    if (c->h_moved) cudaFreeHost(c->h_moved);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->st2) cudaStreamDestroy(c->st2);
    for (cudaEvent_t e : c->ev_copy)
        if (e) cudaEventDestroy(e);
    if (c->st_copy) cudaStreamDestroy(c->st_copy);
    for (cudaGraphExec_t x : c->gx)
        if (x) cudaGraphExecDestroy(x);
    if (c->st_cap) cudaStreamDestroy(c->st_cap);
    if (c->ev_made)
        for (auto &set : c->ev)
            for (cudaEvent_t e : set) cudaEventDestroy(e);
}

extern "C" void mop_destroy(mop_ctx *c) {
    if (!c) return;
    cudaSetDevice(c->p.device);
    cudaStreamSynchronize(c->st);
    if (c->st2) cudaStreamSynchronize(c->st2);
    if (c->st_copy) cudaStreamSynchronize(c->st_copy);
    free_all(c);
    delete c;
}

static mop_status create_impl(mop_ctx **out, const mop_params *p, bool blk, int n0, int Ntot) {
    if (!out || !p) {
        snprintf(g_create_error, sizeof g_create_error, "mop_create: NULL argument");
        return MOP_ERR_INVALID_ARG;
    }
    *out = nullptr;
    auto bad = [&](mop_status s, const char *msg) {
        snprintf(g_create_error, sizeof g_create_error, "mop_create: %s", msg);
        return s;
    };
    if (p->n_atoms < 1 || p->n_beads < 1) return bad(MOP_ERR_INVALID_ARG, "n_atoms and n_beads must be >= 1");
    if (!(p->r_cut > 0.f) || !(p->r_buf >= 0.f)) return bad(MOP_ERR_INVALID_ARG, "need r_cut > 0 and r_buf >= 0");
    if (!(p->dt_path > 0.0) || !(p->nu > 0.0)) return bad(MOP_ERR_INVALID_ARG, "need dt_path > 0 and nu > 0");
    for (int d = 0; d < 3; d++)
        if (!(p->box[d] > 0.f) || !std::isfinite(p->box[d])) return bad(MOP_ERR_INVALID_ARG, "box must be positive");
    const float rl = p->r_cut + p->r_buf;
    for (int d = 0; d < 3; d++)
        if (p->box[d] < 2.0f * rl) return bad(MOP_ERR_BOX_TOO_SMALL, "min(box) < 2 (r_cut + r_buf)");
    if ((double)p->n_atoms * (double)p->n_beads > 1.0e9) return bad(MOP_ERR_INVALID_ARG, "n_atoms * n_beads too large");
    if (blk && (n0 < 0 || Ntot < 1 || n0 + p->n_beads > Ntot))
        return bad(MOP_ERR_INVALID_ARG, "bead block [first_bead, first_bead + n_beads) must lie inside [0, n_beads_path)");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || p->device < 0 || p->device >= ndev) {
        cudaGetLastError();
        return bad(MOP_ERR_CUDA, "no usable CUDA device (the library has no CPU fallback)");
    }
    if (cudaSetDevice(p->device) != cudaSuccess) return bad(MOP_ERR_CUDA, "cudaSetDevice failed");

    mop_ctx *c = new mop_ctx();
    c->p = *p;
    c->Q = p->n_atoms;
    c->N = p->n_beads;
    if (!blk) {
        c->nf = c->nfe = p->n_beads > 1 ? p->n_beads - 1 : 1;
        c->nh = p->n_beads - 1;
    } else {
        // force, eta and H.eta on every bead of the block except the path's last bead (reading G6)
        c->blk = true, c->blk_n0 = n0, c->blk_Ntot = Ntot;
        c->has_u1 = n0 == 0;
        c->nh = Ntot == 1 ? 0 : std::min(p->n_beads, Ntot - 1 - n0);
        c->nfe = Ntot == 1 ? 1 : c->nh;
        c->nf = std::max(c->nfe, 1);
    }
    c->st = (cudaStream_t)p->stream;
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, p->device);
    c->rl = rl;
    c->rl2 = rl * rl * 1.0001f;
    c->rc2 = p->r_cut * p->r_cut; // FP32 product (G8)
    {
        double rc = (double)p->r_cut;
        double krf = p->eps_rf > 0.f ? ((double)p->eps_rf - 1.0) / ((2.0 * (double)p->eps_rf + 1.0) * rc * rc * rc)
                                      : 1.0 / (2.0 * rc * rc * rc);
        c->krf = (float)krf;
        c->krf_d = krf;
        c->crf_d = 1.0 / rc + krf * rc * rc;
    }
    // search grid (S0): columns of side ~ (8/rho)^(1/3) in x,y; thin bins of side/8 along z
    MopGrid &g = c->g;
    {
        double vol = (double)p->box[0] * (double)p->box[1] * (double)p->box[2];
        double side = cbrt((double)MOP_CL * vol / (double)c->Q);
        for (int d = 0; d < 2; d++) {
            int n = (int)floor((double)p->box[d] / side);
            g.dims[d] = n < 1 ? 1 : (n > 1024 ? 1024 : n);
        }
        c->bin_z = (float)(side / 8.0);
        int nz = (int)floor((double)p->box[2] / (double)c->bin_z);
        g.dims[2] = nz < 1 ? 1 : (nz > 4096 ? 4096 : nz);
        for (int d = 0; d < 3; d++) {
            g.box[d] = p->box[d];
            g.inv_box[d] = 1.0f / p->box[d];
            g.sc[d] = (float)g.dims[d] * g.inv_box[d];
        }
        g.ncol = g.dims[0] * g.dims[1];
        g.ncell = g.ncol * g.dims[2];
        g.colw[0] = p->box[0] / (float)g.dims[0];
        g.colw[1] = p->box[1] / (float)g.dims[1];
        g.Q = c->Q;
        g.nf = c->nf;
        size_t S = (size_t)c->Q + (size_t)(MOP_CL - 1) * (size_t)g.ncol;
        g.S = (int)((S + 31) / 32 * 32);
    }
    // what the kernels' index arithmetic assumes: a list entry keeps its j-octet in 24 bits (cj | sid << 24), and the
    // pair kernels address the sorted arrays with 32-bit element offsets bead * S + slot
    if (g.S / MOP_CL >= (1 << 24) || (double)c->nf * (double)g.S >= 2147483648.0) {
        const bool octets = g.S / MOP_CL >= (1 << 24);
        delete c;
        return bad(MOP_ERR_INVALID_ARG, octets ? "more than 2^24 atom octets per bead (n_atoms + padding >= 1.34e8)"
                                               : "force beads * padded slots per bead >= 2^31 (32-bit element offsets)");
    }
    const size_t nf = c->nf, Q = c->Q, S = g.S;
    cudaError_t e = cudaSuccess;
    auto A = [&](cudaError_t r) {
        if (e == cudaSuccess) e = r;
    };
    A(dalloc(&c->d_cell, nf * Q));
    A(dalloc(&c->d_cell_count, nf * g.ncell));
    A(dalloc(&c->d_cell_rel, nf * g.ncell));
    A(dalloc(&c->d_cell_fill, nf * g.ncell));
    A(dalloc(&c->d_col_count, nf * g.ncol));
    A(dalloc(&c->d_col_start, nf * (g.ncol + 1)));
    A(dalloc(&c->d_tmp, nf * S));
    A(dalloc(&c->d_perm, nf * S));
    A(dalloc(&c->d_slot_of, nf * Q));
    A(dalloc(&c->d_typ, nf * S));
    A(dalloc(&c->d_xq, nf * S));
    A(dalloc(&c->d_et, nf * S));
    A(dalloc(&c->d_F4, nf * S));
    A(dalloc(&c->d_H4, nf * S));
    A(dalloc(&c->d_blo, nf * S / MOP_CL));
    A(dalloc(&c->d_bhi, nf * S / MOP_CL));
    A(dalloc(&c->d_ctr, 1));
    A(dalloc(&c->d_slots, 2));
    A(dalloc(&c->d_work, 8));
    A(dalloc(&c->d_energy, 16));   // [0..5] U_lj, U_coul, U_bond, U_angle, E_spring, E_kin; [8..15] scratch
    A(cudaMallocHost((void **)&c->h_energy, 8 * sizeof(double)));
    A(cudaMallocHost((void **)&c->h_ctr, sizeof(MopCounters)));
    A(cudaMallocHost((void **)&c->h_slots, 2 * sizeof(unsigned long long)));
    A(cudaStreamCreateWithFlags(&c->st2, cudaStreamNonBlocking));
    A(cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
    A(cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
    A(cudaStreamCreateWithFlags(&c->st_copy, cudaStreamNonBlocking));
    A(cudaStreamCreateWithFlags(&c->st_cap, cudaStreamNonBlocking));
    for (cudaEvent_t &ev : c->ev_copy) A(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    if (e != cudaSuccess) {
        snprintf(g_create_error, sizeof g_create_error, "mop_create: device allocation failed: %s",
                 cudaGetErrorString(e));
        free_all(c);
        delete c;
        cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? MOP_ERR_OOM : MOP_ERR_CUDA;
    }
    cudaMemsetAsync(c->d_energy, 0, 16 * sizeof(double), c->st);
    cudaMemsetAsync(c->d_ctr, 0, sizeof(MopCounters), c->st);
    cudaMemsetAsync(c->d_slots, 0, 2 * sizeof(unsigned long long), c->st);
    memset(c->h_energy, 0, 8 * sizeof(double));
    memset(c->h_ctr, 0, sizeof(MopCounters));
    c->h_slots[0] = c->h_slots[1] = 0;
    *out = c;
    return MOP_OK;
}

extern "C" mop_status mop_create(mop_ctx **out, const mop_params *p) { return create_impl(out, p, false, 0, 0); }

extern "C" mop_status mop_create_block(mop_ctx **out, const mop_params *p, int first_bead, int n_beads_path) {
    return create_impl(out, p, true, first_bead, n_beads_path);
}

// (re)allocates the pair-list buffers for at least the given numbers of units, entries and exclusion-mask rows
static mop_status alloc_lists(mop_ctx *c, double units, double entries, double masks) {
    auto cap = [](double v) { return (unsigned)std::min(std::max(v, 64.0), 3.5e9); };
    c->cap_units = cap(units), c->cap_entries = cap(entries), c->cap_masks = cap(masks);
    CK(c, dalloc(&c->d_units, (size_t)c->cap_units));
    CK(c, dalloc(&c->d_entries, (size_t)c->cap_entries));
    CK(c, dalloc(&c->d_masks, (size_t)c->cap_masks));
    c->list_valid = false;
    c->gx_valid = false;   // the graphs hold the old buffer addresses
    return MOP_OK;
}

extern "C" mop_status mop_set_topology(mop_ctx *c, const mop_topology *t) {
    if (!c) return MOP_ERR_INVALID_ARG;
    if (c->sticky) return (mop_status)c->sticky;
    if (!t || !t->mass || !t->charge || !t->type || !t->c6 || !t->c12) FAIL(c, MOP_ERR_INVALID_ARG, "NULL topology array");
    const int Q = c->Q;
    if (t->n_types < 1 || t->n_types > MOP_MAX_TYPES) FAIL(c, MOP_ERR_INVALID_ARG, "n_types must be in [1,%d]", MOP_MAX_TYPES);
    if (t->n_bonds < 0 || t->n_angles < 0) FAIL(c, MOP_ERR_INVALID_ARG, "negative term count");
    if ((t->n_bonds > 0 && (!t->bond_ij || !t->bond_b0_kb)) || (t->n_angles > 0 && (!t->angle_ijk || !t->angle_t0_kt)))
        FAIL(c, MOP_ERR_INVALID_ARG, "NULL bonded array");
    const int nt = t->n_types;
    for (int i = 0; i < Q; i++) {
        if (!(t->mass[i] > 0.f) || !std::isfinite(t->mass[i])) FAIL(c, MOP_ERR_INVALID_ARG, "mass[%d] must be > 0", i);
        if (!std::isfinite(t->charge[i])) FAIL(c, MOP_ERR_INVALID_ARG, "charge[%d] not finite", i);
        if (t->type[i] < 0 || t->type[i] >= nt) FAIL(c, MOP_ERR_INVALID_ARG, "type[%d] out of range", i);
    }
    for (int a = 0; a < nt; a++)
        for (int b = 0; b < nt; b++)
            if (t->c6[a * nt + b] != t->c6[b * nt + a] || t->c12[a * nt + b] != t->c12[b * nt + a])
                FAIL(c, MOP_ERR_INVALID_ARG, "c6/c12 table not symmetric at (%d,%d)", a, b);
    for (int b = 0; b < t->n_bonds; b++) {
        int i = t->bond_ij[2 * b], j = t->bond_ij[2 * b + 1];
        if (i < 0 || i >= Q || j < 0 || j >= Q || i == j) FAIL(c, MOP_ERR_INVALID_ARG, "bond %d: bad atom index", b);
    }
    for (int a = 0; a < t->n_angles; a++) {
        int i = t->angle_ijk[3 * a], j = t->angle_ijk[3 * a + 1], k = t->angle_ijk[3 * a + 2];
        if (i < 0 || i >= Q || j < 0 || j >= Q || k < 0 || k >= Q || i == j || j == k || i == k)
            FAIL(c, MOP_ERR_INVALID_ARG, "angle %d: bad atom index", a);
    }
    int n_excl = 0, max_excl = 0;
    if (t->excl_start) {
        if (t->excl_start[0] != 0) FAIL(c, MOP_ERR_INVALID_ARG, "excl_start[0] != 0");
        for (int i = 0; i < Q; i++)
            if (t->excl_start[i + 1] < t->excl_start[i]) FAIL(c, MOP_ERR_INVALID_ARG, "excl_start not monotone at %d", i);
        n_excl = t->excl_start[Q];
        if (n_excl > 0 && !t->excl_list) FAIL(c, MOP_ERR_INVALID_ARG, "excl_list is NULL");
        for (int i = 0; i < Q; i++) {
            int e0 = t->excl_start[i], e1 = t->excl_start[i + 1];
            if (e1 - e0 > max_excl) max_excl = e1 - e0;
            for (int e = e0; e < e1; e++) {
                int j = t->excl_list[e];
                if (j < 0 || j >= Q || j == i) FAIL(c, MOP_ERR_INVALID_ARG, "exclusion of atom %d: bad partner", i);
                if (e > e0 && t->excl_list[e - 1] >= j) FAIL(c, MOP_ERR_INVALID_ARG, "exclusions of atom %d not sorted", i);
                // symmetric: i must be in j's list (binary search)
                int lo = t->excl_start[j], hi = t->excl_start[j + 1] - 1;
                bool found = false;
                while (lo <= hi) {
                    int mid = (lo + hi) / 2;
                    int v = t->excl_list[mid];
                    if (v == i) {
                        found = true;
                        break;
                    }
                    if (v < i) lo = mid + 1;
                    else hi = mid - 1;
                }
                if (!found) FAIL(c, MOP_ERR_INVALID_ARG, "exclusion (%d,%d) not symmetric", i, j);
            }
        }
    }
    CK(c, cudaSetDevice(c->p.device));
    c->nt = nt;
    c->n_bonds = t->n_bonds;
    c->n_angles = t->n_angles;
    c->max_excl = max_excl;
    // derived host arrays
    std::vector<float> inv_m(Q), ai(Q), Ki(Q), tabs(nt * nt);
    std::vector<int> trow(Q);
    std::vector<float2> tab(nt * nt);
    for (int i = 0; i < Q; i++) {
        double m = (double)t->mass[i];
        inv_m[i] = (float)(1.0 / m);
        ai[i] = (float)(c->p.dt_path / (m * c->p.nu));       // L^n_i = a_i F^n_i  (G1)
        Ki[i] = (float)(m * c->p.nu / (2.0 * c->p.dt_path));
        trow[i] = t->type[i];
    }
    const double rc = (double)c->p.r_cut, irc6 = 1.0 / (rc * rc * rc * rc * rc * rc);
    for (int k = 0; k < nt * nt; k++) {
        tab[k] = make_float2(6.0f * t->c6[k], 12.0f * t->c12[k]);
        tabs[k] = c->p.lj_shift ? (float)((double)t->c12[k] * irc6 * irc6 - (double)t->c6[k] * irc6) : 0.0f;
    }
    auto up = [&](auto **dst, const void *src, size_t n, size_t esz) -> cudaError_t {
        cudaError_t r = dalloc(dst, n);
        if (r != cudaSuccess) return r;
        if (n == 0) return cudaSuccess;
        return cudaMemcpyAsync(*dst, src, n * esz, cudaMemcpyHostToDevice, c->st);
    };
    CK(c, up(&c->d_mass, t->mass, Q, 4));
    CK(c, up(&c->d_inv_mass, inv_m.data(), Q, 4));
    CK(c, up(&c->d_charge, t->charge, Q, 4));
    CK(c, up(&c->d_ai, ai.data(), Q, 4));
    CK(c, up(&c->d_Ki, Ki.data(), Q, 4));
    CK(c, up(&c->d_type_row, trow.data(), Q, 4));
    CK(c, up(&c->d_tab, tab.data(), (size_t)nt * nt, 8));
    CK(c, up(&c->d_tabs, tabs.data(), (size_t)nt * nt, 4));
    CK(c, up(&c->d_bond_ij, t->bond_ij, (size_t)2 * t->n_bonds, 4));
    CK(c, up(&c->d_bond_par, t->bond_b0_kb, (size_t)t->n_bonds, 8));
    CK(c, up(&c->d_angle_ijk, t->angle_ijk, (size_t)3 * t->n_angles, 4));
    CK(c, up(&c->d_angle_par, t->angle_t0_kt, (size_t)t->n_angles, 8));
    if (t->excl_start && n_excl > 0) {
        CK(c, up(&c->d_excl_start, t->excl_start, (size_t)Q + 1, 4));
        CK(c, up(&c->d_excl_list, t->excl_list, (size_t)n_excl, 4));
    } else {
        if (c->d_excl_start) cudaFree(c->d_excl_start), c->d_excl_start = nullptr;
        if (c->d_excl_list) cudaFree(c->d_excl_list), c->d_excl_list = nullptr;
    }
    // pair-list capacities (S1): one unit per i-octet (exact bound); entries from the volume of the
    // half shell of octets within reach, masks from the exclusion count, both with head room.  The first evaluation
    // checks them against a real build and regrows them if the estimate was short (inhomogeneous systems).
    {
        const MopGrid &g = c->g;
        const double kPi = 3.14159265358979;
        double vol = (double)g.box[0] * g.box[1] * g.box[2];
        double side = cbrt((double)MOP_CL * vol / (double)Q);
        double reach = c->rl + 1.2 * side;
        double per_ci = 0.5 * ((double)Q / MOP_CL / vol) * (4.0 / 3.0) * kPi * reach * reach * reach * 1.25 + 16.0;
        double nci = (double)c->nf * g.S / MOP_CL;
        int rows = 1 + (max_excl > 0 ? std::min(MOP_EXROWS - 1, 2 * max_excl + 2) : 0);
        mop_status st = alloc_lists(c, nci, nci * per_ci, nci * rows);
        if (st) return st;
        c->caps_checked = false;
    }
    // launch geometry of the persistent pair kernels
    {
        const void *fns[4] = {(const void *)nb_pick(NB_FORCE), (const void *)nb_pick(NB_ENERGY), (const void *)nb_pick(NB_HVP),
                              (const void *)nb_pick(NB_FORCE, true)};
        int *nbs[4] = {&c->nb_blocks_f, &c->nb_blocks_fe, &c->nb_blocks_h, &c->nb_blocks_c};
        for (int k = 0; k < 4; k++) {
            const size_t smem = nb_smem(c);
            CK(c, cudaFuncSetAttribute(fns[k], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            int b = 0;
            CK(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, fns[k], 128, smem));
            *nbs[k] = std::max(1, b) * c->sm_count;
        }
    }
    CK(c, cudaStreamSynchronize(c->st));
    c->has_topology = true;
    c->list_valid = false;
    c->gx_valid = false;
    c->g_current = false;
    return MOP_OK;
}

// ---- stage timing: event k closes stage k-1 of the evaluation in flight (no-ops unless mop_set_timing(1)) ----
static void t_collect(mop_ctx *c, int n_sets) {
    // oldest first; blocks the host until those evaluations have finished
    for (; n_sets > 0 && c->ev_pending > 0; n_sets--, c->ev_pending--) {
        const int set = ((c->ev_head - c->ev_pending) % MOP_TSETS + MOP_TSETS) % MOP_TSETS;
        if (cudaEventSynchronize(c->ev[set][MOP_NSTAGE]) != cudaSuccess) continue;
        for (int k = 0; k < MOP_NSTAGE; k++) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, c->ev[set][k], c->ev[set][k + 1]) == cudaSuccess) c->t_sum[k] += (double)ms;
        }
        c->t_cnt += 1;
    }
}
static void t_mark(mop_ctx *c, int k) {
    if (!c->timing) return;
    if (k == 0 && c->ev_pending == MOP_TSETS) t_collect(c, 1);
    cudaEventRecord(c->ev[c->ev_head % MOP_TSETS][k], c->st);
    if (k == MOP_NSTAGE) {
        c->ev_head = (c->ev_head + 1) % MOP_TSETS;
        c->ev_pending += 1;
    }
}

// ---- S0 + S1 for the first nb beads of R ----
// per-build counters start from zero; the overflow and non-finite words are sticky (only a regrow clears overflow)
__global__ void k_ctr_reset(MopCounters *ctr, unsigned long long *slots) {
    ctr->n_units = ctr->n_entries = ctr->n_masks = ctr->n_units_bead0 = ctr->n_units_mid = 0u;
    slots[0] = slots[1] = 0ull;
}
__global__ void k_ctr_clear_overflow(MopCounters *ctr) { ctr->overflow = 0u; }

// S0 for the beads [b0, b1): cell ids, counting sort, sorted coordinates, octet bounding boxes
static mop_status s0_range(mop_ctx *c, const float *R, int b0, int b1) {
    MopGrid g = c->g;
    g.n0 = b0;
    const int nb = b1 - b0;
    const size_t Q = c->Q;
    CK(c, cudaMemsetAsync(c->d_cell_count + (size_t)b0 * g.ncell, 0, (size_t)nb * g.ncell * sizeof(int), c->st));
    CK(c, cudaMemsetAsync(c->d_cell_fill + (size_t)b0 * g.ncell, 0, (size_t)nb * g.ncell * sizeof(int), c->st));
    dim3 ga(cdiv(Q, 256), nb), gs(cdiv(g.S, 256), nb);
    LAUNCH(c, k_bin, ga, 256, 0, R, g, c->d_cell, c->d_cell_count, &c->d_ctr->nonfinite);
    LAUNCH(c, k_colscan, dim3(cdiv(g.ncol, 4), nb), 128, 0, g, c->d_cell_count, c->d_cell_rel, c->d_col_count);
    LAUNCH(c, k_colstart, nb, 1024, 0, g, c->d_col_count, c->d_col_start);
    LAUNCH(c, k_fill_pad, gs, 256, 0, g, c->d_perm, c->d_xq, c->d_typ);
    LAUNCH(c, k_place, ga, 256, 0, g, c->d_cell, c->d_cell_rel, c->d_col_start, c->d_cell_fill, c->d_tmp);
    LAUNCH(c, k_rank, ga, 256, 0, R, g, c->d_cell, c->d_cell_rel, c->d_col_start, c->d_cell_count, c->d_tmp,
           c->d_charge, c->d_type_row, c->d_perm, c->d_slot_of, c->d_xq, c->d_typ);
    LAUNCH(c, k_bbox, dim3(cdiv(g.S, 128), nb), 128, 0, g, c->d_perm, c->d_xq, c->d_blo, c->d_bhi);
    return MOP_OK;
}

// S1 for the beads [b0, b1): their work units are appended to the list (bead 1 must come first and alone: the units
// before the mark are the energy variant's)
static void s1_range(mop_ctx *c, int b0, int b1) {
    const MopGrid &g = c->g;
    PlArgs a;
    a.g = g;
    a.rl = c->rl;
    a.rl2 = c->rl2;
    a.perm = c->d_perm, a.slot_of = c->d_slot_of, a.xq = c->d_xq;
    a.blo = c->d_blo, a.bhi = c->d_bhi;
    a.col_start = c->d_col_start, a.cell_rel = c->d_cell_rel, a.col_count = c->d_col_count;
    a.excl_start = c->d_excl_start, a.excl_list = c->d_excl_list;
    a.units = c->d_units, a.entries = c->d_entries, a.masks = c->d_masks, a.ctr = c->d_ctr;
    a.slots_active = c->d_slots;
    a.cap_units = c->cap_units, a.cap_entries = c->cap_entries, a.cap_masks = c->cap_masks;
    const unsigned nci_blocks = cdiv(g.S / MOP_CL, MOP_PL_WARPS);
    a.bead0 = b0;
    LAUNCH(c, k_pairlist, dim3(nci_blocks, b1 - b0), 32 * MOP_PL_WARPS, 0, a);
    if (b0 == 0) LAUNCH(c, k_mark_bead0, 1, 1, 0, c->d_ctr, c->cap_units);
}

static mop_status build_list_once(mop_ctx *c, const float *R, int nb, bool timed) {
    LAUNCH(c, k_ctr_reset, 1, 1, 0, c->d_ctr, c->d_slots);
    mop_status s = s0_range(c, R, 0, nb);
    if (s) return s;
    if (timed) t_mark(c, 1);
    s1_range(c, 0, 1);   // bead 1 first: its units come first (energy variant)
    if (nb > 1) s1_range(c, 1, nb);
    c->n_rebuilds += 1;
    if (timed) t_mark(c, 2);
    CK(c, cudaGetLastError());
    return MOP_OK;
}

// the builder keeps counting past the capacities, so an overflowed build tells what a sufficient allocation is
static mop_status regrow_lists(mop_ctx *c) {
    // ... but the counts are those of the LAST build only, while the overflow word is sticky across the builds of one call
    // (the displaced builds of mop_eval_veff_grad_fd, the steps of mop_step): a buffer whose bit is set grows by a factor
    // even when the last build happened to fit, so that repeating the call cannot meet the same overflow for ever
    const MopCounters &h = *c->h_ctr;
    const double gu = (h.overflow & 2u) ? 1.3 : 1.0, ge = (h.overflow & 1u) ? 1.3 : 1.0, gm = (h.overflow & 4u) ? 1.3 : 1.0;
    const double nu = std::max(gu * (double)c->cap_units, 1.05 * h.n_units), ne = std::max(ge * (double)c->cap_entries, 1.3 * h.n_entries),
                 nm = std::max(gm * (double)c->cap_masks, 1.3 * h.n_masks);
    if (h.overflow & 24u) FAIL(c, MOP_ERR_OOM, "pair-list builder: per-octet staging (8) or exclusion rows (16) exhausted, flags 0x%x", h.overflow);
    CK(c, cudaStreamSynchronize(c->st));
    mop_status s = alloc_lists(c, nu, ne, nm);
    if (s) return s;
    LAUNCH(c, k_ctr_clear_overflow, 1, 1, 0, c->d_ctr);
    return MOP_OK;
}

static mop_status build_list(mop_ctx *c, const float *R, int nb, bool timed = false) {
    mop_status s = build_list_once(c, R, nb, timed);
    if (s || c->caps_checked) return s;
    // first build with these capacities: check them on the host (one synchronisation per topology), regrow and rebuild
    for (int attempt = 0; attempt < 3; attempt++) {
        CK(c, cudaMemcpyAsync(c->h_ctr, c->d_ctr, sizeof(MopCounters), cudaMemcpyDeviceToHost, c->st));
        CK(c, cudaStreamSynchronize(c->st));
        if (!c->h_ctr->overflow) break;
        if ((s = regrow_lists(c))) return s;
        if ((s = build_list_once(c, R, nb, false))) return s;
    }
    c->caps_checked = true;
    return MOP_OK;
}

static NbArgs nb_args(mop_ctx *c, float4 *out, int work_slot, int range) {
    NbArgs a;
    a.S = c->g.S, a.nt = c->nt;
    a.rc2 = c->rc2;
    a.k2rf = 2.0f * c->krf, a.krf_d = c->krf_d, a.crf_d = c->crf_d;
    a.xq = c->d_xq, a.typ = c->d_typ, a.et = c->d_et, a.out = out;
    a.units = c->d_units, a.entries = c->d_entries, a.masks = c->d_masks, a.ctr = c->d_ctr;
    a.cap_units = c->cap_units;
    a.cap_entries = c->cap_entries, a.cap_masks = c->cap_masks, a.n_slots = (unsigned)c->nf * (unsigned)c->g.S;
    a.n_inrange = &c->d_ctr->n_inrange;
    a.pair_hash = &c->d_ctr->pair_hash, a.perm = c->d_perm, a.Q = c->Q;
    a.work = c->d_work + work_slot;
    a.range = range;
    a.tab = c->d_tab, a.tabs = c->d_tabs;
    a.energies = c->d_energy;
    for (int d = 0; d < 3; d++) a.box[d] = c->g.box[d];
    return a;
}

static BondedArgs bonded_args(mop_ctx *c, const float *R, float4 *out) {
    BondedArgs b;
    b.Q = c->Q, b.S = c->g.S, b.n_bonds = c->n_bonds, b.n_angles = c->n_angles;
    b.R = R, b.slot_of = c->d_slot_of;
    b.bond_ij = c->d_bond_ij, b.bond_par = c->d_bond_par, b.angle_ijk = c->d_angle_ijk, b.angle_par = c->d_angle_par;
    b.et = c->d_et, b.out = out, b.energies = c->d_energy;
    for (int d = 0; d < 3; d++) b.box[d] = c->g.box[d], b.inv_box[d] = c->g.inv_box[d];
    return b;
}

// pass 1 on the first nb beads: nonbonded (energy variant on bead 1) + bonded.  with_energy = false (displaced
// configurations of the finite-difference mode): plain force kernel on every bead, energy sums go to scratch
static mop_status pass_force(mop_ctx *c, const float *R, int nb, bool timed = false, bool with_energy = true) {
    const size_t smem = nb_smem(c);
    CK(c, cudaMemsetAsync(c->d_F4, 0, (size_t)nb * c->g.S * sizeof(float4), c->st));
    // the bonded terms go first, on the side stream: both kernels accumulate into F4 with reductions, and the few hundred
    // small CTAs of k_bonded are resident before the persistent pair kernel fills the machine
    const int nterm = c->n_bonds + c->n_angles;
    if (nterm > 0) {
        CK(c, cudaEventRecord(c->ev_fork, c->st));
        CK(c, cudaStreamWaitEvent(c->st2, c->ev_fork, 0));
        BondedArgs b = bonded_args(c, R, c->d_F4);
        if (!with_energy) b.energies = c->d_energy + 8;
        k_bonded<false><<<dim3(cdiv(nterm, 128), nb), 128, 0, c->st2>>>(b);
        c->n_launches += 1;
        CK(c, cudaEventRecord(c->ev_join, c->st2));
    }
    if (with_energy) {
        LAUNCH(c, nb_pick(NB_ENERGY), c->nb_blocks_fe, 128, smem, nb_args(c, c->d_F4, 0, 0));
        if (nb > 1) LAUNCH(c, nb_pick(NB_FORCE), c->nb_blocks_f, 128, smem, nb_args(c, c->d_F4, 1, 1));
    } else {
        LAUNCH(c, nb_pick(NB_FORCE), c->nb_blocks_f, 128, smem, nb_args(c, c->d_F4, 0, 2));
    }
    if (timed) t_mark(c, 3);
    if (nterm > 0) CK(c, cudaStreamWaitEvent(c->st, c->ev_join, 0));
    if (timed) t_mark(c, 4);   // S3 = what is left of the bonded kernel after the pair kernels
    return MOP_OK;
}

// pass 2 on the first nb beads: nonbonded + bonded Hessian-vector product with the direction held in et
static mop_status pass_hvp(mop_ctx *c, const float *R, int nb, bool timed = false) {
    const size_t smem = nb_smem(c);
    CK(c, cudaMemsetAsync(c->d_H4, 0, (size_t)nb * c->g.S * sizeof(float4), c->st));
    const int nterm = c->n_bonds + c->n_angles;
    if (nterm > 0) {   // bonded H.eta beside the pair kernel (see pass_force)
        CK(c, cudaEventRecord(c->ev_fork, c->st));
        CK(c, cudaStreamWaitEvent(c->st2, c->ev_fork, 0));
        k_bonded<true><<<dim3(cdiv(nterm, 128), nb), 128, 0, c->st2>>>(bonded_args(c, R, c->d_H4));
        c->n_launches += 1;
        CK(c, cudaEventRecord(c->ev_join, c->st2));
    }
    LAUNCH(c, nb_pick(NB_HVP), c->nb_blocks_h, 128, smem, nb_args(c, c->d_H4, 2, 2));
    if (timed) t_mark(c, 6);
    if (nterm > 0) CK(c, cudaStreamWaitEvent(c->st, c->ev_join, 0));
    if (timed) t_mark(c, 7);
    return MOP_OK;
}

static mop_status read_back(mop_ctx *c) {
    CK(c, cudaMemcpyAsync(c->h_energy, c->d_energy, 8 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaMemcpyAsync(c->h_ctr, c->d_ctr, sizeof(MopCounters), cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaMemcpyAsync(c->h_slots, c->d_slots, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    CK(c, cudaGetLastError());
    if (c->h_ctr->nonfinite) {
        c->sticky = MOP_ERR_NONFINITE;
        FAIL(c, MOP_ERR_NONFINITE, "a coordinate is NaN/Inf or farther than ~1e6 box lengths from the box");
    }
    if (c->h_ctr->overflow) {
        // some build since the last check dropped pairs: the results of this call are invalid.  The buffers are
        // regrown from the builder's own counts, so the caller can simply repeat the evaluation.
        const unsigned fl = c->h_ctr->overflow;
        mop_status s = regrow_lists(c);
        if (s) {
            c->sticky = s;
            return s;
        }
        FAIL(c, MOP_ERR_OOM, "pair-list buffer overflow (flags 0x%x: 1 entries, 2 units, 4 masks); buffers regrown, repeat the call", fl);
    }
    const double *E = c->h_energy;
    c->last_veff = E[0] + E[1] + E[2] + E[3] + E[4];
    c->last_ekin = E[5];
    if (!std::isfinite(c->last_veff)) FAIL(c, MOP_ERR_NONFINITE, "V_eff is not finite (overlapping atoms?)");
    return MOP_OK;
}

// adds dV_bias/dR to grad on beads 1 and N (and deposits a hill at the current S_e2e first when asked to)
static void bias_launch(mop_ctx *c, const float *R, float *grad, bool deposit) {
    BiasArgs b;
    b.Q = c->Q, b.N = c->N, b.na = c->bias_na, b.nb = c->bias_nb;
    b.ga = c->d_bias_ga, b.gb = c->d_bias_gb, b.mass = c->d_mass;
    for (int d = 0; d < 3; d++) b.box[d] = c->g.box[d];
    b.sigma = c->bias_sigma, b.w = c->bias_w;
    b.hills = c->d_bias_hills, b.n_hills = c->d_bias_nh, b.com = c->d_bias_com, b.state = c->d_bias_state;
    LAUNCH(c, k_bias_com, dim3(2, 2), 256, 0, b, R);
    LAUNCH(c, k_bias_cv, 1, 32, 0, b, deposit ? 1 : 0);
    if (grad) LAUNCH(c, k_bias_apply, dim3(cdiv(b.na + b.nb, 256), 2), 256, 0, b, grad);
}

// S0 + S1 of an evaluation.  r_buf = 0: always a fresh build.  r_buf > 0: the list of the last build is kept while no
// atom has moved farther than r_buf / 2 from where it was then (k_refresh re-fills the sorted coordinates in the
// image of that build; the host reads one flag, which synchronises the stream).
static mop_status list_for(mop_ctx *c, const float *R, int nb) {
    if (c->p.r_buf > 0.f && c->list_valid) {
        if (!c->d_moved) {
            CK(c, dalloc(&c->d_moved, 1));
            CK(c, cudaMallocHost((void **)&c->h_moved, sizeof(int)));
        }
        CK(c, cudaMemsetAsync(c->d_moved, 0, sizeof(int), c->st));
        const float hb = 0.5f * c->p.r_buf;
        LAUNCH(c, k_refresh, dim3(cdiv(c->Q, 256), nb), 256, 0, R, c->d_Rref, c->g, hb * hb, c->d_slot_of, c->d_xq,
               c->d_moved);
        CK(c, cudaMemcpyAsync(c->h_moved, c->d_moved, sizeof(int), cudaMemcpyDeviceToHost, c->st));
        CK(c, cudaStreamSynchronize(c->st));
        if (*c->h_moved == 0) {
            c->n_reuses += 1;
            t_mark(c, 1), t_mark(c, 2);
            return MOP_OK;
        }
    }
    mop_status s = build_list(c, R, nb, true);
    if (s) return s;
    if (c->p.r_buf > 0.f) {
        const size_t bytes = (size_t)nb * c->Q * 3 * sizeof(float);
        if (!c->d_Rref) CK(c, dalloc(&c->d_Rref, (size_t)c->nf * c->Q * 3));
        CK(c, cudaMemcpyAsync(c->d_Rref, R, bytes, cudaMemcpyDeviceToDevice, c->st));
        c->list_valid = true;
    }
    return MOP_OK;
}

// One evaluation in three stages (bead-block mode runs them as separate calls with the halo exchange in between):
// 1: S0-S4 (lists, pass 1, eta; R_next = the bead after the block; keta_out = K eta of the block's last bead),
// 2: S5-S6 (pass 2), 3: S7 (assembly; keta_left = K eta of the bead before the block).
static mop_status eval_stage1(mop_ctx *c, const float *R, const float *R_next, float *keta_out, bool want_energy = true) {
    const int nb = c->nfe;
    CK(c, cudaMemsetAsync(c->d_energy, 0, 5 * sizeof(double), c->st));
    CK(c, cudaMemsetAsync(c->d_work, 0, 8 * sizeof(unsigned), c->st));
    t_mark(c, 0);
    mop_status s;
    if (nb > 0) {
        if ((s = list_for(c, R, nb))) return s;
        if ((s = pass_force(c, R, nb, true, c->has_u1 && want_energy))) return s;
    } else {
        t_mark(c, 1), t_mark(c, 2), t_mark(c, 3), t_mark(c, 4);
    }
    if (c->nh > 0) {
        LAUNCH(c, k_eta, dim3(cdiv(c->g.S, 256), c->nh), 256, 0, c->Q, c->g.S, c->N, R, R_next, c->d_perm, c->d_typ, c->d_F4,
               c->d_ai, c->d_Ki, c->d_et, c->d_energy + 4);
        if (keta_out)
            LAUNCH(c, k_keta_out, cdiv(c->Q, 256), 256, 0, c->Q, c->g.S, c->nh - 1, c->d_slot_of, c->d_et, c->d_Ki, keta_out);
    }
    t_mark(c, 5);
    CK(c, cudaGetLastError());
    return MOP_OK;
}

static mop_status eval_stage2(mop_ctx *c, const float *R) {
    if (c->nh > 0) {
        mop_status s = pass_hvp(c, R, c->nh, true);
        if (s) return s;
    } else {
        t_mark(c, 6), t_mark(c, 7);
    }
    return MOP_OK;
}

static mop_status eval_stage3(mop_ctx *c, const float *R, const float *keta_left, float *grad, bool deposit) {
    if (grad)
        LAUNCH(c, k_assemble, dim3(cdiv(c->Q, 256), c->N), 256, 0, c->Q, c->g.S, 0, c->N, c->nh, c->has_u1 ? 1 : 0, c->d_slot_of,
               c->d_F4, c->d_et, c->d_H4, c->d_Ki, keta_left, grad);
    t_mark(c, 8);
    if (c->bias_on && c->N > 1) bias_launch(c, R, grad, deposit);
    CK(c, cudaGetLastError());
    return MOP_OK;
}

// want_energy = false: U(R^1) is not formed (bead 1 takes the plain force kernel): the inner evaluations of mop_step*,
// which need the gradient only
static mop_status eval_async(mop_ctx *c, const float *R, float *grad, bool deposit = false, bool want_energy = true) {
    mop_status s;
    if ((s = eval_stage1(c, R, nullptr, nullptr, want_energy))) return s;
    if ((s = eval_stage2(c, R))) return s;
    return eval_stage3(c, R, nullptr, grad, deposit);
}

#define PRECHECK(c)                                                          \
    do {                                                                     \
        if (!(c)) return MOP_ERR_INVALID_ARG;                                \
        if ((c)->sticky) return (mop_status)(c)->sticky;                     \
        if (!(c)->has_topology) FAIL(c, MOP_ERR_NO_TOPOLOGY, "call mop_set_topology first"); \
        CK(c, cudaSetDevice((c)->p.device));                                 \
    } while (0)

static bool graphs_usable(const mop_ctx *c);
static mop_status graphs_build(mop_ctx *c);

// whole-path calls on a bead-block context are allowed only when the block IS the whole path
#define NOT_A_PARTIAL_BLOCK(c)                                                                                       \
    do {                                                                                                             \
        if ((c)->blk && ((c)->blk_n0 != 0 || (c)->N != (c)->blk_Ntot))                                               \
            FAIL(c, MOP_ERR_INVALID_ARG, "this context holds a bead block of a longer path: use the mop_block_* calls"); \
    } while (0)

extern "C" mop_status mop_eval_veff_grad(mop_ctx *c, const float *R_dev, double *veff_out, float *grad_dev) {
    PRECHECK(c);
    NOT_A_PARTIAL_BLOCK(c);
    if (!R_dev) FAIL(c, MOP_ERR_INVALID_ARG, "R_dev is NULL");
    mop_status s;
    if (graphs_usable(c)) {
        // two graph launches on the staging buffers between two device-to-device copies (a few microseconds each way)
        if ((s = graphs_build(c))) return s;
        const size_t bytes = (size_t)c->N * c->Q * 3 * sizeof(float);
        CK(c, cudaMemcpyAsync(c->d_Rh, R_dev, bytes, cudaMemcpyDeviceToDevice, c->st));
        CK(c, cudaGraphLaunch(c->gx[0], c->st));
        CK(c, cudaGraphLaunch(c->gx[1], c->st));
        c->n_launches += c->gx_launches[0] + c->gx_launches[1];
        c->n_rebuilds += 1;
        if (grad_dev) CK(c, cudaMemcpyAsync(grad_dev, c->d_Gh, bytes, cudaMemcpyDeviceToDevice, c->st));
    } else if ((s = eval_async(c, R_dev, grad_dev))) {
        return s;
    }
    if (veff_out) {
        if ((s = read_back(c))) return s;
        *veff_out = c->last_veff;
    }
    return MOP_OK;
}

// The paper's own form of the gradient: Hessian term by finite differences of two displaced force evaluations
// (eqs (5),(6),(7); PMD kernels 2 and 3).  Three force passes per bead instead of one
// force pass + one H.eta pass; every displaced configuration gets its own cell list and pair list.
extern "C" mop_status mop_eval_veff_grad_fd(mop_ctx *c, const float *R_dev, double eps, double *veff_out, float *grad_dev) {
    PRECHECK(c);
    NOT_A_PARTIAL_BLOCK(c);
    if (!R_dev || !grad_dev) FAIL(c, MOP_ERR_INVALID_ARG, "R_dev or grad_dev is NULL");
    if (!(eps > 0.0) || !std::isfinite(eps)) FAIL(c, MOP_ERR_INVALID_ARG, "need eps > 0");
    const int nb = c->nf;
    const size_t per = (size_t)c->Q * 3, tot = per * nb;
    if (!c->d_fdR) {
        CK(c, dalloc(&c->d_fdR, tot));
        CK(c, dalloc(&c->d_fdEta, tot));
        CK(c, dalloc(&c->d_fdF, tot));
        CK(c, dalloc(&c->d_fdFp, tot));
        CK(c, dalloc(&c->d_fdFm, tot));
    }
    const MopGrid &g = c->g;
    const dim3 gq(cdiv(c->Q, 256), nb);
    CK(c, cudaMemsetAsync(c->d_energy, 0, 5 * sizeof(double), c->st));
    CK(c, cudaMemsetAsync(c->d_work, 0, 8 * sizeof(unsigned), c->st));
    c->list_valid = false;   // the displaced configurations below overwrite the list
    mop_status s = build_list(c, R_dev, nb);
    if (s) return s;
    if ((s = pass_force(c, R_dev, nb))) return s;
    LAUNCH(c, k_gather3, gq, 256, 0, c->Q, g.S, c->d_slot_of, c->d_F4, c->d_fdF, 1.0f);
    if (c->N > 1) {
        LAUNCH(c, k_eta, dim3(cdiv(g.S, 256), nb), 256, 0, c->Q, g.S, c->N, R_dev, (const float *)nullptr, c->d_perm, c->d_typ,
               c->d_F4, c->d_ai, c->d_Ki, c->d_et, c->d_energy + 4);
        LAUNCH(c, k_gather3, gq, 256, 0, c->Q, g.S, c->d_slot_of, c->d_et, c->d_fdEta, 1.0f);
        for (int sign = 0; sign < 2; sign++) {
            LAUNCH(c, k_displace, cdiv(tot, 256), 256, 0, tot, sign ? -(float)eps : (float)eps, R_dev, c->d_fdEta, c->d_fdR);
            CK(c, cudaMemsetAsync(c->d_work, 0, 8 * sizeof(unsigned), c->st));
            if ((s = build_list(c, c->d_fdR, nb))) return s;
            if ((s = pass_force(c, c->d_fdR, nb, false, false))) return s;
            LAUNCH(c, k_gather3, gq, 256, 0, c->Q, g.S, c->d_slot_of, c->d_F4, sign ? c->d_fdFm : c->d_fdFp, 1.0f);
        }
    }
    LAUNCH(c, k_assemble_fd, dim3(cdiv(per, 256), c->N), 256, 0, c->Q, c->N, (float)(1.0 / (4.0 * eps)), c->d_fdF, c->d_fdEta,
           c->d_fdFp, c->d_fdFm, c->d_Ki, grad_dev);
    CK(c, cudaGetLastError());
    if (veff_out) {
        if ((s = read_back(c))) return s;
        *veff_out = c->last_veff;
    }
    return MOP_OK;
}

// ---- one evaluation as two sequences on the context's staging buffers: A = bead 1 alone (S0, S1, force + energy kernel),
// B = the other beads' S0, S1 and force kernel, the bonded terms, eta, pass 2 and the assembly.  The energy kernel thus
// runs before the other beads are sorted, which lets the host entry point copy beads 2..N in behind it; kernels and
// results are those of eval_async.  With mop_set_timing on, the eight timing slots of these sequences are: bead 1's S0 |
// its S1 | its force and energy kernel | (wait for the copy of beads 2..N) | their S0, S1, force kernel | eta | pass 2 |
// assembly.
static mop_status seq_A(mop_ctx *c, const float *R, bool want_energy = true) {
    const int nb = c->nfe;
    mop_status s;
    CK(c, cudaMemsetAsync(c->d_energy, 0, 5 * sizeof(double), c->st));
    CK(c, cudaMemsetAsync(c->d_work, 0, 8 * sizeof(unsigned), c->st));
    CK(c, cudaMemsetAsync(c->d_F4, 0, (size_t)nb * c->g.S * sizeof(float4), c->st));
    LAUNCH(c, k_ctr_reset, 1, 1, 0, c->d_ctr, c->d_slots);
    t_mark(c, 0);
    if ((s = s0_range(c, R, 0, 1))) return s;
    t_mark(c, 1);
    s1_range(c, 0, 1);
    t_mark(c, 2);
    if (want_energy) LAUNCH(c, nb_pick(NB_ENERGY), c->nb_blocks_fe, 128, nb_smem(c), nb_args(c, c->d_F4, 0, 0));
    else LAUNCH(c, nb_pick(NB_FORCE), c->nb_blocks_f, 128, nb_smem(c), nb_args(c, c->d_F4, 0, 0));   // gradient only (inner steps of mop_step)
    t_mark(c, 3);
    CK(c, cudaGetLastError());
    return MOP_OK;
}

// part 0: the whole of B.  Parts 1 and 2 (host entry point): pass 2 and the assembly in two bead groups [0, h) and [h, N),
// so that the gradient rows of the first group travel to the host while the second group's H.eta is computed.
static int split_bead(const mop_ctx *c) { return std::max(1, std::min(c->nh - 1, (7 * c->nh + 9) / 10)); }

static mop_status seq_B(mop_ctx *c, const float *R, float *G, int part = 0) {
    const int nb = c->nfe, N = c->N;
    const int h = part ? split_bead(c) : nb;
    mop_status s;
    if (part == 2) {   // second group: H.eta of beads [h, nh), gradient rows [h, N)
        LAUNCH(c, nb_pick(NB_HVP), c->nb_blocks_h, 128, nb_smem(c), nb_args(c, c->d_H4, 4, 4));
        if (G && N - 1 > h)   // rows [h, N-1): the last row went out with the first group
            LAUNCH(c, k_assemble, dim3(cdiv(c->Q, 256), N - 1 - h), 256, 0, c->Q, c->g.S, h, N, c->nh, 1, c->d_slot_of, c->d_F4,
                   c->d_et, c->d_H4, c->d_Ki, (const float *)nullptr, G);
        CK(c, cudaGetLastError());
        return MOP_OK;
    }
    t_mark(c, 4);
    const int nterm = c->n_bonds + c->n_angles;
    if (nb > 1 && (s = s0_range(c, R, 1, nb))) return s;
    if (nterm > 0) {   // bonded forces of all beads on the side stream (they scatter through slot_of: after S0 of every
                       // bead), beside the list build and the force kernel
        CK(c, cudaEventRecord(c->ev_fork, c->st));
        CK(c, cudaStreamWaitEvent(c->st2, c->ev_fork, 0));
        k_bonded<false><<<dim3(cdiv(nterm, 128), nb), 128, 0, c->st2>>>(bonded_args(c, R, c->d_F4));
        c->n_launches += 1;
        CK(c, cudaEventRecord(c->ev_join, c->st2));
    }
    if (nb > 1) {
        if (part && h > 1) s1_range(c, 1, h);
        if (part) LAUNCH(c, k_mark_mid, 1, 1, 0, c->d_ctr, c->cap_units);
        s1_range(c, part ? h : 1, nb);
        LAUNCH(c, nb_pick(NB_FORCE), c->nb_blocks_f, 128, nb_smem(c), nb_args(c, c->d_F4, 1, 1));
    }
    if (nterm > 0) CK(c, cudaStreamWaitEvent(c->st, c->ev_join, 0));
    t_mark(c, 5);
    if (c->nh > 0) {
        LAUNCH(c, k_eta, dim3(cdiv(c->g.S, 256), c->nh), 256, 0, c->Q, c->g.S, N, R, (const float *)nullptr, c->d_perm,
               c->d_typ, c->d_F4, c->d_ai, c->d_Ki, c->d_et, c->d_energy + 4);
        t_mark(c, 6);
        if (!part) {
            if ((s = pass_hvp(c, R, c->nh, false))) return s;
        } else {   // first group; the bonded H.eta of all beads beside it
            CK(c, cudaMemsetAsync(c->d_H4, 0, (size_t)c->nh * c->g.S * sizeof(float4), c->st));
            if (nterm > 0) {
                CK(c, cudaEventRecord(c->ev_fork, c->st));
                CK(c, cudaStreamWaitEvent(c->st2, c->ev_fork, 0));
                k_bonded<true><<<dim3(cdiv(nterm, 128), c->nh), 128, 0, c->st2>>>(bonded_args(c, R, c->d_H4));
                c->n_launches += 1;
                CK(c, cudaEventRecord(c->ev_join, c->st2));
            }
            LAUNCH(c, nb_pick(NB_HVP), c->nb_blocks_h, 128, nb_smem(c), nb_args(c, c->d_H4, 2, 3));
            if (nterm > 0) CK(c, cudaStreamWaitEvent(c->st, c->ev_join, 0));
        }
    } else {
        t_mark(c, 6);
    }
    t_mark(c, 7);
    if (G) {
        LAUNCH(c, k_assemble, dim3(cdiv(c->Q, 256), part ? h : N), 256, 0, c->Q, c->g.S, 0, N, c->nh, 1, c->d_slot_of, c->d_F4,
               c->d_et, c->d_H4, c->d_Ki, (const float *)nullptr, G);
        if (part)   // the last bead's row is K eta^{N-1} alone (eq. 7): ready now, it leaves with the first group
            LAUNCH(c, k_assemble, dim3(cdiv(c->Q, 256), 1), 256, 0, c->Q, c->g.S, N - 1, N, c->nh, 1, c->d_slot_of, c->d_F4,
                   c->d_et, c->d_H4, c->d_Ki, (const float *)nullptr, G);
    }
    t_mark(c, 8);
    CK(c, cudaGetLastError());
    return MOP_OK;
}

// the two sequences captured as CUDA graphs (one launch each instead of ~25 API calls: on small systems an evaluation is
// bound by launch latency, and so is the start of every host-synchronous call).  Not used while stage timing, a bias or a
// buffered list is on, nor before the first evaluation of a topology has checked the list capacities.
static bool graphs_usable(const mop_ctx *c) {
    return !c->timing && !c->bias_on && !(c->p.r_buf > 0.f) && c->caps_checked && !c->blk;
}

static mop_status graphs_build(mop_ctx *c) {
    if (c->gx_valid) return MOP_OK;
    const size_t tot = (size_t)c->N * c->Q * 3;
    if (!c->d_Rh) CK(c, dalloc(&c->d_Rh, tot));
    if (!c->d_Gh) CK(c, dalloc(&c->d_Gh, tot));   // always with the assembly (15 us): one set of graphs serves every form
    cudaStream_t user = c->st;
    const double l0 = c->n_launches, r0 = c->n_rebuilds;
    for (int k = 0; k < 5; k++) {
        if (c->gx[k]) cudaGraphExecDestroy(c->gx[k]), c->gx[k] = nullptr;
        if ((k == 2 || k == 3) && c->nh < 2) continue;   // nothing to split
        cudaGraph_t g = nullptr;
        const double lk = c->n_launches;
        cudaError_t e = cudaStreamBeginCapture(c->st_cap, cudaStreamCaptureModeThreadLocal);
        mop_status s = MOP_OK;
        if (e == cudaSuccess) {
            c->st = c->st_cap;
            s = k == 0 ? seq_A(c, c->d_Rh) : k == 4 ? seq_A(c, c->d_Rh, false) : seq_B(c, c->d_Rh, c->d_Gh, k - 1);
            c->st = user;
            e = cudaStreamEndCapture(c->st_cap, &g);
        }
        if (s == MOP_OK && e == cudaSuccess) e = cudaGraphInstantiate(&c->gx[k], g, 0);
        if (g) cudaGraphDestroy(g);
        if (s) return s;
        CK(c, e);
        c->gx_launches[k] = c->n_launches - lk;   // kernels in this graph, added to the count at every launch
    }
    c->n_launches = l0, c->n_rebuilds = r0;
    c->gx_valid = true;
    return MOP_OK;
}

// The end-to-end form.  The host->device copy is split: bead 1 first, beads 2..N behind it on the copy stream while the
// main stream already sorts bead 1, builds its list and runs its force + energy kernel (about 0.5 ms of work on the
// 150,000-atom system against 0.25 ms of copy).
extern "C" mop_status mop_eval_veff_grad_host(mop_ctx *c, const float *R_host, double *veff_out, float *grad_host) {
    PRECHECK(c);
    NOT_A_PARTIAL_BLOCK(c);
    if (!R_host || !veff_out) FAIL(c, MOP_ERR_INVALID_ARG, "R_host or veff_out is NULL");
    const size_t bead = (size_t)c->Q * 3, bytes = (size_t)c->N * bead * sizeof(float);
    if (!c->d_Rh) CK(c, dalloc(&c->d_Rh, (size_t)c->N * bead));
    if (grad_host && !c->d_Gh) CK(c, dalloc(&c->d_Gh, (size_t)c->N * bead));
    float *R = c->d_Rh, *G = grad_host ? c->d_Gh : nullptr;
    const int N = c->N;
    mop_status s;
    // the plain sequence for buffered lists (their reuse test needs all beads), while a bias is set, and for the first
    // evaluation of a topology (it checks the list capacities on the host)
    if (c->p.r_buf > 0.f || !c->caps_checked || c->bias_on) {
        CK(c, cudaMemcpyAsync(R, R_host, bytes, cudaMemcpyHostToDevice, c->st));
        if ((s = eval_async(c, R, G))) return s;
        if (grad_host) CK(c, cudaMemcpyAsync(grad_host, G, bytes, cudaMemcpyDeviceToHost, c->st));
        if ((s = read_back(c))) return s;
        *veff_out = c->last_veff;
        return MOP_OK;
    }
    const bool graphs = graphs_usable(c);
    if (graphs && (s = graphs_build(c))) return s;
    const bool split = grad_host && c->nh >= 2;   // pass 2 and the copy out in two bead groups
    // ---- copies in: bead 1 | beads 2..N (ordered after whatever the main stream still does with the staging buffer)
    CK(c, cudaEventRecord(c->ev_copy[0], c->st));
    CK(c, cudaStreamWaitEvent(c->st_copy, c->ev_copy[0], 0));
    CK(c, cudaMemcpyAsync(R, R_host, bead * sizeof(float), cudaMemcpyHostToDevice, c->st_copy));
    CK(c, cudaEventRecord(c->ev_copy[1], c->st_copy));
    if (N > 1) {
        CK(c, cudaMemcpyAsync(R + bead, R_host + bead, (size_t)(N - 1) * bead * sizeof(float), cudaMemcpyHostToDevice, c->st_copy));
        CK(c, cudaEventRecord(c->ev_copy[2], c->st_copy));
    }
    CK(c, cudaStreamWaitEvent(c->st, c->ev_copy[1], 0));
    if (graphs) CK(c, cudaGraphLaunch(c->gx[0], c->st));
    else if ((s = seq_A(c, R))) return s;
    if (N > 1) CK(c, cudaStreamWaitEvent(c->st, c->ev_copy[2], 0));
    if (!split) {
        if (graphs) CK(c, cudaGraphLaunch(c->gx[1], c->st));
        else if ((s = seq_B(c, R, G, 0))) return s;
        if (graphs) c->n_launches += c->gx_launches[0] + c->gx_launches[1];
        if (grad_host) CK(c, cudaMemcpyAsync(grad_host, G, bytes, cudaMemcpyDeviceToHost, c->st));
    } else {
        const size_t h = (size_t)split_bead(c);
        if (graphs) CK(c, cudaGraphLaunch(c->gx[2], c->st));
        else if ((s = seq_B(c, R, G, 1))) return s;
        // gradient rows [0, h) leave on the copy stream while the second group's H.eta runs
        CK(c, cudaEventRecord(c->ev_copy[3], c->st));
        CK(c, cudaStreamWaitEvent(c->st_copy, c->ev_copy[3], 0));
        CK(c, cudaMemcpyAsync(grad_host, G, h * bead * sizeof(float), cudaMemcpyDeviceToHost, c->st_copy));
        CK(c, cudaMemcpyAsync(grad_host + (size_t)(N - 1) * bead, G + (size_t)(N - 1) * bead, bead * sizeof(float),
                              cudaMemcpyDeviceToHost, c->st_copy));   // the last row (eq. 7) is complete already
        CK(c, cudaEventRecord(c->ev_copy[0], c->st_copy));
        if (graphs) CK(c, cudaGraphLaunch(c->gx[3], c->st));
        else if ((s = seq_B(c, R, G, 2))) return s;
        if (graphs) c->n_launches += c->gx_launches[0] + c->gx_launches[2] + c->gx_launches[3];
        if ((size_t)N - 1 > h)
            CK(c, cudaMemcpyAsync(grad_host + h * bead, G + h * bead, ((size_t)N - 1 - h) * bead * sizeof(float),
                                  cudaMemcpyDeviceToHost, c->st));
        CK(c, cudaStreamWaitEvent(c->st, c->ev_copy[0], 0));   // the final synchronisation of st covers both copies
    }
    c->n_rebuilds += 1;
    if ((s = read_back(c))) return s;
    *veff_out = c->last_veff;
    return MOP_OK;
}

// ---- bead-block mode: the paper's parallel layout -- beads spread over processing elements, point-to-point
// exchange between the owners of adjacent beads only -- with a contiguous block of beads per GPU
extern "C" mop_status mop_block_pass1(mop_ctx *c, const float *R_dev, const float *R_right_dev, float *keta_right_out_dev) {
    PRECHECK(c);
    if (!c->blk) FAIL(c, MOP_ERR_INVALID_ARG, "mop_block_pass1: not a bead-block context (mop_create_block)");
    if (!R_dev) FAIL(c, MOP_ERR_INVALID_ARG, "R_dev is NULL");
    const bool has_right = c->blk_n0 + c->N < c->blk_Ntot;
    if (has_right && (!R_right_dev || !keta_right_out_dev))
        FAIL(c, MOP_ERR_INVALID_ARG, "a block that is not the path's last needs R_right_dev and keta_right_out_dev");
    c->blk_stage = 0;
    mop_status s = eval_stage1(c, R_dev, has_right ? R_right_dev : nullptr, has_right ? keta_right_out_dev : nullptr);
    if (s) return s;
    c->blk_stage = 1;
    return MOP_OK;
}

extern "C" mop_status mop_block_pass2(mop_ctx *c, const float *R_dev) {
    PRECHECK(c);
    if (!c->blk || c->blk_stage != 1) FAIL(c, MOP_ERR_INVALID_ARG, "mop_block_pass2 follows mop_block_pass1");
    if (!R_dev) FAIL(c, MOP_ERR_INVALID_ARG, "R_dev is NULL");
    mop_status s = eval_stage2(c, R_dev);
    if (s) return s;
    c->blk_stage = 2;
    return MOP_OK;
}

extern "C" mop_status mop_block_assemble(mop_ctx *c, const float *keta_left_dev, double *veff_local_out, float *grad_dev) {
    PRECHECK(c);
    if (!c->blk || c->blk_stage != 2) FAIL(c, MOP_ERR_INVALID_ARG, "mop_block_assemble follows mop_block_pass2");
    if (c->blk_n0 > 0 && !keta_left_dev) FAIL(c, MOP_ERR_INVALID_ARG, "a block that is not the path's first needs keta_left_dev");
    mop_status s = eval_stage3(c, nullptr, c->blk_n0 > 0 ? keta_left_dev : nullptr, grad_dev, false);
    if (s) return s;
    c->blk_stage = 0;
    if (veff_local_out) {
        if ((s = read_back(c))) return s;
        *veff_local_out = c->last_veff;
    }
    return MOP_OK;
}

extern "C" mop_status mop_block_integrate(mop_ctx *c, float *R_dev, float *V_dev, const float *grad_dev, double dt_pmd, int stage) {
    PRECHECK(c);
    if (!R_dev || !V_dev || !grad_dev) FAIL(c, MOP_ERR_INVALID_ARG, "NULL argument");
    if (!(dt_pmd > 0.0) || (stage != 0 && stage != 1)) FAIL(c, MOP_ERR_INVALID_ARG, "need dt_pmd > 0 and stage 0 or 1");
    const size_t total = (size_t)c->N * c->Q * 3;
    LAUNCH(c, k_verlet, cdiv(total, 256), 256, 0, total, c->Q, (float)dt_pmd, stage, c->d_inv_mass, c->d_mass, grad_dev, R_dev,
           V_dev, (double *)nullptr);
    CK(c, cudaGetLastError());
    return MOP_OK;
}

// the thermostat half of an NVT step on a bead block: the OU update of mop_step_langevin with the generator keyed by the
// coordinate's index in the whole path, so that every rank of a sharded run replays its part of the one noise stream
extern "C" mop_status mop_block_thermostat(mop_ctx *c, float *V_dev, double dt_pmd, double gamma, double temperature,
                                           unsigned long long seed, unsigned long long step) {
    PRECHECK(c);
    if (!V_dev) FAIL(c, MOP_ERR_INVALID_ARG, "V_dev is NULL");
    if (!(dt_pmd > 0.0) || !(gamma >= 0.0) || !(temperature >= 0.0)) FAIL(c, MOP_ERR_INVALID_ARG, "need dt_pmd > 0, gamma >= 0 and temperature >= 0");
    if (gamma == 0.0) return MOP_OK;   // plain velocity Verlet
    const double cc = exp(-gamma * dt_pmd);
    const float amp = (float)sqrt((1.0 - cc * cc) * 0.0083144626 * temperature);   // k_B in kJ mol^-1 K^-1
    const size_t total = (size_t)c->N * c->Q * 3;
    const unsigned long long idx0 = (unsigned long long)(c->blk ? c->blk_n0 : 0) * (unsigned long long)c->Q * 3ull;
    LAUNCH(c, k_ou, cdiv(total, 256), 256, 0, total, c->Q, (float)cc, amp, seed, step, idx0, c->d_inv_mass, c->d_mass, V_dev,
           (double *)nullptr);
    CK(c, cudaGetLastError());
    return MOP_OK;
}

extern "C" mop_status mop_set_timing(mop_ctx *c, int on) {
    if (!c) return MOP_ERR_INVALID_ARG;
    if (c->sticky) return (mop_status)c->sticky;
    CK(c, cudaSetDevice(c->p.device));
    if (on && !c->ev_made) {
        for (auto &set : c->ev)
            for (cudaEvent_t &e : set) CK(c, cudaEventCreate(&e));
        c->ev_made = true;
    }
    if (c->ev_made) t_collect(c, MOP_TSETS);
    c->timing = on != 0;
    for (double &t : c->t_sum) t = 0.0;
    c->t_cnt = 0;
    return MOP_OK;
}

extern "C" mop_status mop_get_timing(mop_ctx *c, double out[16]) {
    if (!c || !out) return MOP_ERR_INVALID_ARG;
    if (c->sticky) return (mop_status)c->sticky;
    CK(c, cudaSetDevice(c->p.device));
    if (c->ev_made) t_collect(c, MOP_TSETS);
    for (int k = 0; k < 16; k++) out[k] = 0.0;
    for (int k = 0; k < MOP_NSTAGE; k++) out[k] = c->t_cnt > 0 ? c->t_sum[k] / c->t_cnt : 0.0;
    out[8] = c->t_cnt;
    return MOP_OK;
}

// one evaluation inside mop_step*: gradient into c->d_G; as CUDA graphs when usable (small systems are launch-bound)
static mop_status eval_for_step(mop_ctx *c, const float *R_dev, bool deposit, bool want_energy) {
    if (!graphs_usable(c)) return eval_async(c, R_dev, c->d_G, deposit, want_energy);
    mop_status s = graphs_build(c);
    if (s) return s;
    const size_t bytes = (size_t)c->N * c->Q * 3 * sizeof(float);
    CK(c, cudaMemcpyAsync(c->d_Rh, R_dev, bytes, cudaMemcpyDeviceToDevice, c->st));
    CK(c, cudaGraphLaunch(c->gx[want_energy ? 0 : 4], c->st));
    CK(c, cudaGraphLaunch(c->gx[1], c->st));
    c->n_launches += c->gx_launches[want_energy ? 0 : 4] + c->gx_launches[1];
    c->n_rebuilds += 1;
    CK(c, cudaMemcpyAsync(c->d_G, c->d_Gh, bytes, cudaMemcpyDeviceToDevice, c->st));
    return MOP_OK;
}

// velocity Verlet on eq. (4) (+ the exact OU velocity update when ou); cont: d_G already holds the gradient at R_dev
static mop_status step_impl(mop_ctx *c, float *R_dev, float *V_dev, double dt_pmd, int n_steps, bool cont, bool ou, double cc,
                            float amp, unsigned long long seed, unsigned long long step0) {
    NOT_A_PARTIAL_BLOCK(c);
    if (!R_dev || !V_dev) FAIL(c, MOP_ERR_INVALID_ARG, "R_dev or V_dev is NULL");
    if (n_steps < 0 || !(dt_pmd > 0.0)) FAIL(c, MOP_ERR_INVALID_ARG, "need n_steps >= 0 and dt_pmd > 0");
    const size_t total = (size_t)c->N * c->Q * 3;
    if (!c->d_G) CK(c, dalloc(&c->d_G, total));
    mop_status s;
    if (cont) {
        if (!c->g_current) FAIL(c, MOP_ERR_INVALID_ARG, "mop_step*_continue: no gradient from a previous mop_step* call is held");
    } else if ((s = eval_for_step(c, R_dev, false, n_steps == 0))) {
        return s;
    }
    c->g_current = false;
    const unsigned nblk = cdiv(total, 256);
    for (int it = 0; it < n_steps; it++) {
        LAUNCH(c, k_verlet, nblk, 256, 0, total, c->Q, (float)dt_pmd, 0, c->d_inv_mass, c->d_mass, c->d_G, R_dev, V_dev,
               (double *)nullptr);
        c->bias_steps += 1;
        const bool last = it == n_steps - 1;   // V_eff (mop_get_stats) is that of the last evaluation of the call: only it forms U(R^1)
        if ((s = eval_for_step(c, R_dev, c->bias_on && c->bias_pace > 0 && c->bias_steps % c->bias_pace == 0, last))) return s;
        if (last) CK(c, cudaMemsetAsync(c->d_energy + 5, 0, sizeof(double), c->st));
        LAUNCH(c, k_verlet, nblk, 256, 0, total, c->Q, (float)dt_pmd, 1, c->d_inv_mass, c->d_mass, c->d_G, R_dev, V_dev,
               (last && !ou) ? c->d_energy + 5 : (double *)nullptr);
        if (ou)
            LAUNCH(c, k_ou, nblk, 256, 0, total, c->Q, (float)cc, amp, seed, step0 + (unsigned long long)it, 0ull, c->d_inv_mass,
                   c->d_mass, V_dev, last ? c->d_energy + 5 : (double *)nullptr);
    }
    CK(c, cudaGetLastError());
    c->g_current = true;   // d_G is the gradient at the R_dev this call leaves behind
    return MOP_OK;
}

extern "C" mop_status mop_step(mop_ctx *c, float *R_dev, float *V_dev, double dt_pmd, int n_steps) {
    PRECHECK(c);
    return step_impl(c, R_dev, V_dev, dt_pmd, n_steps, false, false, 1.0, 0.f, 0ull, 0ull);
}

extern "C" mop_status mop_step_continue(mop_ctx *c, float *R_dev, float *V_dev, double dt_pmd, int n_steps) {
    PRECHECK(c);
    return step_impl(c, R_dev, V_dev, dt_pmd, n_steps, true, false, 1.0, 0.f, 0ull, 0ull);
}

// path MD with the Langevin thermostat of the paper's NVT runs: velocity Verlet, then the exact OU velocity update
static mop_status langevin_impl(mop_ctx *c, float *R_dev, float *V_dev, double dt_pmd, int n_steps, double gamma,
                                double temperature, unsigned long long seed, unsigned long long step0, bool cont) {
    if (!(gamma >= 0.0) || !(temperature >= 0.0)) FAIL(c, MOP_ERR_INVALID_ARG, "need gamma >= 0 and temperature >= 0");
    if (!(dt_pmd > 0.0)) FAIL(c, MOP_ERR_INVALID_ARG, "need n_steps >= 0 and dt_pmd > 0");
    const double cc = exp(-gamma * dt_pmd);
    const float amp = (float)sqrt((1.0 - cc * cc) * 0.0083144626 * temperature);   // k_B in kJ mol^-1 K^-1
    return step_impl(c, R_dev, V_dev, dt_pmd, n_steps, cont, gamma > 0.0, cc, amp, seed, step0);
}

extern "C" mop_status mop_step_langevin(mop_ctx *c, float *R_dev, float *V_dev, double dt_pmd, int n_steps, double gamma,
                                        double temperature, unsigned long long seed, unsigned long long step0) {
    PRECHECK(c);
    return langevin_impl(c, R_dev, V_dev, dt_pmd, n_steps, gamma, temperature, seed, step0, false);
}

extern "C" mop_status mop_step_langevin_continue(mop_ctx *c, float *R_dev, float *V_dev, double dt_pmd, int n_steps,
                                                 double gamma, double temperature, unsigned long long seed,
                                                 unsigned long long step0) {
    PRECHECK(c);
    return langevin_impl(c, R_dev, V_dev, dt_pmd, n_steps, gamma, temperature, seed, step0, true);
}

// debug: raw bits of the thermostat's counter-based generator for idx = 0..n-1 (HOST output)
extern "C" mop_status mop_debug_noise_bits(mop_ctx *c, unsigned long long seed, unsigned long long step, int n,
                                           unsigned long long *host_out) {
    PRECHECK(c);
    if (n < 0 || (n > 0 && !host_out)) FAIL(c, MOP_ERR_INVALID_ARG, "mop_debug_noise_bits: bad argument");
    if (n == 0) return MOP_OK;
    unsigned long long *d = nullptr;
    CK(c, dalloc(&d, (size_t)n));
    LAUNCH(c, k_noise_bits, cdiv(n, 256), 256, 0, n, seed, step, d);
    cudaError_t e = cudaMemcpyAsync(host_out, d, (size_t)n * 8, cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    cudaFree(d);
    CK(c, e);
    return MOP_OK;
}

// ---- metadynamics of paths: Gaussian bias on the end-to-end CV
extern "C" mop_status mop_set_bias(mop_ctx *c, const int *group_a, int n_a, const int *group_b, int n_b, double sigma,
                                   double height, int pace) {
    PRECHECK(c);
    // no block context takes a bias (mop.h), the one that holds the whole path included: mop_block_assemble has no
    // coordinates to form the CV from, and a sharded path would need the owners of beads 1 and N to exchange s(R)
    if (c->blk) FAIL(c, MOP_ERR_INVALID_ARG, "mop_set_bias: bead-block contexts take no bias (use mop_create for a biased path)");
    CK(c, cudaStreamSynchronize(c->st));
    c->bias_on = false;
    c->bias_steps = 0;
    c->g_current = false;
    if (n_a == 0 && n_b == 0) return MOP_OK;   // bias switched off
    if (n_a < 1 || n_b < 1 || !group_a || !group_b) FAIL(c, MOP_ERR_INVALID_ARG, "mop_set_bias: both groups need atoms");
    if (!(sigma > 0.0) || !std::isfinite(height) || pace < 0) FAIL(c, MOP_ERR_INVALID_ARG, "need sigma > 0, finite height, pace >= 0");
    if (c->N < 2) FAIL(c, MOP_ERR_INVALID_ARG, "the end-to-end CV needs n_beads >= 2");
    for (int k = 0; k < n_a; k++)
        if (group_a[k] < 0 || group_a[k] >= c->Q) FAIL(c, MOP_ERR_INVALID_ARG, "group_a[%d] out of range", k);
    for (int k = 0; k < n_b; k++)
        if (group_b[k] < 0 || group_b[k] >= c->Q) FAIL(c, MOP_ERR_INVALID_ARG, "group_b[%d] out of range", k);
    CK(c, dalloc(&c->d_bias_ga, (size_t)n_a));
    CK(c, dalloc(&c->d_bias_gb, (size_t)n_b));
    if (!c->d_bias_hills) {
        CK(c, dalloc(&c->d_bias_hills, (size_t)MOP_MAX_HILLS));
        CK(c, dalloc(&c->d_bias_nh, 1));
        CK(c, dalloc(&c->d_bias_com, 16));
        CK(c, dalloc(&c->d_bias_state, 16));
    }
    CK(c, cudaMemcpyAsync(c->d_bias_ga, group_a, (size_t)n_a * 4, cudaMemcpyHostToDevice, c->st));
    CK(c, cudaMemcpyAsync(c->d_bias_gb, group_b, (size_t)n_b * 4, cudaMemcpyHostToDevice, c->st));
    CK(c, cudaMemsetAsync(c->d_bias_nh, 0, sizeof(int), c->st));
    CK(c, cudaMemsetAsync(c->d_bias_state, 0, 16 * sizeof(double), c->st));
    CK(c, cudaStreamSynchronize(c->st));
    c->bias_na = n_a, c->bias_nb = n_b, c->bias_sigma = sigma, c->bias_w = height, c->bias_pace = pace;
    c->bias_on = true;
    return MOP_OK;
}

extern "C" mop_status mop_add_hill(mop_ctx *c, double s_center) {
    PRECHECK(c);
    if (!c->bias_on) FAIL(c, MOP_ERR_INVALID_ARG, "mop_add_hill: no bias set");
    c->g_current = false;
    int nh = 0;
    CK(c, cudaMemcpyAsync(&nh, c->d_bias_nh, sizeof(int), cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    if (nh >= MOP_MAX_HILLS) FAIL(c, MOP_ERR_OOM, "hill table full (%d)", MOP_MAX_HILLS);
    CK(c, cudaMemcpyAsync(c->d_bias_hills + nh, &s_center, sizeof(double), cudaMemcpyHostToDevice, c->st));
    nh += 1;
    CK(c, cudaMemcpyAsync(c->d_bias_nh, &nh, sizeof(int), cudaMemcpyHostToDevice, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    return MOP_OK;
}

extern "C" mop_status mop_get_bias(mop_ctx *c, double out[8], double *hills_host, int cap, int *n_hills) {
    PRECHECK(c);
    if (!out) FAIL(c, MOP_ERR_INVALID_ARG, "out is NULL");
    for (int k = 0; k < 8; k++) out[k] = 0.0;
    if (n_hills) *n_hills = 0;
    if (!c->bias_on) return MOP_OK;
    double st[16];
    int nh = 0;
    CK(c, cudaMemcpyAsync(st, c->d_bias_state, sizeof st, cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaMemcpyAsync(&nh, c->d_bias_nh, sizeof(int), cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    for (int k = 0; k < 5; k++) out[k] = st[k];
    out[5] = (double)nh;
    if (n_hills) *n_hills = nh;
    if (hills_host && cap > 0 && nh > 0) {
        CK(c, cudaMemcpyAsync(hills_host, c->d_bias_hills, (size_t)std::min(cap, nh) * 8, cudaMemcpyDeviceToHost, c->st));
        CK(c, cudaStreamSynchronize(c->st));
    }
    return MOP_OK;
}

extern "C" mop_status mop_get_stats(mop_ctx *c, double out[16]) {
    PRECHECK(c);
    if (!out) FAIL(c, MOP_ERR_INVALID_ARG, "out is NULL");
    mop_status s = read_back(c);
    if (s && s != MOP_ERR_NONFINITE) return s;
    const double *E = c->h_energy;
    out[0] = c->last_veff;
    out[1] = E[0] + E[1] + E[2] + E[3];
    out[2] = E[4];
    out[3] = E[0], out[4] = E[1], out[5] = E[2], out[6] = E[3];
    out[7] = E[5];
    out[8] = c->n_rebuilds;
    out[9] = (double)c->h_ctr->n_entries;
    out[10] = (double)c->h_ctr->n_units;
    out[11] = (double)c->h_ctr->n_masks;
    out[12] = (double)(*c->h_slots);
    out[13] = c->n_launches;
    out[14] = c->n_reuses;
    out[15] = (double)c->h_slots[1];
    return MOP_OK;
}

extern "C" mop_status mop_debug_get(mop_ctx *c, const char *what, void *host_buf, size_t bytes) {
    PRECHECK(c);
    if (!what || !host_buf) FAIL(c, MOP_ERR_INVALID_ARG, "NULL argument");
    const MopGrid &g = c->g;
    const size_t nf = c->nf, Q = c->Q, S = g.S;
    std::string w(what);
    auto copy = [&](const void *src, size_t n) -> mop_status {
        if (bytes != n) FAIL(c, MOP_ERR_INVALID_ARG, "mop_debug_get(%s): expected %zu bytes, got %zu", what, n, bytes);
        CK(c, cudaMemcpyAsync(host_buf, src, n, cudaMemcpyDeviceToHost, c->st));
        CK(c, cudaStreamSynchronize(c->st));
        return MOP_OK;
    };
    if (w == "dims") {
        int d[8] = {g.dims[0], g.dims[1], g.dims[2], g.S, c->nf, MOP_CL, MOP_NG, 0};
        memcpy(&d[7], &c->bin_z, 4);
        if (bytes != sizeof d) FAIL(c, MOP_ERR_INVALID_ARG, "mop_debug_get(dims): expected %zu bytes", sizeof d);
        memcpy(host_buf, d, sizeof d);
        return MOP_OK;
    }
    if (w == "cell") return copy(c->d_cell, nf * Q * 4);
    if (w == "perm") return copy(c->d_perm, nf * S * 4);
    if (w == "xq") return copy(c->d_xq, nf * S * 16);
    const float4 *src = nullptr;
    if (w == "F") src = c->d_F4;
    else if (w == "eta") src = c->d_et;
    else if (w == "Heta") src = c->d_H4;
    else FAIL(c, MOP_ERR_INVALID_ARG, "mop_debug_get: unknown array '%s'", what);
    if (!c->d_dbg) CK(c, dalloc(&c->d_dbg, nf * Q * 3));
    LAUNCH(c, k_gather3, dim3(cdiv(Q, 256), (unsigned)nf), 256, 0, c->Q, g.S, c->d_slot_of, src, c->d_dbg, 1.0f);
    return copy(c->d_dbg, nf * Q * 12);
}

extern "C" mop_status mop_debug_pairs(mop_ctx *c, int bead, int *pairs, long long cap, long long *n_pairs) {
    PRECHECK(c);
    if (bead < 0 || bead >= c->nf || !n_pairs || cap < 0 || (cap > 0 && !pairs))
        FAIL(c, MOP_ERR_INVALID_ARG, "mop_debug_pairs: bad argument");
    int *d_pairs = nullptr;
    CK(c, dalloc(&d_pairs, (size_t)2 * cap));
    PairDbgArgs a;
    a.S = c->g.S, a.bead = bead, a.rc2 = c->rc2;
    a.xq = c->d_xq, a.perm = c->d_perm, a.units = c->d_units, a.entries = c->d_entries, a.masks = c->d_masks;
    a.ctr = c->d_ctr, a.cap_units = c->cap_units, a.pairs = d_pairs, a.cap = cap;
    for (int d = 0; d < 3; d++) a.box[d] = c->g.box[d];
    cudaMemsetAsync(&c->d_ctr->n_pairs, 0, sizeof(unsigned long long), c->st);
    LAUNCH(c, k_debug_pairs, c->sm_count * 8, 128, 0, a);
    cudaError_t e = cudaMemcpyAsync(c->h_ctr, c->d_ctr, sizeof(MopCounters), cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    if (e == cudaSuccess) {
        *n_pairs = (long long)c->h_ctr->n_pairs;
        long long ncopy = std::min(*n_pairs, cap);
        if (ncopy > 0) e = cudaMemcpy(pairs, d_pairs, (size_t)ncopy * 8, cudaMemcpyDeviceToHost);
    }
    cudaFree(d_pairs);
    CK(c, e);
    return MOP_OK;
}

// The production force kernel's own in-range decisions (its counting instance: same code, plus a population count
// of the per-pair predicate results) over the list of the last evaluation.  which = 0: bead 1; 1: the other force
// beads; 2: all force beads.  The forces it computes go to the H.eta scratch array.  Synchronises.
extern "C" mop_status mop_debug_count_inrange(mop_ctx *c, int which, long long *n_inrange, unsigned long long *pair_hash) {
    PRECHECK(c);
    if (which < 0 || which > 2 || !n_inrange) FAIL(c, MOP_ERR_INVALID_ARG, "mop_debug_count_inrange: bad argument");
    if (c->n_rebuilds == 0) FAIL(c, MOP_ERR_INVALID_ARG, "mop_debug_count_inrange: no evaluation yet");
    CK(c, cudaMemsetAsync(&c->d_ctr->n_inrange, 0, 2 * sizeof(unsigned long long), c->st));   // count and hash
    CK(c, cudaMemsetAsync(c->d_work + 3, 0, sizeof(unsigned), c->st));
    LAUNCH(c, nb_pick(NB_FORCE, true), c->nb_blocks_c, 128, nb_smem(c), nb_args(c, c->d_H4, 3, which));
    CK(c, cudaMemcpyAsync(c->h_ctr, c->d_ctr, sizeof(MopCounters), cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    CK(c, cudaGetLastError());
    *n_inrange = (long long)c->h_ctr->n_inrange;
    if (pair_hash) *pair_hash = c->h_ctr->pair_hash;
    return MOP_OK;
}

// testing aid: replace the pair-list buffers by ones of the given capacities (0: keep that capacity), so that the overflow
// and regrow paths can be driven deterministically.  The automatic check of the first build is switched off.
extern "C" mop_status mop_debug_set_list_capacity(mop_ctx *c, unsigned units, unsigned entries, unsigned masks) {
    PRECHECK(c);
    CK(c, cudaStreamSynchronize(c->st));
    mop_status s = alloc_lists(c, units ? units : c->cap_units, entries ? entries : c->cap_entries, masks ? masks : c->cap_masks);
    if (s) return s;
    c->caps_checked = true;
    return MOP_OK;
}

extern "C" mop_status mop_force_hvp(mop_ctx *c, const float *R_dev, const float *s_dev, float *F_dev, float *Hs_dev) {
    PRECHECK(c);
    if (!R_dev) FAIL(c, MOP_ERR_INVALID_ARG, "R_dev is NULL");
    if (Hs_dev && !s_dev) FAIL(c, MOP_ERR_INVALID_ARG, "Hs_dev needs s_dev");
    CK(c, cudaMemsetAsync(c->d_energy, 0, 5 * sizeof(double), c->st));
    CK(c, cudaMemsetAsync(c->d_work, 0, 8 * sizeof(unsigned), c->st));
    c->list_valid = false;
    mop_status s = build_list(c, R_dev, 1);
    if (s) return s;
    if ((s = pass_force(c, R_dev, 1))) return s;
    const MopGrid &g = c->g;
    if (F_dev) LAUNCH(c, k_gather3, dim3(cdiv(c->Q, 256), 1), 256, 0, c->Q, g.S, c->d_slot_of, c->d_F4, F_dev, 1.0f);
    if (Hs_dev) {
        LAUNCH(c, k_set_dir, cdiv(g.S, 256), 256, 0, g.S, c->d_perm, c->d_typ, s_dev, c->d_et);
        if ((s = pass_hvp(c, R_dev, 1))) return s;
        LAUNCH(c, k_gather3, dim3(cdiv(c->Q, 256), 1), 256, 0, c->Q, g.S, c->d_slot_of, c->d_H4, Hs_dev, 1.0f);
    }
    CK(c, cudaGetLastError());
    return MOP_OK;
}

