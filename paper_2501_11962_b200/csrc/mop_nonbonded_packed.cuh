// mop_nonbonded_packed.cuh -- the production form of S2 (pass 1: force, energy on bead 1) and S5 (pass 2: fused
// force-scalar + Hessian-vector pair kernel), SURVEY.md 8a.  FP32-pipe-bound; no tensor cores.
#pragma once
#include "mop_nonbonded.cuh"
#include "mop_f2.cuh"

// =====================================================================================================
// Packed variant: two i atoms per lane per issue slot (sm_100a FFMA2 / FMUL2 / FADD2 = fma|mul|add.rn.f32x2).
// The pair kernels are bound by issue slots when written with scalar FP32 instructions (profiles/r01_ncu_summary.md);
// the packed form halves the FP issue count, which leaves the FP32 pipe itself (128 lanes/clk/SM) as the bound.
// Lane (jl = lane & 7, g = lane >> 3) owns atom jl of the g-th of the four j-octets of the current step; a packed
// register holds the same quantity for i atoms (2p, 2p+1), p = 0..3.  All packed operations are IEEE
// round-to-nearest per component, so the G8 predicate
// (d = (xw_i - xw_j) - k L, r2 = fma(dz,dz,fma(dy,dy,dx*dx)), r2 < rc*rc) is bit-identical to the scalar form.
// Sign conventions chosen so that no negation is needed in the row body:
//   gn = -g = x (B - A) + C - 2 k_rf ke qi qj,      hn = -h = x (x (8A - 14B) - 3C),      dn = s_j - s_i = -delta
//   F_i += gn d;                (H s)_i += hn (d.dn) d + gn dn;        the j side accumulates the same sums (jn),
//   and the lane's j atom receives -(jn.lo + jn.hi) once per entry.
// staging reads are volatile so that the compiler re-reads shared memory per entry instead of pinning the
// eight i atoms in registers for the whole unit
__device__ __forceinline__ float4 mop_lds_v4(unsigned addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float2 mop_lds_v2(unsigned addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ float mop_lds_f(unsigned addr) {
    float v;
    asm("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}

__device__ __forceinline__ unsigned mop_lds_vu(unsigned addr) {
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint2 mop_lds_vu2(unsigned addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}
#define NBP_NST 2       // stages of the per-warp j-atom ring (one step in flight)

// Shared memory of one CTA (4 warps), bytes:
//   [0, 1024)              i-atom staging, 256 B per warp: for p = 0..3 at float offset 16 p
//                          [0,1] x  [2,3] y  [4,5] z  [6,7] ke q  [8,9] s_x  [10,11] s_y  [12,13] s_z  [14,15] LJ-row address
//   [1024, 2048)           the current chunk of up to 32 list entries (8 steps), 256 B per warp
//   [2048, 3072)           energy variant only: the i atoms in FP64, 256 B per warp: atom k at +32 k: x, y, z, ke q
//   [3072, 3072 + 4 NBP_NST KB)   j-atom ring, per warp NBP_NST stages of 1 KB: xq[32] at +0, eta+type[32] (or type[32]) at +512
//   then the LJ tables: (6 C6, 12 C12)[nt*nt] interleaved (one 8-byte load per pair), energy shift [nt*nt],
//   and one flag per type: its LJ row has a non-zero entry
#define NBP_SM_ENT 1024u
#define NBP_SM_DBL 2048u
#define NBP_SM_RING 3072u
#define NBP_SM_TAB (NBP_SM_RING + 4u * NBP_NST * 1024u)
__host__ __device__ inline size_t nbp_smem_bytes(int nt) { return NBP_SM_TAB + (size_t)nt * nt * 12 + (size_t)nt * 4; }
__device__ __forceinline__ double mop_lds_d(unsigned addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

// One work unit = one i-octet against its list of (j-octet, shift) entries, four entries per step: lane (jl, g) holds
// atom jl of the step's g-th octet.  The builder has ordered the entries by their row-pair pattern, so the union
// pattern of a step (which row pairs the warp evaluates) mostly equals each group's own.  A group whose own pattern
// lacks a row pair of the union evaluates it too; its pairs are out of range there by construction of the pattern
// (the builder's test is a superset of G8), so the exact per-pair predicate masks them.
template <int MODE, bool COUNT>
__device__ __forceinline__ void nbp_unit(const NbArgs &a, const MopUnit &un, float *__restrict__ sw,
                                         const unsigned sw_addr, const unsigned se_addr, const unsigned sr_addr,
                                         const unsigned sd_addr, const unsigned tab6, const unsigned tabS,
                                         const int *__restrict__ tflag, const int lane) {
    constexpr bool HVP = MODE == NB_HVP, ENERGY = MODE == NB_ENERGY;
    // every atom is addressed by its 32-bit element index boff + slot into the [nf][S] arrays (nf * S < 2^31, checked at
    // create): one wide multiply-add per address instead of per-bead 64-bit pointers rebuilt every step
    const unsigned boff = (unsigned)un.bead * (unsigned)a.S;
    const float4 *__restrict__ xq = a.xq;
    const float4 *__restrict__ et = a.et;
    const int *__restrict__ typ = a.typ;
    float4 *__restrict__ out = a.out;
    const int jl = lane & 7, gq = lane >> 3;
    const unsigned ibase = boff + (unsigned)un.ci * MOP_CL;
    MOP_ASSERT(ibase + MOP_CL <= a.n_slots);
    MOP_ASSERT((unsigned long long)un.start + un.count <= a.cap_entries && (un.count % MOP_NG) == 0);

    __syncwarp();
    bool has_lj = false;
    if (lane < MOP_CL) {
        float4 p = xq[ibase + lane];
        float4 e = make_float4(0.f, 0.f, 0.f, 0.f);
        int ti;
        if (HVP) {
            e = et[ibase + lane];
            ti = __float_as_int(e.w);
        } else {
            ti = typ[ibase + lane];
        }
        has_lj = tflag[ti] != 0;
        float *d = sw + (lane >> 1) * 16 + (lane & 1);
        d[0] = p.x, d[2] = p.y, d[4] = p.z;
        d[6] = p.w * MOP_KE;
        d[8] = e.x, d[10] = e.y, d[12] = e.z;
        d[14] = __int_as_float((int)tab6 + ti * a.nt * 8);
        if (COUNT) d[8] = __int_as_float(a.perm[ibase + lane]);   // original index of the i atom (the eta slot is free in force mode)
        if (ENERGY) {
            asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(sd_addr + lane * 32u), "d"((double)p.x), "d"((double)p.y) : "memory");
            asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(sd_addr + lane * 32u + 16u), "d"((double)p.z),
                         "d"(138.935458 * (double)p.w) : "memory");
        }
    }
    __syncwarp();
    const unsigned ljmask = __ballot_sync(0xffffffffu, has_lj) & 0xffu; // bit k: i atom k has a non-zero LJ row

    f2 ax[4], ay[4], az[4];
#pragma unroll
    for (int p = 0; p < 4; p++) ax[p] = ay[p] = az[p] = 0ull;
    double e_lj = 0.0, e_c = 0.0;
    unsigned n_in = 0;
    unsigned long long h_in = 0ull;
    const f2 nk2rf = f2_bc(-a.k2rf);
    const unsigned lane16 = (unsigned)lane * 16u;

    // one step: the lane's j atom (cp, ce, type offset tj8) against the row pairs of the union pattern `upat`.
    // sh*: the lane's periodic shift k L (packed broadcast; zero for most steps: d - 0 = d exactly, so one code path
    // serves both, the shifted form only being compiled into the SHIFTED instance).
    auto step = [&](const uint2 cur, const unsigned upat, const bool shifted, const bool masked, const float4 cp,
                    const float4 ce, const unsigned tj8) {
        const f2 jx = f2_bc(cp.x), jy = f2_bc(cp.y), jz = f2_bc(cp.z), jq = f2_bc(cp.w);
        f2 shx = 0ull, shy = 0ull, shz = 0ull;
        if (shifted) {
            float sx, sy, sz;
            mop_unit_shift((int)(cur.y >> 24), a.box, sx, sy, sz);
            shx = f2_bc(sx), shy = f2_bc(sy), shz = f2_bc(sz);
        }
        f2 nx = 0ull, ny = 0ull, nz = 0ull; // jn: minus the j-side sums
        // energy variant: the lane's j atom and shift in FP64 (see "energy of bead 1" in heavy())
        double jxd = 0.0, jyd = 0.0, jzd = 0.0, acc_c = 0.0;
        f2 eA = 0ull, eB = 0ull, eS = 0ull;   // LJ: FP32 sums of A, B and the shift over the step's in-range pairs
        if (ENERGY) {
            jxd = (double)cp.x, jyd = (double)cp.y, jzd = (double)cp.z;
            if (shifted) {
                float sx, sy, sz;
                mop_unit_shift((int)(cur.y >> 24), a.box, sx, sy, sz);
                jxd += (double)sx, jyd += (double)sy, jzd += (double)sz;   // exact: d = x_i - (x_j + k L)
            }
        }
        // lm: bit k set iff i atom k may interact with this lane's j atom (diagonal block, exclusions)
        // (a padding entry -- pattern 0, it points at the unit's own octet -- allows nothing)
        const int jorig = COUNT ? a.perm[cur.x + jl] : 0;   // counting variant: original index of the lane's j atom
        const bool valid = (cur.y & 15u) != 0u;
        unsigned lm = valid ? 0xffu : 0u;
        if (masked) {
            const unsigned row1 = (cur.y >> 8) & 0xffu;
            if (row1 != 0) {
                MOP_ASSERT(un.excl_base + row1 - 1 < a.cap_masks);
                lm = reinterpret_cast<const unsigned char *>(a.masks)[((size_t)un.excl_base + row1 - 1) * 8 + jl];
            }
        }

        auto heavy = [&](const int p, const bool nolj) {
            const float4 P0 = mop_lds_v4(sw_addr + p * 64), P1 = mop_lds_v4(sw_addr + p * 64 + 16);
            const f2 X = f2_pack(P0.x, P0.y), Y = f2_pack(P0.z, P0.w), Z = f2_pack(P1.x, P1.y);
            f2 dx = f2_sub(X, jx), dy = f2_sub(Y, jy), dz = f2_sub(Z, jz);
            if (shifted) dx = f2_sub(dx, shx), dy = f2_sub(dy, shy), dz = f2_sub(dz, shz); // G8: d = (x_i - x_j) - k L
            const f2 Qi = f2_pack(P1.z, P1.w);
            const f2 r2v = f2_fma(dz, dz, f2_fma(dy, dy, f2_mul(dx, dx)));
            float r2a, r2b;
            f2_unpack(r2v, r2a, r2b);
            bool ina = r2a < a.rc2, inb = r2b < a.rc2; // G8 (padding atoms are never in range: mop_dummy_xq)
            if (masked) {
                ina = ina && ((lm >> (2 * p)) & 1u);
                inb = inb && ((lm >> (2 * p + 1)) & 1u);
            }
            if (COUNT) {
                n_in += (ina ? 1u : 0u) + (inb ? 1u : 0u);
                const float2 io = mop_lds_v2(sw_addr + p * 64 + 32);   // original indices of the two i atoms
                if (ina) h_in += mop_pair_hash((unsigned long long)un.bead, (unsigned long long)a.Q, __float_as_int(io.x), jorig);
                if (inb) h_in += mop_pair_hash((unsigned long long)un.bead, (unsigned long long)a.Q, __float_as_int(io.y), jorig);
            }
            const float ra = mop_rsqrt(r2a), rb = mop_rsqrt(r2b);
            const f2 rinv = f2_pack(ra, rb);
            const f2 qq = f2_mul(Qi, jq);
            f2 S0 = 0ull, S1 = 0ull, S2 = 0ull;
            unsigned ta, tb;
            if (HVP) {
                const float4 E0 = mop_lds_v4(sw_addr + p * 64 + 32), E1 = mop_lds_v4(sw_addr + p * 64 + 48);
                S0 = f2_pack(E0.x, E0.y), S1 = f2_pack(E0.z, E0.w), S2 = f2_pack(E1.x, E1.y);
                ta = (unsigned)__float_as_int(E1.z) + tj8, tb = (unsigned)__float_as_int(E1.w) + tj8;
            } else {
                const float2 T = mop_lds_v2(sw_addr + p * 64 + 56);
                ta = (unsigned)__float_as_int(T.x) + tj8, tb = (unsigned)__float_as_int(T.y) + tj8;
            }
            const f2 x = f2_mul(rinv, rinv);
            const f2 C = f2_mul(qq, f2_mul(x, rinv));
            f2 x3 = 0ull, A = 0ull, B = 0ull, gn;
            if (nolj) { // both i atoms have an all-zero LJ row (water hydrogens): reaction field only
                gn = f2_fma(qq, nk2rf, C);
            } else {
                const float2 la = mop_lds_v2(ta), lb = mop_lds_v2(tb);   // (6 C6, 12 C12) of the two pairs
                const f2 c6 = f2_pack(la.x, lb.x), c12 = f2_pack(la.y, lb.y);
                x3 = f2_mul(f2_mul(x, x), x);
                A = f2_mul(c6, x3);
                B = f2_mul(f2_mul(c12, x3), x3);
                gn = f2_fma(x, f2_sub(B, A), f2_fma(qq, nk2rf, C));
            }
            {
                float ga, gb;
                f2_unpack(gn, ga, gb);
                gn = f2_pack(ina ? ga : 0.f, inb ? gb : 0.f);
            }
            if (!HVP) {
                f2_acc(ax[p], gn, dx), f2_acc(ay[p], gn, dy), f2_acc(az[p], gn, dz);
                f2_acc(nx, gn, dx), f2_acc(ny, gn, dy), f2_acc(nz, gn, dz);
                if (ENERGY) {
                    // Energy of bead 1.  U(R^1) is the small remainder of attractive and repulsive pair terms (sum |u| ~
                    // 1e4 |U| for water-like systems), so FP32 reaction-field pair energies -- 6e-8 relative rounding in
                    // 1/r alone, and the low bits of c_rf lost the same way for every close pair -- leave 3e-6 to 2e-5
                    // of |U(R^1)|; north_star asks for 1e-6 of V_eff, which for N = 1 is U(R^1).  So the reaction-field
                    // term is formed in FP64 (forces stay FP32): d exact from the FP32 coordinates, 1/r = the FP32 rsqrt
                    // refined by one FP64 Newton step (relative error ~ 1e-13), FP64 constants; the lane's q_j multiplies
                    // the step's sum once.  The LJ term has no such cancellation: FP32 sums of A, B and the shift per
                    // step, combined in FP64 (its table constants 6 C6, 12 C12 are exact multiples, so unbiased).
#pragma unroll
                    for (int c = 0; c < 2; c++) {
                        if (c ? inb : ina) {
                            const unsigned ia = sd_addr + (unsigned)(2 * p + c) * 32u;
                            const double ddx = mop_lds_d(ia) - jxd, ddy = mop_lds_d(ia + 8u) - jyd, ddz = mop_lds_d(ia + 16u) - jzd;
                            const double r2d = fma(ddz, ddz, fma(ddy, ddy, ddx * ddx));
                            const double y = (double)(c ? rb : ra);
                            const double t = fma(a.krf_d, r2d, fma(y, fma(-0.5 * (y * y), r2d, 1.5), -a.crf_d));
                            acc_c = fma(mop_lds_d(ia + 24u), t, acc_c);
                        }
                    }
                    if (!nolj) {
                        float v0, v1, w0, w1, s0, s1;
                        f2_unpack(A, v0, v1), f2_unpack(B, w0, w1);
                        s0 = mop_lds_f(tabS + ((ta - tab6) >> 1)), s1 = mop_lds_f(tabS + ((tb - tab6) >> 1));
                        eA = f2_add(eA, f2_pack(ina ? v0 : 0.f, inb ? v1 : 0.f));
                        eB = f2_add(eB, f2_pack(ina ? w0 : 0.f, inb ? w1 : 0.f));
                        eS = f2_add(eS, f2_pack(ina ? s0 : 0.f, inb ? s1 : 0.f));
                    }
                }
            } else {
                f2 hn = nolj ? f2_mul(f2_mul(x, f2_bc(-3.0f)), C)
                             : f2_mul(x, f2_fma(C, f2_bc(-3.0f), f2_mul(x, f2_fma(B, f2_bc(-14.0f), f2_mul(A, f2_bc(8.0f))))));
                {
                    float ha, hb;
                    f2_unpack(hn, ha, hb);
                    hn = f2_pack(ina ? ha : 0.f, inb ? hb : 0.f);
                }
                const f2 ex = f2_sub(f2_bc(ce.x), S0), ey = f2_sub(f2_bc(ce.y), S1), ez = f2_sub(f2_bc(ce.z), S2);
                const f2 tt = f2_mul(hn, f2_fma(dz, ez, f2_fma(dy, ey, f2_mul(dx, ex))));
                // v = tt d + gn e once, then two packed adds: fewer register-file reads than four FFMA2 per
                // component (a three-register FFMA2 costs 3 issue cycles of the FP32 pipe, FMUL2/FADD2 cost 2)
                const f2 vx = f2_fma(tt, dx, f2_mul(gn, ex)), vy = f2_fma(tt, dy, f2_mul(gn, ey)),
                         vz = f2_fma(tt, dz, f2_mul(gn, ez));
                ax[p] = f2_add(ax[p], vx), ay[p] = f2_add(ay[p], vy), az[p] = f2_add(az[p], vz);
                nx = f2_add(nx, vx), ny = f2_add(ny, vy), nz = f2_add(nz, vz);
            }
        };

#pragma unroll
        for (int p = 0; p < 4; p++)
            if ((upat >> p) & 1u) {
                if ((ljmask >> (2 * p)) & 3u) heavy(p, false);
                else heavy(p, true);
            }
        if (valid) {
            float lx, hx, ly, hy, lz, hz;
            f2_unpack(nx, lx, hx), f2_unpack(ny, ly, hy), f2_unpack(nz, lz, hz);
            mop_red_add_f4(out + (cur.x + jl), -lx - hx, -ly - hy, -lz - hz);
        }
        if (ENERGY) {
            auto hsum = [](f2 v) {
                float lo, hi;
                f2_unpack(v, lo, hi);
                return (double)lo + (double)hi;
            };
            e_c = fma((double)cp.w, acc_c, e_c);
            e_lj += hsum(eB) * (1.0 / 12.0) - hsum(eA) * (1.0 / 6.0) - hsum(eS);
        }
    };

    // ---- the unit's entries, 32 at a time (8 steps): the chunk's entry words go to shared memory (one coalesced load;
    // staged as x = element index of the j-octet's first atom, y = flags | shift id << 24), the j atoms of the next step
    // are in flight (cp.async into the warp's two-stage ring; every lane copies and later reads only its own atom, so no
    // cross-lane synchronisation is needed)
    const unsigned eend = un.start + un.count;
    const unsigned se_g = se_addr + gq * 8u;           // this lane group's entry of step 0
    const unsigned infobit = 1u << (16 + jl);          // the bit of the step information this lane contributes to the vote
    const unsigned sr_l = sr_addr + lane16, sr_t = sr_addr + 512u + (HVP ? lane16 : (unsigned)lane * 4u);
    for (unsigned c0 = un.start; c0 < eend; c0 += 32) {
        const int nE = (int)min(32u, eend - c0), nS = nE / MOP_NG;
        __syncwarp();
        if (lane < nE) {
            const uint2 w = a.entries[c0 + lane];
            asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(se_addr + lane * 8), "r"(boff + (w.x & 0xffffffu) * MOP_CL),
                         "r"(w.y | (w.x & 0xff000000u))
                         : "memory");
        }
        __syncwarp();
        auto issue = [&](const int k) { // start the copies of step k's j atoms into stage k % 2
            if (k < nS) {
                const unsigned o = mop_lds_vu(se_g + (unsigned)k * 32u) + jl;
                MOP_ASSERT(o < a.n_slots);
                const unsigned sto = (unsigned)(k & 1) * 1024u;
                mop_cp_async16(sr_l + sto, xq + o);
                if (HVP) mop_cp_async16(sr_t + sto, et + o);
                else mop_cp_async4(sr_t + sto, typ + o);
            }
            mop_cp_commit();
        };
        issue(0);
        for (int i = 0; i < nS; i++) {
            issue(i + 1);
            mop_cp_wait<1>();
            const unsigned sto = (unsigned)(i & 1) * 1024u;
            const uint2 cur = mop_lds_vu2(se_g + (unsigned)i * 32u);
            const float4 cp = mop_lds_v4(sr_l + sto);
            float4 ce = make_float4(0.f, 0.f, 0.f, 0.f);
            unsigned tj8;
            if (HVP) {
                ce = mop_lds_v4(sr_t + sto);
                tj8 = (unsigned)__float_as_int(ce.w) * 8u;
            } else {
                tj8 = mop_lds_vu(sr_t + sto) * 8u;
            }
            // step information from the list builder, the same in all four entries: one vote makes it warp-uniform for
            // the compiler (bits 0-3 union pattern, 4 shifted, 5 masked), so every test below is a uniform branch
            const unsigned info = __ballot_sync(0xffffffffu, (cur.y & infobit) != 0u) & 0x3fu;
            const unsigned upat = info & 15u;
            const bool shifted = (info >> 4) & 1u, masked = (info >> 5) & 1u;
            // two compiled step bodies: the plain one (69 % of the steps on the bench workload) and the general one (periodic
            // shift and exclusion bits).  A third, masked-only body measured the same (3.738 vs 3.734 ms per step), and the
            // kernels are sensitive to code size: with FP64 LJ and reaction-field energies and three bodies the energy variant
            // (4,500 instructions) overflowed the instruction cache ("no instruction" 5 stalls per issue)
            if (shifted || masked) step(cur, upat, true, true, cp, ce, tj8);
            else step(cur, upat, false, false, cp, ce, tj8);
        }
        mop_cp_wait<0>();
    }

    // ---- i side: 24 per-lane partial sums (8 atoms x 3 components) -> atom k = lane / 4.  Three halving
    // exchanges (each lane keeps the half of the values its lane bits select) and two plain butterfly steps.
    float v[24];
#pragma unroll
    for (int p = 0; p < 4; p++) {
        f2_unpack(ax[p], v[6 * p + 0], v[6 * p + 3]);
        f2_unpack(ay[p], v[6 * p + 1], v[6 * p + 4]);
        f2_unpack(az[p], v[6 * p + 2], v[6 * p + 5]);
    }
#pragma unroll
    for (int h = 12, bit = 16; h >= 3; h >>= 1, bit >>= 1) {
        const bool up = (lane & bit) != 0;
#pragma unroll
        for (int j = 0; j < h; j++) {
            const float keep = up ? v[j + h] : v[j], send = up ? v[j] : v[j + h];
            v[j] = keep + __shfl_xor_sync(0xffffffffu, send, bit);
        }
    }
#pragma unroll
    for (int j = 0; j < 3; j++) {
        v[j] += __shfl_xor_sync(0xffffffffu, v[j], 2);
        v[j] += __shfl_xor_sync(0xffffffffu, v[j], 1);
    }
    if ((lane & 3) == 0) mop_red_add_f4(out + (ibase + (lane >> 2)), v[0], v[1], v[2]);
    if (ENERGY) {
        e_lj = mop_warp_sum_d(e_lj), e_c = mop_warp_sum_d(e_c);
        if (lane == 0) {
            atomicAdd(&a.energies[0], e_lj);
            atomicAdd(&a.energies[1], e_c);
        }
    }
    if (COUNT) {
        n_in = (unsigned)__reduce_add_sync(0xffffffffu, n_in);
        if (lane == 0) atomicAdd(a.n_inrange, (unsigned long long)n_in);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) h_in += __shfl_xor_sync(0xffffffffu, h_in, o);
        if (lane == 0) atomicAdd(a.pair_hash, h_in);
    }
}

// persistent grid (resident CTAs x SMs) with a dynamic work counter; CTAS = resident CTAs per SM asked for
template <int MODE, bool COUNT, int CTAS>
__global__ void __launch_bounds__(128, CTAS) k_nonbonded_p(const NbArgs a) {
    extern __shared__ float4 s_dyn[];
    char *sb = reinterpret_cast<char *>(s_dyn);
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float *sw = reinterpret_cast<float *>(sb) + w * 64;
    const int n2 = a.nt * a.nt;
    float2 *t6 = reinterpret_cast<float2 *>(sb + NBP_SM_TAB);
    float *tabs = reinterpret_cast<float *>(t6 + n2);
    int *tflag = reinterpret_cast<int *>(tabs + n2);   // [nt]: 1 iff the type's LJ row has a non-zero entry
    for (int t = threadIdx.x; t < n2; t += blockDim.x) {
        t6[t] = a.tab[t];
        tabs[t] = a.tabs[t];
    }
    for (int t = threadIdx.x; t < a.nt; t += blockDim.x) {
        int f = 0;
        for (int u = 0; u < a.nt; u++) f |= (a.tab[t * a.nt + u].x != 0.f || a.tab[t * a.nt + u].y != 0.f);
        tflag[t] = f;
    }
    __syncthreads();
    const unsigned nu = min(a.ctr->n_units, a.cap_units), nu0 = min(a.ctr->n_units_bead0, a.cap_units);
    unsigned ubeg = 0, uend = nu;
    if (a.range == 0) uend = nu0;
    else if (a.range == 1) ubeg = nu0;
    else if (a.range == 3) uend = min(a.ctr->n_units_mid, a.cap_units);
    else if (a.range == 4) ubeg = min(a.ctr->n_units_mid, a.cap_units);
    const unsigned s0 = (unsigned)__cvta_generic_to_shared(sb);
    const unsigned sw_addr = s0 + w * 256u, se_addr = s0 + NBP_SM_ENT + w * 256u;
    const unsigned sr_addr = s0 + NBP_SM_RING + w * (NBP_NST * 1024u), sd_addr = s0 + NBP_SM_DBL + w * 256u;
    const unsigned tab6 = s0 + NBP_SM_TAB;
    for (;;) {
        unsigned u = 0;
        if (lane == 0) u = atomicAdd(a.work, 1u);
        u = __shfl_sync(0xffffffffu, u, 0) + ubeg;
        if (u >= uend) break;
        MOP_ASSERT(u < a.cap_units);
        const uint4 *up = reinterpret_cast<const uint4 *>(a.units + u);
        const uint4 u0 = up[0], u1 = up[1];
        MopUnit un;
        un.bead = (int)u0.x, un.ci = (int)u0.y, un.start = u0.z, un.count = u0.w;
        un.excl_base = u1.x;
        if (un.count == 0) continue;
        nbp_unit<MODE, COUNT>(a, un, sw, sw_addr, se_addr, sr_addr, sd_addr, tab6, tab6 + (unsigned)n2 * 8u, tflag, lane);
    }
}
